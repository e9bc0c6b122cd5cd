"""Thin Python binding of libfdham (include/fdham.h): argument marshalling only.

Every step of the path (halo resolution, stencil, v_eff multiply-add, store) runs in the CUDA
kernels behind the C ABI; torch is used for device memory and streams.  There is no CPU
fallback: if libfdham.so is missing or no CUDA device is usable this module raises.

Functions mirror the C names: fd_create, fd_apply_kinetic, fd_apply_hamiltonian,
fd_apply_hamiltonian_host, fd_destroy (operation: Eq. 6 first two terms, with
the FD kinetic operator of PAPER.md:232).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

FD_BC_ZERO, FD_BC_PERIODIC = 0, 1
FD_F64, FD_C128, FD_F32, FD_C64 = 0, 1, 2, 3
FD_OK = 0
FD_KERNEL_AUTO, FD_KERNEL_GENERIC, FD_KERNEL_SWEEP = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdham.so")

EXPORTED_SYMBOLS = [
    "fd_create", "fd_create_scaled", "fd_apply_kinetic", "fd_apply_hamiltonian",
    "fd_apply_hamiltonian_host", "fd_workspace_create", "fd_workspace_destroy",
    "fd_apply_hamiltonian_host_ws", "fd_expect_workspace_bytes", "fd_apply_hamiltonian_expect",
    "fd_apply_hamiltonian_expect_static",
    "fd_residual", "fd_jacobi_sweep", "fd_restrict", "fd_interpolate",
    "fd_paw_create", "fd_paw_destroy", "fd_paw_nproj_total", "fd_paw_project", "fd_paw_add_nonlocal",
    "fd_apply_hamiltonian_paw", "fd_apply_overlap", "fd_paw_expect",
    "fd_peak_kernel", "fd_poisson_residual", "fd_mg_create", "fd_mg_destroy", "fd_mg_levels", "fd_mg_vcycle", "fd_mg_get_info",
    "fd_destroy", "fd_strerror", "fd_plan_set_kernel", "fd_plan_get_kernel", "fd_plan_kernel_for", "fd_plan_launches",
    "fd_plan_get_weights", "fd_plan_get_info",
]


class FDError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (fd_status {status})")


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libfdham.so (built in-tree by paper_2310_14776_b200.build). Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2310_14776_b200.build` "
            "(nvcc, sm_100a). libfdham has no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    i32p, f64p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_double)
    lib.fd_create.argtypes = [ctypes.POINTER(vp), i32p, f64p, i32, i32p, f64p, i32, i32]
    lib.fd_create.restype = ctypes.c_int
    lib.fd_create_scaled.argtypes = [ctypes.POINTER(vp), i32p, f64p, i32, i32p, f64p, i32, i32,
                                     ctypes.c_double]
    lib.fd_create_scaled.restype = ctypes.c_int
    lib.fd_apply_kinetic.argtypes = [vp, vp, vp, i64, vp]
    lib.fd_apply_kinetic.restype = ctypes.c_int
    lib.fd_apply_hamiltonian.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.fd_apply_hamiltonian.restype = ctypes.c_int
    lib.fd_apply_hamiltonian_host.argtypes = [vp, vp, vp, vp, i64]
    lib.fd_apply_hamiltonian_host.restype = ctypes.c_int
    lib.fd_workspace_create.argtypes = [ctypes.POINTER(vp), vp, i64]
    lib.fd_workspace_create.restype = ctypes.c_int
    lib.fd_workspace_destroy.argtypes = [vp]
    lib.fd_workspace_destroy.restype = ctypes.c_int
    lib.fd_apply_hamiltonian_host_ws.argtypes = [vp, vp, vp, vp, vp, i64]
    lib.fd_apply_hamiltonian_host_ws.restype = ctypes.c_int
    lib.fd_expect_workspace_bytes.argtypes = [vp, i64]
    lib.fd_expect_workspace_bytes.restype = ctypes.c_int64
    lib.fd_apply_hamiltonian_expect.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, i64, vp]
    lib.fd_apply_hamiltonian_expect.restype = ctypes.c_int
    lib.fd_apply_hamiltonian_expect_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp]
    lib.fd_apply_hamiltonian_expect_static.restype = ctypes.c_int
    lib.fd_residual.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp]
    lib.fd_residual.restype = ctypes.c_int
    lib.fd_jacobi_sweep.argtypes = [vp, vp, vp, vp, i64, ctypes.c_double, vp]
    lib.fd_jacobi_sweep.restype = ctypes.c_int
    lib.fd_restrict.argtypes = [i32p, i32p, i32, vp, vp, i64, vp]
    lib.fd_restrict.restype = ctypes.c_int
    lib.fd_interpolate.argtypes = [i32p, i32p, i32, vp, vp, i64, vp]
    lib.fd_interpolate.restype = ctypes.c_int
    lib.fd_paw_create.argtypes = [ctypes.POINTER(vp), vp, i32, i32p, i32p, i32p, f64p, f64p, f64p]
    lib.fd_paw_create.restype = ctypes.c_int
    lib.fd_paw_destroy.argtypes = [vp]
    lib.fd_paw_destroy.restype = ctypes.c_int
    lib.fd_paw_nproj_total.argtypes = [vp]
    lib.fd_paw_nproj_total.restype = ctypes.c_int32
    lib.fd_paw_project.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.fd_paw_project.restype = ctypes.c_int
    lib.fd_paw_add_nonlocal.argtypes = [vp, vp, vp, vp, vp, i64, vp]
    lib.fd_paw_add_nonlocal.restype = ctypes.c_int
    lib.fd_apply_hamiltonian_paw.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp]
    lib.fd_apply_hamiltonian_paw.restype = ctypes.c_int
    lib.fd_apply_overlap.argtypes = [vp, vp, vp, vp, vp, i64, vp]
    lib.fd_apply_overlap.restype = ctypes.c_int
    lib.fd_paw_expect.argtypes = [vp, vp, i32, vp, vp, i64, vp]
    lib.fd_paw_expect.restype = ctypes.c_int
    lib.fd_poisson_residual.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.fd_poisson_residual.restype = ctypes.c_int
    lib.fd_mg_create.argtypes = [ctypes.POINTER(vp), i32p, f64p, i32, i32p, i32, i32, i64, i32]
    lib.fd_mg_create.restype = ctypes.c_int
    lib.fd_mg_destroy.argtypes = [vp]
    lib.fd_mg_destroy.restype = ctypes.c_int
    lib.fd_mg_levels.argtypes = [vp]
    lib.fd_mg_levels.restype = ctypes.c_int32
    lib.fd_mg_vcycle.argtypes = [vp, vp, vp, i64, i32, i32, i32, ctypes.c_double, vp]
    lib.fd_mg_vcycle.restype = ctypes.c_int
    lib.fd_mg_get_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
    lib.fd_mg_get_info.restype = ctypes.c_int
    lib.fd_peak_kernel.argtypes = [i32, vp, vp, i64, i32, vp]
    lib.fd_peak_kernel.restype = ctypes.c_int
    lib.fd_destroy.argtypes = [vp]
    lib.fd_destroy.restype = ctypes.c_int
    lib.fd_strerror.argtypes = [ctypes.c_int]
    lib.fd_strerror.restype = ctypes.c_char_p
    lib.fd_plan_set_kernel.argtypes = [vp, i32, i32]
    lib.fd_plan_set_kernel.restype = ctypes.c_int
    lib.fd_plan_get_kernel.argtypes = [vp]
    lib.fd_plan_get_kernel.restype = ctypes.c_int
    lib.fd_plan_kernel_for.argtypes = [vp, i64]
    lib.fd_plan_kernel_for.restype = ctypes.c_int
    lib.fd_plan_launches.argtypes = [vp]
    lib.fd_plan_launches.restype = ctypes.c_int64
    lib.fd_plan_get_weights.argtypes = [vp, f64p, i32]
    lib.fd_plan_get_weights.restype = ctypes.c_int
    lib.fd_plan_get_info.argtypes = [vp, i32p]
    lib.fd_plan_get_info.restype = ctypes.c_int
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load_library().fd_strerror(int(status)).decode()


def _check(status: int, where: str) -> None:
    if status != FD_OK:
        raise FDError(status, where)


def fd_create(shape: Sequence[int], h: Sequence[float], nn: int = 3,
              bc: Sequence[int] = (1, 1, 1), k: Optional[Sequence[float]] = None,
              dtype: int = FD_F64, device: int = 0) -> ctypes.c_void_p:
    """Returns an opaque plan handle (see include/fdham.h: fd_create)."""
    lib = load_library()
    plan = ctypes.c_void_p()
    kk = (ctypes.c_double * 3)(*[float(x) for x in k]) if k is not None else None
    rc = lib.fd_create(ctypes.byref(plan), (ctypes.c_int32 * 3)(*[int(s) for s in shape]),
                       (ctypes.c_double * 3)(*[float(x) for x in h]), int(nn),
                       (ctypes.c_int32 * 3)(*[int(b) for b in bc]), kk, int(dtype), int(device))
    _check(rc, "fd_create")
    return plan


def fd_create_scaled(shape: Sequence[int], h: Sequence[float], nn: int = 3,
                     bc: Sequence[int] = (1, 1, 1), k: Optional[Sequence[float]] = None,
                     dtype: int = FD_F64, device: int = 0, scale: float = -0.5) -> ctypes.c_void_p:
    """fd_create with `scale` in place of -1/2 (include/fdham.h: fd_create_scaled)."""
    lib = load_library()
    plan = ctypes.c_void_p()
    kk = (ctypes.c_double * 3)(*[float(x) for x in k]) if k is not None else None
    rc = lib.fd_create_scaled(ctypes.byref(plan), (ctypes.c_int32 * 3)(*[int(s) for s in shape]),
                              (ctypes.c_double * 3)(*[float(x) for x in h]), int(nn),
                              (ctypes.c_int32 * 3)(*[int(b) for b in bc]), kk, int(dtype),
                              int(device), float(scale))
    _check(rc, "fd_create_scaled")
    return plan


def fd_destroy(plan) -> None:
    _PLAN_INFO.pop(plan.value if hasattr(plan, "value") else int(plan), None)
    _check(load_library().fd_destroy(plan), "fd_destroy")


def _stream_ptr(stream) -> ctypes.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    if hasattr(stream, "cuda_stream"):
        return ctypes.c_void_p(stream.cuda_stream)
    return ctypes.c_void_p(int(stream))


def _dev_ptr(t) -> ctypes.c_void_p:
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return ctypes.c_void_p(t.data_ptr())


def fd_plan_get_info(plan) -> dict:
    """shape, nn, dtype, device, bc and kernel family of a plan (include/fdham.h)."""
    buf = (ctypes.c_int32 * 8)()
    _check(load_library().fd_plan_get_info(plan, buf), "fd_plan_get_info")
    return {"shape": (buf[0], buf[1], buf[2]), "nn": buf[3], "dtype": buf[4], "device": buf[5],
            "bc": (buf[6] & 1, (buf[6] >> 1) & 1, (buf[6] >> 2) & 1), "kernel": buf[7]}


# shape / dtype / device of a plan never change after fd_create: one ABI call per handle, not one per
# apply (the launch-bound small batches would pay for it).  Evicted by fd_destroy.
_PLAN_INFO: dict = {}


def _plan_info(plan) -> dict:
    key = plan.value if hasattr(plan, "value") else int(plan)
    info = _PLAN_INFO.get(key)
    if info is None:
        info = fd_plan_get_info(plan)
        _PLAN_INFO[key] = info
    return info


def _torch_dtypes(dtype: int):
    """(torch dtype of psi / out, torch dtype of v_eff) for an FD_* dtype."""
    import torch
    return {FD_F64: (torch.float64, torch.float64), FD_C128: (torch.complex128, torch.float64),
            FD_F32: (torch.float32, torch.float32), FD_C64: (torch.complex64, torch.float32)}[dtype]


def _check_arrays(plan, where: str, batch=(), grid=(), real=()):
    """The C ABI takes raw pointers: a tensor of the wrong shape, dtype or device would become an
    out-of-bounds access on the device, so the binding checks them against the plan first.
    batch: tensors [nbands, nx, ny, nz] of the plan's dtype (same nbands); grid: [nx, ny, nz] of the
    plan's real dtype; real: batch-shaped tensors of the plan's real dtype."""
    info = _plan_info(plan)
    shape, (tdt, rdt) = tuple(info["shape"]), _torch_dtypes(info["dtype"])
    nb = None
    for kind, tensors, want_dt in (("batch", batch, tdt), ("real", real, rdt)):
        for t in tensors:
            if t is None:
                continue
            if t.dim() != 4 or tuple(t.shape[1:]) != shape:
                raise ValueError(f"{where}: expected [nbands, {shape}], got {tuple(t.shape)}")
            if t.dtype != want_dt:
                raise ValueError(f"{where}: expected dtype {want_dt}, got {t.dtype}")
            if nb is not None and t.shape[0] != nb:
                raise ValueError(f"{where}: band counts differ ({t.shape[0]} vs {nb})")
            nb = t.shape[0]
            if t.device.index != info["device"]:
                raise ValueError(f"{where}: tensor on cuda:{t.device.index}, plan on cuda:{info['device']}")
    for t in grid:
        if t is None:
            continue
        if tuple(t.shape) != shape or t.dtype != rdt:
            raise ValueError(f"{where}: v_eff must be {rdt} {shape}, got {t.dtype} {tuple(t.shape)}")
        if t.device.index != info["device"]:
            raise ValueError(f"{where}: tensor on cuda:{t.device.index}, plan on cuda:{info['device']}")


def fd_apply_kinetic(plan, psi, out, stream=None) -> None:
    """out = T psi for torch CUDA tensors psi/out [nbands,nx,ny,nz] (float64 or complex128)."""
    _check_arrays(plan, "fd_apply_kinetic", batch=(psi, out))
    rc = load_library().fd_apply_kinetic(plan, _dev_ptr(psi), _dev_ptr(out), int(psi.shape[0]),
                                         _stream_ptr(stream))
    _check(rc, "fd_apply_kinetic")


def fd_apply_hamiltonian(plan, psi, v_eff, out, stream=None) -> None:
    """out = T psi + v_eff psi; v_eff is a float64 CUDA tensor [nx,ny,nz]."""
    _check_arrays(plan, "fd_apply_hamiltonian", batch=(psi, out), grid=(v_eff,))
    rc = load_library().fd_apply_hamiltonian(plan, _dev_ptr(psi), _dev_ptr(v_eff), _dev_ptr(out),
                                             int(psi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_apply_hamiltonian")


def _host_ptr(a) -> ctypes.c_void_p:
    if a is None:
        return ctypes.c_void_p(0)
    if hasattr(a, "data_ptr"):          # torch CPU tensor (pinned or not)
        if a.is_cuda or not a.is_contiguous():
            raise ValueError("expected a contiguous CPU tensor")
        return ctypes.c_void_p(a.data_ptr())
    if not a.flags.c_contiguous:        # numpy
        raise ValueError("expected a C-contiguous array")
    return ctypes.c_void_p(a.ctypes.data)


def fd_apply_hamiltonian_host(plan, psi_host, v_eff_host, out_host) -> None:
    """End-to-end apply on HOST arrays (numpy or torch CPU, ideally pinned); blocks until done."""
    rc = load_library().fd_apply_hamiltonian_host(plan, _host_ptr(psi_host),
                                                  _host_ptr(v_eff_host), _host_ptr(out_host),
                                                  int(psi_host.shape[0]))
    _check(rc, "fd_apply_hamiltonian_host")


def fd_workspace_create(plan, chunk_bytes: int = 0) -> ctypes.c_void_p:
    """Staging buffers + streams for fd_apply_hamiltonian_host_ws (include/fdham.h)."""
    ws = ctypes.c_void_p()
    _check(load_library().fd_workspace_create(ctypes.byref(ws), plan, int(chunk_bytes)),
           "fd_workspace_create")
    return ws


def fd_workspace_destroy(ws) -> None:
    _check(load_library().fd_workspace_destroy(ws), "fd_workspace_destroy")


def fd_apply_hamiltonian_host_ws(plan, ws, psi_host, v_eff_host, out_host) -> None:
    """fd_apply_hamiltonian_host on a caller-owned workspace (no allocation in the call)."""
    rc = load_library().fd_apply_hamiltonian_host_ws(plan, ws, _host_ptr(psi_host),
                                                     _host_ptr(v_eff_host), _host_ptr(out_host),
                                                     int(psi_host.shape[0]))
    _check(rc, "fd_apply_hamiltonian_host_ws")


def fd_expect_workspace_bytes(plan, nbands: int) -> int:
    n = int(load_library().fd_expect_workspace_bytes(plan, int(nbands)))
    if n < 0:
        raise FDError(n, "fd_expect_workspace_bytes")
    return n


def fd_apply_hamiltonian_expect(plan, psi, v_eff, out, eps, norm, workspace, stream=None) -> None:
    """out = H psi (v_eff None: T psi), eps[b] = Re <psi_b|H psi_b>, norm[b] = <psi_b|psi_b> (grid
    sums) in one pass; eps/norm float64 CUDA tensors [nbands], workspace a CUDA byte/float64 tensor
    of at least fd_expect_workspace_bytes(plan, nbands) bytes."""
    _check_arrays(plan, "fd_apply_hamiltonian_expect", batch=(psi, out), grid=(v_eff,))
    for name, t in (("eps", eps), ("norm", norm)):
        if tuple(t.shape) != (psi.shape[0],) or str(t.dtype) != "torch.float64":
            raise ValueError(f"fd_apply_hamiltonian_expect: {name} must be float64 [nbands]")
    rc = load_library().fd_apply_hamiltonian_expect(
        plan, _dev_ptr(psi), _dev_ptr(v_eff) if v_eff is not None else ctypes.c_void_p(0),
        _dev_ptr(out), _dev_ptr(eps), _dev_ptr(norm), int(psi.shape[0]), _dev_ptr(workspace),
        int(workspace.numel() * workspace.element_size()), _stream_ptr(stream))
    _check(rc, "fd_apply_hamiltonian_expect")


FD_STATIC_SCRATCH_BYTES = 4 * 1024 * 1024  # include/fdham.h
FD_ERR_SCRATCH = -6


def fd_apply_hamiltonian_expect_static(plan, psi, v_eff, out, eps, norm, stream=None) -> None:
    """fd_apply_hamiltonian_expect for callers that cannot allocate device memory (a plug-in under a
    host application that owns the device's memory, a latency path that must not hit the device-wide
    synchronisation of cudaMalloc / cudaFree): no workspace argument, the partial sums go to a
    4 MiB array built into libfdham.so.  Same results, bit for bit.  Batches that need more raise
    FDError with status FD_ERR_SCRATCH; calls that overlap on the GPU race on the shared array; the
    first call per device should come before any stream capture (include/fdham.h has the details)."""
    _check_arrays(plan, "fd_apply_hamiltonian_expect_static", batch=(psi, out), grid=(v_eff,))
    for name, t in (("eps", eps), ("norm", norm)):
        if tuple(t.shape) != (psi.shape[0],) or str(t.dtype) != "torch.float64":
            raise ValueError(f"fd_apply_hamiltonian_expect_static: {name} must be float64 [nbands]")
    rc = load_library().fd_apply_hamiltonian_expect_static(
        plan, _dev_ptr(psi), _dev_ptr(v_eff) if v_eff is not None else ctypes.c_void_p(0),
        _dev_ptr(out), _dev_ptr(eps), _dev_ptr(norm), int(psi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_apply_hamiltonian_expect_static")


def _check_band_vectors(where: str, psi, **vectors) -> None:
    """eps / norm style arguments: float64 [nbands] on the device of psi."""
    for name, t in vectors.items():
        if tuple(t.shape) != (psi.shape[0],) or str(t.dtype) != "torch.float64" or t.device != psi.device:
            raise ValueError(f"{where}: {name} must be float64 [{psi.shape[0]}] on {psi.device}")


def fd_residual(plan, psi, hpsi, eps, norm, r, stream=None) -> None:
    """r_b = hpsi_b - (eps[b] / norm[b]) psi_b; r may be hpsi itself."""
    _check_arrays(plan, "fd_residual", batch=(psi, hpsi, r))
    _check_band_vectors("fd_residual", psi, eps=eps, norm=norm)
    rc = load_library().fd_residual(plan, _dev_ptr(psi), _dev_ptr(hpsi), _dev_ptr(eps),
                                    _dev_ptr(norm), _dev_ptr(r), int(psi.shape[0]),
                                    _stream_ptr(stream))
    _check(rc, "fd_residual")


def fd_jacobi_sweep(plan, phi, rhs, out, omega: float, stream=None) -> None:
    """out = phi + omega (rhs - A phi) / A_ii for the plan's A = scale lap_FD (fd_create_scaled)."""
    _check_arrays(plan, "fd_jacobi_sweep", batch=(phi, rhs, out))
    rc = load_library().fd_jacobi_sweep(plan, _dev_ptr(phi), _dev_ptr(rhs), _dev_ptr(out),
                                        int(phi.shape[0]), float(omega), _stream_ptr(stream))
    _check(rc, "fd_jacobi_sweep")


def coarse_shape(shape_fine: Sequence[int], bc: Sequence[int]):
    """Coarse extents of a fine grid (include/fdham.h: n/2 periodic, (n-1)/2 zero-BC)."""
    return tuple(int(n) // 2 if b else (int(n) - 1) // 2 for n, b in zip(shape_fine, bc))


def _check_transfer(shape_fine, bc, fine, coarse, where: str) -> None:
    nf, nc = tuple(int(n) for n in shape_fine), coarse_shape(shape_fine, bc)
    if not all((n % 2 == 0 and n >= 2) if b else (n % 2 == 1 and n >= 3) for n, b in zip(nf, bc)):
        return  # not a valid fine grid: the library reports it (FD_ERR_INVALID)
    for t, shp, name in ((fine, nf, "fine"), (coarse, nc, "coarse")):
        if t.dim() != 4 or tuple(t.shape[1:]) != shp or str(t.dtype) != "torch.float64":
            raise ValueError(f"{where}: {name} must be float64 [nbands, {shp}], got {t.dtype} {tuple(t.shape)}")
    if fine.shape[0] != coarse.shape[0] or fine.device != coarse.device:
        raise ValueError(f"{where}: fine and coarse differ in band count or device")


def fd_restrict(shape_fine, bc, p: int, fine, coarse, stream=None) -> None:
    """coarse[nbands, nc] <- fine[nbands, nf] (float64 CUDA tensors; include/fdham.h)."""
    _check_transfer(shape_fine, bc, fine, coarse, "fd_restrict")
    rc = load_library().fd_restrict((ctypes.c_int32 * 3)(*[int(s) for s in shape_fine]),
                                    (ctypes.c_int32 * 3)(*[int(b) for b in bc]), int(p),
                                    _dev_ptr(fine), _dev_ptr(coarse), int(fine.shape[0]),
                                    _stream_ptr(stream))
    _check(rc, "fd_restrict")


def fd_interpolate(shape_fine, bc, p: int, coarse, fine, stream=None) -> None:
    """fine[nbands, nf] <- coarse[nbands, nc] (float64 CUDA tensors; include/fdham.h)."""
    _check_transfer(shape_fine, bc, fine, coarse, "fd_interpolate")
    rc = load_library().fd_interpolate((ctypes.c_int32 * 3)(*[int(s) for s in shape_fine]),
                                       (ctypes.c_int32 * 3)(*[int(b) for b in bc]), int(p),
                                       _dev_ptr(coarse), _dev_ptr(fine), int(coarse.shape[0]),
                                       _stream_ptr(stream))
    _check(rc, "fd_interpolate")


def fd_paw_create(plan, box_start, box_size, nproj, proj, dh=None, ds=None) -> ctypes.c_void_p:
    """Projector set on the plan's device (include/fdham.h: fd_paw_create); arguments are host
    arrays (numpy / sequences): box_start, box_size [natoms,3], nproj [natoms], proj and dh / ds
    concatenated per atom."""
    import numpy as np
    bs = np.ascontiguousarray(box_start, dtype=np.int32).reshape(-1, 3)
    bz = np.ascontiguousarray(box_size, dtype=np.int32).reshape(-1, 3)
    npj = np.ascontiguousarray(nproj, dtype=np.int32).reshape(-1)
    pr = np.ascontiguousarray(proj, dtype=np.float64).reshape(-1)
    i32p, f64p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_double)

    def mat(m):
        if m is None:
            return None, None
        a = np.ascontiguousarray(m, dtype=np.float64).reshape(-1)
        return a, a.ctypes.data_as(f64p)
    dh_a, dh_p = mat(dh)
    ds_a, ds_p = mat(ds)
    paw = ctypes.c_void_p()
    rc = load_library().fd_paw_create(ctypes.byref(paw), plan, int(npj.shape[0]),
                                      bs.ctypes.data_as(i32p), bz.ctypes.data_as(i32p),
                                      npj.ctypes.data_as(i32p), pr.ctypes.data_as(f64p), dh_p, ds_p)
    _check(rc, "fd_paw_create")
    return paw


def fd_paw_destroy(paw) -> None:
    _check(load_library().fd_paw_destroy(paw), "fd_paw_destroy")


def fd_paw_nproj_total(paw) -> int:
    n = int(load_library().fd_paw_nproj_total(paw))
    if n < 0:
        raise FDError(n, "fd_paw_nproj_total")
    return n


def _check_coef(paw, psi, coef, where: str) -> None:
    ntot = fd_paw_nproj_total(paw)
    if tuple(coef.shape) != (psi.shape[0], ntot) or coef.dtype != psi.dtype or coef.device != psi.device:
        raise ValueError(f"{where}: coef must be {psi.dtype} [{psi.shape[0]}, {ntot}] on {psi.device}")


def fd_paw_project(plan, paw, psi, coef, stream=None) -> None:
    """coef[nbands, sum n_i] = dv <p~|psi> (dtype of psi)."""
    _check_arrays(plan, "fd_paw_project", batch=(psi,))
    _check_coef(paw, psi, coef, "fd_paw_project")
    rc = load_library().fd_paw_project(plan, paw, _dev_ptr(psi), _dev_ptr(coef), int(psi.shape[0]),
                                       _stream_ptr(stream))
    _check(rc, "fd_paw_project")


def fd_paw_add_nonlocal(plan, paw, psi, out, coef, stream=None) -> None:
    """out += sum |p~> Delta H <p~|psi>; coef is scratch [nbands, sum n_i]."""
    _check_arrays(plan, "fd_paw_add_nonlocal", batch=(psi, out))
    _check_coef(paw, psi, coef, "fd_paw_add_nonlocal")
    rc = load_library().fd_paw_add_nonlocal(plan, paw, _dev_ptr(psi), _dev_ptr(out), _dev_ptr(coef),
                                            int(psi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_paw_add_nonlocal")


def fd_apply_hamiltonian_paw(plan, paw, psi, v_eff, out, coef, stream=None) -> None:
    """out = -1/2 lap psi + v_eff psi + sum |p~> Delta H <p~|psi> (Eq. 6 complete)."""
    _check_arrays(plan, "fd_apply_hamiltonian_paw", batch=(psi, out), grid=(v_eff,))
    _check_coef(paw, psi, coef, "fd_apply_hamiltonian_paw")
    rc = load_library().fd_apply_hamiltonian_paw(
        plan, paw, _dev_ptr(psi), _dev_ptr(v_eff) if v_eff is not None else ctypes.c_void_p(0),
        _dev_ptr(out), _dev_ptr(coef), int(psi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_apply_hamiltonian_paw")


def fd_apply_overlap(plan, paw, psi, out, coef, stream=None) -> None:
    """out = psi + sum |p~> Delta S <p~|psi> (Eq. 7)."""
    _check_arrays(plan, "fd_apply_overlap", batch=(psi, out))
    _check_coef(paw, psi, coef, "fd_apply_overlap")
    rc = load_library().fd_apply_overlap(plan, paw, _dev_ptr(psi), _dev_ptr(out), _dev_ptr(coef),
                                         int(psi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_apply_overlap")


def fd_poisson_residual(plan, phi, rhs, out, stream=None) -> None:
    """out = rhs - A phi for the plan's A = scale lap_FD."""
    _check_arrays(plan, "fd_poisson_residual", batch=(phi, rhs, out))
    rc = load_library().fd_poisson_residual(plan, _dev_ptr(phi), _dev_ptr(rhs), _dev_ptr(out),
                                            int(phi.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_poisson_residual")


def fd_mg_create(shape, h, nn: int = 3, bc=(1, 1, 1), p: int = 2, max_levels: int = 16,
                 max_nbands: int = 1, device: int = 0) -> ctypes.c_void_p:
    """Multigrid hierarchy for lap_FD phi = rhs (include/fdham.h: fd_mg_create)."""
    mg = ctypes.c_void_p()
    rc = load_library().fd_mg_create(ctypes.byref(mg), (ctypes.c_int32 * 3)(*[int(s) for s in shape]),
                                     (ctypes.c_double * 3)(*[float(x) for x in h]), int(nn),
                                     (ctypes.c_int32 * 3)(*[int(b) for b in bc]), int(p),
                                     int(max_levels), int(max_nbands), int(device))
    _check(rc, "fd_mg_create")
    return mg


def fd_mg_destroy(mg) -> None:
    _check(load_library().fd_mg_destroy(mg), "fd_mg_destroy")


def fd_mg_levels(mg) -> int:
    return int(load_library().fd_mg_levels(mg))


def fd_mg_get_info(mg) -> dict:
    """Finest shape, max_nbands, device, levels, graph captures so far, whether capture was given up."""
    buf = (ctypes.c_int64 * 8)()
    _check(load_library().fd_mg_get_info(mg, buf), "fd_mg_get_info")
    return {"shape": (buf[0], buf[1], buf[2]), "max_nbands": buf[3], "device": buf[4], "levels": buf[5],
            "graph_captures": buf[6], "graph_off": bool(buf[7])}


def fd_mg_vcycle(mg, phi, rhs, nu1: int = 2, nu2: int = 2, nu_coarse: int = 8,
                 omega: float = 2.0 / 3.0, stream=None) -> None:
    """One V-cycle in place on phi (float64 CUDA tensors [nbands, nx, ny, nz])."""
    if phi.shape != rhs.shape or phi.dtype != rhs.dtype or str(phi.dtype) != "torch.float64":
        raise ValueError("fd_mg_vcycle: phi and rhs must be float64 tensors of the same shape")
    info = fd_mg_get_info(mg)
    # (nbands > max_nbands is the library's own check: FD_ERR_INVALID, nothing is touched)
    if phi.dim() != 4 or tuple(phi.shape[1:]) != info["shape"]:
        raise ValueError(f"fd_mg_vcycle: expected [nbands, {info['shape']}], got {tuple(phi.shape)}")
    if phi.device.index != info["device"] or rhs.device.index != info["device"]:
        raise ValueError(f"fd_mg_vcycle: tensors must be on cuda:{info['device']}")
    rc = load_library().fd_mg_vcycle(mg, _dev_ptr(phi), _dev_ptr(rhs), int(phi.shape[0]), int(nu1),
                                     int(nu2), int(nu_coarse), float(omega), _stream_ptr(stream))
    _check(rc, "fd_mg_vcycle")


def fd_paw_expect(plan, paw, which: int, coef, out, stream=None) -> None:
    """out[b] += (1/dv) Re P_b^H dO P_b from the projections coef (which: 0 Delta H, 1 Delta S)."""
    info = _plan_info(plan)
    ntot = fd_paw_nproj_total(paw)
    if coef.dim() != 2 or coef.shape[1] != ntot or coef.dtype != _torch_dtypes(info["dtype"])[0] or \
            coef.device.index != info["device"]:
        raise ValueError(f"fd_paw_expect: coef must be [nbands, {ntot}] of the plan's dtype on its device")
    if tuple(out.shape) != (coef.shape[0],) or str(out.dtype) != "torch.float64" or out.device != coef.device:
        raise ValueError("fd_paw_expect: out must be float64 [nbands] on the device of coef")
    rc = load_library().fd_paw_expect(plan, paw, int(which), _dev_ptr(coef), _dev_ptr(out),
                                      int(coef.shape[0]), _stream_ptr(stream))
    _check(rc, "fd_paw_expect")


def fd_peak_kernel(kind: int, a, b, n: int, blocks: int = 0, stream=None) -> None:
    """Micro-benchmark kernels (include/fdham.h: fd_peak_kernel); a, b float64 CUDA tensors."""
    rc = load_library().fd_peak_kernel(int(kind), _dev_ptr(a), _dev_ptr(b) if b is not None else
                                       ctypes.c_void_p(0), int(n), int(blocks), _stream_ptr(stream))
    _check(rc, "fd_peak_kernel")


def fd_plan_set_kernel(plan, kernel: int, param: int = 0) -> None:
    _check(load_library().fd_plan_set_kernel(plan, int(kernel), int(param)), "fd_plan_set_kernel")


def fd_plan_get_kernel(plan) -> int:
    return int(load_library().fd_plan_get_kernel(plan))


def fd_plan_kernel_for(plan, nbands: int) -> int:
    return int(load_library().fd_plan_kernel_for(plan, int(nbands)))


def fd_plan_launches(plan) -> int:
    return int(load_library().fd_plan_launches(plan))


def fd_plan_get_weights(plan, nn: int):
    buf = (ctypes.c_double * (3 * (nn + 1)))()
    n = load_library().fd_plan_get_weights(plan, buf, 3 * (nn + 1))
    if n < 0:
        raise FDError(n, "fd_plan_get_weights")
    return [[buf[d * (nn + 1) + j] for j in range(nn + 1)] for d in range(3)]


class FDHamiltonian:
    """Convenience owner of a plan: `H = FDHamiltonian(shape, h, ...); H.apply(psi, v_eff)`."""

    def __init__(self, shape, h, nn=3, bc=(1, 1, 1), k=None, complex_=False, device=0):
        self.shape = tuple(int(s) for s in shape)
        self.complex = bool(complex_)
        self.plan = fd_create(self.shape, h, nn, bc, k, FD_C128 if complex_ else FD_F64, device)

    def apply(self, psi, v_eff=None, out=None, stream=None):
        import torch
        if out is None:
            out = torch.empty_like(psi)
        if v_eff is None:
            fd_apply_kinetic(self.plan, psi, out, stream)
        else:
            fd_apply_hamiltonian(self.plan, psi, v_eff, out, stream)
        return out

    def close(self):
        if self.plan is not None:
            fd_destroy(self.plan)
            self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
