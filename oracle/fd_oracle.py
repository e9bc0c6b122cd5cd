"""ctypes front end of the CPU oracle (oracle/fd_oracle.c) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2310_14776_b200 and shares no code with it.

The operator is Eq. 6 of the paper without the PAW projector term with the
kinetic operator in its finite-difference representation; see fd_oracle.c for the
definition and DESIGN.md for the readings taken where the paper is silent.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence

import numpy as np

from . import build as _build

BC_ZERO = 0
BC_PERIODIC = 1

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        i32p = ctypes.POINTER(ctypes.c_int32)
        f64p = ctypes.POINTER(ctypes.c_double)
        i64p = ctypes.POINTER(ctypes.c_int64)
        vp = ctypes.c_void_p
        lib.fd_oracle_coeffs.argtypes = [ctypes.c_int, f64p]
        lib.fd_oracle_coeffs.restype = ctypes.c_int
        lib.fd_oracle_apply.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p, ctypes.c_int32,
                                        vp, f64p, vp, ctypes.c_int64, ctypes.c_int32]
        lib.fd_oracle_apply.restype = ctypes.c_int
        lib.fd_oracle_apply_scaled.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p,
                                               ctypes.c_int32, vp, f64p, vp, ctypes.c_int64,
                                               ctypes.c_int32, ctypes.c_double]
        lib.fd_oracle_apply_scaled.restype = ctypes.c_int
        lib.fd_oracle_points.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p, ctypes.c_int32,
                                         vp, f64p, ctypes.c_int64, i64p, ctypes.c_int64, vp]
        lib.fd_oracle_points.restype = ctypes.c_int
        lib.fd_oracle_dense.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p, f64p, vp]
        lib.fd_oracle_dense.restype = ctypes.c_int
        lib.fd_oracle_max_threads.argtypes = []
        lib.fd_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _i32(a):
    return (ctypes.c_int32 * 3)(*[int(x) for x in a])


def _f64(a):
    return (ctypes.c_double * 3)(*[float(x) for x in a])


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _f64ptr(a: Optional[np.ndarray]):
    if a is None:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def max_threads() -> int:
    return int(_load().fd_oracle_max_threads())


def coeffs(nn: int) -> np.ndarray:
    """c_0..c_nn of the order-2nn central second-derivative stencil (fd_oracle.c)."""
    c = (ctypes.c_double * (nn + 1))()
    if _load().fd_oracle_coeffs(int(nn), c) != 0:
        raise ValueError(f"bad nn={nn}")
    return np.array(list(c), dtype=np.float64)


def _check_inputs(shape, psi, v_eff):
    shape = tuple(int(s) for s in shape)
    if psi.ndim != 4 or tuple(psi.shape[1:]) != shape:
        raise ValueError(f"psi must be [nbands,{shape}], got {psi.shape}")
    if psi.dtype not in (np.float64, np.complex128):
        raise ValueError("psi must be float64 or complex128")
    psi = np.ascontiguousarray(psi)
    if v_eff is not None:
        if tuple(v_eff.shape) != shape or v_eff.dtype != np.float64:
            raise ValueError("v_eff must be float64 [nx,ny,nz]")
        v_eff = np.ascontiguousarray(v_eff)
    return shape, psi, v_eff


def apply(shape: Sequence[int], h: Sequence[float], nn: int, bc: Sequence[int],
          k: Optional[Sequence[float]], psi: np.ndarray, v_eff: Optional[np.ndarray] = None,
          nthreads: int = 0, scale: Optional[float] = None) -> np.ndarray:
    """H psi (v_eff given) or T psi (v_eff None) for psi[nbands,nx,ny,nz]; returns a new array.
    scale: prefactor of the FD Laplacian instead of -1/2 (None = the kinetic operator of Eq. 6)."""
    shape, psi, v_eff = _check_inputs(shape, psi, v_eff)
    out = np.empty_like(psi)
    is_c = psi.dtype == np.complex128
    kk = _f64(k) if k is not None else None
    if scale is None:
        rc = _load().fd_oracle_apply(_i32(shape), _f64(h), int(nn), _i32(bc), kk, int(is_c),
                                     _ptr(psi), _f64ptr(v_eff), _ptr(out), psi.shape[0],
                                     int(nthreads))
    else:
        rc = _load().fd_oracle_apply_scaled(_i32(shape), _f64(h), int(nn), _i32(bc), kk,
                                            int(is_c), _ptr(psi), _f64ptr(v_eff), _ptr(out),
                                            psi.shape[0], int(nthreads), float(scale))
    if rc != 0:
        raise ValueError("fd_oracle_apply: invalid argument")
    return out


def points(shape, h, nn, bc, k, psi: np.ndarray, v_eff: Optional[np.ndarray],
           pts: np.ndarray) -> np.ndarray:
    """H psi at sampled outputs pts[s] = (band, ix, iy, iz)."""
    shape, psi, v_eff = _check_inputs(shape, psi, v_eff)
    pts = np.ascontiguousarray(pts, dtype=np.int64).reshape(-1, 4)
    out = np.empty(pts.shape[0], dtype=psi.dtype)
    is_c = psi.dtype == np.complex128
    kk = _f64(k) if k is not None else None
    rc = _load().fd_oracle_points(_i32(shape), _f64(h), int(nn), _i32(bc), kk, int(is_c),
                                  _ptr(psi), _f64ptr(v_eff), psi.shape[0],
                                  pts.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                                  pts.shape[0], _ptr(out))
    if rc != 0:
        raise ValueError("fd_oracle_points: invalid argument")
    return out


def dense(shape, h, nn, bc, k=None, v_eff: Optional[np.ndarray] = None) -> np.ndarray:
    """Explicit P x P complex matrix of H, assembled tap by tap (independent of apply())."""
    shape = tuple(int(s) for s in shape)
    P = shape[0] * shape[1] * shape[2]
    if P > 4096:
        raise ValueError("dense oracle is for tiny grids only")
    if v_eff is not None:
        v_eff = np.ascontiguousarray(v_eff, dtype=np.float64)
        assert v_eff.shape == shape
    M = np.empty((P, P), dtype=np.complex128)
    kk = _f64(k) if k is not None else None
    rc = _load().fd_oracle_dense(_i32(shape), _f64(h), int(nn), _i32(bc), kk, _f64ptr(v_eff),
                                 _ptr(M))
    if rc != 0:
        raise ValueError("fd_oracle_dense: invalid argument")
    return M
