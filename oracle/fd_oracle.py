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
        c128p = ctypes.c_void_p
        lib.fd_oracle_expect.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p, ctypes.c_int32,
                                         vp, f64p, vp, ctypes.c_int64, ctypes.c_double, c128p, f64p]
        lib.fd_oracle_expect.restype = ctypes.c_int
        lib.fd_oracle_residual.argtypes = [ctypes.c_int64, ctypes.c_int32, vp, vp, f64p, vp,
                                           ctypes.c_int64]
        lib.fd_oracle_residual.restype = ctypes.c_int
        lib.fd_oracle_jacobi.argtypes = [i32p, f64p, ctypes.c_int32, i32p, f64p, f64p, f64p,
                                         ctypes.c_int64, ctypes.c_double, ctypes.c_double]
        lib.fd_oracle_jacobi.restype = ctypes.c_int
        lib.fd_oracle_transfer_weights.argtypes = [ctypes.c_int32, f64p]
        lib.fd_oracle_transfer_weights.restype = ctypes.c_int
        lib.fd_oracle_restrict.argtypes = [i32p, i32p, ctypes.c_int32, f64p, f64p, ctypes.c_int64]
        lib.fd_oracle_restrict.restype = ctypes.c_int
        lib.fd_oracle_interpolate.argtypes = [i32p, i32p, ctypes.c_int32, f64p, f64p,
                                              ctypes.c_int64]
        lib.fd_oracle_interpolate.restype = ctypes.c_int
        lib.fd_oracle_paw_apply.argtypes = [i32p, f64p, i32p, f64p, ctypes.c_int32, ctypes.c_int32,
                                            i32p, i32p, i32p, f64p, f64p, vp, vp, vp,
                                            ctypes.c_int64, ctypes.c_int32]
        lib.fd_oracle_paw_apply.restype = ctypes.c_int
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


# ------------------------------------------------------------------------------ SURVEY 8(f) rows

def expect(shape, h, nn, bc, k, psi: np.ndarray, v_eff: Optional[np.ndarray] = None,
           scale: float = -0.5, want_out: bool = False):
    """(eps[nbands] complex, norm[nbands]) = (sum conj(psi) H psi, sum |psi|^2) per band (plain grid
    sums, fd_oracle.c: fd_oracle_expect); with want_out also H psi."""
    shape, psi, v_eff = _check_inputs(shape, psi, v_eff)
    nb = psi.shape[0]
    eps = np.empty(nb, dtype=np.complex128)
    norm = np.empty(nb, dtype=np.float64)
    out = np.empty_like(psi) if want_out else None
    kk = _f64(k) if k is not None else None
    rc = _load().fd_oracle_expect(_i32(shape), _f64(h), int(nn), _i32(bc), kk,
                                  int(psi.dtype == np.complex128), _ptr(psi), _f64ptr(v_eff),
                                  _ptr(out) if out is not None else None, nb, float(scale),
                                  _ptr(eps), _f64ptr(norm))
    if rc != 0:
        raise ValueError("fd_oracle_expect: invalid argument")
    return (eps, norm, out) if want_out else (eps, norm)


def residual(psi: np.ndarray, hpsi: np.ndarray, lam: np.ndarray) -> np.ndarray:
    """r_b = hpsi_b - lam[b] psi_b."""
    psi, hpsi = np.ascontiguousarray(psi), np.ascontiguousarray(hpsi)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    assert psi.shape == hpsi.shape and psi.dtype == hpsi.dtype and lam.shape == (psi.shape[0],)
    out = np.empty_like(psi)
    rc = _load().fd_oracle_residual(int(psi[0].size), int(psi.dtype == np.complex128), _ptr(psi),
                                    _ptr(hpsi), _f64ptr(lam), _ptr(out), psi.shape[0])
    if rc != 0:
        raise ValueError("fd_oracle_residual: invalid argument")
    return out


def jacobi(shape, h, nn, bc, phi: np.ndarray, rhs: np.ndarray, omega: float,
           scale: float = 1.0) -> np.ndarray:
    """One weighted-Jacobi sweep for (scale lap_FD) phi = rhs (fd_oracle.c: fd_oracle_jacobi)."""
    shape, phi, _ = _check_inputs(shape, phi, None)
    rhs = np.ascontiguousarray(rhs, dtype=np.float64)
    assert phi.dtype == np.float64 and rhs.shape == phi.shape
    out = np.empty_like(phi)
    rc = _load().fd_oracle_jacobi(_i32(shape), _f64(h), int(nn), _i32(bc), _f64ptr(phi),
                                  _f64ptr(rhs), _f64ptr(out), phi.shape[0], float(omega),
                                  float(scale))
    if rc != 0:
        raise ValueError("fd_oracle_jacobi: invalid argument")
    return out


def transfer_weights(p: int) -> np.ndarray:
    """b[1..p] (b[0] = 0): midpoint Lagrange weights of the order-p grid transfer."""
    b = (ctypes.c_double * (p + 1))()
    if _load().fd_oracle_transfer_weights(int(p), b) != 0:
        raise ValueError(f"bad transfer order p={p}")
    return np.array(list(b), dtype=np.float64)


def coarse_shape(shape_fine, bc):
    """Coarse extents of a fine grid: n/2 on periodic axes (n even), (n-1)/2 on zero-BC axes."""
    return tuple(int(n) // 2 if b else (int(n) - 1) // 2 for n, b in zip(shape_fine, bc))


def restrict(shape_fine, bc, p: int, fine: np.ndarray) -> np.ndarray:
    fine = np.ascontiguousarray(fine, dtype=np.float64)
    assert fine.ndim == 4 and tuple(fine.shape[1:]) == tuple(shape_fine)
    coarse = np.empty((fine.shape[0],) + coarse_shape(shape_fine, bc), dtype=np.float64)
    rc = _load().fd_oracle_restrict(_i32(shape_fine), _i32(bc), int(p), _f64ptr(fine),
                                    _f64ptr(coarse), fine.shape[0])
    if rc != 0:
        raise ValueError("fd_oracle_restrict: invalid argument")
    return coarse


def interpolate(shape_fine, bc, p: int, coarse: np.ndarray) -> np.ndarray:
    coarse = np.ascontiguousarray(coarse, dtype=np.float64)
    assert coarse.ndim == 4 and tuple(coarse.shape[1:]) == coarse_shape(shape_fine, bc)
    fine = np.empty((coarse.shape[0],) + tuple(int(n) for n in shape_fine), dtype=np.float64)
    rc = _load().fd_oracle_interpolate(_i32(shape_fine), _i32(bc), int(p), _f64ptr(coarse),
                                       _f64ptr(fine), coarse.shape[0])
    if rc != 0:
        raise ValueError("fd_oracle_interpolate: invalid argument")
    return fine


def paw_apply(shape, h, bc, k, psi: np.ndarray, box_start, box_size, nproj, proj, dmat,
              out: Optional[np.ndarray] = None, want_coef: bool = False):
    """Non-local PAW term (fd_oracle.c: fd_oracle_paw_apply).  out None -> returns the term alone;
    out given -> returns out + term (a copy).  With want_coef also the projections
    P[nbands, sum n_i]."""
    shape, psi, _ = _check_inputs(shape, psi, None)
    is_c = psi.dtype == np.complex128
    bs = np.ascontiguousarray(box_start, dtype=np.int32).reshape(-1, 3)
    bz = np.ascontiguousarray(box_size, dtype=np.int32).reshape(-1, 3)
    npj = np.ascontiguousarray(nproj, dtype=np.int32)
    proj = np.ascontiguousarray(proj, dtype=np.float64)
    dmat = np.ascontiguousarray(dmat, dtype=np.float64)
    acc = out is not None
    res = np.array(out, dtype=psi.dtype, copy=True, order="C") if acc else np.empty_like(psi)
    coef = np.empty((psi.shape[0], int(npj.sum())), dtype=psi.dtype) if want_coef else None
    i32p = ctypes.POINTER(ctypes.c_int32)
    kk = _f64(k) if k is not None else None
    rc = _load().fd_oracle_paw_apply(_i32(shape), _f64(h), _i32(bc), kk, int(is_c), len(npj),
                                     bs.ctypes.data_as(i32p), bz.ctypes.data_as(i32p),
                                     npj.ctypes.data_as(i32p), _f64ptr(proj), _f64ptr(dmat),
                                     _ptr(psi), _ptr(res), _ptr(coef) if want_coef else None,
                                     psi.shape[0], int(acc))
    if rc != 0:
        raise ValueError("fd_oracle_paw_apply: invalid argument")
    return (res, coef) if want_coef else res


# ------------------------------------------------------------------------------ multigrid V-cycle

def mg_levels(shape, bc, nn: int, max_levels: int = 16):
    """Grid hierarchy of the V-cycle: level 0 = `shape`; a level is coarsened (n/2 on periodic axes,
    (n-1)/2 on zero-BC axes, fd_oracle.c: fd_oracle_restrict) while every axis allows it (even >= 2
    periodic / odd >= 3 zero-BC) and every coarse axis keeps at least max(nn, 2) points."""
    levels = [tuple(int(n) for n in shape)]
    while len(levels) < max_levels:
        s = levels[-1]
        if not all((n % 2 == 0 and n >= 2) if b else (n % 2 == 1 and n >= 3) for n, b in zip(s, bc)):
            break
        c = coarse_shape(s, bc)
        if min(c) < max(nn, 2):
            break
        levels.append(c)
    return levels


def vcycle(shape, h, nn: int, bc, p: int, phi: np.ndarray, rhs: np.ndarray, nu1: int = 2,
           nu2: int = 2, nu_coarse: int = 8, omega: float = 2.0 / 3.0, scale: float = 1.0,
           max_levels: int = 16, _level: int = 0, _levels=None) -> np.ndarray:
    """One multigrid V-cycle for (scale lap_FD) phi = rhs ("multigrid ... Jacobi"
    Poisson solvers; PAPER.md:93, :150 grid transfer), the textbook algorithm step by step:
        nu1 weighted-Jacobi sweeps;  r = rhs - A phi;  rhs_c = R r,  e_c = 0;
        e_c <- V-cycle on the coarse grid (spacing 2h; nu_coarse sweeps on the coarsest grid);
        phi += I e_c;  nu2 weighted-Jacobi sweeps.
    Every step is the oracle function of that step (jacobi, apply, restrict, interpolate)."""
    if _levels is None:
        _levels = mg_levels(shape, bc, nn, max_levels)
    phi = np.array(phi, dtype=np.float64, copy=True)
    hl = tuple(x * (2 ** _level) for x in h)
    if _level == len(_levels) - 1:
        for _ in range(nu_coarse):
            phi = jacobi(shape, hl, nn, bc, phi, rhs, omega, scale)
        return phi
    for _ in range(nu1):
        phi = jacobi(shape, hl, nn, bc, phi, rhs, omega, scale)
    r = rhs - apply(shape, hl, nn, bc, None, phi, None, scale=scale)
    rhs_c = restrict(shape, bc, p, r)
    e_c = vcycle(_levels[_level + 1], h, nn, bc, p, np.zeros_like(rhs_c), rhs_c, nu1, nu2, nu_coarse,
                 omega, scale, max_levels, _level + 1, _levels)
    phi = phi + interpolate(shape, bc, p, e_c)
    for _ in range(nu2):
        phi = jacobi(shape, hl, nn, bc, phi, rhs, omega, scale)
    return phi


def paw_expect(shape, h, bc, k, psi: np.ndarray, box_start, box_size, nproj, proj, dmat) -> np.ndarray:
    """<psi_b| sum_a sum_ii' |p~_i> dO_ii' <p~_i'| |psi_b> as the plain grid sum
    sum_r conj(psi_b(r)) (N psi_b)(r) of the non-local term above (no dv, like `expect`): the PAW
    part of <psi|H~|psi> (Eq. 6 third term, dO = Delta H) or of <psi|S~|psi> (Eq. 7, dO = Delta S).
    Returned complex; real up to rounding for symmetric dO."""
    npsi = paw_apply(shape, h, bc, k, psi, box_start, box_size, nproj, proj, dmat)
    return np.sum(np.conj(psi) * npsi, axis=(1, 2, 3)).astype(np.complex128)
