"""Pins of fd_oracle_paw_apply: dense P dO P^H dv built here in numpy, Hermiticity,
rank, support, a one-point projector, invariance under lattice translations of a box (Bloch
consistency), projections."""
import numpy as np
import pytest

import workloads as W


def _dense_projectors(cfg, paw):
    """[npoints, ntot] complex matrix of the crystal projectors on the home cell, built with an
    explicit loop over box points (wrap + conj Bloch factor when stored, zero-BC parts dropped)."""
    n = cfg.shape
    Pm = np.zeros((int(np.prod(n)), paw.ntot), dtype=np.complex128)
    col = 0
    for a in range(paw.natoms):
        p = paw.proj_of(a)
        s0, sz = paw.box_start[a], paw.box_size[a]
        for rx in range(sz[0]):
            for ry in range(sz[1]):
                for rz in range(sz[2]):
                    idx, ph, ok = [], 1.0, True
                    for d, r in enumerate((s0[0] + rx, s0[1] + ry, s0[2] + rz)):
                        w = r // n[d]
                        if w != 0:
                            if cfg.bc[d] == 0:
                                ok = False
                                break
                            ph *= np.exp(-2j * np.pi * cfg.k[d] * w)    # e^{ik.R}, R = -w n
                        idx.append(r - w * n[d])
                    if not ok:
                        continue
                    lin = (idx[0] * n[1] + idx[1]) * n[2] + idx[2]
                    Pm[lin, col:col + p.shape[0]] += p[:, rx, ry, rz] * ph
        col += p.shape[0]
    return Pm


def _block_diag(paw):
    D = np.zeros((paw.ntot, paw.ntot))
    o = 0
    for a in range(paw.natoms):
        m = paw.dmat_of(a)
        D[o:o + m.shape[0], o:o + m.shape[0]] = m
        o += m.shape[0]
    return D


@pytest.mark.parametrize("bc,cplx", [((1, 1, 1), True), ((1, 0, 1), True), ((0, 0, 0), False),
                                     ((1, 1, 0), False)])
def test_matches_dense_projector_matrix(oracle, bc, cplx):
    k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc)) if cplx else (0, 0, 0)
    cfg = W.custom((9, 8, 10), (0.2, 0.22, 0.18), bc, k=k, complex_=cplx, nbands=3)
    paw = W.make_paw(cfg, 4, nproj=5)
    psi = W.make_psi(cfg)
    dv = np.prod(cfg.h)
    Pm = _dense_projectors(cfg, paw)
    D = _block_diag(paw)
    N = dv * Pm @ D @ Pm.conj().T
    want = (N @ psi.reshape(3, -1).T).T.reshape(psi.shape)
    got, coef = oracle.paw_apply(cfg.shape, cfg.h, bc, k if cplx else None, psi, paw.box_start,
                                 paw.box_size, paw.nproj, paw.proj, paw.dmat, want_coef=True)
    if not cplx:
        assert np.max(np.abs(want.imag)) < 1e-14
        want = want.real
    assert np.max(np.abs(got - want)) < 1e-12 * max(1.0, np.abs(want).max())
    assert np.max(np.abs(coef - dv * (psi.reshape(3, -1) @ Pm.conj()))) < 1e-12
    # accumulate form: out given -> out + term
    base = W.make_psi(W.custom(cfg.shape, cfg.h_angstrom, bc, k=k, complex_=cplx, nbands=3, index=7))
    got2 = oracle.paw_apply(cfg.shape, cfg.h, bc, k if cplx else None, psi, paw.box_start,
                            paw.box_size, paw.nproj, paw.proj, paw.dmat, out=base)
    assert np.max(np.abs(got2 - (base + got))) < 1e-13 * max(1.0, np.abs(got).max())
    # Hermitian for symmetric dO; rank = number of projectors; zero outside the supports
    assert np.max(np.abs(N - N.conj().T)) < 1e-14
    support = np.abs(Pm).sum(axis=1) > 0
    assert np.all(got.reshape(3, -1)[:, ~support] == 0.0)
    sv = np.linalg.svd(Pm, compute_uv=False)
    assert np.sum(sv > 1e-10 * sv[0]) == paw.ntot


def test_one_point_projector_and_lattice_translation(oracle):
    cfg = W.custom((6, 7, 8), (0.2, 0.2, 0.2), (1, 1, 1), k=(0.25, 0.125, -0.3), complex_=True,
                   nbands=2)
    psi = W.make_psi(cfg)
    dv = np.prod(cfg.h)
    one = dict(box_size=[[1, 1, 1]], nproj=[1], proj=[2.0], dmat=[-1.5])
    got = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, cfg.k, psi, [[2, 3, 4]], **one)
    want = np.zeros_like(psi)
    want[:, 2, 3, 4] = dv * 2.0 * -1.5 * 2.0 * psi[:, 2, 3, 4]
    assert np.max(np.abs(got - want)) < 1e-15
    # the same atom named by a periodic image of its box gives the same operator
    paw = W.make_paw(cfg, 3, nproj=4)
    ref = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, cfg.k, psi, paw.box_start, paw.box_size,
                           paw.nproj, paw.proj, paw.dmat)
    shifted = paw.box_start + np.array([[6, 0, -8], [-6, 7, 0], [12, -7, 8]], dtype=np.int32)
    got = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, cfg.k, psi, shifted, paw.box_size,
                           paw.nproj, paw.proj, paw.dmat)
    assert np.max(np.abs(got - ref)) < 1e-13 * max(1.0, np.abs(ref).max())
    # Hermiticity as a bilinear identity on random vectors
    phi = W.make_psi(W.custom(cfg.shape, cfg.h_angstrom, cfg.bc, k=cfg.k, complex_=True, nbands=2,
                              index=5))
    nphi = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, cfg.k, phi, paw.box_start, paw.box_size,
                            paw.nproj, paw.proj, paw.dmat)
    assert abs(np.vdot(phi, ref) - np.conj(np.vdot(psi, nphi))) < 1e-12


def test_paw_expectation_value_equals_projection_quadratic_form(oracle):
    """sum_r conj(psi) (N psi) = (1/dv) P^H dO P with P = dv <p~|psi>: the grid sum against the
    quadratic form of the projections (two different routes through the oracle's definition)."""
    cfg = W.custom((9, 8, 10), (0.2, 0.22, 0.18), (1, 0, 1), k=(0.25, 0.0, -0.3), complex_=True, nbands=3)
    paw = W.make_paw(cfg, 4, nproj=5)
    psi = W.make_psi(cfg)
    dv = np.prod(cfg.h)
    got = oracle.paw_expect(cfg.shape, cfg.h, cfg.bc, cfg.k, psi, paw.box_start, paw.box_size, paw.nproj,
                            paw.proj, paw.dmat)
    Pm = _dense_projectors(cfg, paw)
    D = _block_diag(paw)
    P = dv * (psi.reshape(3, -1) @ Pm.conj())
    want = np.einsum("bi,ij,bj->b", P.conj(), D, P) / dv
    assert np.max(np.abs(got - want)) < 1e-12 * max(1.0, np.abs(want).max())
    assert np.max(np.abs(got.imag)) < 1e-12 * max(1.0, np.abs(want).max())       # symmetric dO
