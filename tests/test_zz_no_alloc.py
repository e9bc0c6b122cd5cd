"""GPU test of fd_apply_hamiltonian_expect_static, the one entry point of libfdham that brings its
own scratch memory instead of taking a workspace from the caller.

Who needs it: code that is not allowed to allocate device memory.  A plug-in that runs under a host
application whose pool owns the whole device cannot call cudaMalloc; neither can a latency path that
must not hit the device-wide synchronisation cudaMalloc / cudaFree cause, nor a C caller whose
device memory sits behind a caching allocator it cannot reach.  For them the partial sums of the
fused <psi|H|psi>, <psi|psi> go to a fixed 4 MiB array inside the library image
(FD_STATIC_SCRATCH_BYTES, include/fdham.h).

What is checked here: the new call gives what the existing workspace call gives, within the parity
tolerances the other GPU tests use (and, since both run the same kernels in the same order, bit for
bit), on two calls in a row that share the array.  The second call runs a different plan on another
kernel family with a smaller footprint, so anything it wrongly picked up from what the first call
left in the array would show.  Also: the size limit is enforced with its own status code before any
launch, and the largest batch that fits still agrees.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  The test depends on no state left by other tests: the first call on the
device does the one-time address lookup whether or not anything ran before it.
"""
import numpy as np
import pytest

import workloads as W
from helpers import kinetic_row_sum, parity_tol

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def fd():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2310_14776_b200 import build
    build.build()
    import paper_2310_14776_b200 as fd
    fd.load_library()
    return fd


def _tolerances(cfg, psi, v):
    """(out, eps, norm) tolerances as in tests/test_gpu_next.py: north_star's per-point bound for
    H psi, and P max|psi| times it for the grid sums (reading R15)."""
    P = psi[0].size
    mp = float(np.abs(psi).max())
    mv = float(np.abs(v[None] * psi * psi).max())
    t_out = parity_tol(cfg.h, cfg.nn, psi, v)
    t_eps = 1e-12 * P * (mp * mp * kinetic_row_sum(cfg.h, cfg.nn) + mv)
    t_norm = 1e-12 * P * mp * mp
    return t_out, t_eps, t_norm


def _both_paths(fd, cfg, kernel, tyc=0):
    """One batch through the existing call (workspace from torch, filled with NaN) and through the
    no-allocation call; returns whether they agree within tolerance and bit for bit."""
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    dt = fd.FD_C128 if cfg.complex else fd.FD_F64
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None, dt, 0)
    try:
        fd.fd_plan_set_kernel(plan, kernel, tyc)
        nb = psi.shape[0]
        assert fd.fd_plan_kernel_for(plan, nb) == kernel
        d_psi, d_v = torch.from_numpy(psi).cuda(), torch.from_numpy(v).cuda()

        def fresh():
            return (torch.full_like(d_psi, float("nan")),
                    torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda"),
                    torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda"))

        need = fd.fd_expect_workspace_bytes(plan, nb)
        assert 0 < need <= fd.FD_STATIC_SCRATCH_BYTES
        out_a, eps_a, norm_a = fresh()
        ws = torch.full((need // 8 + 1,), float("nan"), dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, d_psi, d_v, out_a, eps_a, norm_a, ws)
        out_b, eps_b, norm_b = fresh()
        fd.fd_apply_hamiltonian_expect_static(plan, d_psi, d_v, out_b, eps_b, norm_b)
        torch.cuda.synchronize()
        for t in (out_a, eps_a, norm_a, out_b, eps_b, norm_b):
            assert bool(torch.isfinite(torch.view_as_real(t) if t.is_complex() else t).all())
        t_out, t_eps, t_norm = _tolerances(cfg, psi, v)
        assert float((out_a - out_b).abs().max()) <= t_out
        assert float((eps_a - eps_b).abs().max()) <= t_eps
        assert float((norm_a - norm_b).abs().max()) <= t_norm
        # same kernels, same order of additions: the stronger statement holds too
        assert torch.equal(eps_a, eps_b) and torch.equal(norm_a, norm_b)
        assert torch.equal(torch.view_as_real(out_a) if out_a.is_complex() else out_a,
                           torch.view_as_real(out_b) if out_b.is_complex() else out_b)
    finally:
        fd.fd_destroy(plan)


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(fd):
    # call 1: the sweep kernel's fused epilogue, several y tiles and band segments (larger footprint)
    big = W.custom((24, 40, 16), (0.2, 0.21, 0.18), (1, 0, 1), nbands=11)
    _both_paths(fd, big, fd.FD_KERNEL_SWEEP, tyc=8)
    # call 2, right after it on the same array: another plan (complex, Bloch phases) on the generic
    # kernel's two-pass form, smaller footprint; stale partial sums of call 1 lie beyond and below it
    small = W.custom((10, 22, 12), (0.2, 0.23, 0.17), (1, 1, 1), k=(0.25, 0.125, -0.3),
                     complex_=True, nbands=4)
    _both_paths(fd, small, fd.FD_KERNEL_GENERIC)
    # and the first plan's shape again on the sweep kernel, complex this time
    again = W.custom((10, 20, 12), (0.2, 0.23, 0.17), (1, 1, 0), k=(0.25, 0.125, 0.0),
                     complex_=True, nbands=4)
    _both_paths(fd, again, fd.FD_KERNEL_SWEEP, tyc=8)


def test_static_scratch_limit_is_enforced_and_the_largest_batch_agrees(fd):
    """On an 8^3 grid the two-pass form needs 16 bytes of scratch per band, so the 4 MiB array
    holds exactly FD_STATIC_SCRATCH_BYTES / 16 bands: that batch runs and agrees with the workspace
    call; one band more is refused with FD_ERR_SCRATCH and nothing is written."""
    limit = fd.FD_STATIC_SCRATCH_BYTES
    nmax = limit // 16
    shape, h = (8, 8, 8), (0.2 / 0.529177210903,) * 3
    plan = fd.fd_create(shape, h, 3, (1, 1, 1), None, fd.FD_F64, 0)
    try:
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_GENERIC, 0)
        assert fd.fd_expect_workspace_bytes(plan, nmax) == limit
        assert fd.fd_expect_workspace_bytes(plan, nmax + 1) > limit
        g = torch.Generator(device="cuda").manual_seed(14776)
        psi = torch.randn((nmax + 1,) + shape, dtype=torch.float64, device="cuda", generator=g)
        v = torch.rand(shape, dtype=torch.float64, device="cuda", generator=g) - 1.0
        out = torch.full_like(psi, float("nan"))
        eps = torch.full((nmax + 1,), float("nan"), dtype=torch.float64, device="cuda")
        norm = torch.full_like(eps, float("nan"))
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_hamiltonian_expect_static(plan, psi, v, out, eps, norm)
        assert ei.value.status == fd.FD_ERR_SCRATCH
        assert "scratch" in fd.strerror(fd.FD_ERR_SCRATCH)
        torch.cuda.synchronize()
        assert bool(torch.isnan(eps).all()) and bool(torch.isnan(out).all())    # nothing ran
        # the largest batch that fits
        fd.fd_apply_hamiltonian_expect_static(plan, psi[:nmax], v, out[:nmax], eps[:nmax], norm[:nmax])
        out_a = torch.full_like(out[:nmax], float("nan"))
        eps_a, norm_a = torch.full_like(eps[:nmax], float("nan")), torch.full_like(eps[:nmax], float("nan"))
        ws = torch.full((limit // 8,), float("nan"), dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, psi[:nmax], v, out_a, eps_a, norm_a, ws)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(eps[:nmax]).all()) and bool(torch.isfinite(norm[:nmax]).all())
        assert torch.equal(eps[:nmax], eps_a) and torch.equal(norm[:nmax], norm_a)
        assert torch.equal(out[:nmax], out_a)
        # the sums themselves, against a plain torch reduction of the stored H psi (float64; the
        # tolerance of tests/test_gpu_next.py's full-size check: 1e-12 P max|psi|^2 (S + max|v|))
        mp = float(psi.abs().max())
        tol = 1e-12 * 512 * mp * mp * (kinetic_row_sum(h, 3) + 1.0)
        ref = (psi[:nmax] * out[:nmax]).sum(dim=(1, 2, 3))
        assert float((ref - eps[:nmax]).abs().max()) <= tol
    finally:
        fd.fd_destroy(plan)
