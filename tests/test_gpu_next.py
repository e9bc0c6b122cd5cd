"""GPU parity of the SURVEY 8(f) rows that ride the stencil kernels: f2 (fused expectation values,
residual) and the f3 weighted-Jacobi sweep, through the C ABI, against the CPU oracle."""
import itertools

import numpy as np
import pytest

import workloads as W
from helpers import kinetic_row_sum, parity_tol, planewave, planewave_eig

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


def expect_tol(h, nn, psi, v, scale=-0.5):
    """|d eps| <= 1e-12 P (max|psi|^2 S + max|v psi^2|): P times the per-point tolerance of H psi
    times max|psi| (reading R15); |d norm| <= 1e-12 P max|psi|^2."""
    P = psi[0].size
    mp = float(np.abs(psi).max())
    mv = float(np.abs(v[None] * psi * psi).max()) if v is not None else 0.0
    return 1e-12 * P * (mp * mp * kinetic_row_sum(h, nn, scale) + mv), 1e-12 * P * mp * mp


def run_expect(fd, cfg, psi, v, kernel, tyc=0, scale=None):
    k = cfg.k if cfg.complex else None
    dt = fd.FD_C128 if cfg.complex else fd.FD_F64
    plan = (fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, dt, 0) if scale is None else
            fd.fd_create_scaled(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, dt, 0, scale))
    try:
        if kernel != "auto":
            fd.fd_plan_set_kernel(plan, kernel, tyc)
        nb = psi.shape[0]
        d_psi = torch.from_numpy(psi).cuda()
        d_v = torch.from_numpy(v).cuda() if v is not None else None
        d_out = torch.full_like(d_psi, float("nan"))
        eps = torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda")
        norm = torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda")
        ws = torch.full((fd.fd_expect_workspace_bytes(plan, nb) // 8 + 1,), float("nan"),
                        dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, d_psi, d_v, d_out, eps, norm, ws)
        torch.cuda.synchronize()
        e1, n1 = eps.cpu().numpy(), norm.cpu().numpy()
        # bit-reproducible: a second call gives identical sums
        eps2, norm2 = torch.empty_like(eps), torch.empty_like(norm)
        fd.fd_apply_hamiltonian_expect(plan, d_psi, d_v, d_out, eps2, norm2, ws)
        torch.cuda.synchronize()
        assert torch.equal(eps, eps2) and torch.equal(norm, norm2)
        return d_out.cpu().numpy(), e1, n1, fd.fd_plan_kernel_for(plan, nb)
    finally:
        fd.fd_destroy(plan)


def check_expect(oracle, fd, cfg, kernel, tyc=0, with_v=True, scale=None):
    psi = W.make_psi(cfg)
    v = W.make_veff(cfg) if with_v else None
    k = cfg.k if cfg.complex else None
    sc = -0.5 if scale is None else scale
    got, eps, norm, used = run_expect(fd, cfg, psi, v, kernel, tyc, scale)
    w_eps, w_norm, want = oracle.expect(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi, v, scale=sc,
                                        want_out=True)
    assert np.max(np.abs(got - want)) <= parity_tol(cfg.h, cfg.nn, psi, v, sc)
    te, tn = expect_tol(cfg.h, cfg.nn, psi, v, sc)
    assert np.max(np.abs(eps - w_eps.real)) <= te, (np.max(np.abs(eps - w_eps.real)), te)
    assert np.max(np.abs(norm - w_norm)) <= tn
    return used


@pytest.mark.parametrize("idx", [1, 2])
@pytest.mark.parametrize("kernel", ["auto", "sweep", "generic"])
def test_expect_small_configs(oracle, fd, idx, kernel):
    cfg = W.get(idx)
    forced = {"auto": "auto", "sweep": fd.FD_KERNEL_SWEEP, "generic": fd.FD_KERNEL_GENERIC}[kernel]
    check_expect(oracle, fd, cfg, forced)


@pytest.mark.parametrize("bc", list(itertools.product((0, 1), repeat=3)))
def test_expect_all_bc_mixes_ragged_tiles(oracle, fd, bc):
    """several y tiles with a ragged one, several bands per team, real and complex Bloch, with and
    without v_eff, nn = 1..3, on the sweep kernel's fused epilogue"""
    for nn in (3, 2, 1):
        # ny = 28: tiles of 8, 8, 8, 4 rows (fused epilogue: ny % 4 == 0); ny = 30: two-pass form
        for ny in (28, 30):
            cfg = W.custom((10, ny, 16), (0.2, 0.23, 0.17), bc, nbands=5, nn=nn)
            assert check_expect(oracle, fd, cfg, fd.FD_KERNEL_SWEEP, tyc=8) == fd.FD_KERNEL_SWEEP
    k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
    ck = W.custom((10, 20, 12), (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=4)
    assert check_expect(oracle, fd, ck, fd.FD_KERNEL_SWEEP, tyc=8) == fd.FD_KERNEL_SWEEP
    check_expect(oracle, fd, ck, fd.FD_KERNEL_SWEEP, tyc=12, with_v=False)
    ck = W.custom((10, 22, 12), (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=4)
    check_expect(oracle, fd, ck, fd.FD_KERNEL_SWEEP, tyc=8)
    check_expect(oracle, fd, W.custom((9, 12, 8), (0.2, 0.23, 0.17), bc, nbands=3), fd.FD_KERNEL_SWEEP,
                 with_v=False, scale=1.0)


@pytest.mark.parametrize("xchunk", [3, 7])
def test_expect_band_segments_split_over_teams(oracle, fd, monkeypatch, xchunk):
    """FDHAM_TUNE=xchunk cuts bands into many team segments: every band's partial sums come from
    several teams and the fixed-order reduction must find all of them."""
    monkeypatch.setenv("FDHAM_TUNE", f"xchunk={xchunk},kernel=2")
    for bc, cplx, k in [((1, 1, 1), False, (0, 0, 0)), ((0, 1, 0), False, (0, 0, 0)),
                        ((1, 1, 1), True, (0.25, 0.125, -0.3))]:
        cfg = W.custom((24, 40, 16), (0.2, 0.21, 0.18), bc, k=k, complex_=cplx, nbands=11)
        assert check_expect(oracle, fd, cfg, "auto") == fd.FD_KERNEL_SWEEP


def test_expect_plane_waves_closed_form(fd):
    """against the closed form directly: eps = lambda P |a|^2, norm = P |a|^2"""
    n, h_ang, k = (24, 16, 32), (0.2, 0.21, 0.18), (0.25, 0.125, -0.4)
    ms = [(1, 2, 3), (0, 0, 0), (3, -2, 1)]
    cfg = W.custom(n, h_ang, (1, 1, 1), k=k, complex_=True, nbands=len(ms))
    psi = np.stack([planewave(n, k, m) for m in ms])
    _, eps, norm, used = run_expect(fd, cfg, psi, None, fd.FD_KERNEL_SWEEP)
    assert used == fd.FD_KERNEL_SWEEP
    P = float(np.prod(n))
    lam = np.array([planewave_eig(n, cfg.h, k, m) for m in ms])
    assert np.max(np.abs(norm - P)) <= 1e-12 * P
    assert np.max(np.abs(eps - lam * P)) <= 1e-12 * P * kinetic_row_sum(cfg.h)


def _big_expect(oracle, fd, cfg, bands):
    """full-size config in the launch configuration bench.py times; every band against the oracle's
    H psi and its grid sums, and `bands` against the oracle's own expect function"""
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None,
                        fd.FD_C128 if cfg.complex else fd.FD_F64, 0)
    try:
        tdt = torch.complex128 if cfg.complex else torch.float64
        d_psi = torch.empty((cfg.nbands,) + cfg.shape, dtype=tdt, device="cuda")
        for b0 in range(0, cfg.nbands, 32):
            bs = range(b0, min(cfg.nbands, b0 + 32))
            d_psi[b0:b0 + len(bs)] = torch.from_numpy(W.make_psi(cfg, bs)).cuda()
        v = W.make_veff(cfg)
        d_v = torch.from_numpy(v).cuda()
        d_out = torch.full_like(d_psi, float("nan"))
        eps = torch.empty(cfg.nbands, dtype=torch.float64, device="cuda")
        norm = torch.empty_like(eps)
        ws = torch.empty(fd.fd_expect_workspace_bytes(plan, cfg.nbands) // 8 + 1,
                         dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, d_psi, d_v, d_out, eps, norm, ws)
        torch.cuda.synchronize()
        # all bands (every team seam of the launch): H psi element by element, and eps / norm against
        # the plain grid sums of the ORACLE's H psi (not of the kernel's own output)
        kk = cfg.k if cfg.complex else None
        g_eps, g_norm = eps.cpu().numpy(), norm.cpu().numpy()
        for b0 in range(0, cfg.nbands, 32):
            bs = list(range(b0, min(cfg.nbands, b0 + 32)))
            psi_c = W.make_psi(cfg, bs)
            want_c = oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, kk, psi_c, v)
            te, tn = expect_tol(cfg.h, cfg.nn, psi_c, v)
            assert np.max(np.abs(d_out[b0:b0 + len(bs)].cpu().numpy() - want_c)) <= \
                parity_tol(cfg.h, cfg.nn, psi_c, v), b0
            w_e = np.array([np.vdot(psi_c[i], want_c[i]).real for i in range(len(bs))])
            w_n = np.array([np.vdot(psi_c[i], psi_c[i]).real for i in range(len(bs))])
            assert np.max(np.abs(g_eps[b0:b0 + len(bs)] - w_e)) <= te, b0
            assert np.max(np.abs(g_norm[b0:b0 + len(bs)] - w_n)) <= tn, b0
        psi_s = W.make_psi(cfg, bands)
        te, tn = expect_tol(cfg.h, cfg.nn, psi_s, v)
        # sampled whole bands against the oracle
        w_eps, w_norm, want = oracle.expect(cfg.shape, cfg.h, cfg.nn, cfg.bc,
                                            cfg.k if cfg.complex else None, psi_s, v, want_out=True)
        got = d_out[list(bands)].cpu().numpy()
        assert np.max(np.abs(got - want)) <= parity_tol(cfg.h, cfg.nn, psi_s, v)
        assert np.max(np.abs(eps[list(bands)].cpu().numpy() - w_eps.real)) <= te
        assert np.max(np.abs(norm[list(bands)].cpu().numpy() - w_norm)) <= tn
    finally:
        fd.fd_destroy(plan)


def test_expect_config3_full_size(oracle, fd):
    _big_expect(oracle, fd, W.get(3), [0, 100, 255])


def test_expect_config4_full_size(oracle, fd):
    _big_expect(oracle, fd, W.get(4), [0, 64, 127])


def test_expect_config5_full_size(oracle, fd):
    _big_expect(oracle, fd, W.get(5), [0, 383])


def test_expect_argument_errors(fd):
    plan = fd.fd_create((16, 16, 16), (0.4,) * 3)
    try:
        x = torch.zeros((2, 16, 16, 16), dtype=torch.float64, device="cuda")
        y = torch.zeros_like(x)
        e = torch.zeros(2, dtype=torch.float64, device="cuda")
        n = torch.zeros(2, dtype=torch.float64, device="cuda")
        need = fd.fd_expect_workspace_bytes(plan, 2)
        assert need >= 16
        small = torch.zeros(1, dtype=torch.float64, device="cuda")
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_hamiltonian_expect(plan, x, None, y, e, n, small)
        assert ei.value.status == -1
        ws = torch.zeros(need // 8 + 1, dtype=torch.float64, device="cuda")
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_hamiltonian_expect(plan, x, None, y, e, e, ws)          # eps aliases norm
        assert ei.value.status == -3
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_hamiltonian_expect(plan, x, None, y, y.view(-1)[:2], n, ws)   # eps inside out
        assert ei.value.status == -3
        fd.fd_apply_hamiltonian_expect(plan, x, None, y, e, n, ws)
        torch.cuda.synchronize()
    finally:
        fd.fd_destroy(plan)


@pytest.mark.parametrize("cplx", [False, True])
def test_residual(oracle, fd, cplx):
    cfg = W.custom((12, 16, 20), (0.2, 0.21, 0.19), (1, 0, 1), complex_=cplx, nbands=5,
                   k=(0.25, 0, 0.125) if cplx else (0, 0, 0))
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    got, eps, norm, _ = run_expect(fd, cfg, psi, v, "auto")
    plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc, cfg.k if cplx else None,
                        fd.FD_C128 if cplx else fd.FD_F64, 0)
    try:
        d_psi, d_h = torch.from_numpy(psi).cuda(), torch.from_numpy(got).cuda()
        d_e, d_n = torch.from_numpy(eps).cuda(), torch.from_numpy(norm).cuda()
        r = torch.full_like(d_psi, float("nan"))
        fd.fd_residual(plan, d_psi, d_h, d_e, d_n, r)
        torch.cuda.synchronize()
        want = oracle.residual(psi, got, eps / norm)
        tol = 1e-13 * (np.abs(got).max() + np.abs(eps / norm).max() * np.abs(psi).max())
        assert np.max(np.abs(r.cpu().numpy() - want)) <= tol
        fd.fd_residual(plan, d_psi, d_h, d_e, d_n, d_h)                        # in place
        torch.cuda.synchronize()
        assert np.max(np.abs(d_h.cpu().numpy() - want)) <= tol
        with pytest.raises(fd.FDError) as ei:
            fd.fd_residual(plan, d_psi, d_h, d_e, d_n, d_psi)
        assert ei.value.status == -3
    finally:
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ f3: Jacobi sweep

def jacobi_tol(h, nn, phi, rhs, omega, scale):
    S = kinetic_row_sum(h, nn, scale)
    c0 = {1: 2.0, 2: 2.5, 3: 49.0 / 18.0, 4: 205.0 / 72.0, 5: 5269.0 / 1800.0, 6: 5369.0 / 1800.0}[nn]
    diag = abs(scale) * c0 * sum(1.0 / (x * x) for x in h)
    return 1e-12 * (np.abs(phi).max() * (1.0 + abs(omega) * S / diag) + abs(omega) * np.abs(rhs).max() / diag)


@pytest.mark.parametrize("bc", list(itertools.product((0, 1), repeat=3)))
def test_jacobi_sweep_both_kernels(oracle, fd, bc):
    for nn, omega, scale, shape in [(3, 2.0 / 3.0, 1.0, (10, 30, 16)), (1, 1.0, 1.0, (9, 12, 8)),
                                    (2, 0.8, -0.5, (12, 10, 14)), (4, 0.7, 1.0, (12, 10, 14))]:
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=4, nn=nn)
        phi = W.make_psi(cfg)
        rhs = W.make_psi(W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=4, nn=nn, index=55)) * 30.0
        want = oracle.jacobi(cfg.shape, cfg.h, nn, bc, phi, rhs, omega, scale)
        tol = jacobi_tol(cfg.h, nn, phi, rhs, omega, scale)
        for kern in (fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create_scaled(cfg.shape, cfg.h, nn, bc, None, fd.FD_F64, 0, scale)
            try:
                try:
                    fd.fd_plan_set_kernel(plan, kern, 8 if kern == fd.FD_KERNEL_SWEEP else 0)
                except fd.FDError:
                    assert nn > 3 and kern == fd.FD_KERNEL_SWEEP
                    continue
                d_phi, d_rhs = torch.from_numpy(phi).cuda(), torch.from_numpy(rhs).cuda()
                d_out = torch.full_like(d_phi, float("nan"))
                fd.fd_jacobi_sweep(plan, d_phi, d_rhs, d_out, omega)
                torch.cuda.synchronize()
                err = float(np.max(np.abs(d_out.cpu().numpy() - want)))
                assert err <= tol, (nn, kern, err, tol)
            finally:
                fd.fd_destroy(plan)


def test_jacobi_converges_to_the_poisson_solution(fd):
    """200 damped sweeps on a periodic 16^3 grid reduce the residual of lap phi = rhs for a smooth
    zero-mean rhs: the kernel is usable as the smoother it is meant to be (no oracle involved)."""
    n, h = (16, 16, 16), (0.3, 0.3, 0.3)
    cfg = W.custom(n, h, (1, 1, 1), nbands=1)
    rhs_np = planewave(n, (0, 0, 0), (1, 0, 0), complex_=False)[None].copy()
    plan = fd.fd_create_scaled(n, cfg.h, 3, (1, 1, 1), None, fd.FD_F64, 0, 1.0)
    try:
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP)
        a = torch.zeros((1,) + n, dtype=torch.float64, device="cuda")
        b = torch.empty_like(a)
        rhs = torch.from_numpy(rhs_np).cuda()
        for _ in range(400):
            fd.fd_jacobi_sweep(plan, a, rhs, b, 0.9)
            a, b = b, a
        lap = torch.empty_like(a)
        fd.fd_apply_kinetic(plan, a, lap)
        torch.cuda.synchronize()
        assert float((lap - rhs).abs().max()) < 1e-2 * float(rhs.abs().max())
    finally:
        fd.fd_destroy(plan)


def test_jacobi_full_size_grid_sampled(oracle, fd):
    """cfg3's grid, 16 right-hand sides, the launch configuration the bench times; one band in full"""
    cfg = W.get(3).with_bands(16)
    phi = W.make_psi(cfg)
    rhs = W.make_psi(W.custom(cfg.shape, cfg.h_angstrom, cfg.bc, nbands=16, index=56))
    plan = fd.fd_create_scaled(cfg.shape, cfg.h, 3, cfg.bc, None, fd.FD_F64, 0, 1.0)
    try:
        assert fd.fd_plan_kernel_for(plan, 16) == fd.FD_KERNEL_SWEEP
        d_out = torch.full((16,) + cfg.shape, float("nan"), dtype=torch.float64, device="cuda")
        fd.fd_jacobi_sweep(plan, torch.from_numpy(phi).cuda(), torch.from_numpy(rhs).cuda(), d_out,
                           2.0 / 3.0)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy()
        assert np.isfinite(got).all()
        for b in (0, 15):
            want = oracle.jacobi(cfg.shape, cfg.h, 3, cfg.bc, phi[b:b + 1], rhs[b:b + 1], 2.0 / 3.0, 1.0)
            assert np.max(np.abs(got[b:b + 1] - want)) <= jacobi_tol(cfg.h, 3, phi, rhs, 2.0 / 3.0, 1.0)
    finally:
        fd.fd_destroy(plan)


def test_jacobi_rejects_complex_plans(fd):
    plan = fd.fd_create((8, 8, 8), (0.4,) * 3, dtype=fd.FD_C128)
    try:
        x = torch.zeros((1, 8, 8, 8), dtype=torch.complex128, device="cuda")
        with pytest.raises(fd.FDError) as ei:
            fd.fd_jacobi_sweep(plan, x, x.clone(), x.clone(), 1.0)
        assert ei.value.status == -2
        with pytest.raises(ValueError):            # the binding checks dtypes against the plan
            fd.fd_jacobi_sweep(plan, x.real.contiguous(), x.real.contiguous(), x.real.contiguous(), 1.0)
    finally:
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ f3: grid transfer

def transfer_tol(p, x):
    """row sum of |weights| of the 3-D operator times 1e-12 max|x| (interpolation: (2 sum|b_j|)^3,
    restriction: (1/2 + sum|b_j|)^3; both <= 2.2 for p <= 3)"""
    return 1e-12 * 2.2 * float(np.abs(x).max())


@pytest.mark.parametrize("bc", list(itertools.product((0, 1), repeat=3)))
@pytest.mark.parametrize("p", [1, 2, 3])
def test_restrict_and_interpolate_all_bc_mixes(oracle, fd, bc, p):
    """several y tiles (ragged), several x chunks, several bands"""
    rng = np.random.default_rng(100 + p)
    nf = tuple(n if b else n + 1 for n, b in zip((44, 36, 24), bc))
    nc = fd.coarse_shape(nf, bc)
    assert nc == oracle.coarse_shape(nf, bc)
    f = rng.standard_normal((3,) + nf)
    c = rng.standard_normal((3,) + nc)
    d_c = torch.full((3,) + nc, float("nan"), dtype=torch.float64, device="cuda")
    fd.fd_restrict(nf, bc, p, torch.from_numpy(f).cuda(), d_c)
    d_f = torch.full((3,) + nf, float("nan"), dtype=torch.float64, device="cuda")
    fd.fd_interpolate(nf, bc, p, torch.from_numpy(c).cuda(), d_f)
    torch.cuda.synchronize()
    got_r, got_i = d_c.cpu().numpy(), d_f.cpu().numpy()
    assert np.isfinite(got_r).all() and np.isfinite(got_i).all()
    assert np.max(np.abs(got_r - oracle.restrict(nf, bc, p, f))) <= transfer_tol(p, f)
    assert np.max(np.abs(got_i - oracle.interpolate(nf, bc, p, c))) <= transfer_tol(p, c)
    # adjointness on the device results: 8 <R f, c> = <f, I c>
    assert abs(8.0 * np.sum(got_r * c) - np.sum(f * got_i)) <= 1e-10 * np.sqrt(f.size)


@pytest.mark.parametrize("nf,bc", [((8, 8, 8), (1, 1, 1)), ((5, 7, 9), (0, 0, 0)), ((6, 9, 130), (1, 0, 1)),
                                   ((20, 70, 12), (1, 1, 1)), ((3, 3, 3), (0, 0, 0)), ((2, 2, 2), (1, 1, 1))])
def test_transfer_awkward_shapes(oracle, fd, nf, bc):
    rng = np.random.default_rng(7)
    nc = fd.coarse_shape(nf, bc)
    for p in (1, 3):
        f = rng.standard_normal((2,) + tuple(nf))
        c = rng.standard_normal((2,) + nc)
        d_c = torch.full((2,) + nc, float("nan"), dtype=torch.float64, device="cuda")
        d_f = torch.full((2,) + tuple(nf), float("nan"), dtype=torch.float64, device="cuda")
        fd.fd_restrict(nf, bc, p, torch.from_numpy(f).cuda(), d_c)
        fd.fd_interpolate(nf, bc, p, torch.from_numpy(c).cuda(), d_f)
        torch.cuda.synchronize()
        assert np.max(np.abs(d_c.cpu().numpy() - oracle.restrict(nf, bc, p, f))) <= transfer_tol(p, f)
        assert np.max(np.abs(d_f.cpu().numpy() - oracle.interpolate(nf, bc, p, c))) <= transfer_tol(p, c)


def test_transfer_full_size_192_to_96(oracle, fd):
    """the fine density grid of cfg3 (2 x 96 per axis) <-> cfg3's grid, the sizes the bench times;
    guard bands around the outputs; one band in full against the oracle"""
    nf, bc, p, nb = (192, 192, 192), (1, 1, 1), 3, 4
    nc = fd.coarse_shape(nf, bc)
    rng = np.random.default_rng(9)
    f = rng.standard_normal((nb,) + nf)
    c = rng.standard_normal((nb,) + nc)
    pad = 4096
    big_c = torch.full((c.size + 2 * pad,), 777.0, dtype=torch.float64, device="cuda")
    big_f = torch.full((f.size + 2 * pad,), 777.0, dtype=torch.float64, device="cuda")
    d_c = big_c[pad:pad + c.size].view(c.shape)
    d_f = big_f[pad:pad + f.size].view(f.shape)
    fd.fd_restrict(nf, bc, p, torch.from_numpy(f).cuda(), d_c)
    fd.fd_interpolate(nf, bc, p, torch.from_numpy(c).cuda(), d_f)
    torch.cuda.synchronize()
    for big, n in ((big_c, c.size), (big_f, f.size)):
        assert bool((torch.cat([big[:pad], big[pad + n:]]) == 777.0).all())
    for b in (0, nb - 1):
        assert np.max(np.abs(d_c[b:b + 1].cpu().numpy() - oracle.restrict(nf, bc, p, f[b:b + 1]))) \
            <= transfer_tol(p, f)
        assert np.max(np.abs(d_f[b:b + 1].cpu().numpy() - oracle.interpolate(nf, bc, p, c[b:b + 1]))) \
            <= transfer_tol(p, c)


def test_transfer_argument_errors(fd):
    x = torch.zeros((1, 8, 8, 8), dtype=torch.float64, device="cuda")
    y = torch.zeros((1, 4, 4, 4), dtype=torch.float64, device="cuda")
    for nf, bc, p, status in [((8, 8, 7), (1, 1, 1), 1, -1),      # odd periodic axis
                              ((8, 8, 8), (1, 1, 0), 1, -1),      # even zero-BC axis
                              ((8, 8, 8), (1, 1, 1), 0, -1), ((8, 8, 8), (1, 1, 1), 4, -2)]:
        with pytest.raises(fd.FDError) as ei:
            fd.fd_restrict(nf, bc, p, x, y)
        assert ei.value.status == status
    with pytest.raises(fd.FDError) as ei:
        fd.fd_interpolate((8, 8, 8), (1, 1, 1), 1, x.view(-1)[:64].view(1, 4, 4, 4), x)
    assert ei.value.status == -3


# ------------------------------------------------------------------------------ f4: PAW non-local term

def paw_bound(oracle, cfg, paw, psi, dmat, want_coef=False):
    """Per output point, the sum of the ABSOLUTE values of every term of the non-local sum:
    the oracle itself on |p~|, |dO|, |psi| with all Bloch factors 1 (k = None, real data).  A sum of n
    terms evaluated in float64 in any order is within n u of that (u = 1.1e-16; n < 4000 here: box
    points + functions), so 1e-12 x this bounds the difference between two correct float64
    evaluations, and it is computed from the data, not from products of maxima.  With want_coef also
    the same bound for the projections, dv sum_r |p~_i(r)| |psi(r)|."""
    return oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, None, np.abs(psi), paw.box_start, paw.box_size,
                            paw.nproj, np.abs(paw.proj), np.abs(dmat), want_coef=want_coef)


def paw_tol(oracle, cfg, paw, psi, dmat):
    """scalar form: 1e-12 x the largest per-point sum of |terms|"""
    return 1e-12 * float(paw_bound(oracle, cfg, paw, psi, dmat).max())


def assert_tolerance_resolves_single_precision(oracle, cfg, k, paw, psi, dmat, want, bound):
    """The gate must be able to tell float64 from float32: psi rounded to single precision (the
    smallest trace fp32 arithmetic could leave) moves the oracle's result by far more than the
    tolerance the kernel is held to."""
    psi32 = psi.astype(np.complex64 if np.iscomplexobj(psi) else np.float32).astype(psi.dtype)
    moved = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, k, psi32, paw.box_start, paw.box_size,
                             paw.nproj, paw.proj, dmat)
    inside = bound > 0
    assert np.max(np.abs(moved - want)[inside] / bound[inside]) > 100 * 1e-12


@pytest.mark.parametrize("bc,cplx", [((1, 1, 1), False), ((1, 1, 1), True), ((1, 0, 1), True),
                                     ((0, 0, 0), False), ((1, 1, 0), False), ((0, 1, 1), True)])
def test_paw_nonlocal_term_overlap_and_full_hamiltonian(oracle, fd, bc, cplx):
    k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc)) if cplx else (0, 0, 0)
    cfg = W.custom((20, 18, 24), (0.2, 0.22, 0.18), bc, k=k, complex_=cplx, nbands=7)
    paw = W.make_paw(cfg, 12, nproj=5)        # 12 atoms in a small cell: boxes overlap, several colours
    ds = W.make_paw(W.custom(cfg.shape, cfg.h_angstrom, bc, k=k, complex_=cplx, nbands=7, index=3),
                    12, nproj=5).dmat * 0.1
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    kk = k if cplx else None
    tdt = torch.complex128 if cplx else torch.float64
    plan = fd.fd_create(cfg.shape, cfg.h, 3, bc, kk, fd.FD_C128 if cplx else fd.FD_F64, 0)
    pw = fd.fd_paw_create(plan, paw.box_start, paw.box_size, paw.nproj, paw.proj, paw.dmat, ds)
    try:
        assert fd.fd_paw_nproj_total(pw) == paw.ntot
        d_psi = torch.from_numpy(psi).cuda()
        coef = torch.full((7, paw.ntot), float("nan"), dtype=tdt, device="cuda")
        want_nl, want_c = oracle.paw_apply(cfg.shape, cfg.h, bc, kk, psi, paw.box_start, paw.box_size,
                                           paw.nproj, paw.proj, paw.dmat, want_coef=True)
        bound, bound_c = paw_bound(oracle, cfg, paw, psi, paw.dmat, want_coef=True)
        tol = 1e-12 * float(bound.max())
        assert_tolerance_resolves_single_precision(oracle, cfg, kk, paw, psi, paw.dmat, want_nl, bound)
        # projections
        fd.fd_paw_project(plan, pw, d_psi, coef)
        torch.cuda.synchronize()
        assert np.all(np.abs(coef.cpu().numpy() - want_c) <= 1e-12 * bound_c)
        # non-local term added to an existing array
        base = W.make_psi(W.custom(cfg.shape, cfg.h_angstrom, bc, k=k, complex_=cplx, nbands=7, index=8))
        d_out = torch.from_numpy(base).cuda()
        fd.fd_paw_add_nonlocal(plan, pw, d_psi, d_out, coef)
        torch.cuda.synchronize()
        # point by point: 1e-12 x the sum of |terms| at that point (+ the rounding of base + term);
        # points outside every box keep base exactly
        assert np.all(np.abs(d_out.cpu().numpy() - (base + want_nl)) <= 1e-12 * bound + 1e-15 * np.abs(base))
        # full H~ psi~ (Eq. 6) and S~ psi~ (Eq. 7)
        want_h = oracle.apply(cfg.shape, cfg.h, 3, bc, kk, psi, v) + want_nl
        d_out = torch.full_like(d_psi, float("nan"))
        fd.fd_apply_hamiltonian_paw(plan, pw, d_psi, torch.from_numpy(v).cuda(), d_out, coef)
        torch.cuda.synchronize()
        assert np.max(np.abs(d_out.cpu().numpy() - want_h)) <= tol + parity_tol(cfg.h, 3, psi, v)
        want_s = oracle.paw_apply(cfg.shape, cfg.h, bc, kk, psi, paw.box_start, paw.box_size, paw.nproj,
                                  paw.proj, ds, out=psi)
        d_out = torch.full_like(d_psi, float("nan"))
        fd.fd_apply_overlap(plan, pw, d_psi, d_out, coef)
        torch.cuda.synchronize()
        assert np.all(np.abs(d_out.cpu().numpy() - want_s) <=
                      1e-12 * paw_bound(oracle, cfg, paw, psi, ds) + 1e-15 * np.abs(psi))
        # deterministic: same bits on a second call
        d_out2 = torch.full_like(d_psi, float("nan"))
        fd.fd_apply_overlap(plan, pw, d_psi, d_out2, coef)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(d_out) if cplx else d_out,
                           torch.view_as_real(d_out2) if cplx else d_out2)
    finally:
        fd.fd_paw_destroy(pw)
        fd.fd_destroy(plan)


def test_paw_full_size_grid_every_band(oracle, fd):
    """cfg3's grid, 128 atoms x up to 13 functions, 256 bands -- the configuration bench.py's
    next_rows times (same seeded projector set): EVERY element of the non-local term of every band
    against the oracle, point by point within 1e-12 x the sum of |terms| at that point."""
    cfg = W.get(3)
    paw = W.make_paw(cfg, 128, nproj=13, radius_angstrom=1.1)
    psi = W.make_psi(cfg)
    nb = cfg.nbands
    plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc)
    pw = fd.fd_paw_create(plan, paw.box_start, paw.box_size, paw.nproj, paw.proj, paw.dmat, None)
    try:
        d_psi = torch.from_numpy(psi).cuda()
        d_out = torch.zeros_like(d_psi)
        coef = torch.empty((nb, paw.ntot), dtype=torch.float64, device="cuda")
        fd.fd_paw_add_nonlocal(plan, pw, d_psi, d_out, coef)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy()
        worst = 0.0
        for b0 in range(0, nb, 32):
            sl = slice(b0, b0 + 32)
            want, want_c = oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, None, psi[sl], paw.box_start,
                                            paw.box_size, paw.nproj, paw.proj, paw.dmat, want_coef=True)
            bound, bound_c = paw_bound(oracle, cfg, paw, psi[sl], paw.dmat, want_coef=True)
            err = np.abs(got[sl] - want)
            assert np.all(err <= 1e-12 * bound), b0
            assert np.all(np.abs(coef[sl].cpu().numpy() - want_c) <= 1e-12 * bound_c), b0
            inside = bound > 0
            worst = max(worst, float(np.max(err[inside] / bound[inside])))
            if b0 == 0:
                assert_tolerance_resolves_single_precision(oracle, cfg, None, paw, psi[sl], paw.dmat,
                                                           want, bound)
        assert worst <= 1e-12
        with pytest.raises(fd.FDError) as ei:                      # Delta S was not given
            fd.fd_apply_overlap(plan, pw, d_psi, d_out, coef)
        assert ei.value.status == -1
    finally:
        fd.fd_paw_destroy(pw)
        fd.fd_destroy(plan)


@pytest.mark.parametrize("k", [(0.5, 0.0, 0.0), (0.0, 0.5, 0.5), (0.5, 0.5, 0.5), (-0.5, 1.0, 1.5)])
def test_paw_real_dtype_at_zone_boundary_k(oracle, fd, k):
    """FD_F64 plans with Bloch factors -1 (2 k_d integer): a box point that wraps a k_d = 1/2 axis
    takes the factor -1, and so does a box whose start lies an odd number of cells away from the home
    cell.  Boxes are placed so that they cross the upper and the lower end of every axis, and some
    start one or two cells below / above the home cell.  The oracle runs the complex definition on
    the real input (its imaginary part must vanish)."""
    for bc in [(1, 1, 1), (1, 0, 1)]:
        kk = tuple(x if b else 0.0 for x, b in zip(k, bc))
        cfg = W.custom((12, 14, 16), (0.2, 0.22, 0.18), bc, nbands=5)
        paw = W.make_paw(cfg, 10, nproj=4)
        start = paw.box_start.copy()
        n = np.array(cfg.shape)
        start[0] = -2                       # crosses the lower end of every axis
        start[1] = n - 3                    # crosses the upper end
        start[2] = start[2] - n             # one cell below the home cell (odd shift)
        start[3] = start[3] + 2 * n         # two cells above (even shift)
        start[4] = start[4] - 3 * n * np.array([1, 0, 1])   # odd shift along x and z only
        for d in range(3):
            if not bc[d]:
                start[:, d] = paw.box_start[:, d]           # zero-BC axis: no lattice shifts
        ds = W.make_paw(W.custom(cfg.shape, cfg.h_angstrom, bc, nbands=5, index=3), 10, nproj=4).dmat * 0.1
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        args = (paw.box_size, paw.nproj, paw.proj)
        want_c, coef_c = oracle.paw_apply(cfg.shape, cfg.h, bc, kk, psi.astype(np.complex128), start,
                                          *args, paw.dmat, want_coef=True)
        assert np.max(np.abs(want_c.imag)) <= 1e-13 * np.abs(want_c).max()
        # the factor matters: the Gamma-point result differs by O(1) where boxes wrap
        gamma = oracle.paw_apply(cfg.shape, cfg.h, bc, None, psi, start, *args, paw.dmat)
        if any(kk):
            assert np.max(np.abs(gamma - want_c.real)) > 1e-3 * np.abs(gamma).max()
        shifted = type(paw)(start, paw.box_size, paw.nproj, paw.proj, paw.dmat)
        bound, bound_c = paw_bound(oracle, cfg, shifted, psi, paw.dmat, want_coef=True)
        plan = fd.fd_create(cfg.shape, cfg.h, 3, bc, kk, fd.FD_F64, 0)
        pw = fd.fd_paw_create(plan, start, paw.box_size, paw.nproj, paw.proj, paw.dmat, ds)
        try:
            d_psi = torch.from_numpy(psi).cuda()
            coef = torch.full((5, paw.ntot), float("nan"), dtype=torch.float64, device="cuda")
            fd.fd_paw_project(plan, pw, d_psi, coef)
            torch.cuda.synchronize()
            assert np.all(np.abs(coef.cpu().numpy() - coef_c.real) <= 1e-12 * bound_c)
            d_out = torch.full_like(d_psi, float("nan"))
            fd.fd_apply_hamiltonian_paw(plan, pw, d_psi, torch.from_numpy(v).cuda(), d_out, coef)
            torch.cuda.synchronize()
            want_h = oracle.apply(cfg.shape, cfg.h, 3, bc, kk, psi.astype(np.complex128), v).real + want_c.real
            assert np.all(np.abs(d_out.cpu().numpy() - want_h) <= 1e-12 * bound + parity_tol(cfg.h, 3, psi, v))
            want_s = oracle.paw_apply(cfg.shape, cfg.h, bc, kk, psi.astype(np.complex128), start, *args, ds,
                                      out=psi.astype(np.complex128)).real
            fd.fd_apply_overlap(plan, pw, d_psi, d_out, coef)
            torch.cuda.synchronize()
            assert np.all(np.abs(d_out.cpu().numpy() - want_s) <=
                          1e-12 * paw_bound(oracle, cfg, shifted, psi, ds) + 1e-15 * np.abs(psi))
            # the PAW part of <psi|H~|psi> from the projections
            e = torch.zeros(5, dtype=torch.float64, device="cuda")
            fd.fd_paw_project(plan, pw, d_psi, coef)
            fd.fd_paw_expect(plan, pw, 0, coef, e)
            torch.cuda.synchronize()
            w_e = np.sum(psi * want_c.real, axis=(1, 2, 3))
            assert np.max(np.abs(e.cpu().numpy() - w_e)) <= 1e-12 * float(np.sum(np.abs(psi) * bound, axis=(1, 2, 3)).max())
        finally:
            fd.fd_paw_destroy(pw)
            fd.fd_destroy(plan)


def test_paw_create_errors(fd):
    plan = fd.fd_create((8, 8, 8), (0.4,) * 3)
    try:
        with pytest.raises(fd.FDError) as ei:                      # box longer than a periodic axis
            fd.fd_paw_create(plan, [[0, 0, 0]], [[9, 2, 2]], [1], np.zeros(36), np.zeros(1))
        assert ei.value.status == -2
        with pytest.raises(fd.FDError) as ei:                      # no matrix at all
            fd.fd_paw_create(plan, [[0, 0, 0]], [[2, 2, 2]], [1], np.zeros(8), None, None)
        assert ei.value.status == -1
        other = fd.fd_create((8, 8, 10), (0.4,) * 3)
        pw = fd.fd_paw_create(plan, [[0, 0, 0]], [[2, 2, 2]], [1], np.ones(8), np.ones(1))
        try:
            x = torch.zeros((1, 8, 8, 10), dtype=torch.float64, device="cuda")
            c = torch.zeros((1, 1), dtype=torch.float64, device="cuda")
            with pytest.raises(fd.FDError) as ei:                  # paw of another grid
                fd.fd_paw_project(other, pw, x, c)
            assert ei.value.status == -1
            # same number of points is not enough: permuted shape, other spacing, other boundaries,
            # other k (float64 at the zone boundary) all carry different tables / factors / dv
            y = torch.zeros((1, 8, 8, 8), dtype=torch.float64, device="cuda")
            for kw in [dict(shape=(8, 8, 8), h=(0.4, 0.4, 0.41)), dict(shape=(8, 8, 8), h=(0.4,) * 3, bc=(1, 0, 1)),
                       dict(shape=(8, 8, 8), h=(0.4,) * 3, k=(0.5, 0.0, 0.0))]:
                p2 = fd.fd_create(**kw)
                try:
                    with pytest.raises(fd.FDError) as ei:
                        fd.fd_paw_project(p2, pw, y, c)
                    assert ei.value.status == -1, kw
                finally:
                    fd.fd_destroy(p2)
            perm_a, perm_b = fd.fd_create((8, 12, 16), (0.4,) * 3), fd.fd_create((16, 12, 8), (0.4,) * 3)
            pw2 = fd.fd_paw_create(perm_a, [[0, 0, 0]], [[2, 2, 2]], [1], np.ones(8), np.ones(1))
            try:
                z = torch.zeros((1, 16, 12, 8), dtype=torch.float64, device="cuda")
                with pytest.raises(fd.FDError) as ei:
                    fd.fd_paw_project(perm_b, pw2, z, c)
                assert ei.value.status == -1
            finally:
                fd.fd_paw_destroy(pw2)
                fd.fd_destroy(perm_a)
                fd.fd_destroy(perm_b)
            # coef may not overlap psi or out (FD_ERR_ALIAS): views into one buffer
            buf = torch.zeros(2 * 512 + 2, dtype=torch.float64, device="cuda")
            psi_v, out_v = buf[:512].view(1, 8, 8, 8), buf[512:1024].view(1, 8, 8, 8)
            for bad_coef in (buf[0:1].view(1, 1), buf[512:513].view(1, 1)):
                with pytest.raises(fd.FDError) as ei:
                    fd.fd_paw_add_nonlocal(plan, pw, psi_v, out_v, bad_coef)
                assert ei.value.status == -3
            fd.fd_paw_add_nonlocal(plan, pw, psi_v, out_v, buf[1024:1025].view(1, 1))
            torch.cuda.synchronize()
        finally:
            fd.fd_paw_destroy(pw)
            fd.fd_destroy(other)
    finally:
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ multigrid V-cycle

@pytest.mark.parametrize("shape,bc,nn,p", [((16, 16, 16), (1, 1, 1), 3, 2), ((15, 15, 15), (0, 0, 0), 2, 2),
                                           ((32, 15, 16), (1, 0, 1), 3, 3), ((24, 20, 16), (1, 1, 1), 1, 1),
                                           ((9, 8, 8), (1, 1, 1), 3, 2)])
def test_vcycle_matches_the_oracle_cycle(oracle, fd, shape, bc, nn, p):
    """One and two V-cycles on the device against the oracle's step-by-step cycle (same hierarchy)"""
    rng = np.random.default_rng(12)
    cfg = W.custom(shape, (0.3, 0.25, 0.35), bc, nbands=3, nn=nn)
    rhs = rng.standard_normal((3,) + tuple(shape))
    if all(bc):
        rhs -= rhs.mean(axis=(1, 2, 3), keepdims=True)
    phi0 = rng.standard_normal((3,) + tuple(shape)) * 0.1
    levels = oracle.mg_levels(shape, bc, nn)
    mg = fd.fd_mg_create(shape, cfg.h, nn, bc, p, 16, 3, 0)
    try:
        assert fd.fd_mg_levels(mg) == len(levels)
        d_phi, d_rhs = torch.from_numpy(phi0).cuda(), torch.from_numpy(rhs).cuda()
        want = phi0
        for cyc in range(2):
            fd.fd_mg_vcycle(mg, d_phi, d_rhs, 2, 1, 6, 2.0 / 3.0)
            torch.cuda.synchronize()
            want = oracle.vcycle(shape, cfg.h, nn, bc, p, want, rhs, nu1=2, nu2=1, nu_coarse=6,
                                 omega=2.0 / 3.0)
            scale = max(np.abs(want).max(), np.abs(phi0).max())
            assert np.max(np.abs(d_phi.cpu().numpy() - want)) <= 1e-11 * scale * (cyc + 1) * len(levels)
    finally:
        fd.fd_mg_destroy(mg)


def test_vcycle_solves_the_poisson_problem_on_the_device(fd):
    """96^3 periodic grid, 4 right-hand sides built from plane waves: 8 cycles reduce the residual by
    > 1e4, a factor < 0.5 per cycle (no oracle involved: the residual is computed by fd_poisson_residual)"""
    n, nn = (96, 96, 96), 3
    cfg = W.custom(n, (0.2, 0.2, 0.2), (1, 1, 1), nbands=4)
    rhs_np = np.stack([planewave(n, (0, 0, 0), m, complex_=False) for m in [(1, 0, 0), (2, 3, 1), (0, 7, 5), (11, 4, 9)]])
    mg = fd.fd_mg_create(n, cfg.h, nn, (1, 1, 1), 3, 16, 4, 0)
    plan = fd.fd_create_scaled(n, cfg.h, nn, (1, 1, 1), None, fd.FD_F64, 0, 1.0)
    try:
        assert fd.fd_mg_levels(mg) == 6
        rhs = torch.from_numpy(rhs_np).cuda()
        phi = torch.zeros_like(rhs)
        res = torch.empty_like(rhs)
        norms = []
        for _ in range(8):
            fd.fd_mg_vcycle(mg, phi, rhs)
            fd.fd_poisson_residual(plan, phi, rhs, res)
            torch.cuda.synchronize()
            norms.append(float(res.abs().max()))
        assert norms[-1] < 1e-4 * float(rhs.abs().max()), norms
        assert all(b < 0.5 * a for a, b in zip(norms[:5], norms[1:6])), norms
    finally:
        fd.fd_destroy(plan)
        fd.fd_mg_destroy(mg)


def test_poisson_residual_parity_and_mg_errors(oracle, fd):
    for bc, nn, shape in [((1, 1, 1), 3, (10, 30, 16)), ((0, 1, 0), 2, (9, 12, 8)), ((1, 0, 1), 4, (12, 10, 14))]:
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=3, nn=nn)
        phi, rhs = W.make_psi(cfg), W.make_psi(W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=3, nn=nn, index=5))
        plan = fd.fd_create_scaled(cfg.shape, cfg.h, nn, bc, None, fd.FD_F64, 0, 1.0)
        try:
            out = torch.full((3,) + shape, float("nan"), dtype=torch.float64, device="cuda")
            fd.fd_poisson_residual(plan, torch.from_numpy(phi).cuda(), torch.from_numpy(rhs).cuda(), out)
            torch.cuda.synchronize()
            want = rhs - oracle.apply(cfg.shape, cfg.h, nn, bc, None, phi, None, scale=1.0)
            assert np.max(np.abs(out.cpu().numpy() - want)) <= parity_tol(cfg.h, nn, phi, None, 1.0) + 1e-15 * np.abs(rhs).max()
        finally:
            fd.fd_destroy(plan)
    mg = fd.fd_mg_create((16, 16, 16), (0.5,) * 3, 3, (1, 1, 1), 2, 16, 2, 0)
    try:
        x = torch.zeros((3, 16, 16, 16), dtype=torch.float64, device="cuda")
        with pytest.raises(fd.FDError) as ei:          # more right-hand sides than the hierarchy holds
            fd.fd_mg_vcycle(mg, x, x.clone())
        assert ei.value.status == -1
        y = torch.zeros((2, 16, 16, 16), dtype=torch.float64, device="cuda")
        with pytest.raises(fd.FDError) as ei:
            fd.fd_mg_vcycle(mg, y, y)
        assert ei.value.status == -3
    finally:
        fd.fd_mg_destroy(mg)
    with pytest.raises(fd.FDError) as ei:
        fd.fd_mg_create((16, 16, 16), (0.5,) * 3, 3, (1, 1, 1), 5, 16, 2, 0)
    assert ei.value.status == -2


def test_mg_create_rejects_hierarchies_whose_transfers_do_not_fit(fd):
    """z rows too long for the transfer kernels (fine nz > ~682): fd_mg_create says
    FD_ERR_UNSUPPORTED itself instead of the first fd_mg_vcycle; a single level (no transfer) and a
    long x or y axis are fine."""
    h = (0.3,) * 3
    with pytest.raises(fd.FDError) as ei:
        fd.fd_mg_create((8, 8, 4096), h, 3, (1, 1, 1), 2, 16, 1, 0)
    assert ei.value.status == -2
    for shape, levels in [((8, 8, 4096), 1), ((1024, 8, 8), 16), ((8, 1024, 8), 16)]:
        mg = fd.fd_mg_create(shape, h, 3, (1, 1, 1), 2, levels, 1, 0)
        try:
            phi = torch.zeros((1,) + shape, dtype=torch.float64, device="cuda")
            rhs = torch.randn((1,) + shape, dtype=torch.float64, device="cuda")
            fd.fd_mg_vcycle(mg, phi, rhs - rhs.mean())
            torch.cuda.synchronize()
            assert bool(torch.isfinite(phi).all())
        finally:
            fd.fd_mg_destroy(mg)


def test_vcycle_graph_replay_on_a_side_stream_matches_direct_launches(fd):
    """On a non-default stream the cycle is captured into a CUDA graph and replayed: same bits as the
    direct launches on the default stream, also after the argument set changes."""
    n, bc = (32, 32, 32), (1, 1, 1)
    cfg = W.custom(n, (0.3, 0.3, 0.3), bc, nbands=2)
    rng = np.random.default_rng(21)
    rhs_np = rng.standard_normal((2,) + n)
    rhs_np -= rhs_np.mean(axis=(1, 2, 3), keepdims=True)
    mg = fd.fd_mg_create(n, cfg.h, 3, bc, 2, 16, 2, 0)
    try:
        rhs = torch.from_numpy(rhs_np).cuda()
        ref = torch.zeros_like(rhs)
        for _ in range(3):
            fd.fd_mg_vcycle(mg, ref, rhs)                       # default stream: direct launches
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        phi = torch.zeros_like(rhs)
        for _ in range(3):
            fd.fd_mg_vcycle(mg, phi, rhs, stream=s)             # capture, then two replays
        s.synchronize()
        assert torch.equal(phi, ref)
        phi2 = torch.zeros_like(rhs)                            # new pointers: re-capture
        fd.fd_mg_vcycle(mg, phi2, rhs, 1, 1, 4, 0.8, stream=s)
        fd.fd_mg_vcycle(mg, phi2, rhs, 1, 1, 4, 0.8, stream=s)
        s.synchronize()
        ref2 = torch.zeros_like(rhs)
        fd.fd_mg_vcycle(mg, ref2, rhs, 1, 1, 4, 0.8)
        fd.fd_mg_vcycle(mg, ref2, rhs, 1, 1, 4, 0.8)
        torch.cuda.synchronize()
        assert torch.equal(phi2, ref2)
        # capture bookkeeping: one capture per argument set, none on replays, and a solver that
        # alternates buffers (here 4 argument sets round robin) re-captures none of them
        info = fd.fd_mg_get_info(mg)
        assert info["shape"] == n and info["max_nbands"] == 2 and info["levels"] == fd.fd_mg_levels(mg)
        assert not info["graph_off"] and info["graph_captures"] == 2
        bufs = [torch.zeros_like(rhs) for _ in range(4)]
        for rounds in range(3):
            for b in bufs:
                fd.fd_mg_vcycle(mg, b, rhs, stream=s)
        s.synchronize()
        assert fd.fd_mg_get_info(mg)["graph_captures"] == 2 + 4
        for b in bufs:
            assert torch.equal(b, ref)                           # 3 cycles each, as ref
        # a stream the caller is capturing: the launches join the caller's graph, nothing breaks
        phi3 = torch.zeros_like(rhs)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            fd.fd_mg_vcycle(mg, phi3, rhs, stream=s)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        assert torch.equal(phi3, ref)
        info = fd.fd_mg_get_info(mg)
        assert not info["graph_off"] and info["graph_captures"] == 6
        # the binding checks phi / rhs against the hierarchy before passing raw pointers on
        with pytest.raises(ValueError):
            fd.fd_mg_vcycle(mg, torch.zeros((2, 32, 32, 16), dtype=torch.float64, device="cuda"),
                            torch.zeros((2, 32, 32, 16), dtype=torch.float64, device="cuda"))
    finally:
        fd.fd_mg_destroy(mg)


@pytest.mark.parametrize("cplx", [False, True])
def test_paw_rayleigh_quotient_and_generalised_residual(oracle, fd, cplx):
    """eps / norm of the stencil pass completed by fd_paw_expect to <psi|H~|psi> / <psi|S~|psi>, and
    the generalised residual H~ psi - lambda S~ psi through fd_residual, against the oracle's sums"""
    bc = (1, 1, 0)
    k = (0.25, 0.125, 0.0) if cplx else (0, 0, 0)
    cfg = W.custom((20, 16, 24), (0.2, 0.22, 0.18), bc, k=k, complex_=cplx, nbands=6)
    paw = W.make_paw(cfg, 10, nproj=5)
    ds = W.make_paw(W.custom(cfg.shape, cfg.h_angstrom, bc, k=k, complex_=cplx, nbands=6, index=3), 10,
                    nproj=5).dmat * 0.1
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    kk = k if cplx else None
    tdt = torch.complex128 if cplx else torch.float64
    plan = fd.fd_create(cfg.shape, cfg.h, 3, bc, kk, fd.FD_C128 if cplx else fd.FD_F64, 0)
    pw = fd.fd_paw_create(plan, paw.box_start, paw.box_size, paw.nproj, paw.proj, paw.dmat, ds)
    try:
        d_psi, d_v = torch.from_numpy(psi).cuda(), torch.from_numpy(v).cuda()
        hpsi, spsi = torch.empty_like(d_psi), torch.empty_like(d_psi)
        eps = torch.empty(6, dtype=torch.float64, device="cuda")
        nrm = torch.empty_like(eps)
        ws = torch.empty(fd.fd_expect_workspace_bytes(plan, 6) // 8 + 2, dtype=torch.float64, device="cuda")
        coef = torch.empty((6, paw.ntot), dtype=tdt, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, d_psi, d_v, hpsi, eps, nrm, ws)     # local part + sums
        fd.fd_paw_project(plan, pw, d_psi, coef)
        fd.fd_paw_expect(plan, pw, 0, coef, eps)                                  # + <psi|N_H|psi>
        fd.fd_paw_expect(plan, pw, 1, coef, nrm)                                  # + <psi|N_S|psi>
        fd.fd_paw_add_nonlocal(plan, pw, d_psi, hpsi, coef)                       # H~ psi
        fd.fd_apply_overlap(plan, pw, d_psi, spsi, coef)                          # S~ psi
        r = torch.empty_like(d_psi)
        fd.fd_residual(plan, spsi, hpsi, eps, nrm, r)
        torch.cuda.synchronize()
        w_eps, w_n = oracle.expect(cfg.shape, cfg.h, 3, bc, kk, psi, v)
        args = (cfg.shape, cfg.h, bc, kk, psi, paw.box_start, paw.box_size, paw.nproj, paw.proj)
        w_eps = w_eps.real + oracle.paw_expect(*args, paw.dmat).real
        w_n = w_n + oracle.paw_expect(*args, ds).real
        te, tn = expect_tol(cfg.h, 3, psi, v)
        tp = paw_tol(oracle, cfg, paw, psi, paw.dmat) * psi[0].size * np.abs(psi).max()
        assert np.max(np.abs(eps.cpu().numpy() - w_eps)) <= te + tp
        assert np.max(np.abs(nrm.cpu().numpy() - w_n)) <= tn + tp
        w_h = oracle.apply(cfg.shape, cfg.h, 3, bc, kk, psi, v) + oracle.paw_apply(*args, paw.dmat)
        w_s = oracle.paw_apply(*args, ds, out=psi)
        lam = w_eps / w_n
        w_r = w_h - lam[:, None, None, None] * w_s
        tol = parity_tol(cfg.h, 3, psi, v) + paw_tol(oracle, cfg, paw, psi, paw.dmat) + \
            np.abs(lam).max() * (paw_tol(oracle, cfg, paw, psi, ds) + 1e-14 * np.abs(psi).max())
        assert np.max(np.abs(r.cpu().numpy() - w_r)) <= tol + 1e-12 * np.abs(w_s).max() * np.abs(lam).max()
        # residual orthogonal to psi: sum conj(psi) r = 0 by construction of lambda
        dots = (d_psi.conj() * r).sum(dim=(1, 2, 3))
        assert float(dots.abs().max()) <= 1e-9 * float(np.abs(w_eps).max())
    finally:
        fd.fd_paw_destroy(pw)
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ seeded random configurations

def test_random_configurations_of_the_next_rows(oracle, fd):
    """40 seeded random cases each of: fused expectation values (any BC mix, nn 1..6, real / complex
    Bloch, random tile height), Jacobi sweeps, restriction + interpolation (any BC mix, p 1..3)."""
    rng = np.random.default_rng(7741)
    for trial in range(40):
        nn = int(rng.integers(1, 7))
        bc = tuple(int(b) for b in rng.integers(0, 2, 3))
        shape = tuple(int(max(rng.integers(8, 33), nn)) for _ in range(3))
        shape = (shape[0], shape[1], shape[2] + (shape[2] & 1))
        cplx = bool(rng.integers(0, 2))
        k = tuple(float(rng.uniform(-0.5, 0.5)) if (b and cplx) else 0.0 for b in bc)
        nb = int(rng.integers(1, 8))
        h = tuple(float(x) for x in rng.uniform(0.15, 0.3, 3))
        cfg = W.custom(shape, h, bc, k=k, complex_=cplx, nbands=nb, nn=nn, index=300 + trial)
        kern = [fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC, "auto"][trial % 3]
        try:
            check_expect(oracle, fd, cfg, kern, tyc=int(rng.choice([0, 4, 8])) if kern == fd.FD_KERNEL_SWEEP else 0,
                         with_v=bool(rng.integers(0, 3)))
        except fd.FDError as e:
            assert e.status == -2 and kern == fd.FD_KERNEL_SWEEP
        if not cplx:
            omega, scale = float(rng.uniform(0.5, 1.0)), float(rng.choice([1.0, -0.5]))
            phi = W.make_psi(cfg)
            rhs = W.make_psi(W.custom(shape, h, bc, nbands=nb, nn=nn, index=400 + trial)) * 10.0
            plan = fd.fd_create_scaled(cfg.shape, cfg.h, nn, bc, None, fd.FD_F64, 0, scale)
            try:
                d_out = torch.full((nb,) + shape, float("nan"), dtype=torch.float64, device="cuda")
                fd.fd_jacobi_sweep(plan, torch.from_numpy(phi).cuda(), torch.from_numpy(rhs).cuda(), d_out, omega)
                torch.cuda.synchronize()
                want = oracle.jacobi(cfg.shape, cfg.h, nn, bc, phi, rhs, omega, scale)
                assert np.max(np.abs(d_out.cpu().numpy() - want)) <= jacobi_tol(cfg.h, nn, phi, rhs, omega, scale)
            finally:
                fd.fd_destroy(plan)
        # grid transfer on an independent random fine grid
        p = int(rng.integers(1, 4))
        nc = tuple(int(rng.integers(1, 21)) for _ in range(3))
        nf = tuple(2 * c if b else 2 * c + 1 for c, b in zip(nc, bc))
        f = rng.standard_normal((nb,) + nf)
        c = rng.standard_normal((nb,) + nc)
        d_c = torch.full((nb,) + nc, float("nan"), dtype=torch.float64, device="cuda")
        d_f = torch.full((nb,) + nf, float("nan"), dtype=torch.float64, device="cuda")
        fd.fd_restrict(nf, bc, p, torch.from_numpy(f).cuda(), d_c)
        fd.fd_interpolate(nf, bc, p, torch.from_numpy(c).cuda(), d_f)
        torch.cuda.synchronize()
        assert np.max(np.abs(d_c.cpu().numpy() - oracle.restrict(nf, bc, p, f))) <= transfer_tol(p, f), (trial, nf, bc, p)
        assert np.max(np.abs(d_f.cpu().numpy() - oracle.interpolate(nf, bc, p, c))) <= transfer_tol(p, c), (trial, nf, bc, p)


def test_peak_microbenchmark_kernels_do_what_they_say(fd):
    """bench.py's hardware_peaks leg times these: write fills, copy copies, read / DFMA leave memory alone"""
    n = 1 << 16
    a = torch.zeros(n, dtype=torch.float64, device="cuda")
    b = torch.zeros(n, dtype=torch.float64, device="cuda")
    fd.fd_peak_kernel(1, a, None, n)
    torch.cuda.synchronize()
    assert bool((a == 1.5).all())
    fd.fd_peak_kernel(2, a, b, n)
    fd.fd_peak_kernel(0, a, b[:2], n)
    torch.cuda.synchronize()
    assert bool((b == 1.5).all())
    sink = torch.zeros(2, dtype=torch.float64, device="cuda")
    fd.fd_peak_kernel(3, sink, None, 64, 4)
    torch.cuda.synchronize()
    assert bool((sink == 0.0).all())
    with pytest.raises(fd.FDError) as ei:
        fd.fd_peak_kernel(7, a, b, n)
    assert ei.value.status == -1
