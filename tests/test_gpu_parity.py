"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerance (north_star):  max|d| <= 1e-12 (max|psi| S + max|v_eff psi|),
S = 1/2 sum_d (|c_0| + 2 sum|c_j|)/h_d^2  (helpers.parity_tol).

Full-size configs 3-5 run on the GPU in the launch configuration bench.py times (all bands, one
apply); the oracle then checks a subset of bands in full plus sampled points from every band.
"""
import itertools

import numpy as np
import pytest

import workloads as W
from helpers import parity_tol, planewave, planewave_eig, kinetic_row_sum

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


def gpu_apply(fd, cfg, psi, v, kernel=None, kinetic=False, tyc=0):
    """psi, v: numpy arrays; returns numpy H psi computed by libfdham on cuda:0.

    kernel: a FD_KERNEL_* family to force, "auto" for the plan's own per-batch choice, or None =
    the sweep kernel wherever the plan supports it (the kernel under test; small batches would
    otherwise be handed to the generic kernel), else the generic one."""
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None,
                        fd.FD_C128 if cfg.complex else fd.FD_F64, 0)
    try:
        if kernel is None:
            try:
                fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP, tyc)
            except fd.FDError:
                fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_GENERIC, 0)
        elif kernel != "auto":
            fd.fd_plan_set_kernel(plan, kernel, tyc)
        d_psi = torch.from_numpy(psi).cuda()
        d_out = torch.full_like(d_psi, float("nan"))
        if kinetic or v is None:
            fd.fd_apply_kinetic(plan, d_psi, d_out)
        else:
            fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v).cuda(), d_out)
        torch.cuda.synchronize()
        used = fd.fd_plan_kernel_for(plan, psi.shape[0])
        return d_out.cpu().numpy(), used
    finally:
        fd.fd_destroy(plan)


def check(oracle, fd, cfg, psi, v, kernel=None, tyc=0):
    got, used = gpu_apply(fd, cfg, psi, v, kernel, tyc=tyc)
    want = oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None, psi, v)
    tol = parity_tol(cfg.h, cfg.nn, psi, v)
    err = float(np.max(np.abs(got - want)))
    assert np.isfinite(got).all()
    assert err <= tol, f"{cfg.name} kernel={used}: max|d|={err:.3e} > tol={tol:.3e}"
    return used


# ------------------------------------------------------------------------------ BASELINE configs

@pytest.mark.parametrize("idx", [1, 2])
@pytest.mark.parametrize("kernel", ["auto", "sweep", "generic"])
def test_small_configs_full_compare(oracle, fd, idx, kernel):
    cfg = W.get(idx)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    forced = {"auto": "auto", "sweep": fd.FD_KERNEL_SWEEP, "generic": fd.FD_KERNEL_GENERIC}[kernel]
    used = check(oracle, fd, cfg, psi, v, forced)
    if kernel == "auto":
        # 24^3 x 8 bands cannot fill the persistent teams: the plan hands it to the generic kernel
        assert used == (fd.FD_KERNEL_GENERIC if idx == 1 else fd.FD_KERNEL_SWEEP)
    else:
        assert used == forced


def _big_config_check(oracle, fd, cfg, chunk=32):
    """All bands on the GPU in one apply (the launch configuration bench.py times); the oracle on
    every band, element by element."""
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None,
                        fd.FD_C128 if cfg.complex else fd.FD_F64, 0)
    try:
        assert fd.fd_plan_get_kernel(plan) == fd.FD_KERNEL_SWEEP
        tdt = torch.complex128 if cfg.complex else torch.float64
        d_psi = torch.empty((cfg.nbands,) + cfg.shape, dtype=tdt, device="cuda")
        for b0 in range(0, cfg.nbands, chunk):
            bands = range(b0, min(cfg.nbands, b0 + chunk))
            d_psi[b0:b0 + len(bands)] = torch.from_numpy(W.make_psi(cfg, bands)).cuda()
        v = W.make_veff(cfg)
        d_v = torch.from_numpy(v).cuda()
        d_out = torch.full_like(d_psi, float("nan"))
        fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(torch.view_as_real(d_out) if cfg.complex else d_out).all())
        k = cfg.k if cfg.complex else None
        # EVERY element of EVERY band against the oracle (OpenMP over bands on the host cores), in
        # chunks of `chunk` bands
        worst = 0.0
        for b0 in range(0, cfg.nbands, chunk):
            bands = list(range(b0, min(cfg.nbands, b0 + chunk)))
            psi_c = W.make_psi(cfg, bands)
            want = oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi_c, v)
            got = d_out[b0:b0 + len(bands)].cpu().numpy()
            tol = parity_tol(cfg.h, cfg.nn, psi_c, v)
            err = float(np.max(np.abs(got - want)))
            assert err <= tol, f"{cfg.name} bands {b0}..: max|d|={err:.3e} > tol={tol:.3e}"
            worst = max(worst, err / tol)
        print(f"{cfg.name}: every element of {cfg.nbands} bands, max|d|/tol = {worst:.3e}")
    finally:
        fd.fd_destroy(plan)


def test_config3_96c_256_bands(oracle, fd):
    _big_config_check(oracle, fd, W.get(3))


def test_config4_bloch_c128_128_bands(oracle, fd):
    _big_config_check(oracle, fd, W.get(4))


def test_config5_slab_384_bands(oracle, fd):
    _big_config_check(oracle, fd, W.get(5))


# ------------------------------------------------------------------------------ shape sweep (M8)

SWEEP_SHAPES = [(8, 8, 8), (9, 8, 10), (8, 17, 12), (33, 10, 8), (12, 50, 14), (16, 16, 16),
                (10, 37, 24), (40, 8, 96)]


@pytest.mark.parametrize("shape", SWEEP_SHAPES)
def test_shape_sweep_all_bc_combinations_real(oracle, fd, shape):
    for bc in itertools.product((0, 1), repeat=3):
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=3)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP)
        assert used == fd.FD_KERNEL_SWEEP


@pytest.mark.parametrize("shape", [(8, 8, 8), (9, 12, 10), (8, 23, 12), (20, 10, 36)])
def test_shape_sweep_complex_bloch(oracle, fd, shape):
    for bc in [(1, 1, 1), (1, 0, 1), (0, 1, 1), (1, 1, 0), (0, 0, 0)]:
        k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=3)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP)
        assert used == fd.FD_KERNEL_SWEEP


@pytest.mark.parametrize("shape", [(3, 4, 5), (7, 7, 7), (6, 6, 6), (5, 9, 11), (3, 3, 3)])
def test_generic_fallback_shapes(oracle, fd, shape):
    """odd nz / tiny axes / n = nn / n = 2nn (double hit) run on the generic kernel."""
    for bc in [(1, 1, 1), (0, 1, 0), (0, 0, 0)]:
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=2)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), "auto")
        assert used == fd.FD_KERNEL_GENERIC
        ck = W.custom(shape, (0.2, 0.23, 0.17), bc, complex_=True, nbands=2,
                      k=tuple(0.3 * b for b in bc))
        check(oracle, fd, ck, W.make_psi(ck), W.make_veff(ck))


@pytest.mark.parametrize("nn", [1, 2, 4, 5, 6])
def test_other_stencil_orders(oracle, fd, nn):
    cfg = W.custom((12, 10, 14), (0.2, 0.23, 0.17), (1, 0, 1), nbands=2, nn=nn)
    used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_GENERIC)
    assert used == fd.FD_KERNEL_GENERIC


@pytest.mark.parametrize("nn", [1, 2])
def test_sweep_kernel_lower_orders(oracle, fd, nn):
    """the sweep kernel for nn = 1, 2 (3- and 5-slot accumulator rotation, nn
    halo rows / planes / z points): all BC mixes, several tiles with a ragged one, real and
    complex with Bloch phases on every axis, several bands per team and several teams."""
    for bc in itertools.product((0, 1), repeat=3):
        cfg = W.custom((9, 26, 12), (0.2, 0.23, 0.17), bc, nbands=7, nn=nn)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP, tyc=8)
        assert used == fd.FD_KERNEL_SWEEP
    for bc in [(1, 1, 1), (0, 1, 1), (1, 1, 0)]:
        k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
        cfg = W.custom((10, 20, 8), (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=5, nn=nn)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP, tyc=8)
        assert used == fd.FD_KERNEL_SWEEP
    cfg = W.custom((40, 48, 64), (0.2, 0.2, 0.18), (1, 1, 0), nbands=40, nn=nn)
    used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP)
    assert used == fd.FD_KERNEL_SWEEP


@pytest.mark.parametrize("tyc", [4, 8, 12, 20])
def test_tile_rows_override_ragged_tiles(oracle, fd, tyc):
    """Several y tiles, ragged last tile, tile seams at different rows."""
    for bc in [(1, 1, 1), (0, 0, 0), (1, 0, 1)]:
        cfg = W.custom((10, 30, 16), (0.2, 0.23, 0.17), bc, nbands=5)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP, tyc)
        assert used == fd.FD_KERNEL_SWEEP
    ck = W.custom((10, 30, 16), (0.2, 0.23, 0.17), (1, 1, 1), k=(0.25, 0.125, 0.4),
                  complex_=True, nbands=3)
    check(oracle, fd, ck, W.make_psi(ck), W.make_veff(ck), fd.FD_KERNEL_SWEEP, tyc)


# ------------------------------------------------------------------------------ metamorphic (M1-M7)

def test_band_independence_and_counts(oracle, fd):
    cfg = W.custom((16, 24, 32), (0.2, 0.2, 0.2), (1, 1, 1), nbands=13)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    full, _ = gpu_apply(fd, cfg, psi, v)
    for sel in ([0], [12], [3, 4], [5, 1, 7, 2, 11]):
        part, _ = gpu_apply(fd, cfg.with_bands(len(sel)), np.ascontiguousarray(psi[sel]), v)
        assert np.max(np.abs(part - full[sel])) <= parity_tol(cfg.h, 3, psi, v)
    for nb in (1, 2, 7, 149, 300):           # more / fewer bands than SMs, primes
        c2 = cfg.with_bands(nb)
        check(oracle, fd, c2, W.make_psi(c2), v)


def test_kinetic_equals_hamiltonian_with_zero_v_and_linearity(oracle, fd):
    cfg = W.custom((12, 16, 20), (0.2, 0.21, 0.19), (1, 0, 1), nbands=4)
    psi, v1 = W.make_psi(cfg), W.make_veff(cfg)
    v2 = np.random.default_rng(4).uniform(-2, 2, cfg.shape)
    t, _ = gpu_apply(fd, cfg, psi, None, kinetic=True)
    h0, _ = gpu_apply(fd, cfg, psi, np.zeros(cfg.shape))
    assert np.max(np.abs(t - h0)) <= 1e-13 * kinetic_row_sum(cfg.h) * np.abs(psi).max()
    ha, _ = gpu_apply(fd, cfg, psi, v1 + v2)
    hb, _ = gpu_apply(fd, cfg, psi, v1)
    assert np.max(np.abs((ha - hb) - v2[None] * psi)) <= parity_tol(cfg.h, 3, psi, v1 + v2)
    want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None, psi)
    assert np.max(np.abs(t - want)) <= parity_tol(cfg.h, 3, psi, None)


def test_complex_gamma_equals_two_real_applies(fd):
    shape, h, bc = (12, 16, 20), (0.2, 0.21, 0.19), (1, 0, 1)
    cr = W.custom(shape, h, bc, nbands=2)
    re, im = W.make_psi(cr), W.make_psi(W.custom(shape, h, bc, nbands=2, index=98))
    v = W.make_veff(cr)
    cc = W.custom(shape, h, bc, complex_=True, nbands=2)
    c, _ = gpu_apply(fd, cc, re + 1j * im, v)
    r, _ = gpu_apply(fd, cr, re, v)
    i, _ = gpu_apply(fd, cr, im, v)
    assert np.max(np.abs(c - (r + 1j * i))) <= parity_tol(h, 3, re + 1j * im, v)


def test_translation_invariance_across_tile_seams(fd):
    cfg = W.custom((16, 40, 24), (0.2, 0.2, 0.2), (1, 1, 1), nbands=2)
    psi = W.make_psi(cfg)
    base, _ = gpu_apply(fd, cfg, psi, None, fd.FD_KERNEL_SWEEP, kinetic=True, tyc=12)
    tol = parity_tol(cfg.h, 3, psi, None)
    for shift, ax in [(1, 1), (5, 1), (11, 2), (13, 2), (3, 3), (23, 3)]:
        got, _ = gpu_apply(fd, cfg, np.ascontiguousarray(np.roll(psi, shift, axis=ax)), None,
                           fd.FD_KERNEL_SWEEP, kinetic=True, tyc=12)
        assert np.max(np.abs(got - np.roll(base, shift, axis=ax))) <= tol


def test_axis_permutation(fd):
    shape, h, bc = (10, 12, 16), (0.2, 0.25, 0.3), (1, 0, 1)
    cfg = W.custom(shape, h, bc, nbands=2)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    base, _ = gpu_apply(fd, cfg, psi, v)
    for perm in [(1, 2, 0), (2, 0, 1), (0, 2, 1)]:
        cp = W.custom([shape[p] for p in perm], [h[p] for p in perm], [bc[p] for p in perm],
                      nbands=2)
        pp = np.ascontiguousarray(psi.transpose((0,) + tuple(1 + p for p in perm)))
        vp = np.ascontiguousarray(v.transpose(perm))
        got, _ = gpu_apply(fd, cp, pp, vp)
        want = base.transpose((0,) + tuple(1 + p for p in perm))
        assert np.max(np.abs(got - want)) <= parity_tol(h, 3, psi, v)


def test_plane_waves_on_device_closed_form(fd):
    """GPU against the closed form directly (not via the oracle): Gamma and Bloch."""
    n, h_ang = (24, 16, 32), (0.2, 0.21, 0.18)
    for k, m in [((0, 0, 0), (1, 2, 3)), ((0.25, 0.125, 0.0), (3, -2, 1)),
                 ((0.25, 0.125, -0.4), (0, 0, 0))]:
        cfg = W.custom(n, h_ang, (1, 1, 1), k=k, complex_=True, nbands=1)
        psi = planewave(n, k, m)[None]
        got, used = gpu_apply(fd, cfg, psi, None, fd.FD_KERNEL_SWEEP, kinetic=True)
        assert used == fd.FD_KERNEL_SWEEP
        lam = planewave_eig(n, cfg.h, k, m)
        assert np.max(np.abs(got - lam * psi)) <= 1e-12 * kinetic_row_sum(cfg.h)


# ------------------------------------------------------------------------------ ABI behaviour on device

def test_alias_and_alignment_errors(fd):
    plan = fd.fd_create((8, 8, 8), (0.4,) * 3)
    try:
        x = torch.zeros((2, 8, 8, 8), dtype=torch.float64, device="cuda")
        v = torch.zeros((8, 8, 8), dtype=torch.float64, device="cuda")
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_kinetic(plan, x, x)
        assert ei.value.status == -3
        ov = x[1].view(8, 8, 8)                             # v_eff inside out
        y = torch.zeros_like(x)
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_hamiltonian(plan, y, ov, x)
        assert ei.value.status == -3
        big = torch.zeros(2 * 512 + 1, dtype=torch.float64, device="cuda")
        mis = big[1:].view(2, 8, 8, 8)                      # 8-byte aligned only
        with pytest.raises(fd.FDError) as ei:
            fd.fd_apply_kinetic(plan, mis, x)
        assert ei.value.status == -1
        lib = fd.load_library()
        assert lib.fd_apply_kinetic(plan, None, None, 0, None) == 0   # nbands == 0: no-op
        assert lib.fd_apply_kinetic(plan, None, None, -1, None) == -1
    finally:
        fd.fd_destroy(plan)


def test_async_on_a_side_stream(oracle, fd):
    cfg = W.custom((16, 16, 16), (0.2,) * 3, (1, 1, 1), nbands=4)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc)
    try:
        s = torch.cuda.Stream()
        d_psi, d_v = torch.from_numpy(psi).cuda(), torch.from_numpy(v).cuda()
        d_out = torch.empty_like(d_psi)
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out)       # picks the current stream
        fd.fd_apply_hamiltonian(plan, d_psi, d_v, torch.empty_like(d_psi), stream=s)
        s.synchronize()
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None, psi, v)
        assert np.max(np.abs(d_out.cpu().numpy() - want)) <= parity_tol(cfg.h, 3, psi, v)
        assert fd.fd_plan_launches(plan) == 2
    finally:
        fd.fd_destroy(plan)


def test_host_buffer_apply(oracle, fd):
    """fd_apply_hamiltonian_host: several chunks, pinned and pageable, real and complex."""
    for cplx in (False, True):
        cfg = W.custom((40, 48, 64), (0.2,) * 3, (1, 1, 0), complex_=cplx, nbands=150,
                       k=(0.25, 0.125, 0.0) if cplx else (0, 0, 0))
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc, cfg.k if cplx else None,
                            fd.FD_C128 if cplx else fd.FD_F64)
        try:
            out = np.empty_like(psi)
            fd.fd_apply_hamiltonian_host(plan, psi, v, out)          # pageable numpy
            want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, cfg.k if cplx else None, psi, v)
            tol = parity_tol(cfg.h, 3, psi, v)
            assert np.max(np.abs(out - want)) <= tol
            p_psi = torch.from_numpy(psi).pin_memory()
            p_out = torch.empty_like(p_psi).pin_memory()
            fd.fd_apply_hamiltonian_host(plan, p_psi, torch.from_numpy(v).pin_memory(), p_out)
            assert np.max(np.abs(p_out.numpy() - want)) <= tol
            fd.fd_apply_hamiltonian_host(plan, p_psi, None, p_out)   # kinetic only
            want_t = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, cfg.k if cplx else None, psi)
            assert np.max(np.abs(p_out.numpy() - want_t)) <= tol
        finally:
            fd.fd_destroy(plan)


@pytest.mark.parametrize("xchunk", [3, 5, 11])
def test_many_short_teams_more_ctas_than_sms(oracle, fd, monkeypatch, xchunk):
    """FDHAM_TUNE=xchunk=n cuts the (band, x) planes into teams of n planes: every team seam, band
    seam and wrap entry of the step table is exercised, with more CTAs than SMs (several waves)."""
    monkeypatch.setenv("FDHAM_TUNE", f"xchunk={xchunk},kernel=2")
    for bc, cplx, k in [((1, 1, 1), False, (0, 0, 0)), ((0, 1, 0), False, (0, 0, 0)),
                        ((1, 1, 1), True, (0.25, 0.125, -0.3))]:
        cfg = W.custom((24, 40, 16), (0.2, 0.21, 0.18), bc, k=k, complex_=cplx, nbands=37)
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        got, used = gpu_apply(fd, cfg, psi, v, "auto")
        assert used == fd.FD_KERNEL_SWEEP
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, cfg.k if cplx else None, psi, v)
        assert np.max(np.abs(got - want)) <= parity_tol(cfg.h, 3, psi, v)


def test_one_plan_two_streams_concurrently(oracle, fd):
    """A plan is immutable: applies of the same plan on two streams may overlap."""
    cfg = W.custom((32, 32, 32), (0.2,) * 3, (1, 1, 1), nbands=24)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc)
    try:
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        a = torch.from_numpy(psi).cuda()
        b = torch.from_numpy(psi[::-1].copy()).cuda()
        d_v = torch.from_numpy(v).cuda()
        oa, ob = torch.empty_like(a), torch.empty_like(b)
        torch.cuda.synchronize()
        for _ in range(5):
            fd.fd_apply_hamiltonian(plan, a, d_v, oa, stream=s1)
            fd.fd_apply_hamiltonian(plan, b, d_v, ob, stream=s2)
        torch.cuda.synchronize()
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None, psi, v)
        tol = parity_tol(cfg.h, 3, psi, v)
        assert np.max(np.abs(oa.cpu().numpy() - want)) <= tol
        assert np.max(np.abs(ob.cpu().numpy() - want[::-1])) <= tol
    finally:
        fd.fd_destroy(plan)


@pytest.mark.parametrize("scale", [1.0, -2.25])
def test_scaled_laplacian_plans(oracle, fd, scale):
    """fd_create_scaled: scale * lap_FD psi + v psi on both kernel families, real
    and complex with Bloch phases, against the oracle's scaled apply."""
    for bc, cplx, k in [((1, 1, 1), False, None), ((1, 0, 1), False, None),
                        ((1, 1, 0), True, (0.25, 0.125, 0.0))]:
        cfg = W.custom((16, 20, 24), (0.2, 0.23, 0.17), bc, k=k or (0, 0, 0), complex_=cplx,
                       nbands=5)
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, k, psi, v, scale=scale)
        tol = parity_tol(cfg.h, 3, psi, v, scale)
        for kern in (fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create_scaled(cfg.shape, cfg.h, 3, cfg.bc, k,
                                       fd.FD_C128 if cplx else fd.FD_F64, 0, scale)
            try:
                fd.fd_plan_set_kernel(plan, kern)
                d_psi = torch.from_numpy(psi).cuda()
                d_out = torch.full_like(d_psi, float("nan"))
                fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v).cuda(), d_out)
                torch.cuda.synchronize()
                assert np.max(np.abs(d_out.cpu().numpy() - want)) <= tol
            finally:
                fd.fd_destroy(plan)
    with pytest.raises(fd.FDError):
        fd.fd_create_scaled((8, 8, 8), (0.2,) * 3, 3, (1, 1, 1), None, fd.FD_F64, 0, float("inf"))


def test_guard_bands_no_out_of_bounds_access(oracle, fd):
    """psi, v_eff and out sit inside larger buffers whose surroundings are NaN (inputs) or a
    sentinel (output): an out-of-bounds read would poison the result, an out-of-bounds write would
    change the guard band.  Ragged y tiles, all boundary mixes, both kernels, both dtypes."""
    pad = 4096  # elements of the buffer's dtype on either side
    for shape, bc, cplx, k, nn in [((12, 26, 16), (1, 1, 1), False, None, 3),
                                   ((9, 22, 12), (0, 1, 0), False, None, 3),
                                   ((10, 18, 8), (1, 1, 1), True, (0.25, 0.125, -0.3), 3),
                                   ((9, 26, 12), (1, 0, 1), False, None, 2),
                                   ((8, 8, 8), (0, 0, 0), False, None, 3)]:
        cfg = W.custom(shape, (0.2, 0.21, 0.18), bc, k=k or (0, 0, 0), complex_=cplx, nbands=5,
                       nn=nn)
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        want = oracle.apply(cfg.shape, cfg.h, nn, cfg.bc, k, psi, v)
        tol = parity_tol(cfg.h, nn, psi, v)
        tdt = torch.complex128 if cplx else torch.float64
        n = psi.size
        big_in = torch.full((n + 2 * pad,), float("nan"), dtype=tdt, device="cuda")
        big_v = torch.full((v.size + 2 * pad,), float("nan"), dtype=torch.float64, device="cuda")
        d_psi = big_in[pad:pad + n].view(psi.shape)
        d_v = big_v[pad:pad + v.size].view(v.shape)
        d_psi.copy_(torch.from_numpy(psi))
        d_v.copy_(torch.from_numpy(v))
        for kern in (fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create(cfg.shape, cfg.h, nn, cfg.bc, k,
                                fd.FD_C128 if cplx else fd.FD_F64, 0)
            try:
                fd.fd_plan_set_kernel(plan, kern, 8 if kern == fd.FD_KERNEL_SWEEP else 0)
                big_out = torch.full((n + 2 * pad,), 12345.0, dtype=tdt, device="cuda")
                d_out = big_out[pad:pad + n].view(psi.shape)
                fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out)
                torch.cuda.synchronize()
                got = d_out.cpu().numpy()
                assert np.isfinite(got).all(), f"{shape} {bc} kernel {kern}: read outside psi/v_eff"
                assert np.max(np.abs(got - want)) <= tol
                guards = torch.cat([big_out[:pad], big_out[pad + n:]])
                assert bool((guards == 12345.0).all()), f"{shape} {bc} kernel {kern}: wrote outside out"
            finally:
                fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ every shipped instantiation

# the pick() tables of csrc/fd_sweep_inst_*.cu: row lengths (doubles per z row) with a compile-time
# pitch.  real: nz; complex: 2 nz.  PH: 0 = Gamma, 1 = k on x / y only, 3 = k_z != 0.
REAL_ROWD = [24, 48, 64, 96, 128, 192]
CPLX_NZ = [24, 48, 72, 96]


@pytest.mark.parametrize("nz", REAL_ROWD)
@pytest.mark.parametrize("has_v", [0, 1])
def test_every_real_row_length_instantiation(oracle, fd, nz, has_v):
    """mixed BCs, several y tiles with a ragged one, fixed-pitch kernel <0, has_v, nz, 0, 3>"""
    for bc in [(1, 1, 1), (0, 1, 0), (1, 0, 1)]:
        cfg = W.custom((9, 22, nz), (0.2, 0.23, 0.17), bc, nbands=3)
        psi = W.make_psi(cfg)
        used = check(oracle, fd, cfg, psi, W.make_veff(cfg) if has_v else None,
                     fd.FD_KERNEL_SWEEP, tyc=8)
        assert used == fd.FD_KERNEL_SWEEP


@pytest.mark.parametrize("nz", CPLX_NZ)
@pytest.mark.parametrize("ph,k", [(0, (0.0, 0.0, 0.0)), (1, (0.25, 0.125, 0.0)), (3, (0.25, 0.0, -0.3))])
@pytest.mark.parametrize("has_v", [0, 1])
def test_every_complex_row_length_and_phase_instantiation(oracle, fd, nz, ph, k, has_v):
    """fixed-pitch kernels <1, has_v, 2 nz, PH, 3> for PH = 0 (Gamma), 1 (x/y phases), 3 (z phase)"""
    for bc in [(1, 1, 1), (1, 1, 0) if ph != 3 else (0, 1, 1)]:
        kk = tuple(x if b else 0.0 for x, b in zip(k, bc))
        cfg = W.custom((9, 22, nz), (0.2, 0.23, 0.17), bc, k=kk, complex_=True, nbands=3)
        psi = W.make_psi(cfg)
        used = check(oracle, fd, cfg, psi, W.make_veff(cfg) if has_v else None,
                     fd.FD_KERNEL_SWEEP, tyc=8)
        assert used == fd.FD_KERNEL_SWEEP


# ------------------------------------------------------------------------------ metamorphic M5, M6

def test_phase_periodicity_and_gauge_M5(fd):
    """k and k + integer vector give the same operator; and e^{-ik.r} H_k e^{ik.r} u for periodic u
    does not depend on which cell the grid origin sits in (shift the origin by one cell: the Bloch
    function picks up e^{ik.L}, a global phase that must come out of H unchanged)."""
    shape, h, bc = (12, 16, 20), (0.2, 0.21, 0.19), (1, 1, 1)
    k = (0.25, 0.125, -0.3)
    cfg = W.custom(shape, h, bc, k=k, complex_=True, nbands=3)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    base, _ = gpu_apply(fd, cfg, psi, v, fd.FD_KERNEL_SWEEP, tyc=8)
    tol = parity_tol(cfg.h, 3, psi, v)
    for shift in [(1, 0, 0), (0, -2, 0), (3, 1, -1)]:
        k2 = tuple(a + b for a, b in zip(k, shift))
        c2 = W.custom(shape, h, bc, k=k2, complex_=True, nbands=3)
        got, _ = gpu_apply(fd, c2, psi, v, fd.FD_KERNEL_SWEEP, tyc=8)
        assert np.max(np.abs(got - base)) <= tol
        gen, _ = gpu_apply(fd, c2, psi, v, fd.FD_KERNEL_GENERIC)
        assert np.max(np.abs(gen - base)) <= tol
    # gauge: psi' = e^{2 pi i k_x} psi is the same Bloch function seen from the next cell along x
    ph = np.exp(2j * np.pi * k[0])
    got, _ = gpu_apply(fd, cfg, np.ascontiguousarray(ph * psi), v, fd.FD_KERNEL_SWEEP, tyc=8)
    assert np.max(np.abs(got - ph * base)) <= tol
    # rolling a Bloch function across the x boundary multiplies the wrapped planes by e^{-ik.L}
    rolled = np.roll(psi, 5, axis=1).copy()
    rolled[:, :5] *= np.exp(-2j * np.pi * k[0])
    vr = np.roll(v, 5, axis=0).copy()
    got, _ = gpu_apply(fd, cfg, rolled, vr, fd.FD_KERNEL_SWEEP, tyc=8)
    want = np.roll(base, 5, axis=1).copy()
    want[:, :5] *= np.exp(-2j * np.pi * k[0])
    assert np.max(np.abs(got - want)) <= tol


def test_separability_with_anisotropic_spacing_M6(fd):
    """psi = f(x) g(y) h(z)  =>  T psi = (T_x f) g h + f (T_y g) h + f g (T_z h), each 1-D factor
    taken from the same library on a grid that is trivial along the other two axes."""
    shape, h, bc = (16, 24, 32), (0.2, 0.26, 0.15), (1, 0, 1)
    rng = np.random.default_rng(8)
    f, g, hh = (rng.standard_normal(n) for n in shape)
    psi = (f[:, None, None] * g[None, :, None] * hh[None, None, :])[None].copy()
    cfg = W.custom(shape, h, bc, nbands=1)
    got, _ = gpu_apply(fd, cfg, psi, None, fd.FD_KERNEL_SWEEP, kinetic=True, tyc=8)
    # 1-D operators from the closed-form weights in helpers (not from the library)
    from helpers import coeffs_f64
    c = coeffs_f64(3)

    def t1d(x, hd, per):
        out = c[0] * x
        for j in (1, 2, 3):
            if per:
                out = out + c[j] * (np.roll(x, j) + np.roll(x, -j))
            else:
                up = np.concatenate([x[j:], np.zeros(j)])
                dn = np.concatenate([np.zeros(j), x[:-j]])
                out = out + c[j] * (up + dn)
        return -0.5 * out / (hd * hd)

    hb = cfg.h
    want = (t1d(f, hb[0], bc[0])[:, None, None] * g[None, :, None] * hh[None, None, :]
            + f[:, None, None] * t1d(g, hb[1], bc[1])[None, :, None] * hh[None, None, :]
            + f[:, None, None] * g[None, :, None] * t1d(hh, hb[2], bc[2])[None, None, :])[None]
    assert np.max(np.abs(got - want)) <= parity_tol(cfg.h, 3, psi, None)


# ------------------------------------------------------------------------------ plans living side by side

def test_two_plans_on_one_instantiation_and_refused_set_kernel(oracle, fd):
    """A later, smaller plan on the same (run-time pitch) instantiation must not break an earlier
    one; a refused fd_plan_set_kernel leaves the plan usable and unchanged."""
    ca = W.custom((24, 128, 40), (0.2, 0.2, 0.2), (1, 1, 1), nbands=6, nn=2)
    cb = W.custom((12, 12, 40), (0.2, 0.2, 0.2), (1, 1, 1), nbands=2, nn=2)
    pa = fd.fd_create(ca.shape, ca.h, 2, ca.bc)
    fd.fd_plan_set_kernel(pa, fd.FD_KERNEL_SWEEP)
    pb = fd.fd_create(cb.shape, cb.h, 2, cb.bc)
    fd.fd_plan_set_kernel(pb, fd.FD_KERNEL_SWEEP, 4)
    try:
        for cfg, plan in ((cb, pb), (ca, pa), (cb, pb)):
            psi, v = W.make_psi(cfg), W.make_veff(cfg)
            d_psi = torch.from_numpy(psi).cuda()
            d_out = torch.full_like(d_psi, float("nan"))
            fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v).cuda(), d_out)
            torch.cuda.synchronize()
            want = oracle.apply(cfg.shape, cfg.h, 2, cfg.bc, None, psi, v)
            assert np.max(np.abs(d_out.cpu().numpy() - want)) <= parity_tol(cfg.h, 2, psi, v)
        # refused request: the sweep family on a plan it cannot run (odd nz); the plan stays usable
        odd = W.custom((8, 12, 9), (0.2, 0.2, 0.2), (1, 1, 1), nbands=2)
        pc = fd.fd_create(odd.shape, odd.h, 3, odd.bc)
        try:
            before = fd.fd_plan_kernel_for(pc, 2)
            with pytest.raises(fd.FDError) as ei:
                fd.fd_plan_set_kernel(pc, fd.FD_KERNEL_SWEEP, 4)
            assert ei.value.status == -2
            assert fd.fd_plan_kernel_for(pc, 2) == before == fd.FD_KERNEL_GENERIC
            psi, v = W.make_psi(odd), W.make_veff(odd)
            d_psi = torch.from_numpy(psi).cuda()
            d_out = torch.full_like(d_psi, float("nan"))
            fd.fd_apply_hamiltonian(pc, d_psi, torch.from_numpy(v).cuda(), d_out)
            torch.cuda.synchronize()
            want = oracle.apply(odd.shape, odd.h, 3, odd.bc, None, psi, v)
            assert np.max(np.abs(d_out.cpu().numpy() - want)) <= parity_tol(odd.h, 3, psi, v)
        finally:
            fd.fd_destroy(pc)
    finally:
        fd.fd_destroy(pa)
        fd.fd_destroy(pb)


def test_host_workspace_reuse(oracle, fd):
    cfg = W.custom((24, 32, 48), (0.2,) * 3, (1, 1, 0), nbands=40)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    plan = fd.fd_create(cfg.shape, cfg.h, 3, cfg.bc)
    ws = fd.fd_workspace_create(plan, 4 << 20)     # 13 bands per chunk: several ring turns
    try:
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None, psi, v)
        p_psi, p_v = torch.from_numpy(psi).pin_memory(), torch.from_numpy(v).pin_memory()
        for _ in range(3):
            out = torch.full(psi.shape, float("nan"), dtype=torch.float64).pin_memory()
            fd.fd_apply_hamiltonian_host_ws(plan, ws, p_psi, p_v, out)
            assert np.max(np.abs(out.numpy() - want)) <= parity_tol(cfg.h, 3, psi, v)
        with pytest.raises(fd.FDError) as ei:                    # v_eff inside out
            big = torch.zeros(psi.size + v.size, dtype=torch.float64)
            fd.fd_apply_hamiltonian_host_ws(plan, ws, p_psi, big[:v.size].view(v.shape),
                                            big[:psi.size].view(psi.shape))
        assert ei.value.status == -3
        other = fd.fd_create((8, 8, 8), (0.4,) * 3)
        try:
            with pytest.raises(fd.FDError) as ei:
                fd.fd_apply_hamiltonian_host_ws(other, ws, p_psi, p_v, out)
            assert ei.value.status == -1
        finally:
            fd.fd_destroy(other)
    finally:
        fd.fd_workspace_destroy(ws)
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ f1: real dtype at k = 1/2

@pytest.mark.parametrize("k", [(0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.0, 0.0, 0.5), (0.5, 0.5, 0.5),
                               (-0.5, 1.0, 1.5)])
def test_real_dtype_at_zone_boundary_k(oracle, fd, k):
    """FD_F64 with Bloch factors -1.  The oracle runs the complex definition on the
    real input (its imaginary part must vanish); both kernel families, nn = 1..3, ragged tiles."""
    for nn, shape, bc in [(3, (10, 22, 16), (1, 1, 1)), (2, (9, 20, 12), (1, 1, 1)), (1, (12, 10, 8), (1, 1, 1)),
                          (3, (12, 18, 24), (1, 0, 1))]:
        kk = tuple(x if b else 0.0 for x, b in zip(k, bc))
        cfg = W.custom(shape, (0.2, 0.23, 0.17), bc, nbands=5, nn=nn)
        psi, v = W.make_psi(cfg), W.make_veff(cfg)
        want_c = oracle.apply(cfg.shape, cfg.h, nn, bc, kk, psi.astype(np.complex128), v)
        assert np.max(np.abs(want_c.imag)) <= 1e-13 * np.abs(want_c).max()
        tol = parity_tol(cfg.h, nn, psi, v)
        for kern in (fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create(cfg.shape, cfg.h, nn, bc, kk, fd.FD_F64, 0)
            try:
                fd.fd_plan_set_kernel(plan, kern, 8 if kern == fd.FD_KERNEL_SWEEP else 0)
                d_psi = torch.from_numpy(psi).cuda()
                d_out = torch.full_like(d_psi, float("nan"))
                fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v).cuda(), d_out)
                torch.cuda.synchronize()
                err = float(np.max(np.abs(d_out.cpu().numpy() - want_c.real)))
                assert err <= tol, (k, nn, kern, err, tol)
                # the other forms fall back to code that knows the sign: expectation values, Jacobi
                eps = torch.empty(5, dtype=torch.float64, device="cuda")
                nrm = torch.empty_like(eps)
                ws = torch.empty(fd.fd_expect_workspace_bytes(plan, 5) // 8 + 1, dtype=torch.float64,
                                 device="cuda")
                fd.fd_apply_hamiltonian_expect(plan, d_psi, torch.from_numpy(v).cuda(), d_out, eps, nrm, ws)
                torch.cuda.synchronize()
                w_eps = np.sum(psi * want_c.real, axis=(1, 2, 3))
                assert np.max(np.abs(eps.cpu().numpy() - w_eps)) <= tol * psi[0].size * np.abs(psi).max()
            finally:
                fd.fd_destroy(plan)
    with pytest.raises(fd.FDError) as ei:
        fd.fd_create((8, 8, 8), (0.4,) * 3, 3, (1, 1, 1), (0.25, 0, 0), fd.FD_F64, 0)
    assert ei.value.status == -1


# ------------------------------------------------------------------------------ f1: nn = 4, 5, 6 on the sweep kernel

@pytest.mark.parametrize("nn", [4, 5, 6])
def test_sweep_kernel_higher_orders(oracle, fd, nn):
    """2 nn + 1 = 9 / 11 / 13 accumulator planes with a 2-row micro tile, 2 nn halo
    rows / planes, the general z-tap form: all BC mixes, several tiles with a ragged one, real and
    complex with Bloch phases on every axis, several bands per team and several teams."""
    for bc in itertools.product((0, 1), repeat=3):
        cfg = W.custom((13, 26, 16), (0.2, 0.23, 0.17), bc, nbands=7, nn=nn)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP, tyc=8)
        assert used == fd.FD_KERNEL_SWEEP
    for bc in [(1, 1, 1), (0, 1, 1), (1, 1, 0)]:
        k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
        cfg = W.custom((14, 20, 12), (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=5, nn=nn)
        used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP, tyc=6)
        assert used == fd.FD_KERNEL_SWEEP
        check(oracle, fd, cfg, W.make_psi(cfg), None, fd.FD_KERNEL_SWEEP)
    cfg = W.custom((40, 48, 64), (0.2, 0.2, 0.18), (1, 1, 0), nbands=40, nn=nn)
    used = check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), "auto")
    assert used == fd.FD_KERNEL_SWEEP
    # n = 2 nn on a periodic axis: taps +nn and -nn hit the same point (R7)
    cfg = W.custom((2 * nn, 2 * nn + 2, 2 * nn), (0.2, 0.23, 0.17), (1, 1, 1), nbands=3, nn=nn)
    if min(cfg.shape) >= 8:
        check(oracle, fd, cfg, W.make_psi(cfg), W.make_veff(cfg), fd.FD_KERNEL_SWEEP)
    # the forms without an nn > 3 instantiation fall back and stay correct
    cfg = W.custom((12, 16, 16), (0.2, 0.23, 0.17), (1, 0, 1), nbands=3, nn=nn)
    psi, v = W.make_psi(cfg), W.make_veff(cfg)
    plan = fd.fd_create(cfg.shape, cfg.h, nn, cfg.bc)
    try:
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP)
        d_psi = torch.from_numpy(psi).cuda()
        d_out = torch.full_like(d_psi, float("nan"))
        eps = torch.empty(3, dtype=torch.float64, device="cuda")
        nrm = torch.empty_like(eps)
        ws = torch.empty(fd.fd_expect_workspace_bytes(plan, 3) // 8 + 1, dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian_expect(plan, d_psi, torch.from_numpy(v).cuda(), d_out, eps, nrm, ws)
        torch.cuda.synchronize()
        w_eps, w_n, want = oracle.expect(cfg.shape, cfg.h, nn, cfg.bc, None, psi, v, want_out=True)
        assert np.max(np.abs(d_out.cpu().numpy() - want)) <= parity_tol(cfg.h, nn, psi, v)
        assert np.max(np.abs(eps.cpu().numpy() - w_eps.real)) <= parity_tol(cfg.h, nn, psi, v) * psi[0].size * np.abs(psi).max()
    finally:
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ f1: float32 / complex64

def tol_f32(h, nn, psi, v):
    """fp32 accumulation of the 6 nn + 2 terms with fp32-rounded weights: |err| <= gamma_n sum|w x|,
    gamma_n = n u / (1 - n u), n = 6 nn + 4, u = 2^-24  (nn = 3: 1.3e-6; reading R18),
    taken as 2e-6 (max|psi| S + max|v psi|), the north_star scale."""
    return 2e-6 / 1e-12 * parity_tol(h, nn, psi.astype(np.complex128 if np.iscomplexobj(psi) else np.float64),
                                     None if v is None else v.astype(np.float64))


def f32_apply(fd, cfg, psi32, v32, kinetic=False, tyc=0):
    k = cfg.k if cfg.complex else None
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, fd.FD_C64 if cfg.complex else fd.FD_F32, 0)
    try:
        assert fd.fd_plan_kernel_for(plan, psi32.shape[0]) == fd.FD_KERNEL_SWEEP
        if tyc:
            fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP, tyc)
        d_psi = torch.from_numpy(psi32).cuda()
        d_out = torch.full_like(d_psi, float("nan"))
        if kinetic:
            fd.fd_apply_kinetic(plan, d_psi, d_out)
        else:
            fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v32).cuda(), d_out)
        torch.cuda.synchronize()
        return d_out.cpu().numpy()
    finally:
        fd.fd_destroy(plan)


@pytest.mark.parametrize("nn", [1, 2, 3])
def test_float32_and_complex64_sweep(oracle, fd, nn):
    """single precision on the sweep kernel against the fp64 oracle on the same (fp32-rounded)
    inputs: all BC mixes, ragged tiles, complex64 with Bloch phases on every axis, several teams"""
    for bc in itertools.product((0, 1), repeat=3):
        cfg = W.custom((10, 26, 16), (0.2, 0.23, 0.17), bc, nbands=5, nn=nn)
        psi32, v32 = W.make_psi(cfg).astype(np.float32), W.make_veff(cfg).astype(np.float32)
        for kin in (False, True):
            got = f32_apply(fd, cfg, psi32, v32, kinetic=kin, tyc=8)
            want = oracle.apply(cfg.shape, cfg.h, nn, bc, None, psi32.astype(np.float64),
                                None if kin else v32.astype(np.float64))
            assert got.dtype == np.float32 and np.isfinite(got).all()
            assert np.max(np.abs(got - want)) <= tol_f32(cfg.h, nn, psi32, None if kin else v32)
        k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
        ck = W.custom((10, 22, 12), (0.2, 0.23, 0.17), bc, k=k, complex_=True, nbands=4, nn=nn)
        psi64c, v32 = W.make_psi(ck).astype(np.complex64), W.make_veff(ck).astype(np.float32)
        got = f32_apply(fd, ck, psi64c, v32, tyc=8)
        want = oracle.apply(ck.shape, ck.h, nn, bc, k, psi64c.astype(np.complex128), v32.astype(np.float64))
        assert got.dtype == np.complex64
        assert np.max(np.abs(got - want)) <= tol_f32(ck.h, nn, psi64c, v32)
    cfg = W.custom((40, 48, 64), (0.2, 0.2, 0.18), (1, 1, 0), nbands=40, nn=nn)
    psi32, v32 = W.make_psi(cfg).astype(np.float32), W.make_veff(cfg).astype(np.float32)
    got = f32_apply(fd, cfg, psi32, v32)
    want = oracle.apply(cfg.shape, cfg.h, nn, cfg.bc, None, psi32.astype(np.float64), v32.astype(np.float64))
    assert np.max(np.abs(got - want)) <= tol_f32(cfg.h, nn, psi32, v32)


def test_float32_full_size_cfg3_grid_and_unsupported_forms(oracle, fd):
    cfg = W.get(3).with_bands(64)
    psi32, v32 = W.make_psi(cfg).astype(np.float32), W.make_veff(cfg).astype(np.float32)
    got = f32_apply(fd, cfg, psi32, v32)
    for b in (0, 63):
        want = oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None, psi32[b:b + 1].astype(np.float64),
                            v32.astype(np.float64))
        assert np.max(np.abs(got[b:b + 1] - want)) <= tol_f32(cfg.h, 3, psi32, v32)
    # the error is single-precision sized, not double-precision sized: the dtype really is fp32
    assert np.max(np.abs(got[:1] - oracle.apply(cfg.shape, cfg.h, 3, cfg.bc, None,
                                                 psi32[:1].astype(np.float64), v32.astype(np.float64)))) \
        > 1e3 * parity_tol(cfg.h, 3, psi32[:1].astype(np.float64), v32.astype(np.float64))
    # shapes / orders the bandwidth kernel does not take run on the generic kernel in the same precision
    for shape, nn, cplx, k in [((8, 8, 10), 3, False, None), ((8, 8, 9), 3, True, (0.25, 0.0, -0.3)),
                               ((12, 12, 12), 4, False, None), ((6, 12, 12), 3, False, None),
                               ((8, 8, 8), 3, False, (0.5, 0.0, 0.5)), ((7, 8, 9), 6, True, (0.1, 0.2, 0.3))]:
        c2 = W.custom(shape, (0.3, 0.31, 0.29), (1, 1, 1), k=k or (0, 0, 0), complex_=cplx, nbands=3, nn=nn)
        p32 = W.make_psi(c2).astype(np.complex64 if cplx else np.float32)
        v32s = W.make_veff(c2).astype(np.float32)
        plan = fd.fd_create(shape, c2.h, nn, (1, 1, 1), k, fd.FD_C64 if cplx else fd.FD_F32, 0)
        try:
            assert fd.fd_plan_kernel_for(plan, 3) == fd.FD_KERNEL_GENERIC
            d_p = torch.from_numpy(p32).cuda()
            d_o = torch.full_like(d_p, float("nan"))
            fd.fd_apply_hamiltonian(plan, d_p, torch.from_numpy(v32s).cuda(), d_o)
            torch.cuda.synchronize()
            want = oracle.apply(shape, c2.h, nn, (1, 1, 1), k if (cplx or k) else None,
                                p32.astype(np.complex128 if (cplx or k) else np.float64), v32s.astype(np.float64))
            got = d_o.cpu().numpy()
            assert got.dtype == p32.dtype
            assert np.max(np.abs(got - (want if cplx else want.real))) <= tol_f32(c2.h, nn, p32, v32s)
        finally:
            fd.fd_destroy(plan)
    plan = fd.fd_create((8, 8, 8), (0.3,) * 3, 3, (1, 1, 1), None, fd.FD_F32, 0)
    try:
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_GENERIC)          # both families exist in fp32
        assert fd.fd_plan_kernel_for(plan, 2) == fd.FD_KERNEL_GENERIC
        fd.fd_plan_set_kernel(plan, fd.FD_KERNEL_SWEEP)
        with pytest.raises(fd.FDError) as ei:
            fd.fd_expect_workspace_bytes(plan, 4)
        assert ei.value.status == -2
    finally:
        fd.fd_destroy(plan)


def test_binding_rejects_arrays_that_do_not_match_the_plan(fd):
    """The C ABI takes raw pointers; the binding checks shape, dtype and band counts first."""
    plan = fd.fd_create((8, 10, 12), (0.4,) * 3)
    try:
        info = fd.fd_plan_get_info(plan)
        assert info["shape"] == (8, 10, 12) and info["nn"] == 3 and info["dtype"] == fd.FD_F64
        assert info["bc"] == (1, 1, 1) and info["device"] == 0
        good = torch.zeros((2, 8, 10, 12), dtype=torch.float64, device="cuda")
        v = torch.zeros((8, 10, 12), dtype=torch.float64, device="cuda")
        fd.fd_apply_hamiltonian(plan, good, v, torch.empty_like(good))
        for bad_psi, bad_out, bad_v in [
                (torch.zeros((2, 8, 10, 10), dtype=torch.float64, device="cuda"), good, v),   # shape
                (good, torch.zeros((1, 8, 10, 12), dtype=torch.float64, device="cuda"), v),   # band count
                (good.to(torch.float32), good, v),                                            # dtype
                (good, torch.empty_like(good), v[:4]),                                        # v_eff shape
                (good, torch.empty_like(good), v.to(torch.float32))]:                        # v_eff dtype
            with pytest.raises(ValueError):
                fd.fd_apply_hamiltonian(plan, bad_psi, bad_v, bad_out)
        with pytest.raises(ValueError):
            fd.fd_apply_kinetic(plan, good, good.cpu())
        # eps / norm of fd_residual, coef / out of fd_paw_expect
        eps = torch.ones(2, dtype=torch.float64, device="cuda")
        r = torch.empty_like(good)
        fd.fd_residual(plan, good, good.clone(), eps, eps.clone(), r)
        for bad_eps in (torch.ones(3, dtype=torch.float64, device="cuda"), eps.to(torch.float32), eps.cpu()):
            with pytest.raises(ValueError):
                fd.fd_residual(plan, good, good.clone(), bad_eps, eps, r)
            with pytest.raises(ValueError):
                fd.fd_residual(plan, good, good.clone(), eps, bad_eps, r)
        pw = fd.fd_paw_create(plan, [[0, 0, 0]], [[2, 2, 2]], [3], np.ones(24), np.eye(3).ravel())
        try:
            coef = torch.zeros((2, 3), dtype=torch.float64, device="cuda")
            fd.fd_paw_expect(plan, pw, 0, coef, eps)
            for bad_coef in (coef[:, :2].contiguous(), coef.to(torch.complex128), coef.cpu()):
                with pytest.raises(ValueError):
                    fd.fd_paw_expect(plan, pw, 0, bad_coef, eps)
            with pytest.raises(ValueError):
                fd.fd_paw_expect(plan, pw, 0, coef, eps.cpu())
        finally:
            fd.fd_paw_destroy(pw)
        # a destroyed plan's cached description must not leak to a new plan at the same address
        for shape in [(8, 8, 8), (8, 8, 16), (16, 8, 8)] * 3:
            p2 = fd.fd_create(shape, (0.4,) * 3)
            x = torch.zeros((1,) + shape, dtype=torch.float64, device="cuda")
            fd.fd_apply_kinetic(p2, x, torch.empty_like(x))
            fd.fd_destroy(p2)
        torch.cuda.synchronize()
    finally:
        fd.fd_destroy(plan)


def test_per_batch_kernel_choice_is_near_the_faster_kernel(fd):
    """fd_plan_kernel_for's crossover (two B200 constants in fd_api.cu): whatever it picks must be
    within 1.6x of the faster family for small and medium batches, and the sweep kernel for big ones."""
    def time_plan(plan, psi, v, out, n=30):
        for _ in range(5):
            fd.fd_apply_hamiltonian(plan, psi, v, out)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fd.fd_apply_hamiltonian(plan, psi, v, out)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n
    for shape, nb in [((24, 24, 24), 8), ((24, 24, 24), 64), ((48, 48, 48), 8), ((48, 48, 48), 64),
                      ((32, 32, 32), 2)]:
        psi = torch.randn((nb,) + shape, dtype=torch.float64, device="cuda")
        v = torch.rand(shape, dtype=torch.float64, device="cuda")
        out = torch.empty_like(psi)
        times = {}
        for kern in ("auto", fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create(shape, (0.4,) * 3)
            try:
                if kern != "auto":
                    fd.fd_plan_set_kernel(plan, kern)
                times[kern] = time_plan(plan, psi, v, out)
            finally:
                fd.fd_destroy(plan)
        best = min(times[fd.FD_KERNEL_SWEEP], times[fd.FD_KERNEL_GENERIC])
        assert times["auto"] <= 1.6 * best + 0.002, (shape, nb, times)
    plan = fd.fd_create((96, 96, 96), (0.4,) * 3)
    try:
        assert fd.fd_plan_kernel_for(plan, 256) == fd.FD_KERNEL_SWEEP
        assert fd.fd_plan_kernel_for(plan, 16) == fd.FD_KERNEL_SWEEP
    finally:
        fd.fd_destroy(plan)


# ------------------------------------------------------------------------------ seeded random configurations

def test_random_configurations_both_kernels_against_the_oracle(oracle, fd):
    """80 seeded random plans (shape 8..40 per axis, even nz, any BC mix, nn 1..6, float64 / complex128
    with random Bloch vectors / float64 at k = 1/2, 1..9 bands, random tile height): the plan's own
    kernel choice, the forced sweep kernel and the generic kernel against the oracle."""
    rng = np.random.default_rng(20231014)
    for trial in range(80):
        nn = int(rng.integers(1, 7))
        bc = tuple(int(b) for b in rng.integers(0, 2, 3))
        shape = tuple(int(max(rng.integers(8, 41), nn)) for _ in range(3))
        shape = (shape[0], shape[1], shape[2] + (shape[2] & 1))
        kind = int(rng.integers(0, 3))                      # 0 real Gamma, 1 complex Bloch, 2 real k = 1/2
        cplx = kind == 1
        if kind == 1:
            k = tuple(float(rng.uniform(-0.5, 0.5)) if b else 0.0 for b in bc)
        elif kind == 2:
            k = tuple(0.5 * int(rng.integers(0, 2)) if b else 0.0 for b in bc)
        else:
            k = (0.0, 0.0, 0.0)
        nb = int(rng.integers(1, 10))
        h = tuple(float(x) for x in rng.uniform(0.15, 0.3, 3))
        cfg = W.custom(shape, h, bc, k=k, complex_=cplx, nbands=nb, nn=nn, index=100 + trial)
        psi, v = W.make_psi(cfg), (W.make_veff(cfg) if rng.integers(0, 4) else None)
        kk = k if (cplx or kind == 2) else None
        want = oracle.apply(cfg.shape, cfg.h, nn, bc, kk, psi.astype(np.complex128) if kind == 2 else psi, v)
        if kind == 2:
            assert np.max(np.abs(want.imag)) <= 1e-12 * max(1.0, np.abs(want).max())
            want = want.real
        tol = parity_tol(cfg.h, nn, psi, v)
        tyc = int(rng.choice([0, 0, 4, 8, 12]))
        for kern in ("auto", fd.FD_KERNEL_SWEEP, fd.FD_KERNEL_GENERIC):
            plan = fd.fd_create(cfg.shape, cfg.h, nn, bc, kk, fd.FD_C128 if cplx else fd.FD_F64, 0)
            try:
                if kern != "auto":
                    try:
                        fd.fd_plan_set_kernel(plan, kern, tyc if kern == fd.FD_KERNEL_SWEEP else 0)
                    except fd.FDError as e:
                        assert e.status == -2 and kern == fd.FD_KERNEL_SWEEP
                        continue
                d_psi = torch.from_numpy(psi).cuda()
                d_out = torch.full_like(d_psi, float("nan"))
                if v is None:
                    fd.fd_apply_kinetic(plan, d_psi, d_out)
                else:
                    fd.fd_apply_hamiltonian(plan, d_psi, torch.from_numpy(v).cuda(), d_out)
                torch.cuda.synchronize()
                err = float(np.max(np.abs(d_out.cpu().numpy() - want)))
                assert err <= tol, (trial, shape, bc, nn, kind, k, nb, tyc, kern, err, tol)
            finally:
                fd.fd_destroy(plan)
