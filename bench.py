#!/usr/bin/env python
"""bench.py -- throughput of the FD Kohn-Sham apply H psi = -1/2 lap_FD psi + v_eff psi on B200.

Contract:
  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfgN]
A "step" is one pass of the whole hot path (halo resolution + 19-point stencil + v_eff multiply-add
+ store, all fused in one kernel launch) over one batch of synthetic wave functions.  The default
workload is BASELINE.json configs[2] (96^3 grid, 256 bands, float64, periodic Gamma): the config
the metric's 70 %-of-HBM target is quoted on.  Inputs (3.6 GB) are larger than the 126 MB L2, so no
L2 flush is needed between steps.

Prints ONE JSON line.  `value` = grid-point x band updates per second (whole job, inputs resident
in HBM); `e2e` = the same through fd_apply_hamiltonian_host_ws with pinned HOST buffers (H2D + D2H
inside the timed region); `roofline` = algorithmic bytes / measured kernel time against the
measured HBM copy peak (`traffic` from profiles/traffic.json when its kernel sha matches);
`cpu_baseline` = the CPU oracle timed on this box's host cores (all cores and one thread).
Beyond the contract (single GPU, default workload): `sustained` = the same apply held for >= 1 s
with its own clock record; `parity` = sampled points of every band against the oracle after
timing; `next_rows` = the SURVEY 8(f) calls on the same grid; `other_workloads` = cfg1, 2, 4, 5.
Multi-GPU (`--gpus N` under torchrun): the path does not shard (north_star: one GPU only), so N
independent replicas run, one per rank, no data-path collective ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FD H.psi apply Gpoint.bands/s"
UNIT = "Gpoint.band/s"
DEFAULT_WORKLOAD = "cfg3"

TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")
KERNEL_SOURCES = ["paper_2310_14776_b200/csrc/fd_sweep_kernel.cuh",   # the kernel
                  "paper_2310_14776_b200/csrc/fd_sweep.cu"]           # its tile / ring / team choice


def kernel_sha() -> str:
    """sha256 (16 hex digits) over the sources of the sweep kernel: profiles/traffic.json records
    the value its ncu capture was taken at."""
    import hashlib
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full`
    capture (profiles/traffic.json), or None when no capture exists for this workload or the kernel
    sources have changed since it was taken."""
    try:
        with open(TRAFFIC_JSON) as f:
            tab = json.load(f)
        ent = tab["workloads"][workload]
        if tab.get("kernel_sha") != kernel_sha():
            return None
        return int(ent["dram_bytes"])
    except Exception:
        return None


def _measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and clock-event reasons through NVML during the timed region."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "app_clocks",
               0x10: "sync_boost"}

    def __init__(self, torch_device_index: int, period_s: float = 0.005):
        self.period = period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = str(torch.cuda.get_device_properties(torch_device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.h is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def _cfg(name):
    import workloads as W
    return W.get(name)


def config_dict(cfg, world: int) -> dict:
    """The `config` object of the JSON line: identical in both arms (ours / --impl reference)."""
    return {"workload": cfg.name, "grid": list(cfg.shape), "nbands": cfg.nbands,
            "bc": list(cfg.bc), "k": list(cfg.k), "nn": cfg.nn,
            "h_angstrom": list(cfg.h_angstrom),
            "parallelism": "replicas only" if world > 1 else "single GPU",
            "l2": "inputs+outputs %.2f GB >> 126 MB L2, no flush between steps" % (cfg.min_bytes / 1e9)
                  if cfg.min_bytes > (256 << 20) else
                  "inputs+outputs %.1f MB fit the 126 MB L2: hot figure; see other_workloads for the "
                  "rotating-buffer cold figure" % (cfg.min_bytes / 1e6)}


def cpu_oracle_rate(cfg, budget_s: float = 10.0, max_bands: int | None = None):
    """Time the CPU oracle (as it stands) on a bounded sample of the workload: OpenMP over bands on
    all host cores (the reported `value`) and one thread (`value_1thread`, a third of the budget)."""
    import workloads as W
    from oracle import fd_oracle
    cores = fd_oracle.max_threads()
    nb = min(cfg.nbands, max(2 * cores, 8))
    if max_bands:
        nb = min(nb, max_bands)
    psi = W.make_psi(cfg, range(nb))
    v = W.make_veff(cfg)
    k = cfg.k if cfg.complex else None
    fd_oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi[:1], v)  # page in / build

    def timed(bands, nthreads, budget):
        passes, t0 = 0, time.perf_counter()
        while True:
            fd_oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi[:bands], v, nthreads=nthreads)
            passes += 1
            el = time.perf_counter() - t0
            if el >= budget or passes >= 50:
                return passes * bands * cfg.npoints / el / 1e9, passes, el

    rate, passes, el = timed(nb, cores, budget_s * 0.7)
    nb1 = max(1, min(nb, 2))
    rate1, passes1, el1 = timed(nb1, 1, budget_s * 0.3)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{nb} of {cfg.nbands} bands of {cfg.name}, {passes} passes, {el:.1f} s, "
                      f"OpenMP over bands",
            "value_1thread": rate1,
            "sample_1thread": f"{nb1} bands, {passes1} passes, {el1:.1f} s, 1 thread"}


def run_reference(args):
    """--impl reference: the oracle, on the host cores, same metric/config (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads as W
    from oracle import fd_oracle
    cfg = _cfg(args.workload)
    cores = fd_oracle.max_threads()
    nb = min(cfg.nbands, max(cores, 8))
    psi = W.make_psi(cfg, range(nb))
    v = W.make_veff(cfg)
    k = cfg.k if cfg.complex else None
    # keep the whole run within a few minutes: cap steps by a 120 s budget
    for _ in range(max(1, min(args.warmup, 2))):
        fd_oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi, v)
    t0 = time.perf_counter()
    done = 0
    for _ in range(args.steps):
        fd_oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi, v)
        done += 1
        if time.perf_counter() - t0 > 120.0:
            break
    el = time.perf_counter() - t0
    value = done * nb * cfg.npoints / el / 1e9
    sample = f"each step = oracle apply on {nb} of {cfg.nbands} bands of {cfg.name}"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": args.gpus, "steps": done, "warmup": args.warmup,
        "ms_per_step": el / done * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "c128" if cfg.complex else "f64", "data": "synthetic",
        "config": config_dict(cfg, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def aggregate(per_rank_ms: float, units_per_rank: float, world: int, reduce_max):
    """Whole-job throughput: all ranks' units / the slowest rank's time (replicas only)."""
    t = reduce_max(per_rank_ms)
    return world * units_per_rank / (t * 1e-3) / 1e9, t


def _kernel_name(fd, plan, nbands):
    return {fd.FD_KERNEL_SWEEP: "sweep", fd.FD_KERNEL_GENERIC: "generic"}[
        fd.fd_plan_kernel_for(plan, nbands)]


def _device_inputs(torch, W, cfg):
    """psi and v_eff of the workload's recipe on the device (generated on the host in band chunks)."""
    tdt = torch.complex128 if cfg.complex else torch.float64
    d_psi = torch.empty((cfg.nbands,) + cfg.shape, dtype=tdt, device="cuda")
    chunk = 32
    for b0 in range(0, cfg.nbands, chunk):
        bands = range(b0, min(cfg.nbands, b0 + chunk))
        d_psi[b0:b0 + len(bands)] = torch.from_numpy(W.make_psi(cfg, bands)).cuda()
    v_host = W.make_veff(cfg)
    return d_psi, torch.from_numpy(v_host).cuda(), v_host


def _time_stream(torch, stream, fn, steps, warmup):
    """mean ms per call of fn, CUDA events on the launch stream."""
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def parity_after_timing(torch, fd, cfg, plan, d_psi, d_v, v_host, h_psi, per_band=16):
    """One apply into a NaN-filled out, then sampled points of EVERY band against the CPU oracle
    (SURVEY 8(d) parity protocol); returns max|d| / tol with tol = 1e-12 (max|psi| S + max|v psi|)."""
    import numpy as np
    from oracle import fd_oracle
    d_out = torch.full_like(d_psi, float("nan"))
    fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out)
    torch.cuda.synchronize()
    finite = bool(torch.isfinite(torch.view_as_real(d_out) if cfg.complex else d_out).all())
    w = fd.fd_plan_get_weights(plan, cfg.nn)
    S = sum(abs(x[0]) + 2.0 * sum(abs(y) for y in x[1:]) for x in w)
    rng = np.random.default_rng(cfg.seed + 17)
    k = cfg.k if cfg.complex else None
    worst, npts, chunk = 0.0, 0, 16
    for b0 in range(0, cfg.nbands, chunk):
        nb = min(chunk, cfg.nbands - b0)
        psi_c = h_psi[b0:b0 + nb].numpy()
        p = np.stack([rng.integers(0, n, nb * per_band) for n in cfg.shape], axis=1)
        edge = rng.integers(0, 3, size=p.shape) == 0          # a third of the coordinates near a face
        lohi = np.where(rng.integers(0, 2, size=p.shape) == 0, rng.integers(0, 4, size=p.shape),
                        np.array(cfg.shape)[None, :] - 1 - rng.integers(0, 4, size=p.shape))
        p = np.where(edge, lohi, p)
        pts = np.concatenate([np.repeat(np.arange(nb), per_band)[:, None], p], axis=1).astype(np.int64)
        want = fd_oracle.points(cfg.shape, cfg.h, cfg.nn, cfg.bc, k, psi_c, v_host, pts)
        idx = torch.from_numpy(pts).cuda()
        got = d_out[idx[:, 0] + b0, idx[:, 1], idx[:, 2], idx[:, 3]].cpu().numpy()
        tol = 1e-12 * (float(np.abs(psi_c).max()) * S + float(np.abs(v_host[None] * psi_c).max()))
        worst = max(worst, float(np.max(np.abs(got - want))) / tol)
        npts += pts.shape[0]
    del d_out
    return {"max_err_over_tol": worst, "ok": bool(finite and worst <= 1.0), "all_finite": finite,
            "points": npts, "bands": cfg.nbands, "oracle": "oracle/fd_oracle.c fd_oracle_points",
            "tolerance": "1e-12 (max|psi| S + max|v_eff psi|), S = abs row sum of T"}


def sampled_parity(torch, fd, shape, h, nn, bc, k, plan, x_dev, v_host, y_dev, rel=1e-12, per_band=8,
                   seed=0):
    """max|d| / tol over sampled points of EVERY band of y_dev = H x_dev (already computed by the timed
    launches) against the oracle's point evaluation on the same inputs brought back to the host (in
    float64; single-precision inputs are converted exactly).  tol = rel (max|x| S + max|v x|) with S
    the absolute row sum of the plan's own weights; rel = 1e-12 (north_star) or 2e-6 (fp32, DESIGN.md
    R18).  k given for a real x: the complex definition on the real input, real part compared."""
    import numpy as np
    from oracle import fd_oracle
    w = fd.fd_plan_get_weights(plan, nn)
    S = sum(abs(r[0]) + 2.0 * sum(abs(t) for t in r[1:]) for r in w)
    rng = np.random.default_rng(seed + 29)
    nbands, worst, npts, chunk = x_dev.shape[0], 0.0, 0, 16
    for b0 in range(0, nbands, chunk):
        nb = min(chunk, nbands - b0)
        xc = x_dev[b0:b0 + nb]
        xc = xc.to(torch.complex128 if xc.is_complex() else torch.float64).cpu().numpy()
        p = np.stack([rng.integers(0, n, nb * per_band) for n in shape], axis=1)
        edge = rng.integers(0, 3, size=p.shape) == 0
        lohi = np.where(rng.integers(0, 2, size=p.shape) == 0, rng.integers(0, 4, size=p.shape),
                        np.array(shape)[None, :] - 1 - rng.integers(0, 4, size=p.shape))
        p = np.where(edge, lohi, p)
        pts = np.concatenate([np.repeat(np.arange(nb), per_band)[:, None], p], axis=1).astype(np.int64)
        real_at_k = k is not None and not np.iscomplexobj(xc)
        want = fd_oracle.points(shape, h, nn, bc, k, xc.astype(np.complex128) if real_at_k else xc,
                                v_host, pts)
        if real_at_k:
            want = want.real
        idx = torch.from_numpy(pts).cuda()
        got = y_dev[idx[:, 0] + b0, idx[:, 1], idx[:, 2], idx[:, 3]]
        got = got.to(torch.complex128 if got.is_complex() else torch.float64).cpu().numpy()
        tol = rel * (float(np.abs(xc).max()) * S + float(np.abs(v_host[None] * xc).max()))
        worst = max(worst, float(np.max(np.abs(got - want))) / tol)
        npts += pts.shape[0]
    return {"max_err_over_tol": worst, "ok": bool(worst <= 1.0), "points": npts, "rel_tol": rel}


def hardware_peaks(torch, fd, stream, local):
    """read-only / write-only / copy bandwidth with float64 vectors and the
    dependent-free DFMA rate, measured here with the library's own micro-benchmark kernels (2 GiB
    arrays >> L2; best of 5, CUDA events), with the SM clock sampled under the DFMA load."""
    n = 1 << 28                                     # doubles per array: 2 GiB
    a = torch.empty(n, dtype=torch.float64, device="cuda").fill_(1.0)
    b = torch.empty(n, dtype=torch.float64, device="cuda")
    sms = torch.cuda.get_device_properties(local).multi_processor_count

    def best(fn, reps=5):
        return min(_time_stream(torch, stream, fn, 1, 1) for _ in range(reps))
    out = {}
    ms = best(lambda: fd.fd_peak_kernel(0, a, b, n, 0, stream))
    out["read_GBps"] = n * 8 / ms / 1e6
    ms = best(lambda: fd.fd_peak_kernel(1, a, None, n, 0, stream))
    out["write_GBps"] = n * 8 / ms / 1e6
    ms = best(lambda: fd.fd_peak_kernel(2, a, b, n, 0, stream))
    out["copy_GBps"] = 2 * n * 8 / ms / 1e6
    iters, blocks = 1 << 14, 8 * sms
    sampler = ClockSampler(local)
    sampler.start()
    ms = best(lambda: fd.fd_peak_kernel(3, a, None, iters, blocks, stream), reps=8)
    out["dfma_clocks"] = sampler.stop()
    out["dfma_TFLOPs"] = 2.0 * 8 * iters * blocks * 256 / ms / 1e9
    out["dfma_Tinstr_per_s"] = out["dfma_TFLOPs"] / 2.0
    out["how"] = ("fd_peak_kernel: 2 GiB float64 arrays, grid-stride 16-byte accesses, 8 CTAs x 256 threads "
                  "per SM, best of 5; DFMA: 8 independent chains per thread")
    del a, b
    return out


def next_rows(torch, W, fd, cfg, plan, d_psi, d_v, d_out, stream, plain_ms, peak):
    """SURVEY 8(f) rows on the headline grid: ms, algorithmic GB/s and fraction of the copy peak."""
    import numpy as np
    rows = {}
    nb, P, E = cfg.nbands, cfg.npoints, cfg.elem_bytes

    def entry(ms, nbytes, **kw):
        gbs = nbytes / (ms * 1e-3) / 1e9
        return {"ms": ms, "algorithmic_bytes": int(nbytes), "GBps": gbs, "frac": gbs / peak, **kw}

    eps = torch.empty(nb, dtype=torch.float64, device="cuda")
    norm = torch.empty_like(eps)
    ws = torch.empty(fd.fd_expect_workspace_bytes(plan, nb) // 8 + 1, dtype=torch.float64, device="cuda")
    ms = _time_stream(torch, stream, lambda: fd.fd_apply_hamiltonian_expect(
        plan, d_psi, d_v, d_out, eps, norm, ws, stream), 20, 3)
    rows["f2_expect"] = entry(ms, cfg.min_bytes, over_plain_apply=ms / plain_ms - 1.0,
                              what="H psi + eps_b + norm_b in one pass (2 launches)")
    ms = _time_stream(torch, stream, lambda: fd.fd_residual(plan, d_psi, d_out, eps, norm, d_out, stream), 20, 3)
    rows["f2_residual"] = entry(ms, 3 * nb * P * E, what="r = H psi - (eps/norm) psi, in place")
    if not cfg.complex:
        pj = fd.fd_create_scaled(cfg.shape, cfg.h, cfg.nn, cfg.bc, None, fd.FD_F64,
                                 torch.cuda.current_device(), 1.0)
        rhs = torch.empty_like(d_psi).normal_()
        ms = _time_stream(torch, stream, lambda: fd.fd_jacobi_sweep(pj, d_psi, rhs, d_out, 2.0 / 3.0, stream), 20, 3)
        rows["f3_jacobi"] = entry(ms, 3 * nb * P * 8, what="weighted-Jacobi sweep, %d right-hand sides" % nb)
        fd.fd_destroy(pj)
        del rhs
        # grid transfer: this grid as the coarse one, its 2x refinement as the fine one
        nf = tuple(2 * n if b else 2 * n + 1 for n, b in zip(cfg.shape, cfg.bc))
        nt = max(1, min(16, nb))
        fine = torch.empty((nt,) + nf, dtype=torch.float64, device="cuda").normal_()
        coarse = d_psi[:nt]
        tb = (fine.numel() + coarse.numel()) * 8
        ms = _time_stream(torch, stream, lambda: fd.fd_restrict(nf, cfg.bc, 3, fine, d_out[:nt], stream), 10, 2)
        rows["f3_restrict"] = entry(ms, tb, what="order p = 3, %s -> %s, %d arrays" % (nf, cfg.shape, nt))
        ms = _time_stream(torch, stream, lambda: fd.fd_interpolate(nf, cfg.bc, 3, coarse, fine, stream), 10, 2)
        rows["f3_interpolate"] = entry(ms, tb, what="order p = 3, %s -> %s, %d arrays" % (cfg.shape, nf, nt))
        del fine
        # one multigrid V-cycle on this grid (2 + 2 sweeps per level, 8 on the coarsest, p = 3)
        mg = fd.fd_mg_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, 3, 16, nt, torch.cuda.current_device())
        nlev = fd.fd_mg_levels(mg)
        rhs = torch.empty((nt,) + cfg.shape, dtype=torch.float64, device="cuda").normal_()
        rhs -= rhs.mean(dim=(1, 2, 3), keepdim=True)
        phi = torch.zeros_like(rhs)
        ms = _time_stream(torch, stream, lambda: fd.fd_mg_vcycle(mg, phi, rhs, 2, 2, 8, 2.0 / 3.0, stream), 10, 2)
        # per fine-level point: 4 sweeps x 24 B + residual 24 + restrict 9 + interpolate 9 + add 24;
        # levels shrink by 8; the coarsest level does 8 sweeps
        pts = [P / 8 ** l for l in range(nlev)]
        vb = nt * (sum(p_ * (4 * 24 + 66) for p_ in pts[:-1]) + pts[-1] * 8 * 24)
        rows["f3_vcycle"] = entry(ms, vb, what="multigrid V-cycle, %d levels, %d right-hand sides, "
                                                "2 + 2 Jacobi sweeps per level, p = 3" % (nlev, nt))
        fd.fd_mg_destroy(mg)
        del rhs, phi
    # f1: the other stencil orders, single precision and the real zone-boundary point on this grid
    for tag, nn_, dt, kvec in (("f1_nn4", 4, None, None), ("f1_nn6", 6, None, None),
                               ("f1_single_precision", cfg.nn, "f32", None),
                               ("f1_real_k_half", cfg.nn, None, (0.5, 0.5, 0.5))):
        if kvec is not None and (cfg.complex or not all(cfg.bc)):
            continue
        if dt == "f32":
            dtype = fd.FD_C64 if cfg.complex else fd.FD_F32
            x = d_psi.to(torch.complex64 if cfg.complex else torch.float32)
            vv = d_v.to(torch.float32)
        else:
            dtype = fd.FD_C128 if cfg.complex else fd.FD_F64
            x, vv = d_psi, d_v
        kk = kvec if kvec is not None else (cfg.k if cfg.complex else None)
        pl = fd.fd_create(cfg.shape, cfg.h, nn_, cfg.bc, kk, dtype, torch.cuda.current_device())
        y = torch.empty_like(x)
        ms = _time_stream(torch, stream, lambda: fd.fd_apply_hamiltonian(pl, x, vv, y, stream), 20, 3)
        nbytes = 2 * x.numel() * x.element_size() + vv.numel() * vv.element_size()
        # the timed launches left y = H x: sampled points of every band against the oracle
        par = sampled_parity(torch, fd, cfg.shape, cfg.h, nn_, cfg.bc, kk, pl, x,
                             vv.to(torch.float64).cpu().numpy(), y, rel=2e-6 if dt == "f32" else 1e-12,
                             seed=cfg.seed + nn_)
        rows[tag] = entry(ms, nbytes, Gpoint_band_per_s=nb * P / (ms * 1e-3) / 1e9,
                          kernel=_kernel_name(fd, pl, nb), parity=par,
                          what="H psi, nn = %d, %s%s" % (nn_, "fp32" if dt else "fp64",
                                                        ", float64 at k = (1/2,1/2,1/2)" if kvec else ""))
        fd.fd_destroy(pl)
        del y
        if dt == "f32":
            del x, vv
    # PAW non-local term: ~1 atom per (9 A)^3 ... synthetic set of 128 atoms x (13 | 11) functions
    paw = W.make_paw(cfg, 128, nproj=13, radius_angstrom=1.1)
    pw = fd.fd_paw_create(plan, paw.box_start, paw.box_size, paw.nproj, paw.proj, paw.dmat, None)
    coef = torch.empty((nb, paw.ntot), dtype=d_psi.dtype, device="cuda")
    box_pts = int(np.prod(paw.box_size, axis=1).sum())
    ms = _time_stream(torch, stream, lambda: fd.fd_paw_add_nonlocal(plan, pw, d_psi, d_out, coef, stream), 10, 2)
    rows["f4_paw_nonlocal"] = entry(ms, 3 * box_pts * E * nb + paw.proj.size * 8,
                                    what="128 atoms, %d projector functions, %d box points: gather psi, "
                                         "read-modify-write out over the boxes" % (paw.ntot, box_pts))
    ms = _time_stream(torch, stream, lambda: fd.fd_apply_hamiltonian_paw(plan, pw, d_psi, d_v, d_out, coef, stream), 10, 2)
    # the timed launches left d_out = H~ psi~: two whole bands against the oracle (stencil + v_eff +
    # non-local term), point by point within 1e-12 x (north_star bound + sum of |terms| of the PAW sum)
    from oracle import fd_oracle
    kk = cfg.k if cfg.complex else None
    sel = sorted({0, nb - 1})
    xs = d_psi[sel].cpu().numpy()
    v_host = d_v.cpu().numpy()
    want = fd_oracle.apply(cfg.shape, cfg.h, cfg.nn, cfg.bc, kk, xs, v_host)
    want = fd_oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, kk, xs, paw.box_start, paw.box_size, paw.nproj,
                               paw.proj, paw.dmat, out=want)
    bound = fd_oracle.paw_apply(cfg.shape, cfg.h, cfg.bc, None, np.abs(xs), paw.box_start, paw.box_size,
                                paw.nproj, np.abs(paw.proj), np.abs(paw.dmat))
    wts = fd.fd_plan_get_weights(plan, cfg.nn)
    S = sum(abs(r[0]) + 2.0 * sum(abs(t) for t in r[1:]) for r in wts)
    tol = 1e-12 * (float(np.abs(xs).max()) * S + float(np.abs(v_host[None] * xs).max()) + bound)
    worst = float(np.max(np.abs(d_out[sel].cpu().numpy() - want) / tol))
    rows["f4_full_paw_hamiltonian"] = entry(ms, cfg.min_bytes + 3 * box_pts * E * nb + paw.proj.size * 8,
                                            what="Eq. 6 complete: stencil + v_eff + non-local term",
                                            parity={"max_err_over_tol": worst, "ok": bool(worst <= 1.0),
                                                    "bands": sel, "points": int(want.size)})
    fd.fd_paw_destroy(pw)
    return rows


def other_workload(torch, W, fd, name, local, peak, steps):
    """ms / value / roofline fraction of another BASELINE config (cfg1, 2: also the rotating-buffer
    'cold' timing SURVEY 8(d) asks for, since they are L2-resident / launch-bound)."""
    cfg = _cfg(name)
    d_psi, d_v, _ = _device_inputs(torch, W, cfg)
    d_out = torch.empty_like(d_psi)
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None,
                        fd.FD_C128 if cfg.complex else fd.FD_F64, local)
    stream = torch.cuda.Stream()
    sampler = ClockSampler(local)
    sampler.start()
    ms = _time_stream(torch, stream, lambda: fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out, stream),
                      steps, 5)
    clocks = sampler.stop()
    units = cfg.npoints * cfg.nbands
    gbs = cfg.min_bytes / (ms * 1e-3) / 1e9
    ent = {"workload": cfg.name, "kernel": _kernel_name(fd, plan, cfg.nbands), "ms": ms,
           "value": units / (ms * 1e-3) / 1e9, "unit": UNIT, "algorithmic_GBps": gbs,
           "frac": gbs / peak, "traffic": ncu_traffic(cfg.name), "clocks": clocks, "steps": steps}
    set_bytes = 2 * d_psi.numel() * d_psi.element_size()
    if set_bytes < (256 << 20):
        # L2-resident: the hot figure above is not an HBM fraction; rotate through buffer sets
        # totalling > 2x the 126 MB L2 so that every apply finds its inputs cold
        nsets = min(400, (256 << 20) // set_bytes + 2)
        sets = [(d_psi.clone(), torch.empty_like(d_out)) for _ in range(nsets)]
        it = {"i": 0}

        def cold():
            a, b = sets[it["i"] % nsets]
            it["i"] += 1
            fd.fd_apply_hamiltonian(plan, a, d_v, b, stream)
        ms_cold = _time_stream(torch, stream, cold, max(steps, 2 * nsets), nsets)
        ent.update({"note": "L2-resident / launch-bound: `frac` of the hot figure is not an HBM fraction",
                    "ms_cold": ms_cold, "value_cold": units / (ms_cold * 1e-3) / 1e9,
                    "frac_cold": cfg.min_bytes / (ms_cold * 1e-3) / 1e9 / peak,
                    "cold": "%d rotating psi/out sets (%.0f MB > 2x L2)" % (nsets, nsets * set_bytes / 1e6)})
        del sets
    fd.fd_destroy(plan)
    return ent


def run_ours(args):
    import torch
    import workloads as W
    import paper_2310_14776_b200 as fd
    from paper_2310_14776_b200 import build as fd_build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libfdham has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        fd_build.build()
    if dist is not None:
        dist.barrier()
    fd.load_library()

    cfg = _cfg(args.workload)
    tdt = torch.complex128 if cfg.complex else torch.float64
    d_psi, d_v, v_host = _device_inputs(torch, W, cfg)
    d_out = torch.empty_like(d_psi)
    plan = fd.fd_create(cfg.shape, cfg.h, cfg.nn, cfg.bc, cfg.k if cfg.complex else None,
                        fd.FD_C128 if cfg.complex else fd.FD_F64, local)
    kernel = _kernel_name(fd, plan, cfg.nbands)
    stream = torch.cuda.Stream()

    def sync_all():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out, stream)
    sync_all()
    sampler = ClockSampler(local)
    l0 = fd.fd_plan_launches(plan)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(args.steps):
            fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out, stream)
        e1.record(stream)
    sync_all()
    clocks = sampler.stop()
    launches = fd.fd_plan_launches(plan) - l0
    ms_local = e0.elapsed_time(e1) / args.steps

    def reduce_max(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    units = cfg.npoints * cfg.nbands
    value, ms_step = aggregate(ms_local, units, world, reduce_max)
    peak, peak_src = _measured_peak_gbs()

    # ---- sustained: the same apply held for >= args.sustain_seconds (own clock record) ---------
    sustained = None
    if args.sustain_seconds > 0:
        n_s = max(args.steps, int(args.sustain_seconds * 1e3 / ms_local) + 1)
        s_sampler = ClockSampler(local)
        s_sampler.start()
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(n_s):
                fd.fd_apply_hamiltonian(plan, d_psi, d_v, d_out, stream)
            e1.record(stream)
        sync_all()
        s_clocks = s_sampler.stop()
        s_ms = reduce_max(e0.elapsed_time(e1) / n_s)
        s_gbs = cfg.min_bytes / (s_ms * 1e-3) / 1e9
        sustained = {"value": world * units / (s_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": s_ms,
                     "steps": n_s, "seconds": n_s * s_ms * 1e-3, "achieved_GBps": s_gbs,
                     "frac": s_gbs / peak, "clocks": s_clocks}

    # ---- end to end: pinned HOST buffers through fd_apply_hamiltonian_host_ws --------------------
    e2e_steps = max(1, min(7, args.steps))
    h_psi = torch.empty(d_psi.shape, dtype=tdt).pin_memory()
    h_psi.copy_(d_psi)
    h_v = torch.from_numpy(v_host).pin_memory()
    h_out = torch.empty(d_psi.shape, dtype=tdt).pin_memory()
    hws = fd.fd_workspace_create(plan, 0)
    fd.fd_apply_hamiltonian_host_ws(plan, hws, h_psi, h_v, h_out)      # warm-up
    sync_all()
    per_step = []
    for _ in range(e2e_steps):
        t0 = time.perf_counter()
        fd.fd_apply_hamiltonian_host_ws(plan, hws, h_psi, h_v, h_out)  # blocks until out is on the host
        per_step.append((time.perf_counter() - t0) * 1e3)
    fd.fd_workspace_destroy(hws)
    # the host side of the box is shared: an occasional call takes 2-3x as long (PCIe / host
    # memory traffic of other tenants), so the median step is reported and the mean kept beside it
    e2e_ms_local = sorted(per_step)[len(per_step) // 2]
    e2e_ms_mean = sum(per_step) / len(per_step)
    e2e_value, _ = aggregate(e2e_ms_local, units, world, reduce_max)
    stride = max(1, cfg.nbands // 16)
    ok = bool(torch.equal(h_out[::stride], d_out[::stride].cpu()))   # host path = device path, bit for bit
    band_bytes = cfg.npoints * cfg.elem_bytes
    e2e = {"value": e2e_value, "unit": UNIT,
           "h2d_bytes_per_step": cfg.nbands * band_bytes + cfg.npoints * 8,
           "d2h_bytes_per_step": cfg.nbands * band_bytes,
           "steps": e2e_steps, "ms_per_step": e2e_ms_local, "ms_per_step_mean": e2e_ms_mean,
           "stat": "median step", "matches_device_path": ok,
           "api": "fd_apply_hamiltonian_host_ws (pinned host buffers, caller-owned workspace, "
                  "3-slot H2D/kernel/D2H ring)"}

    extras = rank == 0 and world == 1 and not args.quick
    parity = rows = peaks = None
    if extras and args.peaks:
        peaks = hardware_peaks(torch, fd, stream, local)
    if extras:
        parity = parity_after_timing(torch, fd, cfg, plan, d_psi, d_v, v_host, h_psi)
    del h_out
    if extras:
        rows = next_rows(torch, W, fd, cfg, plan, d_psi, d_v, d_out, stream, ms_local, peak)
    fd.fd_destroy(plan)
    del d_psi, d_out, d_v, h_psi
    torch.cuda.empty_cache()
    others = None
    if extras and args.workload == DEFAULT_WORKLOAD:
        others = [other_workload(torch, W, fd, n, local, peak, st)
                  for n, st in (("cfg1", 200), ("cfg2", 200), ("cfg4", 50), ("cfg5", 10))]

    if rank == 0:
        achieved = cfg.min_bytes / (ms_local * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": ncu_traffic(cfg.name),
                    "kernel": f"fd_{kernel}_kernel", "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": cfg.min_bytes,
                    "frac_of_nominal_8TBs": achieved / 8000.0,
                    "avg_launch_ms": ms_local, "kernel_sha": kernel_sha()}
        cpu = cpu_oracle_rate(cfg, budget_s=args.cpu_seconds)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128" if cfg.complex else "f64",
            "data": "synthetic",
            "config": config_dict(cfg, world), "kernel": kernel,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "sustained": sustained, "parity": parity,
            "next_rows": rows, "other_workloads": others, "hardware_peaks": peaks,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD,
                    help="cfg1..cfg5 (BASELINE.json configs); default cfg3")
    ap.add_argument("--cpu-seconds", type=float, default=10.0,
                    help="budget of the cpu_baseline leg")
    ap.add_argument("--sustain-seconds", type=float, default=1.0,
                    help="length of the `sustained` leg (0 = skip)")
    ap.add_argument("--peaks", action=argparse.BooleanOptionalAction, default=True,
                    help="measure read / write / copy bandwidth and the DFMA rate (hardware_peaks)")
    ap.add_argument("--quick", action="store_true",
                    help="headline, sustained and e2e only (no parity / next_rows / other_workloads)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
