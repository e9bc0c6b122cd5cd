// Host side of the sweep kernel: tile / ring configuration at plan time and the launch.  The
// kernel itself is the template in fd_sweep_kernel.cuh, instantiated in fd_sweep_inst_*.cu.
#include "fd_internal.h"

namespace {

constexpr int kMaxThreads = kFdSweepMaxThreads;
constexpr int kCtlBytes = kFdSweepCtlBytes;
constexpr int kSmemMax = kFdSweepSmemMax;
constexpr int kPlaneBits = kFdSweepPlaneBits;

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

}  // namespace

void fd_sweep_configure(fd_plan *plan, int tyc_override, int xchunk_override, int stages_override)
{
    FdSweepCfg &c = plan->sweep;
    const FdGeom &g = plan->g;
    c = FdSweepCfg{};
    c.xchunk = xchunk_override;  // 0 = automatic (persistent teams), else planes per team
    c.stages_req = stages_override;
    if (g.nn > 3 && fd_plan_real_phase(plan)) return;  // no sign-flip instantiation for nn > 3
    const int halo = 2 * g.nn;
    if (g.n[0] < 8 || g.n[1] < 8 || g.n[2] < 8 || (g.n[2] & 1)) return;
    if (g.f32 && (g.nn > 3 || fd_plan_real_phase(plan))) return;  // float32: nn <= 3, no sign flips
    if (g.f32 && !g.cplx && (g.n[2] & 3)) return;                  // rows are whole 16-byte chunks
    if (g.n[0] > 65536) return;  // x index + 2 nn in 17 bits of a step-table entry
    // 2 nn + 1 accumulator planes x ty rows per thread must fit the registers (must match the kernel)
    c.ty = g.nn <= 3 ? 4 : ((g.nn == 4 && !g.cplx) ? 3 : 2);
    c.tc = 1;
    const int pitch = g.n[2] * fd_elem_bytes(g.cplx, g.f32);
    const int pitchv = g.n[2] * (g.f32 ? 4 : 8);
    c.lanes = (pitch / 16) / c.tc;
    if (c.lanes > kMaxThreads) return;
    c.zb_bytes = (g.bc[2] == 0) ? (c.ty * pitch + 127) / 128 * 128 : 0;
    const int max_rg = kMaxThreads / c.lanes;
    auto stage_bytes = [&](int tyc) {
        return (c.zb_bytes + (tyc + halo) * pitch + tyc * pitchv + 127) / 128 * 128;
    };
    // fewest y tiles whose stage fits a ring of >= 3 slots beside a 4 KiB (512-step) table
    int tyc = 0;
    const int first = ceil_div(g.n[1], max_rg * c.ty);
    for (int ntiles = first; ntiles <= g.n[1]; ++ntiles) {
        const int t = ceil_div(ceil_div(g.n[1], ntiles), c.ty) * c.ty;
        if (3 * stage_bytes(t) + kCtlBytes + 4096 <= kSmemMax) {
            tyc = t;
            break;
        }
        if (t == c.ty) break;
    }
    if (tyc_override > 0) {
        tyc = ceil_div(tyc_override, c.ty) * c.ty;
        if (tyc > max_rg * c.ty) tyc = max_rg * c.ty;
        if (2 * stage_bytes(tyc) + kCtlBytes + 4096 > kSmemMax) return;
    }
    if (tyc <= 0) return;
    c.tyc = tyc;
    c.rowgroups = tyc / c.ty;
    c.nytiles = ceil_div(g.n[1], tyc);
    c.threads = ceil_div(c.rowgroups * c.lanes, 32) * 32;
    c.threads_wg = ceil_div(c.threads, 128) * 128;
    c.stage_bytes = stage_bytes(tyc);
    c.v_off = c.zb_bytes + (tyc + halo) * pitch;
    int tab_bytes = 16384;
    int stages = (kSmemMax - kCtlBytes - tab_bytes) / c.stage_bytes;
    if (stages < 3) {
        tab_bytes = 4096;
        stages = (kSmemMax - kCtlBytes - tab_bytes) / c.stage_bytes;
    }
    if (stages < 2) return;
    if (stages > 6) stages = 6;
    if (stages_override >= 2 && stages_override < stages) stages = stages_override;
    c.stages = stages;
    tab_bytes = (kSmemMax - kCtlBytes - stages * c.stage_bytes) / 128 * 128;
    if (tab_bytes > 65536) tab_bytes = 65536;
    c.tab_off = kCtlBytes;
    c.tab_cap = tab_bytes / 8;
    c.stage_off = kCtlBytes + tab_bytes;
    c.smem_bytes = c.stage_off + stages * c.stage_bytes;
    c.max_teams = plan->sm_count / c.nytiles > 0 ? plan->sm_count / c.nytiles : 1;
    if (c.smem_bytes > kSmemMax || c.threads > kMaxThreads) return;
    c.supported = 1;
}

bool fd_plan_real_phase(const fd_plan *plan)
{
    const FdGeom &g = plan->g;
    if (g.cplx) return false;
    for (int d = 0; d < 3; ++d)
        if (g.bc[d] && g.ph_re[d] != 1.0) return true;
    return false;
}

namespace {

FdSweepKernelFn kernel_for(const fd_plan *plan, int mode, bool ex)
{
    const FdGeom &g = plan->g;
    const int rowd = g.n[2] * (g.cplx ? 2 : 1);
    if (g.f32) return (mode == 2 || ex) ? nullptr : fd_sweep_pick_f32(g.cplx, mode, g.nn);
    if (g.nn > 3) {  // plain applies only; expectation values and Jacobi fall back (fd_api.cu)
        if (mode == 2 || ex) return nullptr;
        return g.cplx ? fd_sweep_pick_cplx_hi(mode, g.nn) : fd_sweep_pick_real_hi(mode, g.nn);
    }
    if (!g.cplx) {
        if (fd_plan_real_phase(plan))  // plain applies only; the other forms fall back (fd_api.cu)
            return (mode == 2 || ex) ? nullptr : fd_sweep_pick_real_ph(mode, g.nn);
        if (mode == 2) return fd_sweep_pick_real_jacobi(rowd, g.nn);
        return ex ? fd_sweep_pick_real_ex(rowd, mode, g.nn) : fd_sweep_pick_real(rowd, mode, g.nn);
    }
    if (mode == 2) return nullptr;  // the Jacobi sweep is real only
    // which Bloch-phase code the kernel needs: bit 0 = x or y, bit 1 = z
    int ph = 0;
    for (int d = 0; d < 3; ++d)
        if (g.bc[d] && (g.ph_re[d] != 1.0 || g.ph_im[d] != 0.0)) ph |= (d == 2) ? 2 : 1;
    return fd_sweep_pick_cplx(rowd, mode, ph, g.nn, ex);
}

// (band, x) planes per team for a launch of `total` planes (persistent teams unless the xchunk
// tuning knob is set), capped by the step-table capacity.  0 = cannot launch.
long long team_quota(const fd_plan *plan, long long total)
{
    const FdSweepCfg &c = plan->sweep;
    const FdGeom &g = plan->g;
    long long quota;
    if (c.xchunk > 0) {
        quota = c.xchunk;
    } else {
        quota = (total + c.max_teams - 1) / c.max_teams;
        const int min_quota = g.n[0] < 16 ? g.n[0] : 16;  // below this the halo planes dominate
        if (quota < min_quota) quota = min_quota;
    }
    // the team's steps (quota + 2 nn per band touched, + 1 prefetched entry) must fit the table
    const long long quota_cap =
        ((long long)(c.tab_cap - 4 * g.nn - 1) * g.n[0]) / (g.n[0] + 2 * g.nn);
    if (quota > quota_cap) quota = quota_cap;
    return quota < 1 ? 0 : quota;
}

// plane indices in the step table have kPlaneBits bits: very large batches go out in several launches
int64_t bands_per_launch(const fd_plan *plan) { return (1LL << kPlaneBits) / plan->g.n[0]; }

// Sums the per-warp partials of the EX sweep kernel (layout: FdSweepAux) band by band in a fixed
// order.  One warp per band: lane l adds the entries l, l + 32, ... of each team's block in order,
// then a fixed shuffle tree: the same association every run, no atomics.
__global__ void fd_expect_finalize_sweep(const double *__restrict__ ws, double *__restrict__ eps,
                                         double *__restrict__ norm, int nbands, int nx,
                                         long long quota, int maxseg, int nytiles, int nwarps)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (b >= nbands) return;
    const long long l_lo = (long long)b * nx, l_hi = l_lo + nx - 1;
    double e = 0.0, n = 0.0;
    for (long long t = l_lo / quota; t <= l_hi / quota; ++t) {
        const long long seg = b - (t * quota) / nx;  // this band's segment index inside team t
        const double2 *w = reinterpret_cast<const double2 *>(ws) +
                           ((t * maxseg + seg) * nytiles) * (long long)nwarps;
        for (int i = lane; i < nytiles * nwarps; i += 32) {
            const double2 v = w[i];
            e += v.x;
            n += v.y;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_xor_sync(0xffffffffu, e, o);
        n += __shfl_xor_sync(0xffffffffu, n, o);
    }
    if (lane == 0) {
        eps[b] = e;
        norm[b] = n;
    }
}

}  // namespace

// The shared-memory opt-in belongs to the kernel instantiation, not to the plan (plans of different
// shapes share the run-time-pitch instantiations): always the architectural maximum, so that a later
// plan with a smaller footprint never lowers the limit under an earlier one.
cudaError_t fd_sweep_prepare(fd_plan *plan)
{
    for (int mode = 0; mode < 3; ++mode)
        for (int ex = 0; ex < 2; ++ex) {
            if (mode == 2 && (ex || plan->g.cplx)) continue;
            const FdSweepKernelFn fn = kernel_for(plan, mode, ex != 0);
            if (!fn) continue;  // form not on the sweep kernel for this plan
            cudaError_t e = cudaFuncSetAttribute(
                reinterpret_cast<const void *>(fn),
                cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
            if (e != cudaSuccess) return e;
        }
    return cudaSuccess;
}

// Plans on the sweep kernel take the expectation values from the same pass; the others take the
// two-pass form (fd_aux.cu).
bool fd_sweep_expect_fused(const fd_plan *plan)
{
    return plan->sweep.supported != 0 && !fd_plan_real_phase(plan) && plan->g.nn <= 3 && !plan->g.f32;
}

// Bytes of workspace fd_launch_sweep needs for the expectation values of an `nbands` batch.
int64_t fd_sweep_expect_ws_bytes(const fd_plan *plan, int64_t nbands)
{
    const FdSweepCfg &c = plan->sweep;
    const int64_t bpl = bands_per_launch(plan);
    const int64_t nb = nbands < bpl ? nbands : bpl;
    const long long total = (long long)nb * plan->g.n[0];
    const long long quota = team_quota(plan, total);
    if (quota < 1) return 0;
    const long long nteams = (total + quota - 1) / quota;
    const long long maxseg = quota / plan->g.n[0] + 2;
    return (int64_t)(16 * nteams * maxseg * c.nytiles * (c.threads / 32));
}

// mode 0: out = T psi; 1: + second (v_eff[nx,ny,nz]) psi; 2: Jacobi form with second = rhs
// [nbands,nx,ny,nz] (g carries the pre-scaled weights).  eps != nullptr: also the expectation values
// (partials in ws, fd_sweep_expect_ws_bytes), summed by a second small launch.
cudaError_t fd_launch_sweep(const fd_plan *plan, const FdGeom &g, int mode, const void *psi,
                            const double *second, void *out, int64_t nbands, double *eps,
                            double *norm, double *ws, cudaStream_t stream, int *nlaunches)
{
    const FdSweepCfg &c = plan->sweep;
    // 8-byte units per band (the kernel addresses psi / out in 8-byte units for every dtype)
    const long long band_d = (long long)g.n[0] * g.n[1] * g.n[2] * fd_elem_bytes(g.cplx, g.f32) / 8;
    const bool ex = eps != nullptr;
    const FdSweepKernelFn kern = kernel_for(plan, mode, ex);
    if (!kern) return cudaErrorInvalidValue;
    const int64_t bpl = bands_per_launch(plan);
    for (int64_t b0 = 0; b0 < nbands; b0 += bpl) {
        const int64_t nb = (nbands - b0 < bpl) ? nbands - b0 : bpl;
        const long long total = (long long)nb * g.n[0];
        const long long quota = team_quota(plan, total);
        if (quota < 1) return cudaErrorInvalidConfiguration;
        const long long nteams = (total + quota - 1) / quota;
        const long long nblocks = nteams * c.nytiles;
        if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
        const double *p = static_cast<const double *>(psi) + b0 * band_d;
        double *o = static_cast<double *>(out) + b0 * band_d;
        const double *sec = (mode == 2) ? second + b0 * band_d : second;
        FdSweepAux aux;
        aux.ws = ws;
        aux.maxseg = (int)(quota / g.n[0] + 2);
        kern<<<dim3((unsigned)nblocks), dim3((unsigned)(c.threads_wg + kFdSweepProducerThreads)),
               (size_t)c.smem_bytes, stream>>>(g, c, p, sec, o, total, (int)quota, aux);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
        if (nlaunches) ++*nlaunches;
        if (ex) {
            fd_expect_finalize_sweep<<<dim3((unsigned)((nb + 3) / 4)), dim3(128), 0, stream>>>(
                ws, eps + b0, norm + b0, (int)nb, g.n[0], quota, aux.maxseg, c.nytiles,
                c.threads / 32);
            e = cudaPeekAtLastError();
            if (e != cudaSuccess) return e;
            if (nlaunches) ++*nlaunches;
        }
    }
    return cudaSuccess;
}
