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
    if (g.nn > 3) return;  // 2 nn + 1 accumulator planes: the register budget ends at nn = 3
    const int halo = 2 * g.nn;
    if (g.n[0] < 8 || g.n[1] < 8 || g.n[2] < 8 || (g.n[2] & 1)) return;
    if (g.n[0] > 65536) return;  // x index + 2 nn in 17 bits of a step-table entry
    c.ty = 4;
    c.tc = 1;
    const int pitch = g.n[2] * (g.cplx ? 16 : 8);
    const int pitchv = g.n[2] * 8;
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

namespace {

FdSweepKernelFn kernel_for(const fd_plan *plan, bool has_v)
{
    const FdGeom &g = plan->g;
    const int rowd = g.n[2] * (g.cplx ? 2 : 1);
    if (!g.cplx) return fd_sweep_pick_real(rowd, has_v, g.nn);
    // which Bloch-phase code the kernel needs: bit 0 = x or y, bit 1 = z
    int ph = 0;
    for (int d = 0; d < 3; ++d)
        if (g.bc[d] && (g.ph_re[d] != 1.0 || g.ph_im[d] != 0.0)) ph |= (d == 2) ? 2 : 1;
    return fd_sweep_pick_cplx(rowd, has_v, ph, g.nn);
}

}  // namespace

// The shared-memory opt-in belongs to the kernel instantiation, not to the plan (plans of different
// shapes share the run-time-pitch instantiations): always the architectural maximum, so that a later
// plan with a smaller footprint never lowers the limit under an earlier one.
cudaError_t fd_sweep_prepare(fd_plan *plan)
{
    for (int has_v = 0; has_v < 2; ++has_v) {
        cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void *>(kernel_for(plan, has_v)),
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             kSmemMax);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t fd_launch_sweep(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                            int64_t nbands, cudaStream_t stream, int *nlaunches)
{
    const FdSweepCfg &c = plan->sweep;
    const FdGeom &g = plan->g;
    const long long band_d = (long long)g.n[0] * g.n[1] * g.n[2] * (g.cplx ? 2 : 1);
    const FdSweepKernelFn kern = kernel_for(plan, v_eff != nullptr);
    // plane indices in the step table have kPlaneBits bits: very large batches go out in several
    // launches
    const int64_t bands_per_launch = (1LL << kPlaneBits) / g.n[0];
    for (int64_t b0 = 0; b0 < nbands; b0 += bands_per_launch) {
        const int64_t nb = (nbands - b0 < bands_per_launch) ? nbands - b0 : bands_per_launch;
        const long long total = (long long)nb * g.n[0];
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
        if (quota < 1) return cudaErrorInvalidConfiguration;
        const long long nteams = (total + quota - 1) / quota;
        const long long nblocks = nteams * c.nytiles;
        if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
        const double *p = static_cast<const double *>(psi) + b0 * band_d;
        double *o = static_cast<double *>(out) + b0 * band_d;
        kern<<<dim3((unsigned)nblocks), dim3((unsigned)(c.threads_wg + kFdSweepProducerThreads)), (size_t)c.smem_bytes,
               stream>>>(
            g, c, p, v_eff, o, total, (int)quota);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
        if (nlaunches) ++*nlaunches;
    }
    return cudaSuccess;
}
