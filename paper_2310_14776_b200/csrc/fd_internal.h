// Internal declarations of libfdham (not part of the C ABI; see include/fdham.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#define FD_MAX_NN 6

// bytes of one element of psi / out
inline int fd_elem_bytes(int cplx, int f32) { return (cplx ? 16 : 8) >> (f32 ? 1 : 0); }

// Plan constants handed to every kernel by value.
struct FdGeom {
    int n[3];                    // nx, ny, nz
    int bc[3];                   // FD_BC_*
    int nn;
    int cplx;                    // 0: real, 1: complex data
    int f32;                     // 0: float64 / complex128, 1: float32 / complex64 (v_eff float32)
    double w[3][FD_MAX_NN + 1];  // w[d][j] = -1/2 c_j / h_d^2
    double wdiag;                // sum_d w[d][0]
    double ph_re[3], ph_im[3];   // exp(+2 pi i k_d): factor when a tap runs past the UPPER end
    double rhs_coef;             // Jacobi sweep only (sweep MODE 2 / generic): factor of the rhs
};

// Limits shared by the sweep kernel (fd_sweep_kernel.cuh) and its host side (fd_sweep.cu)
constexpr int kFdSweepMaxThreads = 384;      // compute threads per CTA (160 registers each)
constexpr int kFdSweepProducerThreads = 128; // + one warpgroup whose first lane issues the TMA loads
constexpr int kFdSweepMaxStages = 8;         // mbarrier slots reserved per ring
constexpr int kFdSweepCtlBytes = 256;        // full[8] + empty[8] mbarriers, 8 election counters, misc
constexpr int kFdSweepSmemMax = 227 * 1024;  // dynamic shared memory per CTA on sm_100
constexpr int kFdSweepPlaneBits = 26;        // bits of a (band, x) plane index in a step-table entry

// Launch description of the sweep kernel, fixed at plan time (tile choice) -- see fd_sweep.cu.
struct FdSweepCfg {
    int supported;     // 0: plan cannot use the sweep kernel
    int ty, tc;        // thread micro tile: ty rows x tc 16-byte chunks
    int lanes;         // threads per row group  (= chunks per row / tc)
    int rowgroups;     // row groups per CTA; tile rows tyc = rowgroups * ty
    int tyc;           // y rows per CTA tile
    int nytiles;       // ceil(ny / tyc)
    int threads;       // compute threads (multiple of 32)
    int threads_wg;    // the same rounded up to whole warpgroups: first thread of the producer group
    int stages;        // smem ring depth
    int zb_bytes;      // zero block at the start of every stage (zero-BC z halo source), else 0
    int v_off;         // offset of the v_eff rows inside a stage
    int stage_bytes;   // bytes per ring stage
    int tab_off;       // offset of the step table in shared memory
    int tab_cap;       // step table capacity (entries of 8 bytes)
    int stage_off;     // offset of stage 0
    int smem_bytes;    // dynamic shared memory per CTA
    int max_teams;     // teams of nytiles CTAs resident at once (one CTA per SM)
    int xchunk;        // 0 = persistent teams, else x planes per team (tuning knob)
    int stages_req;    // 0 = as many ring slots as fit, else an upper bound (tuning knob)
};

struct fd_plan {
    FdGeom g;
    int device;
    int sm_count;
    int kernel;        // FD_KERNEL_GENERIC | FD_KERNEL_SWEEP: family of the plan
    int forced;        // 1: set explicitly (fd_plan_set_kernel / FDHAM_TUNE), no per-batch choice
    FdSweepCfg sweep;
    double h[3];
    double k[3];
    long long launches;  // kernels launched so far (diagnostic)
};

// fd_generic.cu
cudaError_t fd_launch_generic(const fd_plan *plan, const FdGeom &g, int mode, const void *psi,
                              const double *second, void *out, int64_t nbands, cudaStream_t stream);
// fd_aux.cu: streaming helper kernels (two-pass expectation values, residual)
int64_t fd_dot_ws_bytes(const fd_plan *plan, int64_t nbands);
cudaError_t fd_launch_dot(const fd_plan *plan, const void *psi, const void *hpsi, double *eps,
                          double *norm, double *ws, int64_t nbands, cudaStream_t stream,
                          int *nlaunches);
cudaError_t fd_launch_add(double *y, const double *x, long long n, int sm_count, cudaStream_t stream);
cudaError_t fd_launch_residual(const fd_plan *plan, const void *psi, const void *hpsi,
                               const double *eps, const double *norm, void *r, int64_t nbands,
                               cudaStream_t stream);
// Extra arguments of the sweep kernel's EX instantiations (fd_apply_hamiltonian_expect): where the
// per-warp partial sums go.  Entry ((team * maxseg + segment) * nytiles + ytile) * nwarps + warp
// holds the pair (sum conj(psi) H psi, sum |psi|^2) of that warp for that band segment.
struct FdSweepAux {
    double *ws;
    int maxseg;  // band segments a team can touch: quota / nx + 2
};

// fd_sweep_inst_*.cu: instantiations of the sweep kernel template (fd_sweep_kernel.cuh).
// mode: 0 kinetic, 1 + v_eff psi, 2 Jacobi sweep (real, not EX); ex: with the expectation values.
typedef void (*FdSweepKernelFn)(const FdGeom, const FdSweepCfg, const double *, const double *,
                                double *, const long long, const int, const FdSweepAux);
FdSweepKernelFn fd_sweep_pick_real(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_real_ex(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_real_jacobi(int rowd, int nn);
FdSweepKernelFn fd_sweep_pick_real_ph(int mode, int nn);
FdSweepKernelFn fd_sweep_pick_real_hi(int mode, int nn);  // nn = 4..6, float64
FdSweepKernelFn fd_sweep_pick_cplx_hi(int mode, int nn);
FdSweepKernelFn fd_sweep_pick_f32(int cplx, int mode, int nn);  // float32 / complex64, nn = 1..3  // nn = 4..6, complex128 (all phase code)  // float64, Bloch factors -1 (k = 1/2)
FdSweepKernelFn fd_sweep_pick_cplx_ph0(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_cplx_ph1(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_cplx_ph3(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_cplx_ph0_ex(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_cplx_ph1_ex(int rowd, int mode, int nn);
FdSweepKernelFn fd_sweep_pick_cplx_ph3_ex(int rowd, int mode, int nn);
inline FdSweepKernelFn fd_sweep_pick_cplx(int rowd, int mode, int ph, int nn, int ex)
{
    if (ex) {
        if (ph == 0) return fd_sweep_pick_cplx_ph0_ex(rowd, mode, nn);
        if (ph == 1) return fd_sweep_pick_cplx_ph1_ex(rowd, mode, nn);
        return fd_sweep_pick_cplx_ph3_ex(rowd, mode, nn);
    }
    if (ph == 0) return fd_sweep_pick_cplx_ph0(rowd, mode, nn);
    if (ph == 1) return fd_sweep_pick_cplx_ph1(rowd, mode, nn);
    return fd_sweep_pick_cplx_ph3(rowd, mode, nn);
}
// fd_api.cu: integer value of `key` in the FDHAM_TUNE environment variable (0 if absent)
int fd_tune_value(const char *key);
// fd_sweep.cu
void fd_sweep_configure(fd_plan *plan, int tyc_override, int xchunk_override, int stages_override);
cudaError_t fd_sweep_prepare(fd_plan *plan);  // shared-memory opt-in of the plan's kernels
bool fd_plan_real_phase(const fd_plan *plan);      // float64 plan with a Bloch factor -1
bool fd_sweep_expect_fused(const fd_plan *plan);  // else: two passes (sweep, then fd_launch_dot)
int64_t fd_sweep_expect_ws_bytes(const fd_plan *plan, int64_t nbands);
cudaError_t fd_launch_sweep(const fd_plan *plan, const FdGeom &g, int mode, const void *psi,
                            const double *second, void *out, int64_t nbands, double *eps,
                            double *norm, double *ws, cudaStream_t stream, int *nlaunches);
// fd_transfer.cu: restriction (interp = 0) / interpolation (interp = 1) between the fine grid
// `shape_fine` and its coarse grid; returns an fd_status value
int fd_transfer_run(int interp, const int32_t shape_fine[3], const int32_t bc[3], int p,
                    const double *src, double *dst, int64_t nbands, cudaStream_t stream);
int fd_transfer_check(int interp, const int32_t shape_fine[3], const int32_t bc[3], int p,
                      int64_t nbands);  // same status without launching (tile / shared-memory fit)
// fd_paw.cu: PAW non-local term
struct fd_paw;
int fd_paw_build(fd_paw **out, const fd_plan *plan, int natoms, const int32_t *box_start,
                 const int32_t *box_size, const int32_t *nproj, const double *proj_host,
                 const double *dh_host, const double *ds_host);  // returns an fd_status value
void fd_paw_free(fd_paw *w);
int fd_paw_ntot(const fd_paw *w);
int fd_paw_has(const fd_paw *w, int which);            // which: 0 = Delta H, 1 = Delta S
int fd_paw_matches(const fd_paw *w, const fd_plan *plan);
cudaError_t fd_paw_launch_project(const fd_paw *w, const void *psi, void *coef, int64_t nbands,
                                  cudaStream_t stream, int *nlaunches);
cudaError_t fd_paw_launch_expect(const fd_paw *w, int which, const void *coef, double *out, int64_t nbands,
                                 cudaStream_t stream, int *nlaunches);
cudaError_t fd_paw_launch_add(const fd_paw *w, int which, const void *coef, void *out, int64_t nbands,
                              cudaStream_t stream, int *nlaunches);
// fd_peaks.cu: bandwidth / DFMA micro-benchmarks (bench.py --peaks)
cudaError_t fd_peak_launch(int kind, double *a, double *b, long long n, int blocks, int sm_count,
                           cudaStream_t stream);
