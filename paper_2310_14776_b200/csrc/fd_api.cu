// C ABI of libfdham (declared and documented in include/fdham.h): plan construction, argument
// checking, kernel dispatch, and the host-buffer (end-to-end) variant.  No CPU compute path exists
// here on purpose: without a CUDA device every entry point fails with FD_ERR_CUDA.
#include <math.h>
#include <mutex>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "../../include/fdham.h"
#include "fd_internal.h"

namespace {

const double kPi = 3.14159265358979323846264338327950288;

double factorial(int n)
{
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= i;
    return f;
}

// Central 2nd-derivative weights of order 2*nn (reading R1): c_0 = -2 sum 1/j^2,
// c_j = 2 (-1)^(j+1) (nn!)^2 / (j^2 (nn-j)! (nn+j)!).
void stencil_coeffs(int nn, double *c)
{
    double s = 0.0;
    for (int j = 1; j <= nn; ++j) {
        const double sign = (j & 1) ? 1.0 : -1.0;
        c[j] = 2.0 * sign * factorial(nn) * factorial(nn) /
               ((double)j * j * factorial(nn - j) * factorial(nn + j));
        s += 1.0 / ((double)j * j);
    }
    c[0] = -2.0 * s;
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

int check_apply_args(const fd_plan *plan, const void *psi, const double *v_eff, bool need_v,
                     const void *out, int64_t nbands)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!psi || !out || (need_v && !v_eff)) return FD_ERR_INVALID;
    if (((uintptr_t)psi | (uintptr_t)out | (uintptr_t)v_eff) & 15) return FD_ERR_INVALID;
    const size_t P = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2];
    const size_t nb = P * (size_t)nbands * (size_t)fd_elem_bytes(plan->g.cplx, plan->g.f32);
    if (overlaps(out, nb, psi, nb)) return FD_ERR_ALIAS;
    if (v_eff && overlaps(out, nb, v_eff, P * (plan->g.f32 ? 4 : 8))) return FD_ERR_ALIAS;
    return FD_OK;
}

// Kernel family for a batch of `nbands`.  The sweep kernel pays ~1.2 us per x plane of a team's
// share plus 6 halo planes per band segment whatever the grid size, so a batch that is far too
// small to fill the persistent teams goes to the one-thread-per-point kernel (measured on B200:
// 24^3 x 8 bands takes 8 us there against 27 us; 48^3 x 64 bands 115 us against 39 us).
int kernel_for_batch(const fd_plan *plan, int64_t nbands)
{
    if (plan->kernel != FD_KERNEL_SWEEP || plan->forced || plan->g.f32) return plan->kernel;
    const FdGeom &g = plan->g;
    const double units = (double)g.n[0] * g.n[1] * g.n[2] * (double)nbands * (g.cplx ? 2.0 : 1.0);
    const double total = (double)nbands * g.n[0];
    double quota = ceil(total / plan->sweep.max_teams);
    const double min_quota = g.n[0] < 16 ? g.n[0] : 16;
    if (quota < min_quota) quota = min_quota;
    const double nseg = 1.0 + floor(quota / g.n[0]);
    const double t_sweep_us = 5.0 + 1.2 * (quota + 2.0 * g.nn * nseg + 4.0);
    const double t_generic_us = 4.0 + units / 60.0e3;
    return t_generic_us < t_sweep_us ? FD_KERNEL_GENERIC : FD_KERNEL_SWEEP;
}

// The device the plan was built for must be current in the calling thread (the launches below go
// to the current device): FD_ERR_INVALID otherwise, instead of a launch in the wrong context.
int check_device(const fd_plan *plan)
{
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    return cur == plan->device ? FD_OK : FD_ERR_INVALID;
}

// mode 0: T psi, 1: + v_eff psi, 2: Jacobi form (g = pre-scaled copy of the plan's geometry, second =
// rhs).  eps != nullptr: also the expectation values (fused in the sweep kernel, or a second pass
// over the stored H psi when the batch runs on the generic kernel); ws as fd_expect_workspace_bytes.
int apply_device(const fd_plan *plan, const FdGeom &g, int mode, const void *psi, const double *second,
                 void *out, int64_t nbands, double *eps, double *norm, double *ws,
                 cudaStream_t stream)
{
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;
    cudaError_t e;
    int n = 0;
    // float64 plans with a Bloch factor -1 and nn > 3 have no Jacobi instantiation of the sweep kernel
    const bool sweep_ok = !(mode == 2 && (fd_plan_real_phase(plan) || plan->g.nn > 3));
    if (sweep_ok && kernel_for_batch(plan, nbands) == FD_KERNEL_SWEEP) {
        const bool fused = eps && fd_sweep_expect_fused(plan);
        e = fd_launch_sweep(plan, g, mode, psi, second, out, nbands, fused ? eps : nullptr, norm, ws,
                            stream, &n);
        if (e == cudaSuccess && eps && !fused)
            e = fd_launch_dot(plan, psi, out, eps, norm, ws, nbands, stream, &n);
    } else {
        e = fd_launch_generic(plan, g, mode, psi, second, out, nbands, stream);
        n = 1;
        if (e == cudaSuccess && eps) e = fd_launch_dot(plan, psi, out, eps, norm, ws, nbands, stream, &n);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    __atomic_add_fetch(&const_cast<fd_plan *>(plan)->launches, (long long)n, __ATOMIC_RELAXED);
    return FD_OK;
}

}  // namespace

// "tyc=24,xchunk=32,kernel=1": debugging / tuning knob read once at fd_create.
int fd_tune_value(const char *key)
{
    const char *env = getenv("FDHAM_TUNE");
    if (!env) return 0;
    const size_t kl = strlen(key);
    for (const char *p = env; *p;) {
        if (!strncmp(p, key, kl) && p[kl] == '=') return atoi(p + kl + 1);
        p = strchr(p, ',');
        if (!p) break;
        ++p;
    }
    return 0;
}

namespace {
int tune_value(const char *key) { return fd_tune_value(key); }
}  // namespace

extern "C" {

int fd_create(fd_plan **plan_out, const int32_t shape[3], const double h[3], int32_t nn,
              const int32_t bc[3], const double k_reduced[3], int32_t dtype, int32_t device)
{
    return fd_create_scaled(plan_out, shape, h, nn, bc, k_reduced, dtype, device, -0.5);
}

int fd_create_scaled(fd_plan **plan_out, const int32_t shape[3], const double h[3], int32_t nn,
                     const int32_t bc[3], const double k_reduced[3], int32_t dtype, int32_t device,
                     double scale)
{
    if (!plan_out || !shape || !h || !bc || !isfinite(scale)) return FD_ERR_INVALID;
    if (nn < 1 || nn > FD_MAX_NN) return FD_ERR_INVALID;
    if (dtype != FD_F64 && dtype != FD_C128 && dtype != FD_F32 && dtype != FD_C64) return FD_ERR_INVALID;
    const bool real_dtype = (dtype == FD_F64 || dtype == FD_F32);
    for (int d = 0; d < 3; ++d) {
        if (shape[d] < 1) return FD_ERR_INVALID;
        if (!(h[d] > 0.0) || !isfinite(h[d])) return FD_ERR_INVALID;
        if (bc[d] != FD_BC_ZERO && bc[d] != FD_BC_PERIODIC) return FD_ERR_INVALID;
        if (bc[d] == FD_BC_PERIODIC && shape[d] < nn) return FD_ERR_INVALID;
        const double kd = k_reduced ? k_reduced[d] : 0.0;
        if (!isfinite(kd)) return FD_ERR_INVALID;
        if (kd != 0.0 && bc[d] == FD_BC_ZERO) return FD_ERR_INVALID;
        // real data: the Bloch factor exp(2 pi i k_d) must be real: +-1, i.e. 2 k_d an integer
        if (real_dtype && 2.0 * kd != rint(2.0 * kd)) return FD_ERR_INVALID;
    }
    if ((long long)shape[0] * shape[1] * shape[2] > (1LL << 40)) return FD_ERR_INVALID;

    // shapes the one-thread-per-point kernel cannot launch (its grid is (nz/64, ny/4, nx * groups))
    if (shape[0] > 65535 || (shape[1] + 3) / 4 > 65535) return FD_ERR_UNSUPPORTED;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    // the plan is built with `device` current; the caller's current device is restored on return
    int prev_device = -1;
    if (cudaGetDevice(&prev_device) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    struct DeviceGuard {
        int prev, now;
        ~DeviceGuard() { if (prev >= 0 && prev != now) cudaSetDevice(prev); }
    } guard{prev_device, device};
    if (prev_device != device && cudaSetDevice(device) != cudaSuccess) return FD_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return FD_ERR_CUDA;

    fd_plan *p = new (std::nothrow) fd_plan();
    if (!p) return FD_ERR_NOMEM;
    memset(p, 0, sizeof(*p));
    p->device = device;
    p->sm_count = prop.multiProcessorCount;
    FdGeom &g = p->g;
    g.nn = nn;
    g.cplx = (dtype == FD_C128 || dtype == FD_C64);
    g.f32 = (dtype == FD_F32 || dtype == FD_C64);
    double c[FD_MAX_NN + 1];
    stencil_coeffs(nn, c);
    g.wdiag = 0.0;
    for (int d = 0; d < 3; ++d) {
        g.n[d] = shape[d];
        g.bc[d] = bc[d];
        p->h[d] = h[d];
        p->k[d] = k_reduced ? k_reduced[d] : 0.0;
        for (int j = 0; j <= nn; ++j) g.w[d][j] = (scale * c[j]) / (h[d] * h[d]);
        g.wdiag += g.w[d][0];
        // exp(+2 pi i k_d); exact 1 at Gamma so real-valued data stays phase free
        if (p->k[d] == 0.0) {
            g.ph_re[d] = 1.0;
            g.ph_im[d] = 0.0;
        } else if (2.0 * p->k[d] == rint(2.0 * p->k[d])) {
            // integer or half-integer k: exactly +1 / -1 (float64 plans rely on it)
            g.ph_re[d] = (fmod(fabs(2.0 * p->k[d]), 2.0) == 1.0) ? -1.0 : 1.0;
            g.ph_im[d] = 0.0;
        } else {
            g.ph_re[d] = cos(2.0 * kPi * p->k[d]);
            g.ph_im[d] = sin(2.0 * kPi * p->k[d]);
        }
    }

    fd_sweep_configure(p, tune_value("tyc"), tune_value("xchunk"), tune_value("stages"));
    p->kernel = p->sweep.supported ? FD_KERNEL_SWEEP : FD_KERNEL_GENERIC;
    if (tune_value("kernel") == FD_KERNEL_GENERIC) p->kernel = FD_KERNEL_GENERIC;
    if (tune_value("kernel") != 0) p->forced = 1;

    if (p->sweep.supported && fd_sweep_prepare(p) != cudaSuccess) {
        cudaGetLastError();
        delete p;
        return FD_ERR_CUDA;
    }
    *plan_out = p;
    return FD_OK;
}

int fd_apply_kinetic(const fd_plan *plan, const void *psi, void *out, int64_t nbands,
                     void *cuda_stream)
{
    const int rc = check_apply_args(plan, psi, nullptr, false, out, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    return apply_device(plan, plan->g, 0, psi, nullptr, out, nbands, nullptr, nullptr, nullptr,
                        (cudaStream_t)cuda_stream);
}

int fd_apply_hamiltonian(const fd_plan *plan, const void *psi, const void *v_eff_any, void *out,
                         int64_t nbands, void *cuda_stream)
{
    // float for single-precision plans (the kernels reinterpret it), double otherwise
    const double *v_eff = static_cast<const double *>(v_eff_any);
    const int rc = check_apply_args(plan, psi, v_eff, true, out, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    return apply_device(plan, plan->g, 1, psi, v_eff, out, nbands, nullptr, nullptr, nullptr,
                        (cudaStream_t)cuda_stream);
}

// Device staging buffers and streams of the host-buffer applies: created once, reused by every
// fd_apply_hamiltonian_host_ws call (one call at a time per workspace).
struct fd_workspace {
    static const int kSlots = 3;
    int device;
    size_t npoints;       // grid points of the plan it was created for
    size_t band_bytes;
    int64_t chunk;        // bands per ring slot
    double *v_dev;
    char *in_dev[kSlots], *out_dev[kSlots];
    cudaStream_t st[kSlots];
    cudaEvent_t v_ready;
};

int fd_workspace_destroy(fd_workspace *ws)
{
    if (!ws) return FD_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != ws->device) cudaSetDevice(ws->device);
    if (ws->v_ready) cudaEventDestroy(ws->v_ready);
    for (int i = 0; i < fd_workspace::kSlots; ++i) {
        if (ws->st[i]) cudaStreamDestroy(ws->st[i]);
        if (ws->in_dev[i]) cudaFree(ws->in_dev[i]);
        if (ws->out_dev[i]) cudaFree(ws->out_dev[i]);
    }
    if (ws->v_dev) cudaFree(ws->v_dev);
    if (prev >= 0 && prev != ws->device) cudaSetDevice(prev);
    cudaGetLastError();
    delete ws;
    return FD_OK;
}

int fd_workspace_create(fd_workspace **ws_out, const fd_plan *plan, int64_t chunk_bytes)
{
    if (!ws_out || !plan || chunk_bytes < 0) return FD_ERR_INVALID;
    if (plan->g.f32) return FD_ERR_UNSUPPORTED;
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;
    fd_workspace *w = new (std::nothrow) fd_workspace();
    if (!w) return FD_ERR_NOMEM;
    memset(w, 0, sizeof(*w));
    w->device = plan->device;
    w->npoints = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2];
    w->band_bytes = w->npoints * (plan->g.cplx ? 16 : 8);
    if (chunk_bytes == 0) chunk_bytes = 64 << 20;
    w->chunk = (int64_t)((size_t)chunk_bytes / w->band_bytes);
    if (w->chunk < 1) w->chunk = 1;
    int rc = FD_OK;
    if (cudaMalloc(&w->v_dev, w->npoints * 8) != cudaSuccess) rc = FD_ERR_NOMEM;
    for (int i = 0; i < fd_workspace::kSlots && rc == FD_OK; ++i) {
        if (cudaMalloc(&w->in_dev[i], w->band_bytes * w->chunk) != cudaSuccess ||
            cudaMalloc(&w->out_dev[i], w->band_bytes * w->chunk) != cudaSuccess)
            rc = FD_ERR_NOMEM;
        else if (cudaStreamCreateWithFlags(&w->st[i], cudaStreamNonBlocking) != cudaSuccess)
            rc = FD_ERR_CUDA;
    }
    if (rc == FD_OK && cudaEventCreateWithFlags(&w->v_ready, cudaEventDisableTiming) != cudaSuccess)
        rc = FD_ERR_CUDA;
    if (rc != FD_OK) {
        cudaGetLastError();
        fd_workspace_destroy(w);
        return rc;
    }
    *ws_out = w;
    return FD_OK;
}

int fd_apply_hamiltonian_host_ws(const fd_plan *plan, fd_workspace *ws, const void *psi_host,
                                 const double *v_eff_host, void *out_host, int64_t nbands)
{
    if (!plan || !ws || nbands < 0) return FD_ERR_INVALID;
    if (plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (nbands == 0) return FD_OK;
    if (!psi_host || !out_host) return FD_ERR_INVALID;
    const size_t P = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2];
    const size_t band_bytes = P * (plan->g.cplx ? 16 : 8);
    if (ws->device != plan->device || ws->npoints != P || ws->band_bytes != band_bytes)
        return FD_ERR_INVALID;
    if (overlaps(out_host, band_bytes * nbands, psi_host, band_bytes * nbands)) return FD_ERR_ALIAS;
    if (v_eff_host && overlaps(out_host, band_bytes * nbands, v_eff_host, P * 8)) return FD_ERR_ALIAS;
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;

    // Band chunks ride a 3-slot ring; each slot has its own stream running H2D -> kernel -> D2H, so
    // the copy engines (both directions) and the SMs overlap.
    const int kSlots = fd_workspace::kSlots;
    const int64_t chunk = ws->chunk;
    int rc = FD_OK;
    auto fail = [&](int code) { if (rc == FD_OK) rc = code; };
    double *v_dev = v_eff_host ? ws->v_dev : nullptr;
    if (v_dev) {
        if (cudaMemcpyAsync(v_dev, v_eff_host, P * 8, cudaMemcpyHostToDevice, ws->st[0]) != cudaSuccess ||
            cudaEventRecord(ws->v_ready, ws->st[0]) != cudaSuccess)
            fail(FD_ERR_CUDA);
    }
    int64_t b0 = 0;
    for (int i = 0; rc == FD_OK && b0 < nbands; ++i, b0 += chunk) {
        const int s = i % kSlots;
        const int64_t nb = (nbands - b0 < chunk) ? nbands - b0 : chunk;
        const char *src = static_cast<const char *>(psi_host) + (size_t)b0 * band_bytes;
        char *dst = static_cast<char *>(out_host) + (size_t)b0 * band_bytes;
        if (cudaMemcpyAsync(ws->in_dev[s], src, band_bytes * nb, cudaMemcpyHostToDevice, ws->st[s]) !=
            cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
        if (v_dev && s != 0 && i < kSlots && cudaStreamWaitEvent(ws->st[s], ws->v_ready, 0) != cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
        const int arc = apply_device(plan, plan->g, v_dev ? 1 : 0, ws->in_dev[s], v_dev, ws->out_dev[s],
                                     nb, nullptr, nullptr, nullptr, ws->st[s]);
        if (arc != FD_OK) {
            fail(arc);
            break;
        }
        if (cudaMemcpyAsync(dst, ws->out_dev[s], band_bytes * nb, cudaMemcpyDeviceToHost, ws->st[s]) !=
            cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
    }
    for (int i = 0; i < kSlots; ++i)
        if (cudaStreamSynchronize(ws->st[i]) != cudaSuccess) fail(FD_ERR_CUDA);
    if (rc == FD_ERR_CUDA) cudaGetLastError();
    return rc;
}

int fd_apply_hamiltonian_host(const fd_plan *plan, const void *psi_host, const double *v_eff_host,
                              void *out_host, int64_t nbands)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    fd_workspace *ws = nullptr;
    int rc = fd_workspace_create(&ws, plan, 0);
    if (rc != FD_OK) return rc;
    rc = fd_apply_hamiltonian_host_ws(plan, ws, psi_host, v_eff_host, out_host, nbands);
    fd_workspace_destroy(ws);
    return rc;
}

// ---- expectation values and residual ---------------------------------------------

int64_t fd_expect_workspace_bytes(const fd_plan *plan, int64_t nbands)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (nbands == 0) return 0;
    const int64_t n = (kernel_for_batch(plan, nbands) == FD_KERNEL_SWEEP && fd_sweep_expect_fused(plan))
                          ? fd_sweep_expect_ws_bytes(plan, nbands)
                          : fd_dot_ws_bytes(plan, nbands);
    return n < 16 ? 16 : n;
}

int fd_apply_hamiltonian_expect(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                                double *eps, double *norm, int64_t nbands, void *workspace,
                                int64_t workspace_bytes, void *cuda_stream)
{
    if (plan && plan->g.f32) return FD_ERR_UNSUPPORTED;
    const int rc = check_apply_args(plan, psi, v_eff, false, out, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    if (!eps || !norm || !workspace) return FD_ERR_INVALID;
    if ((((uintptr_t)eps | (uintptr_t)norm) & 7) || ((uintptr_t)workspace & 15)) return FD_ERR_INVALID;
    if (workspace_bytes < fd_expect_workspace_bytes(plan, nbands)) return FD_ERR_INVALID;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands *
                      (plan->g.cplx ? 16 : 8);
    if (overlaps(out, nb, eps, 8 * (size_t)nbands) || overlaps(out, nb, norm, 8 * (size_t)nbands) ||
        overlaps(out, nb, workspace, (size_t)workspace_bytes) ||
        overlaps(eps, 8 * (size_t)nbands, norm, 8 * (size_t)nbands))
        return FD_ERR_ALIAS;
    return apply_device(plan, plan->g, v_eff ? 1 : 0, psi, v_eff, out, nbands, eps, norm,
                        static_cast<double *>(workspace), (cudaStream_t)cuda_stream);
}

int fd_residual(const fd_plan *plan, const void *psi, const void *hpsi, const double *eps,
                const double *norm, void *r, int64_t nbands, void *cuda_stream)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (nbands == 0) return FD_OK;
    if (!psi || !hpsi || !eps || !norm || !r) return FD_ERR_INVALID;
    if (((uintptr_t)psi | (uintptr_t)hpsi | (uintptr_t)r) & 15) return FD_ERR_INVALID;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands *
                      (plan->g.cplx ? 16 : 8);
    if (overlaps(r, nb, psi, nb)) return FD_ERR_ALIAS;
    if (r != hpsi && overlaps(r, nb, hpsi, nb)) return FD_ERR_ALIAS;  // exactly in place is allowed
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;
    if (fd_launch_residual(plan, psi, hpsi, eps, norm, r, nbands, (cudaStream_t)cuda_stream) !=
        cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    __atomic_add_fetch(&const_cast<fd_plan *>(plan)->launches, 1LL, __ATOMIC_RELAXED);
    return FD_OK;
}

// ---- weighted-Jacobi sweep ---------------------------------------------------------

int fd_jacobi_sweep(const fd_plan *plan, const double *phi, const double *rhs, double *out,
                    int64_t nbands, double omega, void *cuda_stream)
{
    if (!plan || nbands < 0 || !isfinite(omega)) return FD_ERR_INVALID;
    if (plan->g.cplx || plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (nbands == 0) return FD_OK;
    if (!phi || !rhs || !out) return FD_ERR_INVALID;
    if (((uintptr_t)phi | (uintptr_t)rhs | (uintptr_t)out) & 15) return FD_ERR_INVALID;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands * 8;
    if (overlaps(out, nb, phi, nb) || overlaps(out, nb, rhs, nb)) return FD_ERR_ALIAS;
    if (plan->g.wdiag == 0.0) return FD_ERR_INVALID;
    // out = phi + omega (rhs - A phi) / A_ii = (1 - omega) phi - (omega / A_ii) A_offdiag phi
    //       + (omega / A_ii) rhs : the stencil kernels with rescaled weights and an additive term
    FdGeom gj = plan->g;
    const double f = omega / plan->g.wdiag;
    for (int d = 0; d < 3; ++d)
        for (int j = 0; j <= gj.nn; ++j) gj.w[d][j] = -f * plan->g.w[d][j];
    gj.wdiag = 1.0 - omega;
    gj.rhs_coef = f;
    return apply_device(plan, gj, 2, phi, rhs, out, nbands, nullptr, nullptr, nullptr,
                        (cudaStream_t)cuda_stream);
}

int fd_poisson_residual(const fd_plan *plan, const double *phi, const double *rhs, double *out,
                        int64_t nbands, void *cuda_stream)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (plan->g.cplx || plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (nbands == 0) return FD_OK;
    if (!phi || !rhs || !out) return FD_ERR_INVALID;
    if (((uintptr_t)phi | (uintptr_t)rhs | (uintptr_t)out) & 15) return FD_ERR_INVALID;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands * 8;
    if (overlaps(out, nb, phi, nb) || overlaps(out, nb, rhs, nb)) return FD_ERR_ALIAS;
    // out = rhs - A phi: the Jacobi form of the stencil kernels with weights -w and coefficient 1
    FdGeom gr = plan->g;
    for (int d = 0; d < 3; ++d)
        for (int j = 0; j <= gr.nn; ++j) gr.w[d][j] = -plan->g.w[d][j];
    gr.wdiag = -plan->g.wdiag;
    gr.rhs_coef = 1.0;
    return apply_device(plan, gr, 2, phi, rhs, out, nbands, nullptr, nullptr, nullptr,
                        (cudaStream_t)cuda_stream);
}

// ---- multigrid V-cycle on the f3 kernels ------------------------------------------------------------

struct fd_mg {
    static const int kMaxLevels = 16;
    int nlevels, p, device;
    int32_t bc[3];
    int32_t shape[kMaxLevels][3];
    size_t npoints[kMaxLevels];
    fd_plan *plan[kMaxLevels];
    double *phi[kMaxLevels], *rhs[kMaxLevels], *tmp[kMaxLevels];  // phi / rhs of level 0: the caller's
    int64_t max_nbands;
    // The cycle is ~15 launches per level and launch bound on the coarse levels: it is captured once
    // into a CUDA graph per argument set and replayed; the last kGraphSlots argument sets are kept
    // (a solver that alternates a few right-hand-side buffers re-captures none of them).
    struct GraphKey {
        const void *phi, *rhs;
        int64_t nbands;
        int nu1, nu2, nu_coarse;
        double omega;
        // field by field: the struct has padding bytes, which a memcmp would compare too
        bool same(const GraphKey &o) const
        {
            return phi == o.phi && rhs == o.rhs && nbands == o.nbands && nu1 == o.nu1 &&
                   nu2 == o.nu2 && nu_coarse == o.nu_coarse && omega == o.omega;
        }
    };
    static const int kGraphSlots = 4;
    mutable std::mutex graph_mutex;
    mutable GraphKey graph_key[kGraphSlots];
    mutable cudaGraphExec_t graph_exec[kGraphSlots];
    mutable unsigned long long graph_used[kGraphSlots];  // tick of the last launch (least recent goes)
    mutable unsigned long long graph_tick;
    mutable long long graph_captures;  // captures so far (diagnostic, fd_mg_get_info)
    mutable bool graph_off;  // capture failed once (e.g. an unsupported stream): launch directly
};

int fd_mg_destroy(fd_mg *mg)
{
    if (!mg) return FD_OK;
    for (int i = 0; i < fd_mg::kGraphSlots; ++i)
        if (mg->graph_exec[i]) cudaGraphExecDestroy(mg->graph_exec[i]);
    for (int l = 0; l < mg->nlevels; ++l) {
        if (mg->plan[l]) fd_destroy(mg->plan[l]);
        if (l > 0) {
            cudaFree(mg->phi[l]);
            cudaFree(mg->rhs[l]);
        }
        cudaFree(mg->tmp[l]);
    }
    cudaGetLastError();
    delete mg;
    return FD_OK;
}

int fd_mg_create(fd_mg **mg_out, const int32_t shape[3], const double h[3], int32_t nn,
                 const int32_t bc[3], int32_t p, int32_t max_levels, int64_t max_nbands, int32_t device)
{
    if (!mg_out || !shape || !h || !bc || max_nbands < 1 || max_levels < 1) return FD_ERR_INVALID;
    if (p < 1 || p > 3) return (p >= 1 && p <= 6) ? FD_ERR_UNSUPPORTED : FD_ERR_INVALID;
    int cur = -1;  // the level buffers are allocated on the current device: it must be `device`
    if (cudaGetDevice(&cur) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    if (cur != device) return FD_ERR_INVALID;
    fd_mg *mg = new (std::nothrow) fd_mg();
    if (!mg) return FD_ERR_NOMEM;
    mg->nlevels = 0;
    for (int i = 0; i < fd_mg::kGraphSlots; ++i) {
        mg->graph_exec[i] = nullptr;
        mg->graph_used[i] = 0;
        mg->graph_key[i] = fd_mg::GraphKey{nullptr, nullptr, 0, 0, 0, 0, 0.0};
    }
    mg->graph_tick = 0;
    mg->graph_captures = 0;
    mg->graph_off = false;
    for (int l = 0; l < fd_mg::kMaxLevels; ++l) {
        mg->plan[l] = nullptr;
        mg->phi[l] = mg->rhs[l] = mg->tmp[l] = nullptr;
        mg->npoints[l] = 0;
    }
    mg->p = p;
    mg->device = device;
    mg->max_nbands = max_nbands;
    if (max_levels > fd_mg::kMaxLevels) max_levels = fd_mg::kMaxLevels;
    int32_t s[3] = {shape[0], shape[1], shape[2]};
    double hl[3] = {h[0], h[1], h[2]};
    int rc = FD_OK;
    for (int l = 0; l < max_levels && rc == FD_OK; ++l) {
        for (int d = 0; d < 3; ++d) {
            mg->bc[d] = bc[d];
            mg->shape[l][d] = s[d];
        }
        mg->npoints[l] = (size_t)s[0] * s[1] * s[2];
        rc = fd_create_scaled(&mg->plan[l], s, hl, nn, bc, nullptr, FD_F64, device, 1.0);
        if (rc != FD_OK) break;
        mg->nlevels = l + 1;
        const size_t bytes = mg->npoints[l] * 8 * (size_t)max_nbands;
        if (cudaMalloc(&mg->tmp[l], bytes) != cudaSuccess ||
            (l > 0 && (cudaMalloc(&mg->phi[l], bytes) != cudaSuccess ||
                       cudaMalloc(&mg->rhs[l], bytes) != cudaSuccess))) {
            rc = FD_ERR_NOMEM;
            break;
        }
        // the next level: every axis must allow coarsening and keep max(nn, 2) points
        bool ok = true;
        int32_t c[3];
        for (int d = 0; d < 3; ++d) {
            ok = ok && (bc[d] ? (s[d] % 2 == 0 && s[d] >= 2) : (s[d] % 2 == 1 && s[d] >= 3));
            c[d] = bc[d] ? s[d] / 2 : (s[d] - 1) / 2;
            ok = ok && c[d] >= (nn > 2 ? nn : 2);
        }
        if (!ok || l + 1 >= max_levels) break;
        // both transfers between this level and the next must fit the kernels (z-row limits): fail
        // here with FD_ERR_UNSUPPORTED rather than in the first fd_mg_vcycle
        // (the tile choice depends on the batch size: both ends of the allowed range are checked)
        for (int interp = 0; interp < 2 && rc == FD_OK; ++interp) {
            rc = fd_transfer_check(interp, s, bc, p, max_nbands);
            if (rc == FD_OK) rc = fd_transfer_check(interp, s, bc, p, 1);
        }
        if (rc != FD_OK) break;
        for (int d = 0; d < 3; ++d) {
            s[d] = c[d];
            hl[d] *= 2.0;
        }
    }
    if (rc != FD_OK) {
        cudaGetLastError();
        fd_mg_destroy(mg);
        return rc;
    }
    *mg_out = mg;
    return FD_OK;
}

int32_t fd_mg_levels(const fd_mg *mg) { return mg ? mg->nlevels : FD_ERR_INVALID; }

namespace {

// nu weighted-Jacobi sweeps on level l, result in phi (tmp is the other buffer of the ping-pong)
int mg_smooth(const fd_mg *mg, int l, double *phi, const double *rhs, int64_t nbands, int nu,
              double omega, void *stream)
{
    double *src = phi, *dst = mg->tmp[l];
    for (int s = 0; s < nu; ++s) {
        const int rc = fd_jacobi_sweep(mg->plan[l], src, rhs, dst, nbands, omega, stream);
        if (rc != FD_OK) return rc;
        double *t = src;
        src = dst;
        dst = t;
    }
    if (src != phi &&
        cudaMemcpyAsync(phi, src, mg->npoints[l] * 8 * (size_t)nbands, cudaMemcpyDeviceToDevice,
                        (cudaStream_t)stream) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    return FD_OK;
}

}  // namespace

namespace {

// the launches of one cycle, in order, on stream cuda_stream
int mg_cycle_launches(const fd_mg *mg, double *phi, const double *rhs, int64_t nbands, int32_t nu1,
                      int32_t nu2, int32_t nu_coarse, double omega, void *cuda_stream)
{
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int L = mg->nlevels;
    double *ph[fd_mg::kMaxLevels];
    const double *rh[fd_mg::kMaxLevels];
    for (int l = 0; l < L; ++l) {
        ph[l] = l ? mg->phi[l] : phi;
        rh[l] = l ? mg->rhs[l] : rhs;
    }
    int rc;
    for (int l = 0; l + 1 < L; ++l) {  // down: smooth, residual, restrict, zero initial guess
        if ((rc = mg_smooth(mg, l, ph[l], rh[l], nbands, nu1, omega, cuda_stream)) != FD_OK) return rc;
        if ((rc = fd_poisson_residual(mg->plan[l], ph[l], rh[l], mg->tmp[l], nbands, cuda_stream)) != FD_OK)
            return rc;
        if ((rc = fd_transfer_run(0, mg->shape[l], mg->bc, mg->p, mg->tmp[l], mg->rhs[l + 1], nbands, st)) != 0)
            return rc;
        if (cudaMemsetAsync(mg->phi[l + 1], 0, mg->npoints[l + 1] * 8 * (size_t)nbands, st) != cudaSuccess) {
            cudaGetLastError();
            return FD_ERR_CUDA;
        }
    }
    if ((rc = mg_smooth(mg, L - 1, ph[L - 1], rh[L - 1], nbands, nu_coarse, omega,
                        cuda_stream)) != FD_OK)
        return rc;
    for (int l = L - 2; l >= 0; --l) {  // up: interpolate the correction, add, smooth
        if ((rc = fd_transfer_run(1, mg->shape[l], mg->bc, mg->p, ph[l + 1], mg->tmp[l], nbands, st)) != 0)
            return rc;
        if (fd_launch_add(ph[l], mg->tmp[l], (long long)(mg->npoints[l] * (size_t)nbands),
                          mg->plan[l]->sm_count, st) != cudaSuccess) {
            cudaGetLastError();
            return FD_ERR_CUDA;
        }
        if ((rc = mg_smooth(mg, l, ph[l], rh[l], nbands, nu2, omega, cuda_stream)) != FD_OK) return rc;
    }
    return FD_OK;
}

}  // namespace

int fd_mg_vcycle(const fd_mg *mg, double *phi, const double *rhs, int64_t nbands, int32_t nu1,
                 int32_t nu2, int32_t nu_coarse, double omega, void *cuda_stream)
{
    if (!mg || nbands < 0 || nu1 < 0 || nu2 < 0 || nu_coarse < 0 || !isfinite(omega)) return FD_ERR_INVALID;
    if (nbands > mg->max_nbands) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!phi || !rhs) return FD_ERR_INVALID;
    if (((uintptr_t)phi | (uintptr_t)rhs) & 15) return FD_ERR_INVALID;
    const size_t nb0 = mg->npoints[0] * 8 * (size_t)nbands;
    if (overlaps(phi, nb0, rhs, nb0)) return FD_ERR_ALIAS;
    const int drc = check_device(mg->plan[0]);
    if (drc != FD_OK) return drc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The legacy default stream cannot be captured: launch directly there.
    if (st == nullptr || st == cudaStreamLegacy || mg->graph_off)
        return mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);
    // A stream the caller is capturing already: the launches simply join the caller's graph.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    if (cap != cudaStreamCaptureStatusNone)
        return mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);

    std::lock_guard<std::mutex> lock(mg->graph_mutex);
    const fd_mg::GraphKey key = {phi, rhs, nbands, nu1, nu2, nu_coarse, omega};
    int slot = -1;
    for (int i = 0; i < fd_mg::kGraphSlots; ++i)
        if (mg->graph_exec[i] && mg->graph_key[i].same(key)) slot = i;
    if (slot < 0) {
        // an empty slot, else the least recently launched one
        slot = 0;
        for (int i = 0; i < fd_mg::kGraphSlots; ++i) {
            if (!mg->graph_exec[i]) {
                slot = i;
                break;
            }
            if (mg->graph_used[i] < mg->graph_used[slot]) slot = i;
        }
        if (mg->graph_exec[slot]) {
            cudaGraphExecDestroy(mg->graph_exec[slot]);
            mg->graph_exec[slot] = nullptr;
        }
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            mg->graph_off = true;
            return mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);
        }
        const int rc = mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        if (rc != FD_OK || ce != cudaSuccess || !graph) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            // nothing was enqueued; whatever went wrong (a call that is not allowed inside a capture, a
            // real launch error) shows again, with its proper status, in the direct launch
            mg->graph_off = true;
            return mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);
        }
        const cudaError_t ie = cudaGraphInstantiate(&mg->graph_exec[slot], graph, 0);
        cudaGraphDestroy(graph);
        if (ie != cudaSuccess) {
            cudaGetLastError();
            mg->graph_exec[slot] = nullptr;
            mg->graph_off = true;
            return mg_cycle_launches(mg, phi, rhs, nbands, nu1, nu2, nu_coarse, omega, cuda_stream);
        }
        mg->graph_key[slot] = key;
        ++mg->graph_captures;
    }
    mg->graph_used[slot] = ++mg->graph_tick;
    if (cudaGraphLaunch(mg->graph_exec[slot], st) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    return FD_OK;
}

int fd_mg_get_info(const fd_mg *mg, int64_t info[8])
{
    if (!mg || !info) return FD_ERR_INVALID;
    info[0] = mg->shape[0][0];
    info[1] = mg->shape[0][1];
    info[2] = mg->shape[0][2];
    info[3] = mg->max_nbands;
    info[4] = mg->device;
    info[5] = mg->nlevels;
    {
        std::lock_guard<std::mutex> lock(mg->graph_mutex);
        info[6] = mg->graph_captures;
        info[7] = mg->graph_off ? 1 : 0;
    }
    return FD_OK;
}

// ---- grid transfer ---------------------------------------------------------------

static int transfer_call(int interp, const int32_t shape_fine[3], const int32_t bc[3], int32_t p,
                         const double *src, double *dst, int64_t nbands, void *cuda_stream)
{
    if (!shape_fine || !bc || nbands < 0) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!src || !dst) return FD_ERR_INVALID;
    if (((uintptr_t)src | (uintptr_t)dst) & 7) return FD_ERR_INVALID;
    size_t pf = 1, pc = 1;
    for (int d = 0; d < 3; ++d) {
        if (shape_fine[d] < 2) return FD_ERR_INVALID;
        pf *= (size_t)shape_fine[d];
        pc *= (size_t)(bc[d] ? shape_fine[d] / 2 : (shape_fine[d] - 1) / 2);
    }
    const size_t nsrc = (interp ? pc : pf) * 8 * (size_t)nbands, ndst = (interp ? pf : pc) * 8 * (size_t)nbands;
    if (overlaps(dst, ndst, src, nsrc)) return FD_ERR_ALIAS;
    return fd_transfer_run(interp, shape_fine, bc, p, src, dst, nbands, (cudaStream_t)cuda_stream);
}

int fd_restrict(const int32_t shape_fine[3], const int32_t bc[3], int32_t p, const double *fine,
                double *coarse, int64_t nbands, void *cuda_stream)
{
    return transfer_call(0, shape_fine, bc, p, fine, coarse, nbands, cuda_stream);
}

int fd_interpolate(const int32_t shape_fine[3], const int32_t bc[3], int32_t p, const double *coarse,
                   double *fine, int64_t nbands, void *cuda_stream)
{
    return transfer_call(1, shape_fine, bc, p, coarse, fine, nbands, cuda_stream);
}

// ---- PAW non-local term ----------------------------------------------------------

int fd_paw_create(fd_paw **paw, const fd_plan *plan, int32_t natoms, const int32_t *box_start,
                  const int32_t *box_size, const int32_t *nproj, const double *proj_host,
                  const double *dh_host, const double *ds_host)
{
    if (!paw || !plan || natoms < 0) return FD_ERR_INVALID;
    if (plan->g.f32) return FD_ERR_UNSUPPORTED;
    if (natoms > 0 && (!box_start || !box_size || !nproj || !proj_host)) return FD_ERR_INVALID;
    if (!dh_host && !ds_host && natoms > 0) return FD_ERR_INVALID;
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;
    return fd_paw_build(paw, plan, natoms, box_start, box_size, nproj, proj_host, dh_host, ds_host);
}

int fd_paw_destroy(fd_paw *paw)
{
    fd_paw_free(paw);
    return FD_OK;
}

int32_t fd_paw_nproj_total(const fd_paw *paw) { return paw ? fd_paw_ntot(paw) : FD_ERR_INVALID; }

static int paw_args(const fd_plan *plan, const fd_paw *paw, const void *psi, const void *coef,
                    int64_t nbands)
{
    if (!plan || !paw || nbands < 0) return FD_ERR_INVALID;
    if (!fd_paw_matches(paw, plan)) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!psi || !coef) return FD_ERR_INVALID;
    if (((uintptr_t)psi | (uintptr_t)coef) & 15) return FD_ERR_INVALID;
    return check_device(plan);
}

// coef (nbands x ntot elements, written by the projection) must not overlap psi or out
static int paw_coef_alias(const fd_plan *plan, const fd_paw *paw, const void *psi, const void *out,
                          const void *coef, int64_t nbands)
{
    const size_t elem = plan->g.cplx ? 16 : 8;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands * elem;
    const size_t nc = (size_t)nbands * (size_t)fd_paw_ntot(paw) * elem;
    if (overlaps(coef, nc, psi, nb) || (out && overlaps(coef, nc, out, nb))) return FD_ERR_ALIAS;
    return FD_OK;
}

static int paw_finish(const fd_plan *plan, cudaError_t e, int n)
{
    if (e != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    __atomic_add_fetch(&const_cast<fd_plan *>(plan)->launches, (long long)n, __ATOMIC_RELAXED);
    return FD_OK;
}

int fd_paw_project(const fd_plan *plan, const fd_paw *paw, const void *psi, void *coef,
                   int64_t nbands, void *cuda_stream)
{
    int rc = paw_args(plan, paw, psi, coef, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    rc = paw_coef_alias(plan, paw, psi, nullptr, coef, nbands);
    if (rc != FD_OK) return rc;
    int n = 0;
    return paw_finish(plan, fd_paw_launch_project(paw, psi, coef, nbands, (cudaStream_t)cuda_stream, &n), n);
}

int fd_paw_expect(const fd_plan *plan, const fd_paw *paw, int32_t which, const void *coef, double *out,
                  int64_t nbands, void *cuda_stream)
{
    if (!plan || !paw || nbands < 0 || (which != 0 && which != 1)) return FD_ERR_INVALID;
    if (!fd_paw_matches(paw, plan) || !fd_paw_has(paw, which)) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!coef || !out || ((uintptr_t)coef & 15) || ((uintptr_t)out & 7)) return FD_ERR_INVALID;
    const int drc = check_device(plan);
    if (drc != FD_OK) return drc;
    int n = 0;
    return paw_finish(plan, fd_paw_launch_expect(paw, which, coef, out, nbands, (cudaStream_t)cuda_stream, &n), n);
}

// out += sum |p~> dO <p~|psi>, which: 0 = Delta H, 1 = Delta S
static int paw_add(const fd_plan *plan, const fd_paw *paw, int which, const void *psi, void *out,
                   void *coef, int64_t nbands, cudaStream_t stream)
{
    if (!fd_paw_has(paw, which)) return FD_ERR_INVALID;
    int n = 0;
    cudaError_t e = fd_paw_launch_project(paw, psi, coef, nbands, stream, &n);
    if (e == cudaSuccess) e = fd_paw_launch_add(paw, which, coef, out, nbands, stream, &n);
    return paw_finish(plan, e, n);
}

int fd_paw_add_nonlocal(const fd_plan *plan, const fd_paw *paw, const void *psi, void *out, void *coef,
                        int64_t nbands, void *cuda_stream)
{
    int rc = paw_args(plan, paw, psi, coef, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    rc = check_apply_args(plan, psi, nullptr, false, out, nbands);
    if (rc != FD_OK) return rc;
    rc = paw_coef_alias(plan, paw, psi, out, coef, nbands);
    if (rc != FD_OK) return rc;
    return paw_add(plan, paw, 0, psi, out, coef, nbands, (cudaStream_t)cuda_stream);
}

int fd_apply_hamiltonian_paw(const fd_plan *plan, const fd_paw *paw, const void *psi,
                             const double *v_eff, void *out, void *coef, int64_t nbands,
                             void *cuda_stream)
{
    int rc = paw_args(plan, paw, psi, coef, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    rc = check_apply_args(plan, psi, v_eff, false, out, nbands);
    if (rc != FD_OK) return rc;
    rc = paw_coef_alias(plan, paw, psi, out, coef, nbands);
    if (rc != FD_OK) return rc;
    rc = apply_device(plan, plan->g, v_eff ? 1 : 0, psi, v_eff, out, nbands, nullptr, nullptr, nullptr,
                      (cudaStream_t)cuda_stream);
    if (rc != FD_OK) return rc;
    return paw_add(plan, paw, 0, psi, out, coef, nbands, (cudaStream_t)cuda_stream);
}

int fd_apply_overlap(const fd_plan *plan, const fd_paw *paw, const void *psi, void *out, void *coef,
                     int64_t nbands, void *cuda_stream)
{
    int rc = paw_args(plan, paw, psi, coef, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    rc = check_apply_args(plan, psi, nullptr, false, out, nbands);
    if (rc != FD_OK) return rc;
    rc = paw_coef_alias(plan, paw, psi, out, coef, nbands);
    if (rc != FD_OK) return rc;
    const size_t nb = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (size_t)nbands *
                      (plan->g.cplx ? 16 : 8);
    if (cudaMemcpyAsync(out, psi, nb, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    return paw_add(plan, paw, 1, psi, out, coef, nbands, (cudaStream_t)cuda_stream);
}

int fd_peak_kernel(int32_t kind, void *a, void *b, int64_t n, int32_t blocks, void *cuda_stream)
{
    if (kind < 0 || kind > 3 || n < 0 || !a || (kind != 1 && kind != 3 && !b)) return FD_ERR_INVALID;
    if (((uintptr_t)a | (uintptr_t)b) & 15) return FD_ERR_INVALID;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    if (fd_peak_launch(kind, static_cast<double *>(a), static_cast<double *>(b), n, blocks, sms,
                       (cudaStream_t)cuda_stream) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    return FD_OK;
}

int fd_destroy(fd_plan *plan)
{
    delete plan;
    return FD_OK;
}

const char *fd_strerror(int status)
{
    switch (status) {
    case FD_OK: return "success";
    case FD_ERR_INVALID: return "invalid argument";
    case FD_ERR_UNSUPPORTED: return "unsupported by this plan or build";
    case FD_ERR_ALIAS: return "output overlaps an input";
    case FD_ERR_CUDA: return "CUDA error (no device, or launch/copy failure)";
    case FD_ERR_NOMEM: return "out of memory";
    case FD_ERR_SCRATCH: return "batch needs more scratch than the library's built-in array holds";
    default: return "unknown fd_status";
    }
}

int fd_plan_set_kernel(fd_plan *plan, int32_t kernel, int32_t param)
{
    if (!plan) return FD_ERR_INVALID;
    if (kernel == FD_KERNEL_GENERIC) {
        plan->kernel = FD_KERNEL_GENERIC;
        plan->forced = 1;
        return FD_OK;
    }
    if (kernel != FD_KERNEL_AUTO && kernel != FD_KERNEL_SWEEP) return FD_ERR_INVALID;
    if (param != 0 || kernel == FD_KERNEL_SWEEP) {
        // configure a copy: a refused request leaves the plan exactly as it was
        fd_plan trial = *plan;
        fd_sweep_configure(&trial, param, plan->sweep.xchunk, plan->sweep.stages_req);
        if (!trial.sweep.supported) return FD_ERR_UNSUPPORTED;
        const int drc = check_device(plan);
        if (drc != FD_OK) return drc;
        if (fd_sweep_prepare(&trial) != cudaSuccess) {
            cudaGetLastError();
            return FD_ERR_CUDA;
        }
        plan->sweep = trial.sweep;
    }
    if (!plan->sweep.supported && kernel == FD_KERNEL_SWEEP) return FD_ERR_UNSUPPORTED;
    plan->kernel = plan->sweep.supported ? FD_KERNEL_SWEEP : FD_KERNEL_GENERIC;
    plan->forced = (kernel != FD_KERNEL_AUTO);
    return FD_OK;
}

int fd_plan_get_kernel(const fd_plan *plan) { return plan ? plan->kernel : FD_ERR_INVALID; }

int fd_plan_get_info(const fd_plan *plan, int32_t info[8])
{
    if (!plan || !info) return FD_ERR_INVALID;
    const FdGeom &g = plan->g;
    info[0] = g.n[0];
    info[1] = g.n[1];
    info[2] = g.n[2];
    info[3] = g.nn;
    info[4] = g.f32 ? (g.cplx ? FD_C64 : FD_F32) : (g.cplx ? FD_C128 : FD_F64);
    info[5] = plan->device;
    info[6] = g.bc[0] | (g.bc[1] << 1) | (g.bc[2] << 2);
    info[7] = plan->kernel;
    return FD_OK;
}

int fd_plan_kernel_for(const fd_plan *plan, int64_t nbands)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    return kernel_for_batch(plan, nbands);
}

int64_t fd_plan_launches(const fd_plan *plan) { return plan ? plan->launches : 0; }

int fd_plan_get_weights(const fd_plan *plan, double *w, int32_t capacity)
{
    if (!plan || !w) return FD_ERR_INVALID;
    const int n = 3 * (plan->g.nn + 1);
    if (capacity < n) return FD_ERR_INVALID;
    for (int d = 0; d < 3; ++d)
        for (int j = 0; j <= plan->g.nn; ++j) w[d * (plan->g.nn + 1) + j] = plan->g.w[d][j];
    return n;
}

}  // extern "C"
