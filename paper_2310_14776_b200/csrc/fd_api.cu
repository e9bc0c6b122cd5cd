// C ABI of libfdham (declared and documented in include/fdham.h): plan construction, argument
// checking, kernel dispatch, and the host-buffer (end-to-end) variant.  No CPU compute path exists
// here on purpose: without a CUDA device every entry point fails with FD_ERR_CUDA.
#include <math.h>
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
    const size_t nb = P * (size_t)nbands * (plan->g.cplx ? 16 : 8);
    if (overlaps(out, nb, psi, nb)) return FD_ERR_ALIAS;
    if (v_eff && overlaps(out, nb, v_eff, P * 8)) return FD_ERR_ALIAS;
    return FD_OK;
}

// Kernel family for a batch of `nbands`.  The sweep kernel pays ~1.2 us per x plane of a team's
// share plus 6 halo planes per band segment whatever the grid size, so a batch that is far too
// small to fill the persistent teams goes to the one-thread-per-point kernel (measured on B200:
// 24^3 x 8 bands takes 8 us there against 27 us; 48^3 x 64 bands 115 us against 39 us).
int kernel_for_batch(const fd_plan *plan, int64_t nbands)
{
    if (plan->kernel != FD_KERNEL_SWEEP || plan->forced) return plan->kernel;
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

int apply_device(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                 int64_t nbands, cudaStream_t stream)
{
    cudaError_t e;
    int n = 0;
    if (kernel_for_batch(plan, nbands) == FD_KERNEL_SWEEP) {
        e = fd_launch_sweep(plan, psi, v_eff, out, nbands, stream, &n);
    } else {
        e = fd_launch_generic(plan, psi, v_eff, out, nbands, stream);
        n = 1;
    }
    if (e != cudaSuccess) return FD_ERR_CUDA;
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
    if (dtype != FD_F64 && dtype != FD_C128) return FD_ERR_INVALID;
    for (int d = 0; d < 3; ++d) {
        if (shape[d] < 1) return FD_ERR_INVALID;
        if (!(h[d] > 0.0) || !isfinite(h[d])) return FD_ERR_INVALID;
        if (bc[d] != FD_BC_ZERO && bc[d] != FD_BC_PERIODIC) return FD_ERR_INVALID;
        if (bc[d] == FD_BC_PERIODIC && shape[d] < nn) return FD_ERR_INVALID;
        const double kd = k_reduced ? k_reduced[d] : 0.0;
        if (!isfinite(kd)) return FD_ERR_INVALID;
        if (kd != 0.0 && (bc[d] == FD_BC_ZERO || dtype == FD_F64)) return FD_ERR_INVALID;
    }
    if ((long long)shape[0] * shape[1] * shape[2] > (1LL << 40)) return FD_ERR_INVALID;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    if (cudaSetDevice(device) != cudaSuccess) return FD_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return FD_ERR_CUDA;

    fd_plan *p = new (std::nothrow) fd_plan();
    if (!p) return FD_ERR_NOMEM;
    memset(p, 0, sizeof(*p));
    p->device = device;
    p->sm_count = prop.multiProcessorCount;
    FdGeom &g = p->g;
    g.nn = nn;
    g.cplx = (dtype == FD_C128);
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
    return apply_device(plan, psi, nullptr, out, nbands, (cudaStream_t)cuda_stream);
}

int fd_apply_hamiltonian(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                         int64_t nbands, void *cuda_stream)
{
    const int rc = check_apply_args(plan, psi, v_eff, true, out, nbands);
    if (rc != FD_OK || nbands == 0) return rc;
    return apply_device(plan, psi, v_eff, out, nbands, (cudaStream_t)cuda_stream);
}

int fd_apply_hamiltonian_host(const fd_plan *plan, const void *psi_host, const double *v_eff_host,
                              void *out_host, int64_t nbands)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    if (nbands == 0) return FD_OK;
    if (!psi_host || !out_host) return FD_ERR_INVALID;
    const size_t P = (size_t)plan->g.n[0] * plan->g.n[1] * plan->g.n[2];
    const size_t band_bytes = P * (plan->g.cplx ? 16 : 8);
    if (overlaps(out_host, band_bytes * nbands, psi_host, band_bytes * nbands)) return FD_ERR_ALIAS;
    if (cudaSetDevice(plan->device) != cudaSuccess) return FD_ERR_CUDA;

    // Band chunks of ~64 MiB ride a 3-slot ring; each slot has its own stream running
    // H2D -> kernel -> D2H, so the copy engines (both directions) and the SMs overlap.
    constexpr int kSlots = 3;
    int64_t chunk = (int64_t)((64u << 20) / band_bytes);
    if (chunk < 1) chunk = 1;
    if (chunk > nbands) chunk = nbands;
    const int nslots = (int)((nbands + chunk - 1) / chunk < kSlots ? (nbands + chunk - 1) / chunk
                                                                   : kSlots);
    int rc = FD_OK;
    double *v_dev = nullptr;
    char *in_dev[kSlots] = {nullptr, nullptr, nullptr};
    char *out_dev[kSlots] = {nullptr, nullptr, nullptr};
    cudaStream_t st[kSlots] = {nullptr, nullptr, nullptr};
    cudaEvent_t v_ready = nullptr;
    auto fail = [&](int code) { if (rc == FD_OK) rc = code; };

    if (v_eff_host && cudaMalloc(&v_dev, P * 8) != cudaSuccess) fail(FD_ERR_NOMEM);
    for (int i = 0; i < nslots && rc == FD_OK; ++i) {
        if (cudaMalloc(&in_dev[i], band_bytes * chunk) != cudaSuccess ||
            cudaMalloc(&out_dev[i], band_bytes * chunk) != cudaSuccess)
            fail(FD_ERR_NOMEM);
        else if (cudaStreamCreateWithFlags(&st[i], cudaStreamNonBlocking) != cudaSuccess)
            fail(FD_ERR_CUDA);
    }
    if (rc == FD_OK && cudaEventCreateWithFlags(&v_ready, cudaEventDisableTiming) != cudaSuccess)
        fail(FD_ERR_CUDA);
    if (rc == FD_OK && v_dev) {
        if (cudaMemcpyAsync(v_dev, v_eff_host, P * 8, cudaMemcpyHostToDevice, st[0]) != cudaSuccess ||
            cudaEventRecord(v_ready, st[0]) != cudaSuccess)
            fail(FD_ERR_CUDA);
    }
    int64_t b0 = 0;
    for (int i = 0; rc == FD_OK && b0 < nbands; ++i, b0 += chunk) {
        const int s = i % nslots;
        const int64_t nb = (nbands - b0 < chunk) ? nbands - b0 : chunk;
        const char *src = static_cast<const char *>(psi_host) + (size_t)b0 * band_bytes;
        char *dst = static_cast<char *>(out_host) + (size_t)b0 * band_bytes;
        if (cudaMemcpyAsync(in_dev[s], src, band_bytes * nb, cudaMemcpyHostToDevice, st[s]) !=
            cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
        if (v_dev && s != 0 && i < nslots && cudaStreamWaitEvent(st[s], v_ready, 0) != cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
        const int arc = apply_device(plan, in_dev[s], v_dev, out_dev[s], nb, st[s]);
        if (arc != FD_OK) {
            fail(arc);
            break;
        }
        if (cudaMemcpyAsync(dst, out_dev[s], band_bytes * nb, cudaMemcpyDeviceToHost, st[s]) !=
            cudaSuccess) {
            fail(FD_ERR_CUDA);
            break;
        }
    }
    for (int i = 0; i < nslots; ++i)
        if (st[i] && cudaStreamSynchronize(st[i]) != cudaSuccess) fail(FD_ERR_CUDA);
    if (v_ready) cudaEventDestroy(v_ready);
    for (int i = 0; i < kSlots; ++i) {
        if (st[i]) cudaStreamDestroy(st[i]);
        if (in_dev[i]) cudaFree(in_dev[i]);
        if (out_dev[i]) cudaFree(out_dev[i]);
    }
    if (v_dev) cudaFree(v_dev);
    if (rc == FD_ERR_CUDA) cudaGetLastError();
    return rc;
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
        fd_sweep_configure(plan, param, plan->sweep.xchunk, plan->sweep.stages_req);
        if (plan->sweep.supported && fd_sweep_prepare(plan) != cudaSuccess) {
            cudaGetLastError();
            return FD_ERR_CUDA;
        }
    }
    if (!plan->sweep.supported && kernel == FD_KERNEL_SWEEP) return FD_ERR_UNSUPPORTED;
    // a failed request above leaves the family and the per-batch choice as they were
    plan->kernel = plan->sweep.supported ? FD_KERNEL_SWEEP : FD_KERNEL_GENERIC;
    plan->forced = (kernel != FD_KERNEL_AUTO);
    return FD_OK;
}

int fd_plan_get_kernel(const fd_plan *plan) { return plan ? plan->kernel : FD_ERR_INVALID; }

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
