// Streaming helper kernels of the eigensolver epilogue:
//   * the two-pass form of the expectation values (plans / batches that run on the generic kernel:
//     eps_b = sum Re conj(psi_b) (H psi)_b and norm_b = sum |psi_b|^2 from the stored H psi), with a
//     deterministic two-stage reduction (fixed chunking, fixed tree, no atomics);
//   * the residual r_b = H psi_b - (eps_b / norm_b) psi_b.
// The fused form (sums taken inside the sweep kernel while psi is in registers) is in
// fd_sweep_kernel.cuh.
#include "fd_internal.h"

namespace {

constexpr int kDotThreads = 256;
constexpr int kDotChunk = 16384;  // doubles per CTA

// complex data: Re conj(a) b = a.re b.re + a.im b.im, so both dtypes are a plain product over doubles
__global__ void __launch_bounds__(kDotThreads)
fd_dot_partial_kernel(const double *__restrict__ psi, const double *__restrict__ hpsi,
                      double *__restrict__ ws, long long band_d, int nchunk)
{
    const int chunk = blockIdx.x;
    const long long b = blockIdx.y;
    const double *a = psi + b * band_d;
    const double *h = hpsi + b * band_d;
    const long long lo = (long long)chunk * kDotChunk;
    const long long hi = (lo + kDotChunk < band_d) ? lo + kDotChunk : band_d;
    double e = 0.0, n = 0.0;
    // band_d is even and 16-byte aligned for every plan (complex, or real with the library's
    // alignment rule); odd real sizes take the scalar tail
    long long i = lo + 2 * threadIdx.x;
    for (; i + 1 < hi; i += 2 * kDotThreads) {
        if (((reinterpret_cast<uintptr_t>(a + i) | reinterpret_cast<uintptr_t>(h + i)) & 15) == 0) {
            const double2 x = __ldcs(reinterpret_cast<const double2 *>(a + i));
            const double2 y = __ldcs(reinterpret_cast<const double2 *>(h + i));
            e = fma(x.x, y.x, fma(x.y, y.y, e));
            n = fma(x.x, x.x, fma(x.y, x.y, n));
        } else {
            e = fma(a[i], h[i], fma(a[i + 1], h[i + 1], e));
            n = fma(a[i], a[i], fma(a[i + 1], a[i + 1], n));
        }
    }
    if (i < hi) {
        e = fma(a[i], h[i], e);
        n = fma(a[i], a[i], n);
    }
    __shared__ double se[kDotThreads / 32], sn[kDotThreads / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_xor_sync(0xffffffffu, e, o);
        n += __shfl_xor_sync(0xffffffffu, n, o);
    }
    if ((threadIdx.x & 31) == 0) {
        se[threadIdx.x >> 5] = e;
        sn[threadIdx.x >> 5] = n;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double te = 0.0, tn = 0.0;
        for (int w = 0; w < kDotThreads / 32; ++w) {
            te += se[w];
            tn += sn[w];
        }
        ws[2 * (b * nchunk + chunk)] = te;
        ws[2 * (b * nchunk + chunk) + 1] = tn;
    }
}

__global__ void fd_dot_finalize_kernel(const double *__restrict__ ws, double *__restrict__ eps,
                                       double *__restrict__ norm, long long nbands, int nchunk)
{
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbands) return;
    double e = 0.0, n = 0.0;
    for (int c = 0; c < nchunk; ++c) {
        e += ws[2 * (b * nchunk + c)];
        n += ws[2 * (b * nchunk + c) + 1];
    }
    eps[b] = e;
    norm[b] = n;
}

// r = hpsi - (eps_b / norm_b) psi, over doubles (real lambda: the same for re and im parts)
__global__ void __launch_bounds__(256)
fd_residual_kernel(const double *__restrict__ psi, const double *hpsi, const double *__restrict__ eps,
                   const double *__restrict__ norm, double *r, long long band_d, int per_band)
{
    const long long b = blockIdx.y;
    const double lam = eps[b] / norm[b];
    const double *a = psi + b * band_d;
    const double *h = hpsi + b * band_d;
    double *o = r + b * band_d;
    const bool vec = (((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(h) |
                        reinterpret_cast<uintptr_t>(o)) & 15) == 0) && !(band_d & 1);
    const long long lo = (long long)blockIdx.x * per_band;
    const long long hi = (lo + per_band < band_d) ? lo + per_band : band_d;
    if (vec) {
        for (long long i = lo + 2 * threadIdx.x; i < hi; i += 2 * blockDim.x) {
            const double2 x = __ldcs(reinterpret_cast<const double2 *>(a + i));
            const double2 y = __ldcs(reinterpret_cast<const double2 *>(h + i));
            __stcs(reinterpret_cast<double2 *>(o + i),
                   make_double2(fma(-lam, x.x, y.x), fma(-lam, x.y, y.y)));
        }
    } else {
        for (long long i = lo + threadIdx.x; i < hi; i += blockDim.x) o[i] = fma(-lam, a[i], h[i]);
    }
}

// y += x over n doubles (the coarse-grid correction of the V-cycle)
__global__ void __launch_bounds__(256) fd_add_kernel(double *__restrict__ y, const double *__restrict__ x, long long n)
{
    const long long stride = (long long)gridDim.x * blockDim.x * 2;
    long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 2;
    const bool vec = ((reinterpret_cast<uintptr_t>(y) | reinterpret_cast<uintptr_t>(x)) & 15) == 0;
    for (; i + 1 < n; i += stride) {
        if (vec) {
            double2 a = *reinterpret_cast<double2 *>(y + i);
            const double2 b = __ldcs(reinterpret_cast<const double2 *>(x + i));
            a.x += b.x;
            a.y += b.y;
            *reinterpret_cast<double2 *>(y + i) = a;
        } else {
            y[i] += x[i];
            y[i + 1] += x[i + 1];
        }
    }
    if (i < n) y[i] += x[i];
}

inline int dot_chunks(const fd_plan *plan)
{
    const long long band_d =
        (long long)plan->g.n[0] * plan->g.n[1] * plan->g.n[2] * (plan->g.cplx ? 2 : 1);
    return (int)((band_d + kDotChunk - 1) / kDotChunk);
}

}  // namespace

int64_t fd_dot_ws_bytes(const fd_plan *plan, int64_t nbands)
{
    return (int64_t)16 * nbands * dot_chunks(plan);
}

cudaError_t fd_launch_dot(const fd_plan *plan, const void *psi, const void *hpsi, double *eps,
                          double *norm, double *ws, int64_t nbands, cudaStream_t stream,
                          int *nlaunches)
{
    const FdGeom &g = plan->g;
    const long long band_d = (long long)g.n[0] * g.n[1] * g.n[2] * (g.cplx ? 2 : 1);
    const int nchunk = dot_chunks(plan);
    for (int64_t b0 = 0; b0 < nbands; b0 += 65535) {
        const int64_t nb = (nbands - b0 < 65535) ? nbands - b0 : 65535;
        fd_dot_partial_kernel<<<dim3((unsigned)nchunk, (unsigned)nb), kDotThreads, 0, stream>>>(
            static_cast<const double *>(psi) + b0 * band_d,
            static_cast<const double *>(hpsi) + b0 * band_d, ws + 2 * b0 * nchunk, band_d, nchunk);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
        if (nlaunches) ++*nlaunches;
    }
    fd_dot_finalize_kernel<<<dim3((unsigned)((nbands + 127) / 128)), 128, 0, stream>>>(
        ws, eps, norm, nbands, nchunk);
    if (nlaunches) ++*nlaunches;
    return cudaPeekAtLastError();
}

cudaError_t fd_launch_residual(const fd_plan *plan, const void *psi, const void *hpsi,
                               const double *eps, const double *norm, void *r, int64_t nbands,
                               cudaStream_t stream)
{
    const FdGeom &g = plan->g;
    const long long band_d = (long long)g.n[0] * g.n[1] * g.n[2] * (g.cplx ? 2 : 1);
    // enough CTAs per band to fill the device even for a single band
    int per_band = 1 << 15;
    while (per_band > 2048 && (band_d + per_band - 1) / per_band * nbands < 4LL * plan->sm_count)
        per_band >>= 1;
    const unsigned gx = (unsigned)((band_d + per_band - 1) / per_band);
    for (int64_t b0 = 0; b0 < nbands; b0 += 65535) {
        const int64_t nb = (nbands - b0 < 65535) ? nbands - b0 : 65535;
        fd_residual_kernel<<<dim3(gx, (unsigned)nb), 256, 0, stream>>>(
            static_cast<const double *>(psi) + b0 * band_d,
            static_cast<const double *>(hpsi) + b0 * band_d, eps + b0, norm + b0,
            static_cast<double *>(r) + b0 * band_d, band_d, per_band);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t fd_launch_add(double *y, const double *x, long long n, int sm_count, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    long long blocks = (n / 2 + 255) / 256;
    const long long cap = 8LL * sm_count;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    fd_add_kernel<<<(unsigned)blocks, 256, 0, stream>>>(y, x, n);
    return cudaPeekAtLastError();
}
