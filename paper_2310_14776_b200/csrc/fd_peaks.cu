// Micro-benchmarks behind the roofline denominators: read-only, write-only
// and copy bandwidth with float64 vectors, and the dependent-free DFMA rate.  Not part of the hot
// path; bench.py --peaks times them with CUDA events and reports them beside MEASURED_PEAKS.json.
#include "fd_internal.h"

namespace {

// grid-stride read of n double2: every value is consumed (sum), one store per thread at the end
__global__ void __launch_bounds__(256) fd_peak_read(const double2 *__restrict__ a, long long n, double *sink)
{
    double s = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double2 v = __ldcs(a + i);
        s += v.x + v.y;
    }
    if (s == 123.456) sink[0] = s;  // never true for the fill pattern: keeps the loads alive
}

__global__ void __launch_bounds__(256) fd_peak_write(double2 *__restrict__ a, long long n, double val)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        __stcs(a + i, make_double2(val, val));
}

__global__ void __launch_bounds__(256) fd_peak_copy(const double2 *__restrict__ a, double2 *__restrict__ b,
                                                    long long n)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        __stcs(b + i, __ldcs(a + i));
}

// 8 independent DFMA chains per thread, `iters` rounds of 8: 2 flop per DFMA
__global__ void __launch_bounds__(256) fd_peak_dfma(long long iters, double x, double *sink)
{
    double a0 = x, a1 = x + 1, a2 = x + 2, a3 = x + 3, a4 = x + 4, a5 = x + 5, a6 = x + 6, a7 = x + 7;
    const double m = 1.0000001, c = 1e-9;
    for (long long i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) sink[0] = s;
}

}  // namespace

// kind 0: read `n` doubles of a; 1: write n doubles to a; 2: copy n doubles a -> b; 3: DFMA, n = rounds
// of 8 DFMA per thread on `blocks` x 256 threads (blocks = 0: 8 per SM).  Returns a cudaError_t.
cudaError_t fd_peak_launch(int kind, double *a, double *b, long long n, int blocks, int sm_count,
                           cudaStream_t stream)
{
    if (blocks <= 0) blocks = 8 * sm_count;
    switch (kind) {
    case 0: fd_peak_read<<<blocks, 256, 0, stream>>>(reinterpret_cast<const double2 *>(a), n / 2, b); break;
    case 1: fd_peak_write<<<blocks, 256, 0, stream>>>(reinterpret_cast<double2 *>(a), n / 2, 1.5); break;
    case 2: fd_peak_copy<<<blocks, 256, 0, stream>>>(reinterpret_cast<const double2 *>(a),
                                                     reinterpret_cast<double2 *>(b), n / 2); break;
    case 3: fd_peak_dfma<<<blocks, 256, 0, stream>>>(n, 0.5, a); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaPeekAtLastError();
}
