// Generic FD Hamiltonian kernel: one thread per grid point, any nn (1..6), any shape, any mix of
// boundary conditions, float64 or complex128.  It is the correctness baseline and the fallback
// for shapes the sweep kernel does not take (odd nz, tiny axes, nn != 3); every neighbour is
// fetched through L1/L2, so it is NOT the bandwidth path.
//
// Operation: include/fdham.h (Eq. 6 first two terms; FD kinetic operator,
// PAPER.md:232; halo rules SURVEY 8(a) step a2).
#include "fd_internal.h"

namespace {

// One grid value: T = double (float64 / complex128) or float (float32 / complex64); CPLX = (re, im).
template <bool CPLX, typename T>
struct Val;
template <typename T>
struct Val<false, T> {
    T x;
    __device__ __forceinline__ static Val zero() { return {T(0)}; }
    __device__ __forceinline__ void fma(T w, const Val &o) { x = w * o.x + x; }  // contracted to an FMA
    // real data: the Bloch factor is +1 or -1 (k_d = 1/2), its imaginary part 0
    __device__ __forceinline__ Val mulphase(T pr, T) const { return {x * pr}; }
};
template <typename T>
struct Val<true, T> {
    T x, y;
    __device__ __forceinline__ static Val zero() { return {T(0), T(0)}; }
    __device__ __forceinline__ void fma(T w, const Val &o)
    {
        x = w * o.x + x;
        y = w * o.y + y;
    }
    __device__ __forceinline__ Val mulphase(T pr, T pi) const
    {
        return {x * pr - y * pi, x * pi + y * pr};
    }
};

template <typename T>
struct Pair;  // the 2-vector of T: one complex value moves as one 16- / 8-byte access
template <>
struct Pair<double> {
    typedef double2 type;
};
template <>
struct Pair<float> {
    typedef float2 type;
};

template <bool CPLX, typename T>
__device__ __forceinline__ Val<CPLX, T> load(const T *p, long long idx)
{
    if constexpr (CPLX) {
        const typename Pair<T>::type t = __ldg(reinterpret_cast<const typename Pair<T>::type *>(p) + idx);
        return {t.x, t.y};
    } else {
        return {__ldg(p + idx)};
    }
}
template <bool CPLX, typename T>
__device__ __forceinline__ void store(T *p, long long idx, const Val<CPLX, T> &v)
{
    if constexpr (CPLX) {
        typename Pair<T>::type t;
        t.x = v.x;
        t.y = v.y;
        reinterpret_cast<typename Pair<T>::type *>(p)[idx] = t;
    } else {
        p[idx] = v.x;
    }
}

// Block = 64 z-points x 4 rows of one x plane (neighbours along z and y share L1 lines); the
// stencil half width is a template parameter so the tap loops unroll and the weights come
// straight from the constant bank.  blockIdx.z = x plane * band groups + band group.
constexpr int kBx = 64, kBy = 4;

// MODE 0: T psi; 1: + v_eff psi (v_eff[nx,ny,nz]); 2: the weighted-Jacobi form, v_eff = the right-hand
// side [nbands,nx,ny,nz], added as g.rhs_coef * rhs (g carries the pre-scaled weights; real only).
// T: double, or float for FD_F32 / FD_C64 (psi, out AND v_eff are then float, fp32 accumulation).
template <bool CPLX, int MODE, int NN, typename T>
__global__ void __launch_bounds__(kBx * kBy)
fd_generic_kernel(const __grid_constant__ FdGeom g, const T *__restrict__ psi,
                  const T *__restrict__ v_eff, T *__restrict__ out, long long nbands, int bgroups)
{
    constexpr bool HAS_V = MODE == 1;
    const int iz = blockIdx.x * kBx + threadIdx.x;
    const int iy = blockIdx.y * kBy + threadIdx.y;
    const int ix = blockIdx.z / bgroups;
    const int bg = blockIdx.z - ix * bgroups;
    if (iz >= g.n[2] || iy >= g.n[1]) return;
    const long long P = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long lin = ((long long)ix * g.n[1] + iy) * g.n[2] + iz;
    const int idx[3] = {ix, iy, iz};
    const long long stride[3] = {(long long)g.n[1] * g.n[2], (long long)g.n[2], 1};
    T diag = (T)g.wdiag;
    if (HAS_V) diag += __ldg(v_eff + lin);

    for (long long b = bg; b < nbands; b += bgroups) {
        const T *pb = psi + (CPLX ? 2 : 1) * b * P;
        const Val<CPLX, T> c = load<CPLX, T>(pb, lin);
        Val<CPLX, T> acc = Val<CPLX, T>::zero();
        acc.fma(diag, c);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int n = g.n[d];
#pragma unroll
            for (int j = 1; j <= NN; ++j) {
                const T w = (T)g.w[d][j];
                // upper tap i + j
                int p = idx[d] + j;
                if (p < n) {
                    acc.fma(w, load<CPLX, T>(pb, lin + j * stride[d]));
                } else if (g.bc[d] == 1) {
                    const Val<CPLX, T> t = load<CPLX, T>(pb, lin + (long long)(j - n) * stride[d]);
                    acc.fma(w, t.mulphase((T)g.ph_re[d], (T)g.ph_im[d]));
                }
                // lower tap i - j
                p = idx[d] - j;
                if (p >= 0) {
                    acc.fma(w, load<CPLX, T>(pb, lin - j * stride[d]));
                } else if (g.bc[d] == 1) {
                    const Val<CPLX, T> t = load<CPLX, T>(pb, lin + (long long)(n - j) * stride[d]);
                    acc.fma(w, t.mulphase((T)g.ph_re[d], -(T)g.ph_im[d]));
                }
            }
        }
        if constexpr (MODE == 2 && !CPLX) acc.x = (T)g.rhs_coef * __ldg(v_eff + b * P + lin) + acc.x;
        store<CPLX, T>(out, b * P + lin, acc);
    }
}

template <bool CPLX, int MODE, typename T>
cudaError_t launch_nn(const FdGeom &g, const T *p, const T *v_eff, T *o, long long nbands,
                      cudaStream_t stream)
{
    // band groups: enough CTAs to fill the device, blockIdx.z <= 65535
    long long bgroups = nbands;
    const long long cap = 65535 / g.n[0];
    if (bgroups > cap) bgroups = cap;
    if (bgroups < 1) return cudaErrorInvalidConfiguration;
    const dim3 block(kBx, kBy);
    const dim3 grid((unsigned)((g.n[2] + kBx - 1) / kBx), (unsigned)((g.n[1] + kBy - 1) / kBy),
                    (unsigned)(g.n[0] * bgroups));
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    const int bgi = (int)bgroups;
    switch (g.nn) {
    case 1: fd_generic_kernel<CPLX, MODE, 1, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    case 2: fd_generic_kernel<CPLX, MODE, 2, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    case 3: fd_generic_kernel<CPLX, MODE, 3, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    case 4: fd_generic_kernel<CPLX, MODE, 4, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    case 5: fd_generic_kernel<CPLX, MODE, 5, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    case 6: fd_generic_kernel<CPLX, MODE, 6, T><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands, bgi); break;
    default: return cudaErrorInvalidConfiguration;
    }
    return cudaPeekAtLastError();
}

}  // namespace

cudaError_t fd_launch_generic(const fd_plan *plan, const FdGeom &g, int mode, const void *psi,
                              const double *second, void *out, int64_t nbands, cudaStream_t stream)
{
    (void)plan;
    if (g.n[0] > 65535) return cudaErrorInvalidConfiguration;
    if (g.f32) {  // float32 / complex64: plain applies only (second = float v_eff)
        const float *p = static_cast<const float *>(psi);
        const float *v = reinterpret_cast<const float *>(second);
        float *o = static_cast<float *>(out);
        if (mode == 2) return cudaErrorInvalidValue;
        if (g.cplx)
            return mode ? launch_nn<true, 1, float>(g, p, v, o, nbands, stream)
                        : launch_nn<true, 0, float>(g, p, nullptr, o, nbands, stream);
        return mode ? launch_nn<false, 1, float>(g, p, v, o, nbands, stream)
                    : launch_nn<false, 0, float>(g, p, nullptr, o, nbands, stream);
    }
    const double *p = static_cast<const double *>(psi);
    double *o = static_cast<double *>(out);
    if (g.cplx) {
        if (mode == 2) return cudaErrorInvalidValue;
        return mode ? launch_nn<true, 1, double>(g, p, second, o, nbands, stream)
                    : launch_nn<true, 0, double>(g, p, nullptr, o, nbands, stream);
    }
    if (mode == 2) return launch_nn<false, 2, double>(g, p, second, o, nbands, stream);
    return mode ? launch_nn<false, 1, double>(g, p, second, o, nbands, stream)
                : launch_nn<false, 0, double>(g, p, nullptr, o, nbands, stream);
}
