// Generic FD Hamiltonian kernel: one thread per grid point, any nn (1..6), any shape, any mix of
// boundary conditions, float64 or complex128.  It is the correctness baseline and the fallback
// for shapes the sweep kernel does not take (odd nz, tiny axes, nn != 3); every neighbour is
// fetched through L1/L2, so it is NOT the bandwidth path.
//
// Operation: include/fdham.h (Eq. 6 first two terms; FD kinetic operator,
// PAPER.md:232; halo rules SURVEY 8(a) step a2).
#include "fd_internal.h"

namespace {

template <bool CPLX>
struct Val;
template <>
struct Val<false> {
    double x;
    __device__ __forceinline__ static Val zero() { return {0.0}; }
    __device__ __forceinline__ void fma(double w, const Val &o) { x = ::fma(w, o.x, x); }
    __device__ __forceinline__ Val mulphase(double, double) const { return *this; }
};
template <>
struct Val<true> {
    double x, y;
    __device__ __forceinline__ static Val zero() { return {0.0, 0.0}; }
    __device__ __forceinline__ void fma(double w, const Val &o)
    {
        x = ::fma(w, o.x, x);
        y = ::fma(w, o.y, y);
    }
    __device__ __forceinline__ Val mulphase(double pr, double pi) const
    {
        return {x * pr - y * pi, x * pi + y * pr};
    }
};

template <bool CPLX>
__device__ __forceinline__ Val<CPLX> load(const double *p, long long idx);
template <>
__device__ __forceinline__ Val<false> load<false>(const double *p, long long idx)
{
    return {__ldg(p + idx)};
}
template <>
__device__ __forceinline__ Val<true> load<true>(const double *p, long long idx)
{
    const double2 t = __ldg(reinterpret_cast<const double2 *>(p) + idx);
    return {t.x, t.y};
}

template <bool CPLX>
__device__ __forceinline__ void store(double *p, long long idx, const Val<CPLX> &v);
template <>
__device__ __forceinline__ void store<false>(double *p, long long idx, const Val<false> &v)
{
    p[idx] = v.x;
}
template <>
__device__ __forceinline__ void store<true>(double *p, long long idx, const Val<true> &v)
{
    reinterpret_cast<double2 *>(p)[idx] = make_double2(v.x, v.y);
}

template <bool CPLX, bool HAS_V>
__global__ void __launch_bounds__(256)
fd_generic_kernel(const FdGeom g, const double *__restrict__ psi, const double *__restrict__ v_eff,
                  double *__restrict__ out, long long nbands)
{
    const long long P = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long lin = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (lin >= P) return;
    const int iz = (int)(lin % g.n[2]);
    const int iy = (int)((lin / g.n[2]) % g.n[1]);
    const int ix = (int)(lin / ((long long)g.n[2] * g.n[1]));
    const int idx[3] = {ix, iy, iz};
    const long long stride[3] = {(long long)g.n[1] * g.n[2], (long long)g.n[2], 1};
    double diag = g.wdiag;
    if (HAS_V) diag += __ldg(v_eff + lin);

    for (long long b = blockIdx.y; b < nbands; b += gridDim.y) {
        const double *pb = psi + (CPLX ? 2 : 1) * b * P;
        const Val<CPLX> c = load<CPLX>(pb, lin);
        Val<CPLX> acc = Val<CPLX>::zero();
        acc.fma(diag, c);
        for (int d = 0; d < 3; ++d) {
            const int n = g.n[d];
            for (int j = 1; j <= g.nn; ++j) {
                const double w = g.w[d][j];
                // upper tap i + j
                int p = idx[d] + j;
                if (p < n) {
                    acc.fma(w, load<CPLX>(pb, lin + j * stride[d]));
                } else if (g.bc[d] == 1) {
                    const Val<CPLX> t = load<CPLX>(pb, lin + (long long)(j - n) * stride[d]);
                    acc.fma(w, t.mulphase(g.ph_re[d], g.ph_im[d]));
                }
                // lower tap i - j
                p = idx[d] - j;
                if (p >= 0) {
                    acc.fma(w, load<CPLX>(pb, lin - j * stride[d]));
                } else if (g.bc[d] == 1) {
                    const Val<CPLX> t = load<CPLX>(pb, lin + (long long)(n - j) * stride[d]);
                    acc.fma(w, t.mulphase(g.ph_re[d], -g.ph_im[d]));
                }
            }
        }
        store<CPLX>(out, b * P + lin, acc);
    }
}

}  // namespace

cudaError_t fd_launch_generic(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                              int64_t nbands, cudaStream_t stream)
{
    const FdGeom &g = plan->g;
    const long long P = (long long)g.n[0] * g.n[1] * g.n[2];
    dim3 block(256);
    dim3 grid((unsigned)((P + 255) / 256), (unsigned)(nbands < 32768 ? nbands : 32768));
    const double *p = static_cast<const double *>(psi);
    double *o = static_cast<double *>(out);
    if (g.cplx) {
        if (v_eff)
            fd_generic_kernel<true, true><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands);
        else
            fd_generic_kernel<true, false><<<grid, block, 0, stream>>>(g, p, nullptr, o, nbands);
    } else {
        if (v_eff)
            fd_generic_kernel<false, true><<<grid, block, 0, stream>>>(g, p, v_eff, o, nbands);
        else
            fd_generic_kernel<false, false><<<grid, block, 0, stream>>>(g, p, nullptr, o, nbands);
    }
    return cudaPeekAtLastError();
}
