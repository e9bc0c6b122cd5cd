// PAW non-local term with localised projector functions: the third term of Eq. 6,
//     out_b += sum_a sum_{i,i'} |p~^a_i> dO^a_{i i'} <p~^a_i'|psi_b>
// with dO = Delta H (Hamiltonian) or Delta S (overlap operator, Eq. 7);
// "overlaps between projector functions and wave functions" is the third C hot spot.
// Conventions (box of grid points per atom, Bloch factors on wrapped points, dv in the projection):
// include/fdham.h (fd_paw_create ...).  PAW data sets are not available: the projector functions
// are whatever the caller supplies (synthetic in tests and bench).
//
// Two kernels.  project: gather psi over each atom's box (an index table built at fd_paw_create
// resolves wrap / zero-BC clipping once), P_b[a,i] = dv sum_r p~_i(r) psi^_b(r); one warp per 4 bands
// of an atom, lanes over box points, 8 projector functions at a time in registers, fixed-order warp
// reduction (deterministic).
// add: out_b(r) += conj(phase) sum_i p~_i(r) (dO P_b)_i, one thread per box point; atoms are greedily
// coloured at create so that the boxes of one launch are disjoint: plain read-modify-write, no
// atomics, results independent of scheduling.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>

#include "fd_internal.h"

struct PawAtom {
    int npts;            // box points
    int ni;              // projector functions
    long long proj_off;  // first double of [ni][npts] in proj
    long long idx_off;   // first entry of the index / wrap-code tables
    int coef_off;        // first projector of this atom in a row of P
    int dmat_off;        // first double of [ni][ni] in dH / dS
    double ph0_re, ph0_im;  // Bloch factor of the lattice vector that moved the box start into the
                            // home cell: the projections are reported for the box as given
};

struct fd_paw {
    int device;
    int cplx;
    int natoms, ntot, ncolours;
    int has_phase;
    int n[3], bc[3];     // of the plan the tables were built for (fd_paw_matches)
    double h[3], k[3];
    size_t npoints;
    double dv;
    double ph_re[3], ph_im[3];
    PawAtom *atoms;      // device
    int *idx;            // device: home-cell linear index of every box point, -1 = dropped (zero BC)
    unsigned char *code; // device: bit d set = wrapped along axis d (nullptr when no Bloch phases)
    double *proj, *dH, *dS;
    int *colour_atoms;   // device: atom ids grouped by colour
    int *row_atom;       // device: atom of every row of P (ntot entries)
    std::vector<int> colour_start;  // host: ncolours + 1 offsets into colour_atoms
};

namespace {

constexpr int kPawThreads = 256;
constexpr int kMaxNi = 32;

template <bool CPLX>
struct Acc;
template <>
struct Acc<false> {
    double x;
    __device__ __forceinline__ void zero() { x = 0.0; }
    __device__ __forceinline__ void reduce()
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    }
};
template <>
struct Acc<true> {
    double x, y;
    __device__ __forceinline__ void zero() { x = y = 0.0; }
    __device__ __forceinline__ void reduce()
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            x += __shfl_xor_sync(0xffffffffu, x, o);
            y += __shfl_xor_sync(0xffffffffu, y, o);
        }
    }
};

struct Phases {
    double re[3], im[3];
};

// Bloch factor of a box point from its wrap code (box starts are normalised into the home cell at
// create, so a point wraps at most once, upwards, along each axis)
__device__ __forceinline__ void phase_of(unsigned code, const Phases &ph, double &pr, double &pi)
{
    pr = 1.0;
    pi = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d)
        if (code & (1u << d)) {
            const double r = pr * ph.re[d] - pi * ph.im[d];
            pi = pr * ph.im[d] + pi * ph.re[d];
            pr = r;
        }
}

// float64 plans at k_d = 1/2 (Bloch factors -1): the factor of a wrapped box point is the product of
// the +-1 of the wrapped axes
__device__ __forceinline__ double sign_of(unsigned code, const Phases &ph)
{
    double s = 1.0;
#pragma unroll
    for (int d = 0; d < 3; ++d)
        if (code & (1u << d)) s *= ph.re[d];
    return s;
}

// grid (atoms, tiles of 8 NB bands); coef[b][coef_off + i] = dv sum_r p~_i(r) psi^_b(r).
// A warp owns NB bands of the atom: lanes run over the box points, every lane keeps NI x NB partial
// sums (psi is gathered once per point and meets NI projector values), projector functions go by
// in chunks of NI; fixed shuffle tree at the end of a chunk.  The 8 warps of a CTA share the atom's
// projector values through L1.
// SG (float64 only): the plan has Bloch factors -1; a separate instantiation so that the Gamma-point
// code stays exactly what it was (the gather loop is sensitive to anything added to it).
template <bool CPLX, int NB, int NI, bool SG>
__global__ void __launch_bounds__(kPawThreads)
fd_paw_project_kernel(const PawAtom *__restrict__ atoms, const int *__restrict__ idx,
                      const unsigned char *__restrict__ code, const double *__restrict__ proj,
                      const double *__restrict__ psi, double *__restrict__ coef, long long band_d,
                      long long nbands, int ntot, double dv, const Phases ph)
{
    const PawAtom at = atoms[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long b0 = ((long long)blockIdx.y * (kPawThreads / 32) + warp) * NB;
    if (b0 >= nbands) return;
    const int *ix = idx + at.idx_off;
    const double *pb[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b)  // bands past the end re-read the last one and are not written
        pb[b] = psi + ((b0 + b < nbands) ? (b0 + b) : (nbands - 1)) * band_d;
    for (int i0 = 0; i0 < at.ni; i0 += NI) {
        const double *p = proj + at.proj_off + (long long)i0 * at.npts;
        Acc<CPLX> acc[NI][NB];
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int b = 0; b < NB; ++b) acc[i][b].zero();
        // dropped points (zero-BC clipping) take weight 0 at a valid address: no branch in the loop
#pragma unroll 2
        for (int r = lane; r < at.npts; r += 32) {
            const int gr = ix[r];
            const int gi = gr < 0 ? 0 : gr;
            Acc<CPLX> v[NB];
            if constexpr (CPLX) {
                double pr = 1.0, pi = 0.0;
                if (code) phase_of(code[at.idx_off + r], ph, pr, pi);
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    const double2 t = *reinterpret_cast<const double2 *>(pb[b] + 2LL * gi);
                    v[b].x = t.x * pr - t.y * pi;
                    v[b].y = t.x * pi + t.y * pr;
                }
            } else {
                if constexpr (SG) {
                    const double sg = sign_of(code[at.idx_off + r], ph);
#pragma unroll
                    for (int b = 0; b < NB; ++b) v[b].x = pb[b][gi] * sg;
                } else {
#pragma unroll
                    for (int b = 0; b < NB; ++b) v[b].x = pb[b][gi];
                }
            }
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                const double w = (gr < 0 || i0 + i >= at.ni) ? 0.0 : p[(long long)i * at.npts + r];
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    acc[i][b].x = fma(w, v[b].x, acc[i][b].x);
                    if constexpr (CPLX) acc[i][b].y = fma(w, v[b].y, acc[i][b].y);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                acc[i][b].reduce();
                if (lane == 0 && i0 + i < at.ni && b0 + b < nbands) {
                    double *c = coef + ((b0 + b) * ntot + at.coef_off + i0 + i) * (CPLX ? 2 : 1);
                    if constexpr (CPLX) {
                        c[0] = dv * (acc[i][b].x * at.ph0_re - acc[i][b].y * at.ph0_im);
                        c[1] = dv * (acc[i][b].x * at.ph0_im + acc[i][b].y * at.ph0_re);
                    } else {
                        if constexpr (SG)
                            c[0] = dv * (acc[i][b].x * at.ph0_re);  // +-1 (lattice shift at k = 1/2)
                        else
                            c[0] = dv * acc[i][b].x;
                    }
                }
            }
    }
}

// grid (atoms of one colour, band tiles); out_b(r') += conj(phase) sum_i p~_i(r) (dO P_b)_i
template <bool CPLX, int NB, bool SG>
__global__ void __launch_bounds__(kPawThreads)
fd_paw_add_kernel(const PawAtom *__restrict__ atoms, const int *__restrict__ colour_atoms,
                  const int *__restrict__ idx, const unsigned char *__restrict__ code,
                  const double *__restrict__ proj, const double *__restrict__ dmat,
                  const double *__restrict__ coef, double *__restrict__ out, long long band_d,
                  long long nbands, int ntot, const Phases ph)
{
    constexpr int E = CPLX ? 2 : 1;
    __shared__ double d[kMaxNi][NB][E];  // d[i][b] = sum_i' dO[i][i'] P_b[i']
    const PawAtom at = atoms[colour_atoms[blockIdx.x]];
    const long long b0 = (long long)blockIdx.y * NB;
    for (int e = threadIdx.x; e < at.ni * NB; e += kPawThreads) {
        const int i = e / NB, b = e - i * NB;
        double sx = 0.0, sy = 0.0;
        if (b0 + b < nbands) {
            const double *c = coef + ((b0 + b) * ntot + at.coef_off) * E;
            const double *m = dmat + at.dmat_off + i * at.ni;
            for (int i2 = 0; i2 < at.ni; ++i2) {
                sx = fma(m[i2], c[i2 * E], sx);
                if (CPLX) sy = fma(m[i2], c[i2 * E + 1], sy);
            }
        }
        if (CPLX) {  // back to the home-cell box: times conj(ph0)
            d[i][b][0] = sx * at.ph0_re + sy * at.ph0_im;
            d[i][b][E - 1] = sy * at.ph0_re - sx * at.ph0_im;
        } else {
            d[i][b][0] = SG ? sx * at.ph0_re : sx;
        }
    }
    __syncthreads();
    const int *ix = idx + at.idx_off;
    for (int r = threadIdx.x; r < at.npts; r += kPawThreads) {
        const int gi = ix[r];
        if (gi < 0) continue;  // dropped by zero-BC clipping
        double sx[NB], sy[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) sx[b] = sy[b] = 0.0;
#pragma unroll 4
        for (int i = 0; i < at.ni; ++i) {
            const double w = proj[at.proj_off + (long long)i * at.npts + r];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                sx[b] = fma(w, d[i][b][0], sx[b]);
                if (CPLX) sy[b] = fma(w, d[i][b][E - 1], sy[b]);
            }
        }
        if constexpr (CPLX) {
            double pr = 1.0, pi = 0.0;
            if (code) phase_of(code[at.idx_off + r], ph, pr, pi);
#pragma unroll
            for (int b = 0; b < NB; ++b)
                if (b0 + b < nbands) {
                    double2 *o = reinterpret_cast<double2 *>(out + (b0 + b) * band_d + 2LL * gi);
                    double2 v = *o;
                    v.x += sx[b] * pr + sy[b] * pi;   // times conj(phase)
                    v.y += sy[b] * pr - sx[b] * pi;
                    *o = v;
                }
        } else {
            if constexpr (SG) {
                const double sg = sign_of(code[at.idx_off + r], ph);
#pragma unroll
                for (int b = 0; b < NB; ++b)
                    if (b0 + b < nbands) out[(b0 + b) * band_d + gi] += sx[b] * sg;
            } else {
#pragma unroll
                for (int b = 0; b < NB; ++b)
                    if (b0 + b < nbands) out[(b0 + b) * band_d + gi] += sx[b];
            }
        }
    }
}

// grid (bands): out[b] += (1/dv) Re sum_a sum_ii' conj(P_b[a,i]) dO^a_ii' P_b[a,i'] -- the PAW part of
// <psi_b|H~|psi_b> (or of <psi_b|S~|psi_b>) from the projections.  One CTA per band, threads over
// (atom, i) rows in a fixed order, fixed shuffle / shared-memory tree: deterministic.
template <bool CPLX>
__global__ void __launch_bounds__(kPawThreads)
fd_paw_expect_kernel(const PawAtom *__restrict__ atoms, int natoms, const int *__restrict__ row_atom,
                     const double *__restrict__ dmat, const double *__restrict__ coef,
                     double *__restrict__ out, int ntot, double inv_dv)
{
    constexpr int E = CPLX ? 2 : 1;
    const long long b = blockIdx.x;
    const double *c = coef + b * ntot * E;
    double s = 0.0;
    for (int row = threadIdx.x; row < ntot; row += kPawThreads) {
        const PawAtom at = atoms[row_atom[row]];
        const int i = row - at.coef_off;
        const double *m = dmat + at.dmat_off + i * at.ni;
        const double *ca = c + at.coef_off * E;
        double tx = 0.0, ty = 0.0;
        for (int i2 = 0; i2 < at.ni; ++i2) {
            tx = fma(m[i2], ca[i2 * E], tx);
            if (CPLX) ty = fma(m[i2], ca[i2 * E + 1], ty);
        }
        s = fma(ca[i * E], tx, s);                 // Re conj(P_i) t
        if (CPLX) s = fma(ca[i * E + 1], ty, s);
    }
    (void)natoms;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ double part[kPawThreads / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < kPawThreads / 32; ++w) t += part[w];
        out[b] += inv_dv * t;
    }
}

template <typename T>
bool upload(T **dev, const void *host, size_t count)
{
    *dev = nullptr;
    if (count == 0) return true;
    if (cudaMalloc(dev, count * sizeof(T)) != cudaSuccess) return false;
    return cudaMemcpy(*dev, host, count * sizeof(T), cudaMemcpyHostToDevice) == cudaSuccess;
}

// do the index intervals [s, s + len) of two boxes meet along an axis of n points?
bool axis_overlap(int s1, int l1, int s2, int l2, int n, int periodic)
{
    if (!periodic) return s1 < s2 + l2 && s2 < s1 + l1;  // clipping to [0, n) cannot create overlap
    if (l1 >= n || l2 >= n) return true;
    // starts are normalised into [0, n): compare on the circle
    for (int shift = -1; shift <= 1; ++shift) {
        const int t2 = s2 + shift * n;
        if (s1 < t2 + l2 && t2 < s1 + l1) return true;
    }
    return false;
}

}  // namespace

int fd_paw_build(fd_paw **out, const fd_plan *plan, int natoms, const int32_t *box_start,
                 const int32_t *box_size, const int32_t *nproj, const double *proj_host,
                 const double *dh_host, const double *ds_host)
{
    const FdGeom &g = plan->g;
    const long long P = (long long)g.n[0] * g.n[1] * g.n[2];
    if (P >= (1LL << 31)) return -2;
    fd_paw *w = new (std::nothrow) fd_paw();
    if (!w) return -5;
    w->device = plan->device;
    w->cplx = g.cplx;
    w->natoms = natoms;
    w->npoints = (size_t)P;
    w->dv = plan->h[0] * plan->h[1] * plan->h[2];
    w->has_phase = 0;
    for (int d = 0; d < 3; ++d) {
        w->n[d] = g.n[d];
        w->bc[d] = g.bc[d];
        w->h[d] = plan->h[d];
        w->k[d] = plan->k[d];
        w->ph_re[d] = g.ph_re[d];
        w->ph_im[d] = g.ph_im[d];
        if (g.bc[d] && (g.ph_re[d] != 1.0 || g.ph_im[d] != 0.0)) w->has_phase = 1;
    }
    w->atoms = nullptr;
    w->idx = nullptr;
    w->code = nullptr;
    w->proj = w->dH = w->dS = nullptr;
    w->colour_atoms = nullptr;
    w->row_atom = nullptr;

    std::vector<PawAtom> atoms((size_t)natoms);
    std::vector<int> start((size_t)natoms * 3);
    long long npts_total = 0, proj_total = 0, dmat_total = 0;
    int ntot = 0;
    for (int a = 0; a < natoms; ++a) {
        const int32_t *sz = box_size + 3 * a;
        if (nproj[a] < 1 || nproj[a] > kMaxNi) { delete w; return nproj[a] > kMaxNi ? -2 : -1; }
        double shift_phase = 0.0;
        int shift_odd = 0;  // float64 plans: parity of the cells moved along the axes with factor -1
        for (int d = 0; d < 3; ++d) {
            if (sz[d] < 1) { delete w; return -1; }
            if (g.bc[d] && sz[d] > g.n[d]) { delete w; return -2; }  // a box may not meet itself
            int s = box_start[3 * a + d];
            if (g.bc[d]) {  // lattice translations leave the operator unchanged: home-cell start
                int w0 = s / g.n[d];
                if (s - w0 * g.n[d] < 0) --w0;  // floor
                s -= w0 * g.n[d];
                shift_phase += 2.0 * 3.14159265358979323846264338327950288 * plan->k[d] * (double)w0;
                if (g.ph_re[d] < 0.0) shift_odd ^= (w0 & 1);
            }
            start[3 * a + d] = s;
        }
        atoms[a].ph0_re = (shift_phase == 0.0) ? 1.0 : cos(shift_phase);
        atoms[a].ph0_im = (shift_phase == 0.0) ? 0.0 : sin(shift_phase);
        if (!g.cplx) {  // Bloch factors are exactly +-1 (2 k_d integer): no rounding from cos / sin
            atoms[a].ph0_re = shift_odd ? -1.0 : 1.0;
            atoms[a].ph0_im = 0.0;
        }
        const long long np = (long long)sz[0] * sz[1] * sz[2];
        if (np > (1LL << 30)) { delete w; return -2; }
        atoms[a].npts = (int)np;
        atoms[a].ni = nproj[a];
        atoms[a].proj_off = proj_total;
        atoms[a].idx_off = npts_total;
        atoms[a].coef_off = ntot;
        atoms[a].dmat_off = (int)dmat_total;
        npts_total += np;
        proj_total += np * nproj[a];
        dmat_total += (long long)nproj[a] * nproj[a];
        ntot += nproj[a];
    }
    w->ntot = ntot;
    std::vector<int> idx((size_t)npts_total);
    std::vector<unsigned char> code((size_t)npts_total);
    for (int a = 0; a < natoms; ++a) {
        const int32_t *sz = box_size + 3 * a;
        long long e = atoms[a].idx_off;
        for (int rx = 0; rx < sz[0]; ++rx)
            for (int ry = 0; ry < sz[1]; ++ry)
                for (int rz = 0; rz < sz[2]; ++rz, ++e) {
                    int p[3] = {start[3 * a] + rx, start[3 * a + 1] + ry, start[3 * a + 2] + rz};
                    unsigned c = 0;
                    bool dropped = false;
                    for (int d = 0; d < 3; ++d)
                        if (p[d] < 0 || p[d] >= g.n[d]) {
                            if (!g.bc[d]) { dropped = true; break; }
                            p[d] -= g.n[d];
                            c |= 1u << d;
                        }
                    idx[e] = dropped ? -1 : (int)(((long long)p[0] * g.n[1] + p[1]) * g.n[2] + p[2]);
                    code[e] = (unsigned char)c;
                }
    }
    // greedy colouring: atoms of one colour have pairwise disjoint boxes
    std::vector<int> colour((size_t)natoms, -1);
    int ncol = 0;
    for (int a = 0; a < natoms; ++a) {
        std::vector<char> used((size_t)ncol + 1, 0);
        for (int b = 0; b < a; ++b) {
            bool meet = true;
            for (int d = 0; d < 3 && meet; ++d)
                meet = axis_overlap(start[3 * a + d], box_size[3 * a + d], start[3 * b + d],
                                    box_size[3 * b + d], g.n[d], g.bc[d]);
            if (meet) used[colour[b]] = 1;
        }
        int c = 0;
        while (used[c]) ++c;
        colour[a] = c;
        if (c == ncol) ++ncol;
    }
    w->ncolours = ncol;
    std::vector<int> order;
    w->colour_start.assign((size_t)ncol + 1, 0);
    for (int c = 0; c < ncol; ++c) {
        w->colour_start[c] = (int)order.size();
        for (int a = 0; a < natoms; ++a)
            if (colour[a] == c) order.push_back(a);
    }
    w->colour_start[ncol] = (int)order.size();

    bool ok = upload(&w->atoms, atoms.data(), atoms.size()) && upload(&w->idx, idx.data(), idx.size()) &&
              upload(&w->proj, proj_host, (size_t)proj_total) &&
              upload(&w->colour_atoms, order.data(), order.size());
    std::vector<int> row_atom;
    for (int a = 0; a < natoms; ++a)
        for (int i = 0; i < atoms[a].ni; ++i) row_atom.push_back(a);
    if (ok) ok = upload(&w->row_atom, row_atom.data(), row_atom.size());
    if (ok && w->has_phase) ok = upload(&w->code, code.data(), code.size());
    if (ok && dh_host) ok = upload(&w->dH, dh_host, (size_t)dmat_total);
    if (ok && ds_host) ok = upload(&w->dS, ds_host, (size_t)dmat_total);
    if (!ok) {
        cudaGetLastError();
        fd_paw_free(w);
        return -5;
    }
    *out = w;
    return 0;
}

void fd_paw_free(fd_paw *w)
{
    if (!w) return;
    cudaFree(w->atoms);
    cudaFree(w->idx);
    cudaFree(w->code);
    cudaFree(w->proj);
    cudaFree(w->dH);
    cudaFree(w->dS);
    cudaFree(w->colour_atoms);
    cudaFree(w->row_atom);
    cudaGetLastError();
    delete w;
}

int fd_paw_ntot(const fd_paw *w) { return w->ntot; }
int fd_paw_has(const fd_paw *w, int which) { return which ? w->dS != nullptr : w->dH != nullptr; }
// The index tables, Bloch factors and dv belong to the plan the set was built for: another plan is
// accepted only if it describes the same grid (shape, spacing, boundaries, k, dtype, device).
int fd_paw_matches(const fd_paw *w, const fd_plan *plan)
{
    if (w->device != plan->device || w->cplx != plan->g.cplx) return 0;
    for (int d = 0; d < 3; ++d)
        if (w->n[d] != plan->g.n[d] || w->bc[d] != plan->g.bc[d] || w->h[d] != plan->h[d] ||
            w->k[d] != plan->k[d])
            return 0;
    return 1;
}

cudaError_t fd_paw_launch_project(const fd_paw *w, const void *psi, void *coef, int64_t nbands,
                                  cudaStream_t stream, int *nlaunches)
{
    if (w->natoms == 0 || nbands == 0) return cudaSuccess;
    Phases ph;
    for (int d = 0; d < 3; ++d) {
        ph.re[d] = w->ph_re[d];
        ph.im[d] = w->ph_im[d];
    }
    const long long band_d = (long long)w->npoints * (w->cplx ? 2 : 1);
    const int tile = 2 * (kPawThreads / 32);  // bands per CTA: 2 per warp
    for (int64_t b0 = 0; b0 < nbands; b0 += 65535LL * tile) {
        const int64_t nb = (nbands - b0 < 65535LL * tile) ? nbands - b0 : 65535LL * tile;
        const dim3 grid((unsigned)w->natoms, (unsigned)((nb + tile - 1) / tile));
        const double *p = static_cast<const double *>(psi) + b0 * band_d;
        double *c = static_cast<double *>(coef) + b0 * w->ntot * (w->cplx ? 2 : 1);
        if (w->cplx)
            fd_paw_project_kernel<true, 2, 8, false><<<grid, kPawThreads, 0, stream>>>(
                w->atoms, w->idx, w->code, w->proj, p, c, band_d, nb, w->ntot, w->dv, ph);
        else if (w->code)  // float64 at k = 1/2
            fd_paw_project_kernel<false, 2, 16, true><<<grid, kPawThreads, 0, stream>>>(
                w->atoms, w->idx, w->code, w->proj, p, c, band_d, nb, w->ntot, w->dv, ph);
        else
            fd_paw_project_kernel<false, 2, 16, false><<<grid, kPawThreads, 0, stream>>>(
                w->atoms, w->idx, w->code, w->proj, p, c, band_d, nb, w->ntot, w->dv, ph);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
        if (nlaunches) ++*nlaunches;
    }
    return cudaSuccess;
}

cudaError_t fd_paw_launch_add(const fd_paw *w, int which, const void *coef, void *out, int64_t nbands,
                              cudaStream_t stream, int *nlaunches)
{
    if (w->natoms == 0 || nbands == 0) return cudaSuccess;
    Phases ph;
    for (int d = 0; d < 3; ++d) {
        ph.re[d] = w->ph_re[d];
        ph.im[d] = w->ph_im[d];
    }
    const double *dm = which ? w->dS : w->dH;
    const long long band_d = (long long)w->npoints * (w->cplx ? 2 : 1);
    const int NB = w->cplx ? 4 : 8;
    for (int c = 0; c < w->ncolours; ++c) {
        const int na = w->colour_start[c + 1] - w->colour_start[c];
        for (int64_t b0 = 0; b0 < nbands; b0 += 65535LL * NB) {
            const int64_t nb = (nbands - b0 < 65535LL * NB) ? nbands - b0 : 65535LL * NB;
            const dim3 grid((unsigned)na, (unsigned)((nb + NB - 1) / NB));
            const double *cf = static_cast<const double *>(coef) + b0 * w->ntot * (w->cplx ? 2 : 1);
            double *o = static_cast<double *>(out) + b0 * band_d;
            if (w->cplx)
                fd_paw_add_kernel<true, 4, false><<<grid, kPawThreads, 0, stream>>>(
                    w->atoms, w->colour_atoms + w->colour_start[c], w->idx, w->code, w->proj, dm, cf,
                    o, band_d, nb, w->ntot, ph);
            else if (w->code)  // float64 at k = 1/2
                fd_paw_add_kernel<false, 8, true><<<grid, kPawThreads, 0, stream>>>(
                    w->atoms, w->colour_atoms + w->colour_start[c], w->idx, w->code, w->proj, dm, cf,
                    o, band_d, nb, w->ntot, ph);
            else
                fd_paw_add_kernel<false, 8, false><<<grid, kPawThreads, 0, stream>>>(
                    w->atoms, w->colour_atoms + w->colour_start[c], w->idx, w->code, w->proj, dm, cf,
                    o, band_d, nb, w->ntot, ph);
            cudaError_t e = cudaPeekAtLastError();
            if (e != cudaSuccess) return e;
            if (nlaunches) ++*nlaunches;
        }
    }
    return cudaSuccess;
}

cudaError_t fd_paw_launch_expect(const fd_paw *w, int which, const void *coef, double *out, int64_t nbands,
                                 cudaStream_t stream, int *nlaunches)
{
    if (w->natoms == 0 || nbands == 0) return cudaSuccess;
    const double *dm = which ? w->dS : w->dH;
    for (int64_t b0 = 0; b0 < nbands; b0 += 0x7fffffffLL) {
        const int64_t nb = (nbands - b0 < 0x7fffffffLL) ? nbands - b0 : 0x7fffffffLL;
        const double *c = static_cast<const double *>(coef) + b0 * w->ntot * (w->cplx ? 2 : 1);
        if (w->cplx)
            fd_paw_expect_kernel<true><<<(unsigned)nb, kPawThreads, 0, stream>>>(
                w->atoms, w->natoms, w->row_atom, dm, c, out + b0, w->ntot, 1.0 / w->dv);
        else
            fd_paw_expect_kernel<false><<<(unsigned)nb, kPawThreads, 0, stream>>>(
                w->atoms, w->natoms, w->row_atom, dm, c, out + b0, w->ntot, 1.0 / w->dv);
        cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
        if (nlaunches) ++*nlaunches;
    }
    return cudaSuccess;
}
