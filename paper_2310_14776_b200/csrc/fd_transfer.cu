// Grid transfer between a fine grid (spacing h) and the coarse grid of spacing 2h: restriction and
// interpolation ("interpolating from one uniform grid to another" is the second C
// hot spot the paper lists; multigrid Poisson / preconditioner).
// Operation and index conventions: include/fdham.h (fd_restrict / fd_interpolate), DESIGN.md
// readings R13 (midpoint Lagrange weights b_j of order p, restriction = interpolation^T / 8) and
// R14 (coarse point I on fine point 2I + off, off = 0 periodic / 1 zero-BC).
//
// Both kernels are tensor-product sweeps along x.  A CTA owns a tile of coarse y rows x the full
// z row and a chunk of coarse x planes; every plane it brings in is staged in shared memory with
// its z halo resolved (wrapped or zero), reduced / expanded along z and then along y by two small
// separable passes, and combined along x in REGISTERS:
//   restriction   -- scatter: the y-z-restricted fine plane adds r_a s to the 2p coarse planes in
//                    flight (a shifting register queue); a coarse plane is stored when complete;
//   interpolation -- gather: the y-z-interpolated coarse plane enters a queue of 2p planes; the
//                    even fine plane is the plane itself, the odd one the b_j-weighted sum.
// Each fine value therefore crosses HBM once (plus the tile / chunk halos, which hit L2).
#include <atomic>

#include "fd_internal.h"

namespace {

constexpr int kThreads = 512;
constexpr int kMaxPt = 8;   // output points of the swept plane per thread

struct TGeom {
    int nf[3], nc[3], bc[3], off[3];
    double b[4];  // b[1..p]: midpoint Lagrange weights
};

// z index of a padded row -> source index in [0, n) or -1 (zero)
// (one wrap by an add / subtract; the integer modulo -- ~40 instructions, and this is called for every
// halo word of every staged row -- only for grids shorter than the halo)
__device__ __forceinline__ int wrap_or_zero(int i, int n, int periodic)
{
    if (i >= 0 && i < n) return i;
    if (!periodic) return -1;
    i += (i < 0) ? n : -n;
    if (i >= 0 && i < n) return i;
    i %= n;
    return i < 0 ? i + n : i;
}

// Stage `rows` rows of a plane in shared memory, z halo resolved: dst[rr][0 .. n + 2 pad), source row
// index y0 + rr and z index zp - pad, both wrapped (periodic) or zero.  One warp per row, lanes
// along z: coalesced, no division.
__device__ __forceinline__ void stage_rows(double *dst, const double *__restrict__ plane, int rows,
                                           int y0, int ny, int per_y, int n, int pad, int per_z)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int pitch = n + 2 * pad;
    for (int rr = warp; rr < rows; rr += kThreads / 32) {
        const int y = wrap_or_zero(y0 + rr, ny, per_y);
        double *d = dst + rr * pitch;
        if (y < 0) {
            for (int z = lane; z < pitch; z += 32) d[z] = 0.0;
            continue;
        }
        const double *srow = plane + (long long)y * n;
        for (int z = lane; z < n; z += 32) d[pad + z] = __ldg(srow + z);
        if (lane < 2 * pad) {  // pad <= 5: one lane per halo word
            const int zp = (lane < pad) ? lane : n + lane;          // padded index
            const int z = wrap_or_zero(zp - pad, n, per_z);
            d[zp] = z < 0 ? 0.0 : __ldg(srow + z);
        }
    }
}

// The same, asynchronously: every in-range word is an 8-byte cp.async (LDGSTS: no registers, the
// thread goes on), zeros are stored directly; the caller commits the group and waits for it one
// plane later, so the loads of plane t + 1 overlap the passes over plane t.
__device__ __forceinline__ void cp_async8(double *dst, const double *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(
                     static_cast<uint32_t>(__cvta_generic_to_shared(dst))),
                 "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void cp_async16(double *dst, const double *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(
                     static_cast<uint32_t>(__cvta_generic_to_shared(dst))),
                 "l"(src)
                 : "memory");
}
// pitch >= n + 2 pad: words per staged row (the caller may add slack / keep it even)
__device__ __forceinline__ void stage_rows_async(double *dst, const double *__restrict__ plane,
                                                 int rows, int y0, int ny, int per_y, int n, int pad,
                                                 int per_z, int pitch)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // 16-byte copies when every source row and every destination row start is 16-byte aligned
    const bool vec = !(n & 1) && !(pad & 1) && !(pitch & 1) &&
                     !(reinterpret_cast<uintptr_t>(plane) & 15);
    for (int rr = warp; rr < rows; rr += kThreads / 32) {
        const int y = wrap_or_zero(y0 + rr, ny, per_y);
        double *d = dst + rr * pitch;
        if (y < 0) {
            for (int z = lane; z < n + 2 * pad; z += 32) d[z] = 0.0;
            continue;
        }
        const double *srow = plane + (long long)y * n;
        if (vec) {
            for (int z = 2 * lane; z < n; z += 64) cp_async16(d + pad + z, srow + z);
        } else {
            for (int z = lane; z < n; z += 32) cp_async8(d + pad + z, srow + z);
        }
        if (lane < 2 * pad) {  // pad <= 5: one lane per halo word
            const int zp = (lane < pad) ? lane : n + lane;          // padded index
            const int z = wrap_or_zero(zp - pad, n, per_z);
            if (z < 0) d[zp] = 0.0;
            else cp_async8(d + zp, srow + z);
        }
    }
}

// ---------------------------------------------------------------------------------- restriction
// blockIdx.x: coarse y tile (jt rows), blockIdx.y: chunk of ic coarse x planes, blockIdx.z: band.
// NPT: coarse points of the swept plane per thread (point e = tid + n * kThreads of the jt x kc tile).
// Two CTAs per SM (64 registers; measured +17 % over one CTA at 110 registers).
template <int P, int NPT>
__global__ void __launch_bounds__(kThreads, 2)
fd_restrict_kernel(const __grid_constant__ TGeom g, const double *__restrict__ fine,
                   double *__restrict__ coarse, int jt, int ic)
{
    constexpr int M = 2 * P - 1;  // reach of the 1-D restriction in fine points
    extern __shared__ double sm[];
    const int nzf = g.nf[2], kc = g.nc[2];
    // z halo of pad >= M words per side, chosen so that the word under coarse point k sits at the even
    // index 2 P + 2 k of the staged row (16-byte window loads in the z pass); + 4 words of slack for
    // the window of the last run
    const int pad = M + 1 - g.off[2];
    const int fp = (nzf + 2 * pad + 4 + 1) & ~1;  // words per staged fine row
    const int rows = 2 * jt - 1 + 2 * M;      // fine rows staged per plane
    double *F0 = sm;                          // 2 x [rows][fp]: the plane in use and the plane in flight
    double *T = sm + 2 * (size_t)rows * fp;   // [rows][kc]  z-restricted rows
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int J0 = blockIdx.x * jt, nj = min(jt, g.nc[1] - J0);
    const int I0 = blockIdx.y * ic, ni = min(ic, g.nc[0] - I0);
    const long long band = blockIdx.z;
    const double *fb = fine + band * ((long long)g.nf[0] * g.nf[1] * nzf);
    double *cb = coarse + band * ((long long)g.nc[0] * g.nc[1] * kc);
    const int yf0 = 2 * J0 + g.off[1] - M;    // fine row of staged row 0
    const int oz = g.off[2];
    double r[P + 1];                          // 1-D restriction weights: 1/2 and b_j / 2
    r[0] = 0.5;
#pragma unroll
    for (int j = 1; j <= P; ++j) r[j] = 0.5 * g.b[j];

    // this thread's points: offset of the centre row in T, offset in a coarse plane (-1: none)
    int toff[NPT], coff[NPT];
#pragma unroll
    for (int n = 0; n < NPT; ++n) {
        const int e = tid + n * kThreads;
        const int j = e / kc, k = e - j * kc;
        const bool in_tile = e < jt * kc;
        toff[n] = in_tile ? (2 * j + M) * kc + k : M * kc;
        coff[n] = (in_tile && j < nj) ? (J0 + j) * kc + k : -1;
    }
    double acc[2 * P][NPT];                   // coarse planes base .. base + 2P - 1 in flight
#pragma unroll
    for (int a = 0; a < 2 * P; ++a)
#pragma unroll
        for (int n = 0; n < NPT; ++n) acc[a][n] = 0.0;

    // The planes the sweep consumes, in order: step t = 2 (c - c0) + phase, phase 0 = the odd plane
    // d = 2c + 1, phase 1 = the even plane d = 2c + 2 (used only when coarse c + 1 is in the chunk).
    const int c0 = I0 - P, nsteps = 2 * (ni + 2 * P - 1);
    auto plane_of = [&](int t) -> int {  // fine x index of step t, or -1 when the step has no plane
        const int c = c0 + (t >> 1);
        if ((t & 1) && !(c + 1 >= I0 && c + 1 < I0 + ni)) return -1;
        return wrap_or_zero(2 * c + 1 + (t & 1) + g.off[0], g.nf[0], g.bc[0]);
    };
    auto next_plane = [&](int t) -> int {  // first step after t that has a plane (nsteps: none)
        for (++t; t < nsteps && plane_of(t) < 0; ++t) {
        }
        return t;
    };
    auto issue = [&](int t, int buf) {
        stage_rows_async(F0 + (size_t)buf * rows * fp, fb + (long long)plane_of(t) * g.nf[1] * nzf, rows,
                         yf0, g.nf[1], g.bc[1], nzf, pad, g.bc[2], fp);
        cp_async_commit();
    };
    int t_next = next_plane(-1), buf = 0;  // the plane in flight into F0[buf]
    if (t_next < nsteps) issue(t_next, 0);

    // y-z restriction of the next plane of the sequence into s[] for the owned points
    auto plane = [&](double (&s)[NPT]) {
        const double *F = F0 + (size_t)buf * rows * fp;
        const int t_after = next_plane(t_next);
        if (t_after < nsteps) {  // F0[buf ^ 1] was last read before the previous plane's second barrier
            issue(t_after, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        t_next = t_after;
        buf ^= 1;
        __syncthreads();  // this plane has landed for every thread; the previous T is no longer read
        // z pass: a lane takes runs of 3 adjacent coarse points; their 4 P + 4 fine words start at the
        // even word 2 k0 of the staged row: 2 P + 2 conflict-free 16-byte loads for 3 outputs
        for (int rr = warp; rr < rows; rr += kThreads / 32) {
            const double *row = F + rr * fp;
            for (int k0 = 3 * lane; k0 < kc; k0 += 96) {
                double win[4 * P + 4];
#pragma unroll
                for (int i = 0; i < 2 * P + 2; ++i) {
                    const double2 w2 = *reinterpret_cast<const double2 *>(row + 2 * k0 + 2 * i);
                    win[2 * i] = w2.x;
                    win[2 * i + 1] = w2.y;
                }
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    double t = r[0] * win[2 * P + 2 * q];
#pragma unroll
                    for (int j = 1; j <= P; ++j)
                        t = fma(r[j], win[2 * P + 2 * q - (2 * j - 1)] + win[2 * P + 2 * q + (2 * j - 1)], t);
                    if (k0 + q < kc) T[rr * kc + k0 + q] = t;
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int n = 0; n < NPT; ++n) {
            const double *col = T + toff[n];
            double t = r[0] * col[0];
#pragma unroll
            for (int q = 1; q <= P; ++q)
                t = fma(r[q], col[-(2 * q - 1) * kc] + col[(2 * q - 1) * kc], t);
            s[n] = t;
        }
    };

    // iteration c: odd fine plane d = 2c + 1 (between coarse c and c + 1), then even plane d = 2c + 2
    // (on coarse c + 1); d = fine x index - off_x.  acc[0] is coarse plane base = c + 1 - P.
    for (int c = I0 - P; c <= I0 + ni + P - 2; ++c) {
        double s[NPT];
        {
            if (plane_of(2 * (c - c0)) >= 0) {
                plane(s);
#pragma unroll
                for (int j = 1; j <= P; ++j)
#pragma unroll
                    for (int n = 0; n < NPT; ++n) {
                        acc[P - j][n] = fma(r[j], s[n], acc[P - j][n]);          // coarse c + 1 - j
                        acc[P + j - 1][n] = fma(r[j], s[n], acc[P + j - 1][n]);  // coarse c + j
                    }
            }
        }
        const int base = c + 1 - P;  // complete after the odd plane
        if (base >= I0 && base < I0 + ni) {
            double *cp = cb + (long long)base * g.nc[1] * kc;
#pragma unroll
            for (int n = 0; n < NPT; ++n)
                if (coff[n] >= 0) __stcs(cp + coff[n], acc[0][n]);
        }
#pragma unroll
        for (int a = 0; a + 1 < 2 * P; ++a)
#pragma unroll
            for (int n = 0; n < NPT; ++n) acc[a][n] = acc[a + 1][n];
#pragma unroll
        for (int n = 0; n < NPT; ++n) acc[2 * P - 1][n] = 0.0;
        // even plane on coarse c + 1 (slot P - 1 after the shift)
        if (plane_of(2 * (c - c0) + 1) >= 0) {
            plane(s);
#pragma unroll
            for (int n = 0; n < NPT; ++n) acc[P - 1][n] = fma(r[0], s[n], acc[P - 1][n]);
        }
    }
}

// -------------------------------------------------------------------------------- interpolation
// blockIdx.x: coarse y tile (jt rows -> 2 jt fine rows, + the fine row below the first coarse row
// on a zero-BC axis), blockIdx.y: chunk of ic coarse x planes, blockIdx.z: band.
// NPT: fine-plane points per thread (point e = tid + n * kThreads of the (2 jt + 1) x nzf tile).
template <int P, int NPT>
__global__ void __launch_bounds__(kThreads)
fd_interp_kernel(const __grid_constant__ TGeom g, const double *__restrict__ coarse,
                 double *__restrict__ fine, int jt, int ic)
{
    extern __shared__ double sm[];
    const int nzf = g.nf[2], kc = g.nc[2];
    const int cp = kc + 2 * P;                // padded coarse row
    const int rows = jt + 2 * P;              // coarse rows staged per plane: J0 - P .. J0 + jt + P - 1
    double *C0 = sm;                          // 2 x [rows][cp]: the plane in use and the plane in flight
    double *T = sm + 2 * (size_t)rows * cp;   // [rows][nzf]  z-interpolated rows
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int J0 = blockIdx.x * jt, nj = min(jt, g.nc[1] - J0);
    const int I0 = blockIdx.y * ic, ni = min(ic, g.nc[0] - I0);
    const long long band = blockIdx.z;
    const double *cb = coarse + band * ((long long)g.nc[0] * g.nc[1] * kc);
    double *fb = fine + band * ((long long)g.nf[0] * g.nf[1] * nzf);
    const int oy = g.off[1], oz = g.off[2], ox = g.off[0];
    double b[P + 1];
#pragma unroll
    for (int j = 1; j <= P; ++j) b[j] = g.b[j];

    // local fine rows l = 0 .. 2 jt: e_y = 2 J0 - 1 + l (e = fine index - off); row 0 is the midpoint
    // below the tile's first coarse row: it belongs to this tile only at a zero-BC lower wall.
    const int ey_lo = (J0 == 0 && oy == 1) ? -1 : 2 * J0;
    const int ey_hi = min(2 * (J0 + nj), g.nf[1] - oy);  // exclusive
    // this thread's points: T offset of the (lower) coarse row, odd-row flag, fine-plane offset (-1: none)
    int toff[NPT], foff[NPT];
    unsigned oddmask = 0;
#pragma unroll
    for (int n = 0; n < NPT; ++n) {
        const int e = tid + n * kThreads;
        const int l = e / nzf, fz = e - l * nzf;
        const bool in_tile = e < (2 * jt + 1) * nzf;
        const int ey = 2 * J0 - 1 + l;
        const bool odd = (ey & 1) != 0;
        // staged row of coarse row cy is cy - J0 + P; odd rows: lower neighbour c = (ey - 1) / 2
        const int crow = (odd ? ((ey - 1) >> 1) : (ey >> 1)) - J0 + P;
        toff[n] = in_tile ? crow * nzf + fz : P * nzf;
        if (odd && in_tile) oddmask |= 1u << n;
        foff[n] = (in_tile && ey >= ey_lo && ey < ey_hi) ? (ey + oy) * nzf + fz : -1;
    }

    double sq[2 * P][NPT];  // y-z-interpolated coarse planes i - 2P + 1 .. i
#pragma unroll
    for (int a = 0; a < 2 * P; ++a)
#pragma unroll
        for (int n = 0; n < NPT; ++n) sq[a][n] = 0.0;

    // the chunk owns the even planes e_x = 2 i, i in [I0, I0 + ni), and the odd planes e_x = 2 c + 1,
    // c in [c_first, I0 + ni): c_first = -1 for the first chunk on a zero-BC axis (the wall), else I0
    const int c_first = (I0 == 0 && ox == 1) ? -1 : I0;
    const int i_lo = c_first + 1 - P, i_hi = I0 + ni - 1 + P;  // coarse planes the sweep brings in
    auto next_plane = [&](int i) -> int {  // first plane after i that exists (i_hi + 1: none)
        for (++i; i <= i_hi && wrap_or_zero(i, g.nc[0], g.bc[0]) < 0; ++i) {
        }
        return i;
    };
    auto issue = [&](int i, int buf) {
        stage_rows_async(C0 + (size_t)buf * rows * cp,
                         cb + (long long)wrap_or_zero(i, g.nc[0], g.bc[0]) * g.nc[1] * kc, rows, J0 - P,
                         g.nc[1], g.bc[1], kc, P, g.bc[2], cp);
        cp_async_commit();
    };
    int i_next = next_plane(i_lo - 1), buf = 0;
    if (i_next <= i_hi) issue(i_next, 0);

    auto plane = [&](double (&s)[NPT]) {
        const double *C = C0 + (size_t)buf * rows * cp;
        const int i_after = next_plane(i_next);
        if (i_after <= i_hi) {
            issue(i_after, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        i_next = i_after;
        buf ^= 1;
        __syncthreads();
        for (int rr = warp; rr < rows; rr += kThreads / 32) {
            const double *row = C + rr * cp + P;
            for (int fz = lane; fz < nzf; fz += 32) {
                const int ez = fz - oz;            // >= -1
                double t;
                if ((ez & 1) == 0) {
                    t = row[ez >> 1];
                } else {
                    const int c = (ez - 1) >> 1;   // lower coarse neighbour (-1 at a zero-BC wall)
                    t = 0.0;
#pragma unroll
                    for (int j = 1; j <= P; ++j) t = fma(b[j], row[c + 1 - j] + row[c + j], t);
                }
                T[rr * nzf + fz] = t;
            }
        }
        __syncthreads();
#pragma unroll
        for (int n = 0; n < NPT; ++n) {
            const double *col = T + toff[n];
            if (oddmask & (1u << n)) {
                double t = 0.0;
#pragma unroll
                for (int j = 1; j <= P; ++j) t = fma(b[j], col[(1 - j) * nzf] + col[j * nzf], t);
                s[n] = t;
            } else {
                s[n] = col[0];
            }
        }
    };
    auto store_plane = [&](int ex, const double (&s)[NPT]) {
        const int fx = ex + ox;
        if (fx < 0 || fx >= g.nf[0]) return;
        double *fpx = fb + (long long)fx * g.nf[1] * nzf;
#pragma unroll
        for (int n = 0; n < NPT; ++n)
            if (foff[n] >= 0) __stcs(fpx + foff[n], s[n]);
    };

    for (int i = i_lo; i <= i_hi; ++i) {
        double s[NPT];
        const int xc = wrap_or_zero(i, g.nc[0], g.bc[0]);
        if (xc >= 0) {
            plane(s);
        } else {
#pragma unroll
            for (int n = 0; n < NPT; ++n) s[n] = 0.0;
        }
#pragma unroll
        for (int a = 0; a + 1 < 2 * P; ++a)
#pragma unroll
            for (int n = 0; n < NPT; ++n) sq[a][n] = sq[a + 1][n];
#pragma unroll
        for (int n = 0; n < NPT; ++n) sq[2 * P - 1][n] = s[n];
        if (i >= I0 && i < I0 + ni) store_plane(2 * i, s);
        const int c = i - P;  // odd plane between coarse c and c + 1: sq[P - j] and sq[P + j - 1]
        if (c >= c_first && c < I0 + ni) {
            double o[NPT];
#pragma unroll
            for (int n = 0; n < NPT; ++n) {
                double t = 0.0;
#pragma unroll
                for (int j = 1; j <= P; ++j) t = fma(b[j], sq[P - j][n] + sq[P + j - 1][n], t);
                o[n] = t;
            }
            store_plane(2 * c + 1, o);
        }
    }
}

// midpoint Lagrange weights b_1 .. b_p (reading R13), closed form of the product
void transfer_weights(int p, double *b)
{
    for (int j = 1; j <= p; ++j) {
        const double tj = j - 0.5;
        double w = 1.0;
        for (int m = 1; m <= p; ++m) {
            const double tm = m - 0.5;
            if (m != j) w *= (-tm / (tj - tm));   // node +t_m
            w *= (tm / (tj + tm));                // node -t_m
        }
        b[j] = w;
    }
}

int fill_geom(TGeom &g, const int32_t shape_fine[3], const int32_t bc[3], int p)
{
    for (int d = 0; d < 3; ++d) {
        if (bc[d] != 0 && bc[d] != 1) return -1;
        g.nf[d] = shape_fine[d];
        g.bc[d] = bc[d];
        if (bc[d]) {
            if (shape_fine[d] < 2 || (shape_fine[d] & 1)) return -1;
            g.nc[d] = shape_fine[d] / 2;
            g.off[d] = 0;
        } else {
            if (shape_fine[d] < 3 || !(shape_fine[d] & 1)) return -1;
            g.nc[d] = (shape_fine[d] - 1) / 2;
            g.off[d] = 1;
        }
    }
    g.b[0] = 0.0;
    transfer_weights(p, g.b);
    return 0;
}

// coarse rows per tile and coarse planes per chunk: the swept plane's points fit kMaxPt per thread
// and the grid has a few CTAs per SM where the problem allows it
void tile_choice(int pts_per_row, bool interp, int ncx, int ncy, int64_t nbands, int sm_count,
                 int *jt, int *ic)
{
    // 8 coarse rows per tile where the swept plane fits (16 was measured: fewer halo rows, but too few
    // CTAs for single arrays and small grids)
    int t = 8;
    while (t > 1 && (interp ? (2 * t + 1) : t) * pts_per_row > kThreads * kMaxPt) t >>= 1;
    if (t > ncy) t = ncy;
    const long long ytiles = (ncy + t - 1) / t;
    long long chunks = (4LL * sm_count + ytiles * nbands - 1) / (ytiles * nbands);
    const long long max_chunks = (ncx + 7) / 8;  // at least 8 coarse planes per chunk: halo planes
    if (chunks > max_chunks) chunks = max_chunks;
    if (chunks < 1) chunks = 1;
    *jt = t;
    *ic = (int)((ncx + chunks - 1) / chunks);
}

// Current device and its SM count; the count is looked up once per device.
cudaError_t device_sms(int *dev_out, int *sms_out)
{
    static std::atomic<int> cached[64];  // 0 = not looked up yet
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    int sms = (dev >= 0 && dev < 64) ? cached[dev].load(std::memory_order_relaxed) : 0;
    if (sms == 0) {
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) cached[dev].store(sms, std::memory_order_relaxed);
    }
    *dev_out = dev;
    *sms_out = sms;
    return cudaSuccess;
}

template <int P, int NPT>
cudaError_t launch_npt(bool interp, const TGeom &g, const double *src, double *dst, int64_t nbands,
                       int jt, int ic, size_t smem, int dev, cudaStream_t stream)
{
    const void *fn = interp ? (const void *)fd_interp_kernel<P, NPT> : (const void *)fd_restrict_kernel<P, NPT>;
    // The two function attributes belong to (instantiation, device): set once each, not per call
    // (the coarse levels of a V-cycle are launch bound).  Bit d of prepared[k]: done on device d.
    static std::atomic<unsigned long long> prepared[2];
    const bool tracked = dev >= 0 && dev < 64;
    if (!tracked || !((prepared[interp ? 1 : 0].load(std::memory_order_acquire) >> dev) & 1ULL)) {
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kFdSweepSmemMax);
        if (e != cudaSuccess) return e;
        // two CTAs per SM need the shared-memory carve-out at its maximum
        e = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        if (tracked) prepared[interp ? 1 : 0].fetch_or(1ULL << dev, std::memory_order_release);
    }
    const unsigned gx = (unsigned)((g.nc[1] + jt - 1) / jt), gy = (unsigned)((g.nc[0] + ic - 1) / ic);
    if (gy > 65535) return cudaErrorInvalidConfiguration;
    const long long band_f = (long long)g.nf[0] * g.nf[1] * g.nf[2];
    const long long band_c = (long long)g.nc[0] * g.nc[1] * g.nc[2];
    for (int64_t b0 = 0; b0 < nbands; b0 += 65535) {
        const unsigned nb = (unsigned)((nbands - b0 < 65535) ? nbands - b0 : 65535);
        if (interp)
            fd_interp_kernel<P, NPT><<<dim3(gx, gy, nb), kThreads, smem, stream>>>(
                g, src + b0 * band_c, dst + b0 * band_f, jt, ic);
        else
            fd_restrict_kernel<P, NPT><<<dim3(gx, gy, nb), kThreads, smem, stream>>>(
                g, src + b0 * band_f, dst + b0 * band_c, jt, ic);
        const cudaError_t e = cudaPeekAtLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// Tile and shared-memory footprint of a transfer; cudaErrorInvalidConfiguration when a z row is too
// long for the kernels (fine nz > 682 or so for restriction, coarse nz > 2048 for interpolation).
template <int P>
cudaError_t transfer_cfg(bool interp, const TGeom &g, int64_t nbands, int sms, int *jt_out, int *ic_out,
                         size_t *smem_out, int *npt_out)
{
    int jt, ic;
    tile_choice(interp ? g.nf[2] : g.nc[2], interp, g.nc[0], g.nc[1], nbands, sms, &jt, &ic);
    const int pts = interp ? (2 * jt + 1) * g.nf[2] : jt * g.nc[2];
    if (pts > kThreads * kMaxPt) return cudaErrorInvalidConfiguration;
    size_t smem;
    if (interp)
        smem = sizeof(double) * ((size_t)(jt + 2 * P) * 2 * (g.nc[2] + 2 * P) + (size_t)(jt + 2 * P) * g.nf[2]);
    else
        smem = sizeof(double) * (size_t)(2 * jt - 1 + 2 * (2 * P - 1)) *
               (2 * (size_t)((g.nf[2] + 2 * (2 * P - g.off[2]) + 5) & ~1) + g.nc[2]);
    if (smem > (size_t)kFdSweepSmemMax) return cudaErrorInvalidConfiguration;
    *jt_out = jt;
    *ic_out = ic;
    *smem_out = smem;
    *npt_out = (pts + kThreads - 1) / kThreads;
    return cudaSuccess;
}

template <int P>
cudaError_t launch(bool interp, const TGeom &g, const double *src, double *dst, int64_t nbands,
                   cudaStream_t stream)
{
    int dev = 0, sms = 148;
    cudaError_t e = device_sms(&dev, &sms);
    if (e != cudaSuccess) return e;
    int jt, ic, npt;
    size_t smem;
    e = transfer_cfg<P>(interp, g, nbands, sms, &jt, &ic, &smem, &npt);
    if (e != cudaSuccess) return e;
    if (npt <= 1) return launch_npt<P, 1>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
    if (npt <= 2) return launch_npt<P, 2>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
    if (npt <= 3) return launch_npt<P, 3>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
    if (npt <= 4) return launch_npt<P, 4>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
    if (npt <= 6) return launch_npt<P, 6>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
    return launch_npt<P, 8>(interp, g, src, dst, nbands, jt, ic, smem, dev, stream);
}

}  // namespace

// rc: 0 ok, -1 invalid argument, -2 unsupported, -4 CUDA
int fd_transfer_run(int interp, const int32_t shape_fine[3], const int32_t bc[3], int p,
                    const double *src, double *dst, int64_t nbands, cudaStream_t stream)
{
    TGeom g;
    if (p < 1 || p > 3) return (p >= 1 && p <= 6) ? -2 : -1;
    if (fill_geom(g, shape_fine, bc, p) != 0) return -1;
    for (int d = 0; d < 3; ++d)
        if (g.nc[d] < 1) return -1;
    cudaError_t e;
    switch (p) {
    case 1: e = launch<1>(interp != 0, g, src, dst, nbands, stream); break;
    case 2: e = launch<2>(interp != 0, g, src, dst, nbands, stream); break;
    default: e = launch<3>(interp != 0, g, src, dst, nbands, stream); break;
    }
    if (e == cudaErrorInvalidConfiguration) {
        cudaGetLastError();
        return -2;
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return -4;
    }
    return 0;
}

// Would fd_transfer_run accept this transfer on the current device?  0 yes, -1 / -2 / -4 as there.
// Nothing is launched (fd_mg_create asks for every level, so that a hierarchy whose z rows are too
// long for the kernels fails at create and not in the first cycle).
int fd_transfer_check(int interp, const int32_t shape_fine[3], const int32_t bc[3], int p, int64_t nbands)
{
    TGeom g;
    if (p < 1 || p > 3) return (p >= 1 && p <= 6) ? -2 : -1;
    if (fill_geom(g, shape_fine, bc, p) != 0) return -1;
    for (int d = 0; d < 3; ++d)
        if (g.nc[d] < 1) return -1;
    int dev = 0, sms = 148, jt, ic, npt;
    size_t smem;
    if (device_sms(&dev, &sms) != cudaSuccess) {
        cudaGetLastError();
        return -4;
    }
    cudaError_t e;
    switch (p) {
    case 1: e = transfer_cfg<1>(interp != 0, g, nbands, sms, &jt, &ic, &smem, &npt); break;
    case 2: e = transfer_cfg<2>(interp != 0, g, nbands, sms, &jt, &ic, &smem, &npt); break;
    default: e = transfer_cfg<3>(interp != 0, g, nbands, sms, &jt, &ic, &smem, &npt); break;
    }
    return e == cudaSuccess ? 0 : -2;
}
