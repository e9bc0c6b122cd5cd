// Sweep kernel: the bandwidth path of libfdham (nn = 3, i.e. GPAW's default 19-point star).
//
// Operation: include/fdham.h -- out = -1/2 lap_FD psi + v_eff psi (Eq. 6 first two terms,
// PAPER.md:187-188; FD kinetic operator PAPER.md:232; the stencil hot spot PAPER.md:150).
// Steps a2..a6 of SURVEY 8(a) are all fused here: halo/boundary resolution, the 19 taps, the
// v_eff multiply-add, the store, and the band-batched tiling.
//
// Design:
//   * A CTA owns one y-tile (tyc rows x the full z row) and sweeps along x.  The y-z tile of each
//     x plane, with 3 halo rows on either side, is staged in shared memory by the TMA unit
//     (cp.async.bulk, completion on an mbarrier) through a 4-deep ring, so HBM reads are deep,
//     asynchronous and fully coalesced (whole rows), and each psi value crosses HBM once.
//   * x direction: scatter form.  When plane xl arrives its value u adds w_x[|j|] u to the seven
//     in-flight output accumulators xl-3..xl+3 held in REGISTERS; output xl-3 is then complete
//     and is stored.  The accumulator slots rotate by compile-time index (loop unrolled x7).
//   * y and z directions: read from the shared-memory tile of the centre plane.  Each thread owns
//     a micro tile of TY rows x TC 16-byte chunks (real: 4 rows x 2 points, complex: 2 rows x 2
//     points) to amortise halo reads: ~3.3 (real) / 3.5 (complex) LDS.128 per point pair.
//   * Boundaries are resolved while staging / addressing, never by a padded copy:
//       periodic y  -> the wrapped halo rows are a separate bulk copy from the other end;
//       zero y      -> those shared-memory rows are zeroed once and never overwritten;
//       periodic z  -> per-thread precomputed wrapped chunk offsets inside the row;
//       zero z      -> the out-of-range chunk address points at a 16-byte zero word (stride 0);
//       periodic x  -> the sweep prologue/epilogue read planes from the other end;
//       zero x      -> those steps are skipped (accumulators are born zero);
//       Bloch phase -> multiply only wrapped rows / chunks / planes (complex128 only).
//   * Persistent teams: the (band, x) planes are split evenly over floor(#SM / nytiles) teams of
//     nytiles CTAs; the CTAs of a team sweep the same planes for adjacent y-tiles at the same
//     time, so the y-halo rows they share are L2 hits, and every SM gets the same amount of work.
#include "fd_internal.h"

namespace {

constexpr int kStages = 4;       // ring depth (power of two)
constexpr int kStagesLog2 = 2;
constexpr int kMaxThreads = 384;
constexpr int kBarBytes = 128;   // full[4] + empty[4] mbarriers at the start of shared memory
constexpr int kRowOff = 128;     // rows start here inside a stage; bytes [0,16) are a zero word

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {
    }
}
// TMA 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void fma2(double2 &a, double w, const double2 &x)
{
    a.x = fma(w, x.x, a.x);
    a.y = fma(w, x.y, a.y);
}
__device__ __forceinline__ double2 mul2(double w, const double2 &x)
{
    return make_double2(w * x.x, w * x.y);
}
__device__ __forceinline__ double2 cmul(const double2 &a, double pr, double pi)
{
    return make_double2(a.x * pr - a.y * pi, a.x * pi + a.y * pr);
}

// Walks the planes a CTA has to LOAD, in consumption order: for each segment (band, [x0, x0+len))
// of its linear (band, x) range the steps s = 0..len+5 with plane xl = x0 - 3 + s; planes outside
// [0, nx) wrap on a periodic x axis and are skipped on a zero one.
struct PlaneIter {
    long long L, L1;
    long long band;
    int nx, per_x;
    int x0, len, s;
    __device__ void init(long long l0, long long l1, int nx_, int per)
    {
        L = l0;
        L1 = l1;
        nx = nx_;
        per_x = per;
        seg();
    }
    __device__ void seg()
    {
        s = 0;
        if (L < L1) {
            band = L / nx;
            x0 = (int)(L - band * nx);
            const long long rem = L1 - L;
            len = (rem < (long long)(nx - x0)) ? (int)rem : (nx - x0);
        } else {
            band = 0;
            x0 = 0;
            len = 0;
        }
    }
    // next plane to load: returns false when exhausted
    __device__ bool next(long long &b, int &xg)
    {
        while (L < L1) {
            if (s >= len + 6) {
                L += len;
                seg();
                continue;
            }
            const int xl = x0 - 3 + s;
            ++s;
            if (xl < 0) {
                if (!per_x) continue;
                xg = xl + nx;
            } else if (xl >= nx) {
                if (!per_x) continue;
                xg = xl - nx;
            } else {
                xg = xl;
            }
            b = band;
            return true;
        }
        return false;
    }
};

template <bool CPLX, bool HAS_V>
__global__ void __launch_bounds__(kMaxThreads, 1)
fd_sweep_kernel(const FdGeom g, const FdSweepCfg cfg, const double *__restrict__ psi,
                const double *__restrict__ v_eff, double *__restrict__ out,
                const long long total_planes, const int quota)
{
    constexpr int TY = CPLX ? 2 : 4;   // rows per thread
    constexpr int TC = CPLX ? 2 : 1;   // 16-byte chunks per thread per row
    constexpr int ZH = CPLX ? 3 : 2;   // halo chunks per side along z
    constexpr int NP = TY * TC;

    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t full_bar = smem_base;        // kStages x 8 bytes
    const uint32_t empty_bar = smem_base + 64;  // kStages x 8 bytes
    const uint32_t stage0 = smem_base + kBarBytes;

    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int pitch = nz * (CPLX ? 16 : 8);  // bytes per z row
    const int cpr = pitch >> 4;              // 16-byte chunks per row
    const int rowd = pitch >> 3;             // doubles per row
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int nwarps = blockDim.x >> 5;

    const int yt = (int)(blockIdx.x % (unsigned)cfg.nytiles);
    const long long team = blockIdx.x / (unsigned)cfg.nytiles;
    const int y0 = yt * cfg.tyc;
    const int rows_valid = min(cfg.tyc, ny - y0);
    const long long L0 = team * (long long)quota;
    const long long L1 = (L0 + quota < total_planes) ? (L0 + quota) : total_planes;
    if (L0 >= L1) return;  // whole CTA exits together

    // ---- y segments of the staged tile: smem row R <-> global row y0 - 3 + R ------------------
    const int per_y = g.bc[1], per_x = g.bc[0], per_z = g.bc[2];
    const int nlo = max(0, 3 - y0);                     // rows below row 0
    const int nhi = max(0, y0 + rows_valid + 3 - ny);   // rows past row ny-1
    const int nmid = rows_valid + 6 - nlo - nhi;
    const uint32_t stage_bytes = (uint32_t)cfg.stage_bytes;
    const uint32_t tx_bytes = (uint32_t)((nmid + (per_y ? nlo + nhi : 0)) * pitch);

    // ---- one-time shared memory setup ------------------------------------------------------
    if (tid == 0) {
        for (int i = 0; i < kStages; ++i) {
            mbar_init(full_bar + 8 * i, 1);
            mbar_init(empty_bar + 8 * i, nwarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int st = 0; st < kStages; ++st) {
        unsigned char *sb = smem + kBarBytes + (size_t)st * stage_bytes;
        if (tid < 2) reinterpret_cast<double *>(sb)[tid] = 0.0;  // the zero word
        if (!per_y) {                                            // zero halo rows, written once
            for (int i = tid; i < nlo * rowd; i += blockDim.x)
                reinterpret_cast<double *>(sb + kRowOff)[i] = 0.0;
            for (int i = tid; i < nhi * rowd; i += blockDim.x)
                reinterpret_cast<double *>(sb + kRowOff + (size_t)(nlo + nmid) * pitch)[i] = 0.0;
        }
        // rows past the ragged end of the last tile are never loaded: define them
        for (int i = tid; i < (cfg.tyc - rows_valid) * rowd; i += blockDim.x)
            reinterpret_cast<double *>(sb + kRowOff + (size_t)(rows_valid + 6) * pitch)[i] = 0.0;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // ---- thread -> micro tile ---------------------------------------------------------------
    int rg = tid / cfg.lanes;
    const int lz = tid - rg * cfg.lanes;
    const bool tactive = rg < cfg.rowgroups;
    if (!tactive) rg = cfg.rowgroups - 1;  // surplus threads shadow the last row group, never store
    const int r0 = rg * TY;                // first halo row (smem row index) of this thread
    const int zc0 = lz * TC;               // first own chunk in the row
    const uint32_t own_off = kRowOff + (uint32_t)(r0 * pitch + zc0 * 16);

    // halo chunks along z: k < ZH left of the own chunks, k >= ZH right of them
    uint32_t hb[2 * ZH], hs[2 * ZH];
    int zwrap = 0;  // 2 bits per halo chunk: 1 = wrapped below 0, 2 = wrapped past nz (complex only)
#pragma unroll
    for (int k = 0; k < 2 * ZH; ++k) {
        int cz = zc0 + ((k < ZH) ? (k - ZH) : (k - ZH + TC));
        bool valid = true;
        if (cz < 0) {
            if (per_z) { cz += cpr; zwrap |= 1 << (2 * k); } else valid = false;
        } else if (cz >= cpr) {
            if (per_z) { cz -= cpr; zwrap |= 2 << (2 * k); } else valid = false;
        }
        hb[k] = valid ? (uint32_t)(kRowOff + (r0 + 3) * pitch + cz * 16) : 0u;
        hs[k] = valid ? (uint32_t)pitch : 0u;
    }
    const bool zphase = CPLX && per_z && (g.ph_re[2] != 1.0 || g.ph_im[2] != 0.0);
    const bool yphase = CPLX && per_y && (g.ph_re[1] != 1.0 || g.ph_im[1] != 0.0);
    const bool xphase = CPLX && per_x && (g.ph_re[0] != 1.0 || g.ph_im[0] != 0.0);

    // store / v_eff addressing: row i of the micro tile is global row y0 + r0 + i
    bool row_ok[TY];
    long long row_goff[TY];  // offset in doubles of (y, own chunk) inside an x plane of psi / out
    long long row_voff[TY];  // offset in doubles inside an x plane of v_eff
#pragma unroll
    for (int i = 0; i < TY; ++i) {
        const int yl = r0 + i;
        row_ok[i] = tactive && (yl < rows_valid) && (zc0 < cpr);
        const int y = min(y0 + yl, ny - 1);
        const int zc = min(zc0, cpr - TC);
        row_goff[i] = (long long)y * rowd + zc * 2;
        row_voff[i] = (long long)y * nz + (CPLX ? zc : zc * 2);
    }
    const long long plane_d = (long long)ny * rowd;  // doubles per x plane of psi / out
    const long long plane_v = (long long)ny * nz;

    const double wx1 = g.w[0][1], wx2 = g.w[0][2], wx3 = g.w[0][3];
    const double wy1 = g.w[1][1], wy2 = g.w[1][2], wy3 = g.w[1][3];
    const double wz1 = g.w[2][1], wz2 = g.w[2][2], wz3 = g.w[2][3];
    const double wdiag = g.wdiag;

    // ---- producer state (thread 0) -------------------------------------------------------------
    PlaneIter it;
    long long q_issued = 0;
    auto issue = [&](long long qi, long long b, int xg) {
        const uint32_t st = (uint32_t)(qi & (kStages - 1));
        const uint32_t bar = full_bar + 8 * st;
        const uint32_t dst = stage0 + st * stage_bytes + kRowOff;
        const double *src = psi + ((b * nx + xg) * (long long)ny) * rowd;
        mbar_expect_tx(bar, tx_bytes);
        if (per_y && nlo > 0)
            bulk_g2s(dst, src + (long long)(ny - nlo) * rowd, (uint32_t)(nlo * pitch), bar);
        bulk_g2s(dst + nlo * pitch, src + (long long)(y0 - 3 + nlo) * rowd, (uint32_t)(nmid * pitch),
                 bar);
        if (per_y && nhi > 0)
            bulk_g2s(dst + (nlo + nmid) * pitch, src, (uint32_t)(nhi * pitch), bar);
    };
    if (tid == 0) {
        it.init(L0, L1, nx, per_x);
        long long b;
        int xg;
        for (int i = 0; i < kStages; ++i) {
            if (!it.next(b, xg)) break;
            issue(q_issued, b, xg);
            ++q_issued;
        }
    }

    // ---- consumer sweep ----------------------------------------------------------------------
    long long q = 0;  // planes consumed so far by this thread
    double2 acc[7][NP];
#pragma unroll
    for (int a = 0; a < 7; ++a)
#pragma unroll
        for (int p = 0; p < NP; ++p) acc[a][p] = make_double2(0.0, 0.0);

    for (long long L = L0; L < L1;) {
        const long long band = L / nx;
        const int x0 = (int)(L - band * nx);
        const int len = ((L1 - L) < (long long)(nx - x0)) ? (int)(L1 - L) : (nx - x0);
        const int nsteps = len + 6;
        const double *vplane = HAS_V ? v_eff + (long long)x0 * plane_v : nullptr;
        double *oplane = out + (band * nx + x0) * plane_d;

        for (int s7 = 0; s7 < nsteps; s7 += 7) {
#pragma unroll
            for (int J = 0; J < 7; ++J) {
                const int s = s7 + J;
                if (s < nsteps) {
                    const int xl = x0 - 3 + s;
                    const bool center = (s >= 3) && (s < 3 + len);
                    const bool valid = per_x || (xl >= 0 && xl < nx);
                    if (valid) {
                        // producer: refill the stage plane q-1 lived in with plane q-1+kStages
                        if (tid == 0 && q >= 1 && q_issued == q - 1 + kStages) {
                            long long b;
                            int xg;
                            if (it.next(b, xg)) {
                                const long long qp = q - 1;
                                mbar_wait(empty_bar + 8 * (uint32_t)(qp & (kStages - 1)),
                                          (uint32_t)((qp >> kStagesLog2) & 1));
                                issue(q_issued, b, xg);
                                ++q_issued;
                            }
                        }
                        double2 vv[TY];
                        if (HAS_V && center) {
#pragma unroll
                            for (int i = 0; i < TY; ++i)
                                vv[i] = __ldg(reinterpret_cast<const double2 *>(
                                    vplane + (long long)(s - 3) * plane_v + row_voff[i]));
                        }
                        const uint32_t st = (uint32_t)(q & (kStages - 1));
                        mbar_wait(full_bar + 8 * st, (uint32_t)((q >> kStagesLog2) & 1));
                        const uint32_t sb = stage0 + st * stage_bytes;
                        double2 u[NP];
                        if (center) {
                            // ---- y taps (+ own values) from the staged tile
                            double2 c[TY + 6][TC];
#pragma unroll
                            for (int rr = 0; rr < TY + 6; ++rr)
#pragma unroll
                                for (int t = 0; t < TC; ++t)
                                    c[rr][t] = lds128(sb + own_off + rr * pitch + t * 16);
                            if (yphase) {
#pragma unroll
                                for (int rr = 0; rr < TY + 6; ++rr) {
                                    const int R = r0 + rr;
                                    if (R < nlo) {
#pragma unroll
                                        for (int t = 0; t < TC; ++t)
                                            c[rr][t] = cmul(c[rr][t], g.ph_re[1], -g.ph_im[1]);
                                    } else if (R >= nlo + nmid) {
#pragma unroll
                                        for (int t = 0; t < TC; ++t)
                                            c[rr][t] = cmul(c[rr][t], g.ph_re[1], g.ph_im[1]);
                                    }
                                }
                            }
#pragma unroll
                            for (int i = 0; i < TY; ++i)
#pragma unroll
                                for (int t = 0; t < TC; ++t) {
                                    double2 &a = acc[J][i * TC + t];
                                    u[i * TC + t] = c[3 + i][t];
                                    fma2(a, wy1, c[2 + i][t]);
                                    fma2(a, wy1, c[4 + i][t]);
                                    fma2(a, wy2, c[1 + i][t]);
                                    fma2(a, wy2, c[5 + i][t]);
                                    fma2(a, wy3, c[i][t]);
                                    fma2(a, wy3, c[6 + i][t]);
                                }
                            // ---- z taps
#pragma unroll
                            for (int i = 0; i < TY; ++i) {
                                double2 hz[2 * ZH];
#pragma unroll
                                for (int k = 0; k < 2 * ZH; ++k)
                                    hz[k] = lds128(sb + hb[k] + i * hs[k]);
                                if (zphase && zwrap != 0) {
#pragma unroll
                                    for (int k = 0; k < 2 * ZH; ++k) {
                                        const int wbits = (zwrap >> (2 * k)) & 3;
                                        if (wbits == 1) hz[k] = cmul(hz[k], g.ph_re[2], -g.ph_im[2]);
                                        if (wbits == 2) hz[k] = cmul(hz[k], g.ph_re[2], g.ph_im[2]);
                                    }
                                }
                                if constexpr (CPLX) {
                                    // chunks are complex points: own C0,C1; hz = L3,L2,L1,R1,R2,R3
                                    double2 &a0 = acc[J][i * TC + 0];
                                    double2 &a1 = acc[J][i * TC + (TC - 1)];
                                    const double2 C0 = u[i * TC + 0], C1 = u[i * TC + (TC - 1)];
                                    fma2(a0, wz1, hz[ZH - 1]);
                                    fma2(a0, wz1, C1);
                                    fma2(a0, wz2, hz[ZH - 2]);
                                    fma2(a0, wz2, hz[ZH]);
                                    fma2(a0, wz3, hz[0]);
                                    fma2(a0, wz3, hz[ZH + 1]);
                                    fma2(a1, wz1, C0);
                                    fma2(a1, wz1, hz[ZH]);
                                    fma2(a1, wz2, hz[ZH - 1]);
                                    fma2(a1, wz2, hz[ZH + 1]);
                                    fma2(a1, wz3, hz[ZH - 2]);
                                    fma2(a1, wz3, hz[2 * ZH - 1]);
                                } else {
                                    // chunk = points (z, z+1); hz = L2,L1,R1,R2
                                    double2 &a = acc[J][i];
                                    const double2 o = u[i];
                                    a.x = fma(wz1, hz[1].y, a.x);
                                    a.x = fma(wz1, o.y, a.x);
                                    a.x = fma(wz2, hz[1].x, a.x);
                                    a.x = fma(wz2, hz[2].x, a.x);
                                    a.x = fma(wz3, hz[0].y, a.x);
                                    a.x = fma(wz3, hz[2].y, a.x);
                                    a.y = fma(wz1, o.x, a.y);
                                    a.y = fma(wz1, hz[2].x, a.y);
                                    a.y = fma(wz2, hz[1].y, a.y);
                                    a.y = fma(wz2, hz[2].y, a.y);
                                    a.y = fma(wz3, hz[1].x, a.y);
                                    a.y = fma(wz3, hz[3].x, a.y);
                                }
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < TY; ++i)
#pragma unroll
                                for (int t = 0; t < TC; ++t)
                                    u[i * TC + t] = lds128(sb + own_off + (3 + i) * pitch + t * 16);
                            if (xphase && (xl < 0 || xl >= nx)) {
                                const double pi_ = (xl < 0) ? -g.ph_im[0] : g.ph_im[0];
#pragma unroll
                                for (int p = 0; p < NP; ++p) u[p] = cmul(u[p], g.ph_re[0], pi_);
                            }
                        }
                        // done with the stage: release it to the producer
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty_bar + 8 * st);
                        ++q;

                        // ---- diagonal (+ v_eff) and x taps (scatter into the 7 in-flight outputs)
                        if (center) {
#pragma unroll
                            for (int i = 0; i < TY; ++i) {
                                if constexpr (CPLX) {
                                    const double d0 = HAS_V ? wdiag + vv[i].x : wdiag;
                                    const double d1 = HAS_V ? wdiag + vv[i].y : wdiag;
                                    fma2(acc[J][i * TC + 0], d0, u[i * TC + 0]);
                                    fma2(acc[J][i * TC + (TC - 1)], d1, u[i * TC + (TC - 1)]);
                                } else {
                                    const double d0 = HAS_V ? wdiag + vv[i].x : wdiag;
                                    const double d1 = HAS_V ? wdiag + vv[i].y : wdiag;
                                    acc[J][i].x = fma(d0, u[i].x, acc[J][i].x);
                                    acc[J][i].y = fma(d1, u[i].y, acc[J][i].y);
                                }
                            }
                        }
#pragma unroll
                        for (int p = 0; p < NP; ++p) {
                            acc[(J + 3) % 7][p] = mul2(wx3, u[p]);
                            fma2(acc[(J + 2) % 7][p], wx2, u[p]);
                            fma2(acc[(J + 1) % 7][p], wx1, u[p]);
                            fma2(acc[(J + 6) % 7][p], wx1, u[p]);
                            fma2(acc[(J + 5) % 7][p], wx2, u[p]);
                            fma2(acc[(J + 4) % 7][p], wx3, u[p]);
                        }
                    } else {
#pragma unroll
                        for (int p = 0; p < NP; ++p) acc[(J + 3) % 7][p] = make_double2(0.0, 0.0);
                    }
                    // ---- output x0 + s - 6 is complete
                    if (s >= 6) {
                        double *o = oplane + (long long)(s - 6) * plane_d;
#pragma unroll
                        for (int i = 0; i < TY; ++i)
                            if (row_ok[i]) {
#pragma unroll
                                for (int t = 0; t < TC; ++t)
                                    __stcs(reinterpret_cast<double2 *>(o + row_goff[i]) + t,
                                           acc[(J + 4) % 7][i * TC + t]);
                            }
                    }
                }
            }
        }
        L += len;
    }
}

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

}  // namespace

void fd_sweep_configure(fd_plan *plan, int tyc_override, int xchunk_override)
{
    FdSweepCfg &c = plan->sweep;
    const FdGeom &g = plan->g;
    c = FdSweepCfg{};
    c.xchunk = xchunk_override;  // 0 = automatic (persistent teams), else planes per CTA
    if (g.nn != 3) return;
    if (g.n[0] < 8 || g.n[1] < 8 || g.n[2] < 8 || (g.n[2] & 1)) return;
    c.ty = g.cplx ? 2 : 4;
    c.tc = g.cplx ? 2 : 1;
    const int pitch = g.n[2] * (g.cplx ? 16 : 8);
    const int cpr = pitch / 16;
    c.lanes = ceil_div(cpr, c.tc);
    if (c.lanes > kMaxThreads) return;
    const int smem_cap = 227 * 1024 - kBarBytes;
    const int rows_cap = (smem_cap / kStages - kRowOff) / pitch - 6;  // tile rows that fit a stage
    int max_rg = kMaxThreads / c.lanes;
    if (max_rg * c.ty > rows_cap) max_rg = rows_cap / c.ty;
    if (max_rg < 1) return;
    int tyc;
    if (tyc_override > 0) {
        tyc = ceil_div(tyc_override, c.ty) * c.ty;
        if (tyc > max_rg * c.ty) tyc = max_rg * c.ty;
    } else {
        const int ntiles = ceil_div(g.n[1], max_rg * c.ty);
        tyc = ceil_div(ceil_div(g.n[1], ntiles), c.ty) * c.ty;
    }
    if (tyc < 4) tyc = 4;
    c.tyc = tyc;
    c.rowgroups = tyc / c.ty;
    c.nytiles = ceil_div(g.n[1], tyc);
    c.threads = ceil_div(c.rowgroups * c.lanes, 32) * 32;
    c.stages = kStages;
    c.stage_bytes = ((kRowOff + (tyc + 6) * pitch) + 127) / 128 * 128;
    c.smem_bytes = kBarBytes + kStages * c.stage_bytes;
    if (c.smem_bytes > 227 * 1024 || c.threads > kMaxThreads) return;
    c.supported = 1;
}

cudaError_t fd_sweep_prepare(const fd_plan *plan)
{
    const int bytes = plan->sweep.smem_bytes;
    cudaError_t e;
    e = cudaFuncSetAttribute(fd_sweep_kernel<false, false>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fd_sweep_kernel<false, true>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fd_sweep_kernel<true, false>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(fd_sweep_kernel<true, true>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

cudaError_t fd_launch_sweep(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                            int64_t nbands, cudaStream_t stream)
{
    const FdSweepCfg &c = plan->sweep;
    const FdGeom &g = plan->g;
    const long long total = (long long)nbands * g.n[0];
    // persistent teams: one CTA per SM, nytiles CTAs per team, equal plane quota per team
    long long nteams = plan->sm_count / c.nytiles;
    if (nteams < 1) nteams = 1;
    long long quota;
    if (c.xchunk > 0) {
        quota = c.xchunk;
    } else {
        quota = (total + nteams - 1) / nteams;
        const int min_quota = g.n[0] < 16 ? g.n[0] : 16;  // below this the 6 halo planes dominate
        if (quota < min_quota) quota = min_quota;
    }
    nteams = (total + quota - 1) / quota;
    const long long nblocks = nteams * c.nytiles;
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)nblocks), block((unsigned)c.threads);
    const double *p = static_cast<const double *>(psi);
    double *o = static_cast<double *>(out);
    const int qi = (int)quota;
    if (g.cplx) {
        if (v_eff)
            fd_sweep_kernel<true, true><<<grid, block, c.smem_bytes, stream>>>(g, c, p, v_eff, o, total, qi);
        else
            fd_sweep_kernel<true, false><<<grid, block, c.smem_bytes, stream>>>(g, c, p, nullptr, o, total, qi);
    } else {
        if (v_eff)
            fd_sweep_kernel<false, true><<<grid, block, c.smem_bytes, stream>>>(g, c, p, v_eff, o, total, qi);
        else
            fd_sweep_kernel<false, false><<<grid, block, c.smem_bytes, stream>>>(g, c, p, nullptr, o, total, qi);
    }
    return cudaPeekAtLastError();
}
