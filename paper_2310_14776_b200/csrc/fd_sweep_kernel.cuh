// fd_sweep_kernel.cuh -- the sweep kernel template (included by the fd_sweep_inst_*.cu translation
// units, which instantiate it, so that they compile in parallel).
//
// Sweep kernel: the bandwidth path of libfdham (nn = 1..6; nn = 3 is GPAW's default 19-point star,
// which the comments below use for concreteness: halo 3, seven accumulators).  The same template
// also carries the SURVEY 8(f) forms that ride the stencil: the weighted-Jacobi / residual form
// (MODE 2), the fused expectation values (EX), real Bloch factors -1 (PH on float64), nn = 4..6
// (2-row micro tile) and float32 / complex64 (F32); see the template parameter list below.
//
// Operation: include/fdham.h -- out = -1/2 lap_FD psi + v_eff psi (Eq. 6 first two terms,
// PAPER.md:187-188; FD kinetic operator PAPER.md:232; the stencil hot spot PAPER.md:150).
// Steps a2..a6 of SURVEY 8(a) are all fused here: halo/boundary resolution, the 19 taps, the
// v_eff multiply-add, the store, and the band-batched tiling.
//
// Design:
//   * A CTA owns one y-tile (tyc rows x the full z row) and sweeps along x.  The y-z tile of each
//     x plane, with 3 halo rows on either side, and the matching v_eff rows are staged in shared
//     memory by the TMA unit (cp.async.bulk, completion on an mbarrier) through a ring of
//     `stages` slots, so HBM reads are deep, asynchronous and fully coalesced (whole rows), and
//     each psi value crosses HBM once.
//   * The whole schedule of a CTA (which plane to load, which output plane completes, which
//     v_eff plane, which Bloch factor, which L2 policy) is a table in shared memory built once at
//     kernel start: the sweep itself is one flat loop over table entries with no index
//     arithmetic; the next entry is fetched one step ahead.
//   * x direction: scatter form.  When plane xl arrives its value u adds w_x[|j|] u to the seven
//     in-flight output accumulators xl-3..xl+3 held in REGISTERS; output xl-3 is then complete
//     and is stored (streaming store).  The accumulator slots rotate by compile-time index
//     (loop unrolled x7).
//   * y and z directions: read from the shared-memory tile of the centre plane.  Each thread owns
//     a micro tile of 4 rows x one 16-byte chunk (real: 2 points, complex: 1 point) to amortise
//     the y-halo reads; consecutive lanes own consecutive chunks, so every 16-byte shared-memory
//     access of a warp is conflict free (the shared-memory data pipe is what bounds this kernel).
//   * The row length is a template parameter for the common grids (ROWD doubles per z row; 0 =
//     run time), so every shared-memory and store address of a step is base register + immediate.
//   * Warp specialisation: a fourth warpgroup's first lane is the producer.  It waits on the
//     `empty` mbarrier of a slot (one arrival per compute warp) and issues that slot's bulk copies,
//     v_eff rows first; setmaxnreg hands its registers to the 12 compute warps (24 / 160).  The
//     compute warps never issue a load and never wait for each other.
//   * Boundaries are resolved while staging / addressing, never by a padded copy:
//       periodic y  -> the wrapped halo rows are a separate bulk copy from the other end;
//       zero y      -> those shared-memory rows are zeroed once and never overwritten;
//       periodic z  -> per-thread precomputed wrapped chunk offsets inside the row;
//       zero z      -> the out-of-range chunk address points at a zero block of the stage;
//       periodic x  -> the table's prologue/epilogue entries load planes from the other end;
//       zero x      -> those entries carry no load (the value is taken as zero);
//       Bloch phase -> multiply only wrapped rows / chunks / planes (complex; sign flips for
//                      float64 at k = 1/2).
//   * Persistent teams: the (band, x) planes are split evenly over sm_count / nytiles teams of
//     nytiles CTAs (one CTA per SM, plain launch, no cluster: 147 of 148 SMs for 3 tiles).  The
//     CTAs of a team sweep the same planes for adjacent y-tiles; the y-halo rows they share are
//     fetched from HBM once and hit L2 the second time.  Nothing synchronises the CTAs of a
//     team: a CTA that falls behind finds its halo rows in L2 (its neighbours loaded them), runs
//     faster and catches up, so the drift stays far below what the 126 MB L2 retains (measured:
//     DRAM reads 1.92 GB against 1.82 GB algorithmic on the 96^3 x 256 workload).  A progress
//     throttle through global memory was tried and removed: its polls sit behind the bulk
//     traffic in the memory system and cost more than 2x (dropped variants).
//   * L2 policy: planes that the periodic x wrap reads twice (the first and last three of a band)
//     are loaded evict_last the first time, as is v_eff (shared by all bands).
#pragma once
#include "fd_internal.h"

namespace {

constexpr int kMaxThreads = kFdSweepMaxThreads;          // compute threads
constexpr int kProducerThreads = kFdSweepProducerThreads;  // one more warpgroup: its first lane issues the loads
constexpr int kMaxStages = kFdSweepMaxStages;
constexpr int kCtlBytes = kFdSweepCtlBytes;
constexpr int kSmemMax = kFdSweepSmemMax;

// Step-table entry (8 bytes): .x = flags | (xl + nn), xl = x index of the plane the step brings in
// (-nn .. nx+nn-1: the halo steps of a band segment lie outside the band), .y = band * nx (plane
// index of the band's first plane).  Load plane = .y + xl (+- nx when wrapped), completed output
// plane = .y + xl - nn (flag kOut), v_eff plane of a centre step = xl.
constexpr unsigned kXMask = (1u << 17) - 1u;
constexpr unsigned kWrapLo = 1u << 26;   // plane wrapped from below 0: Bloch factor conj(ph_x)
constexpr unsigned kWrapHi = 1u << 27;   // plane wrapped from past nx-1: Bloch factor ph_x
constexpr unsigned kKeepL2 = 1u << 28;   // load evict_last: the x wrap reads this plane again
constexpr unsigned kZero = 1u << 29;     // no load: the plane lies outside a zero-BC x axis
constexpr unsigned kCentre = 1u << 30;   // centre plane: y/z taps, diagonal and v_eff this step
constexpr unsigned kOut = 1u << 31;      // the step completes output plane xl - nn

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
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void *src, uint32_t bytes,
                                              uint32_t bar, unsigned long long policy)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ unsigned long long policy_evict_last()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// one lane of the (converged) warp
__device__ __forceinline__ bool elect_one()
{
    uint32_t p;
    asm volatile(
        "{\n"
        ".reg .pred P;\n"
        "elect.sync _|P, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, P;\n"
        "}\n"
        : "=r"(p));
    return p != 0;
}

__device__ __forceinline__ double2 lds128(const unsigned char *p)
{
    return *reinterpret_cast<const double2 *>(p);
}
__device__ __forceinline__ double lds64(const unsigned char *p)
{
    return *reinterpret_cast<const double *>(p);
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
__device__ __forceinline__ float4 lds128f(const unsigned char *p)
{
    return *reinterpret_cast<const float4 *>(p);
}
__device__ __forceinline__ void fma4(float4 &a, float w, const float4 &x)
{
    a.x = fmaf(w, x.x, a.x);
    a.y = fmaf(w, x.y, a.y);
    a.z = fmaf(w, x.z, a.z);
    a.w = fmaf(w, x.w, a.w);
}
// two complex64 points times one phase
__device__ __forceinline__ float4 cmul4(const float4 &a, float pr, float pi)
{
    return make_float4(a.x * pr - a.y * pi, a.x * pi + a.y * pr, a.z * pr - a.w * pi, a.z * pi + a.w * pr);
}
template <bool F32>
struct FdVec;
template <>
struct FdVec<false> {
    typedef double2 type;
    typedef double scalar;
    __device__ __forceinline__ static double2 zero() { return make_double2(0.0, 0.0); }
};
template <>
struct FdVec<true> {
    typedef float4 type;
    typedef float scalar;
    __device__ __forceinline__ static float4 zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }
};
__device__ __forceinline__ double2 cmul(const double2 &a, double pr, double pi)
{
    return make_double2(a.x * pr - a.y * pi, a.x * pi + a.y * pr);
}

// The linear (band, x) plane range [L0, L1) of a team, cut into segments of one band each:
// segment 0 = (b0, [x00, x00+len0)), segment k >= 1 = (b0+k, [0, len_k)).  A segment of `len`
// output planes takes len + 2 nn steps s = 0..len+2nn-1; step s brings in plane xl = x0 - nn + s.
struct TeamRange {
    long long L0, L1;
    int nx;
    int b0, x00, len0;
    int nsteps;
    int hn;  // stencil half width nn: a segment has 2 nn halo steps
    __device__ void init(long long l0, long long l1, int nx_, int nn_)
    {
        hn = nn_;
        L0 = l0;
        L1 = l1;
        nx = nx_;
        b0 = (int)(l0 / nx_);
        x00 = (int)(l0 - (long long)b0 * nx_);
        const long long n = l1 - l0;
        len0 = (n < (long long)(nx_ - x00)) ? (int)n : (nx_ - x00);
        const long long rest = n - len0;
        const int nseg = 1 + (int)((rest + nx_ - 1) / nx_);
        nsteps = (int)n + 2 * hn * nseg;
    }
    // Table entry of step e (layout above).
    __device__ uint2 entry(int e, int per_x) const
    {
        int band, x0, len, s;
        if (e < len0 + 2 * hn) {
            band = b0;
            x0 = x00;
            len = len0;
            s = e;
        } else {
            const int e2 = e - (len0 + 2 * hn);
            const int k = e2 / (nx + 2 * hn);
            s = e2 - k * (nx + 2 * hn);
            band = b0 + 1 + k;
            x0 = 0;
            const long long rem = L1 - (L0 + len0 + (long long)k * nx);
            len = (rem < (long long)nx) ? (int)rem : nx;
        }
        const int xl = x0 - hn + s;
        uint2 m;
        m.x = (unsigned)(xl + hn);
        m.y = (unsigned)(band * nx);
        if (xl < 0) m.x |= per_x ? kWrapLo : kZero;
        if (xl >= nx) m.x |= per_x ? kWrapHi : kZero;
        // a whole periodic band: its last three planes (read first, as the wrap) and its first
        // three come round again ~nx steps later
        if (per_x && x0 == 0 && len == nx && s < 2 * hn) m.x |= kKeepL2;
        if (s >= hn && s < len + hn) m.x |= kCentre;
        if (s >= 2 * hn) m.x |= kOut;
        return m;
    }
};

// MODE: what rides the second staged array -- 0: nothing (kinetic), 1: v_eff[nx,ny,nz], added to
//   the diagonal (H psi), 2: a right-hand side rhs[nbands,nx,ny,nz] added as g.rhs_coef * rhs (the
//   weighted-Jacobi sweep of fd_jacobi_sweep: the plan's weights arrive pre-scaled in g; real only).
// PH (complex only): which Bloch-phase code is compiled in -- bit 0: x and y wraps, bit 1: z wraps.
// NN: stencil half width (1..6); 2 NN + 1 register accumulators per point, unrolled 2 NN + 1 times.
//   nn = 4..6 run with a 2-row micro tile and the general z-tap form.
// EX: also accumulate sum conj(psi) H psi and sum |psi|^2 per band (fd_apply_hamiltonian_expect).
//   H is Hermitian: sum_i conj(psi_i) (F psi)_i = conj( sum_i conj(psi_i) (B psi)_i ) for the
//   forward / backward halves F, B of the taps along an axis (wrapped taps carry conjugate Bloch
//   factors), so  eps = sum_i [ d_i |psi_i|^2 + 2 Re conj(psi_i) (B psi)_i ]  needs only taps that
//   are already in the accumulator when psi_i is in registers (x: the planes that arrived before).
//   Each warp writes one partial (eps, norm) pair per band segment; fd_expect_finalize_sweep adds
//   them in a fixed order (deterministic, no atomics).
// F32: float32 / complex64 data: the staging, ring and step table are unchanged (rows
//   are counted in 8-byte units); the arithmetic is a separate body on 16-byte chunks of 4 floats
//   (4 real points or 2 complex points), fp32 accumulation.  Plain applies only (MODE 0 / 1, no EX).
template <bool CPLX, int MODE, int ROWD, int PH, int NN, bool EX, bool F32 = false>
__global__ void __launch_bounds__(kMaxThreads + kProducerThreads, 1)
fd_sweep_kernel(const __grid_constant__ FdGeom g, const __grid_constant__ FdSweepCfg cfg,
                const double *__restrict__ psi, const double *__restrict__ v_eff,
                double *__restrict__ out, const long long total_planes, const int quota,
                const FdSweepAux aux)
{
    constexpr bool HAS_V = MODE != 0;
    static_assert(!(CPLX && MODE == 2), "the Jacobi sweep is real only");
    static_assert(!(F32 && (MODE == 2 || EX)), "float32: plain applies only");
    using VT = typename FdVec<F32>::type;  // one 16-byte chunk: double2 or float4
    using WT = typename FdVec<F32>::scalar;
    // rows per thread: 2 NN + 1 accumulator planes x TY rows must fit the registers
    // (nn <= 3: 4 rows, 7 planes; float64 nn = 4: 3 rows, 9 planes; else 2 rows, 9 / 11 / 13 planes:
    // complex128 nn = 4 with 3 rows spills and runs at half the speed)
    constexpr int TY = (NN <= 3) ? 4 : ((NN == 4 && !CPLX) ? 3 : 2);
    constexpr int TC = 1;              // 16-byte chunks per thread per row (lane stride 16 B)
    // halo chunks per side along z (a chunk holds 2 / 1 points in double, 4 / 2 points in float)
    constexpr int ZH = F32 ? (NN * (CPLX ? 2 : 1) + 3) / 4 : (CPLX ? NN : (NN + 1) / 2);
    constexpr int NS = 2 * NN + 1;     // in-flight output planes (accumulator slots)
    constexpr int NP = TY * TC;

    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t full_bar = smem_base;         // kMaxStages x 8 bytes
    const uint32_t empty_bar = smem_base + 64;   // kMaxStages x 8 bytes
    const uint2 *const tabp = reinterpret_cast<const uint2 *>(smem + cfg.tab_off);
    const unsigned char *const stage0p = smem + cfg.stage_off;
    const uint32_t stage0 = smem_base + (uint32_t)cfg.stage_off;
    const uint32_t stage_bytes = (uint32_t)cfg.stage_bytes;
    const int K = cfg.stages;

    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    // 8-byte units per z row of psi (doubles; for F32 two floats each)
    const int rowd = ROWD ? ROWD : (F32 ? nz * (CPLX ? 2 : 1) / 2 : nz * (CPLX ? 2 : 1));
    const int pitch = rowd * 8;                          // bytes per z row of psi
    const int pitchv = CPLX ? pitch / 2 : pitch;         // bytes per z row of v_eff
    const int cpr = rowd >> 1;                           // 16-byte chunks per row
    const int tid = threadIdx.x;
    const unsigned nwarps = (unsigned)cfg.threads >> 5;  // compute warps (the empty barriers count them)

    const int yt = (int)(blockIdx.x % (unsigned)cfg.nytiles);
    const long long team = blockIdx.x / (unsigned)cfg.nytiles;
    const int y0 = yt * cfg.tyc;
    const int rows_valid = min(cfg.tyc, ny - y0);
    const long long L0 = team * (long long)quota;
    const long long L1 = (L0 + quota < total_planes) ? (L0 + quota) : total_planes;
    if (L0 >= L1) return;

    // ---- y segments of the staged tile: smem row R <-> global row y0 - 3 + R ------------------
    const int per_y = g.bc[1], per_x = g.bc[0], per_z = g.bc[2];
    const int nlo = max(0, NN - y0);                     // rows below row 0
    const int nhi = max(0, y0 + rows_valid + NN - ny);   // rows past row ny-1
    const int nmid = rows_valid + 2 * NN - nlo - nhi;
    const uint32_t zb = (uint32_t)cfg.zb_bytes;
    const uint32_t tx_psi = (uint32_t)((nmid + (per_y ? nlo + nhi : 0)) * pitch);
    const uint32_t tx_v = (uint32_t)(rows_valid * pitchv);
    const long long plane_d = (long long)ny * rowd;  // doubles per x plane of psi / out

    TeamRange tr;
    tr.init(L0, L1, nx, NN);
    const int nsteps = tr.nsteps;

    // ---- one-time shared memory setup ------------------------------------------------------
    if (tid == 0) {
        for (int i = 0; i < K; ++i) {
            mbar_init(full_bar + 8 * i, 1);
            mbar_init(empty_bar + 8 * i, nwarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int e = tid; e <= nsteps; e += blockDim.x)  // one entry past the end: prefetched, unused
        reinterpret_cast<uint2 *>(smem + cfg.tab_off)[e] =
            (e < nsteps) ? tr.entry(e, per_x) : make_uint2(kZero, 0u);
    for (int st = 0; st < K; ++st) {
        unsigned char *sb = smem + cfg.stage_off + (size_t)st * stage_bytes;
        for (int i = tid; i < (int)(zb >> 3); i += blockDim.x)  // the zero block
            reinterpret_cast<double *>(sb)[i] = 0.0;
        double *rows = reinterpret_cast<double *>(sb + zb);
        if (!per_y) {  // zero halo rows, written once
            for (int i = tid; i < nlo * rowd; i += blockDim.x) rows[i] = 0.0;
            for (int i = tid; i < nhi * rowd; i += blockDim.x)
                rows[(size_t)(nlo + nmid) * rowd + i] = 0.0;
        }
        // rows past the ragged end of the last tile are never loaded: define them
        for (int i = tid; i < (cfg.tyc - rows_valid) * rowd; i += blockDim.x)
            rows[(size_t)(rows_valid + 2 * NN) * rowd + i] = 0.0;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // ---- producer: the first lane of the extra warpgroup refills every slot as soon as the compute
    // warps have released it.  (Issuing from a compute warp put ~10 % on the step: the warp that
    // releases a slot last is the one every other warp is waiting for.)  The v_eff rows (L2 hits) go
    // first: behind the psi rows (DRAM) they would arrive last and hold the stage back.
    if (tid >= cfg.threads_wg) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (tid != cfg.threads_wg) return;
        const unsigned long long pol = policy_evict_last();
        uint32_t s = 0, ph = 0;  // ring slot and pass parity: pass p waits for the release of pass p - 1
        for (int e = 0; e < nsteps; ++e) {
            if (e >= K) mbar_wait(empty_bar + 8 * s, ph ^ 1u);
            const uint2 me = tabp[e];
            const unsigned mx = me.x;
            const uint32_t bar = full_bar + 8 * s;
            if (mx & kZero) {
                mbar_arrive(bar);
            } else {
                const uint32_t dst = stage0 + s * stage_bytes + zb;
                const int xl = (int)(mx & kXMask) - NN;  // wrapped planes come from the other end
                const int xs = xl + ((mx & kWrapLo) ? nx : 0) - ((mx & kWrapHi) ? nx : 0);
                const double *src = psi + (long long)(me.y + (unsigned)xs) * plane_d;
                const bool with_v = HAS_V && (mx & kCentre);
                mbar_expect_tx(bar, tx_psi + (with_v ? tx_v : 0u));
                if (with_v) {
                    if (MODE == 2)  // the band's own right-hand side plane: streamed once
                        bulk_g2s(stage0 + s * stage_bytes + (uint32_t)cfg.v_off,
                                 v_eff + ((long long)(me.y + (unsigned)xl) * ny + y0) * nz, tx_v, bar);
                    else
                        bulk_g2s_hint(stage0 + s * stage_bytes + (uint32_t)cfg.v_off,
                                      reinterpret_cast<const unsigned char *>(v_eff) +
                                          ((long long)xl * ny + y0) * pitchv,
                                      tx_v, bar, pol);
                }
                if (mx & kKeepL2) {
                    if (per_y && nlo > 0)
                        bulk_g2s_hint(dst, src + (long long)(ny - nlo) * rowd, (uint32_t)(nlo * pitch),
                                      bar, pol);
                    bulk_g2s_hint(dst + nlo * pitch, src + (long long)(y0 - NN + nlo) * rowd,
                                  (uint32_t)(nmid * pitch), bar, pol);
                    if (per_y && nhi > 0)
                        bulk_g2s_hint(dst + (nlo + nmid) * pitch, src, (uint32_t)(nhi * pitch), bar, pol);
                } else {
                    if (per_y && nlo > 0)
                        bulk_g2s(dst, src + (long long)(ny - nlo) * rowd, (uint32_t)(nlo * pitch), bar);
                    bulk_g2s(dst + nlo * pitch, src + (long long)(y0 - NN + nlo) * rowd,
                             (uint32_t)(nmid * pitch), bar);
                    if (per_y && nhi > 0)
                        bulk_g2s(dst + (nlo + nmid) * pitch, src, (uint32_t)(nhi * pitch), bar);
                }
            }
            if (++s == (uint32_t)K) {
                s = 0;
                ph ^= 1u;
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
    if (tid >= cfg.threads) return;  // warps that only fill up the last compute warpgroup

    // ---- thread -> micro tile ---------------------------------------------------------------
    int rg = tid / cfg.lanes;
    const int lz = tid - rg * cfg.lanes;
    const bool tactive = rg < cfg.rowgroups;
    if (!tactive) rg = cfg.rowgroups - 1;  // surplus threads shadow the last row group, never store
    const int r0 = rg * TY;                // first halo row (smem row index) of this thread
    const int zc0 = lz * TC;               // first own chunk in the row
    const int own_off = (int)zb + r0 * pitch + zc0 * 16;
    const int v_off = cfg.v_off + r0 * pitchv + lz * (CPLX ? 8 : 16);

    // halo chunks along z: k < ZH left of the own chunks, k >= ZH right of them; an out-of-range
    // chunk on a zero-BC axis reads the zero block at the start of the stage (offset 0).
    int hb[2 * ZH];
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
        hb[k] = valid ? (int)zb + (r0 + NN) * pitch + cz * 16 : 0;
    }
    // real: lanes of odd 8-lane groups fetch z+4 first and z-3 second (see the z taps)
    const bool swp = !CPLX && (tid & 8) != 0;
    const int off8a = swp ? hb[2 * ZH - 1] : hb[0] + 8;
    const int off8b = swp ? hb[0] + 8 : hb[2 * ZH - 1];
    // float64 with PH != 0: real Bloch factors -1 (k_d = 1/2): the same wraps flip a sign instead
    const bool zphase = (PH & 2) && per_z && (g.ph_re[2] != 1.0 || g.ph_im[2] != 0.0) && zwrap != 0;
    const bool yphase = (PH & 1) && per_y && (g.ph_re[1] != 1.0 || g.ph_im[1] != 0.0);
    const bool xphase = (PH & 1) && per_x && (g.ph_re[0] != 1.0 || g.ph_im[0] != 0.0);

    // only the first row group of tile 0 has wrapped rows below, only row groups reaching past the
    // last valid row of the last tile have wrapped rows above
    const bool ylo = yphase && r0 < nlo;
    const bool yhi = yphase && r0 + TY + 2 * NN > nlo + nmid;

    // store addressing: row i of the micro tile is global row y0 + r0 + i
    unsigned row_ok = 0;
#pragma unroll
    for (int i = 0; i < TY; ++i)
        if (tactive && (r0 + i) < rows_valid) row_ok |= 1u << i;
    double *const obase = out + (long long)(y0 + r0) * rowd + zc0 * 2;

    WT wx[NN + 1], wy[NN + 1], wz[NN + 1];  // w[j] = scale c_j / h_d^2, j = 1..NN
#pragma unroll
    for (int j = 1; j <= NN; ++j) {
        wx[j] = (WT)g.w[0][j];
        wy[j] = (WT)g.w[1][j];
        wz[j] = (WT)g.w[2][j];
    }
    const WT wdiag = (WT)g.wdiag;

    // ---- the sweep: one flat loop over the step table ------------------------------------------
    VT acc[NS][NP];
#pragma unroll
    for (int a = 0; a < NS; ++a)
#pragma unroll
        for (int p = 0; p < NP; ++p) acc[a][p] = FdVec<F32>::zero();

    // EX: this thread's share of eps / norm of the current band segment.  One chain each: more
    // chains spill at 160 registers (float64) or run slower (complex128: measured).  Rows outside the
    // grid (surplus threads, ragged last tile) are masked per row; dropping the masks for grids with
    // ny % 4 == 0 was measured slower (ptxas schedules the select form better), so they stay.
    constexpr int EXC = 1;
    double ex_e[EXC], ex_n[EXC];
#pragma unroll
    for (int i = 0; i < EXC; ++i) ex_e[i] = ex_n[i] = 0.0;
    int ex_seg = 0;
    uint32_t st = 0, par = 0;  // ring slot and mbarrier phase parity of the current step
    uint2 m = tabp[0];         // .x flags (| load plane), .y out plane of the current step
    for (int q7 = 0; q7 < nsteps; q7 += NS) {
#pragma unroll
        for (int J = 0; J < NS; ++J) {
            const int q = q7 + J;
            if (q < nsteps) {
                const uint2 mn = tabp[q + 1];
                mbar_wait(full_bar + 8 * st, par);
                const unsigned char *const sb = stage0p + st * stage_bytes;
                const unsigned char *const ub = sb + own_off;

                VT u[NP];  // float64 / float32 paths: own values of the incoming plane
                if constexpr (F32) {
                    // ---- float32 / complex64: 16-byte chunk = 4 floats = 4 real or 2 complex points
                    constexpr int ST = CPLX ? 2 : 1;  // floats per point
                    const float pxr = (float)g.ph_re[0], pxi = (float)g.ph_im[0];
                    const float pyr = (float)g.ph_re[1], pyi = (float)g.ph_im[1];
                    const float pzr = (float)g.ph_re[2], pzi = (float)g.ph_im[2];
                    if (!(m.x & kZero)) {
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            u[i] = lds128f(ub + (NN + i) * pitch);
                            if constexpr (CPLX) {
                                if (yhi && r0 + NN + i >= nlo + nmid) u[i] = cmul4(u[i], pyr, pyi);
                                if (xphase && (m.x & (kWrapLo | kWrapHi)))
                                    u[i] = cmul4(u[i], pxr, (m.x & kWrapLo) ? -pxi : pxi);
                            }
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < TY; ++i) u[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    // x taps, oldest output first: it is complete after this and leaves
#pragma unroll
                    for (int i = 0; i < TY; ++i) fma4(acc[(J + NN + 1) % NS][i], wx[NN], u[i]);
                    if (m.x & kOut) {
                        double *o = obase + (long long)(m.y + (m.x & kXMask) - 2 * NN) * plane_d;
#pragma unroll
                        for (int i = 0; i < TY; ++i)
                            if (row_ok & (1u << i))
                                __stcs(reinterpret_cast<float4 *>(o + i * rowd), acc[(J + NN + 1) % NS][i]);
                    }
#pragma unroll
                    for (int i = 0; i < TY; ++i)
#pragma unroll
                        for (int d = 1; d < NN; ++d) {
                            fma4(acc[(J + NS - d) % NS][i], wx[d], u[i]);
                            fma4(acc[(J + d) % NS][i], wx[d], u[i]);
                        }
                    if (m.x & kCentre) {
                        // diagonal (+ v_eff: one float per point)
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            float4 d4 = make_float4(wdiag, wdiag, wdiag, wdiag);
                            if (HAS_V) {
                                if constexpr (CPLX) {
                                    const float2 vv = *reinterpret_cast<const float2 *>(sb + v_off + i * pitchv);
                                    d4.x += vv.x; d4.y += vv.x; d4.z += vv.y; d4.w += vv.y;
                                } else {
                                    const float4 vv = lds128f(sb + v_off + i * pitchv);
                                    d4.x += vv.x; d4.y += vv.y; d4.z += vv.z; d4.w += vv.w;
                                }
                            }
                            acc[J][i].x = fmaf(d4.x, u[i].x, acc[J][i].x);
                            acc[J][i].y = fmaf(d4.y, u[i].y, acc[J][i].y);
                            acc[J][i].z = fmaf(d4.z, u[i].z, acc[J][i].z);
                            acc[J][i].w = fmaf(d4.w, u[i].w, acc[J][i].w);
                        }
                        // y taps: halo rows of the thread's column
#pragma unroll
                        for (int rr = 0; rr < TY + 2 * NN; ++rr) {
                            if (rr >= NN && rr < NN + TY) continue;  // own rows: already in u
                            float4 c = lds128f(ub + rr * pitch);
                            if constexpr (CPLX) {
                                if (rr < NN) {
                                    if (ylo && r0 + rr < nlo) c = cmul4(c, pyr, -pyi);
                                } else if (yhi && r0 + rr >= nlo + nmid) {
                                    c = cmul4(c, pyr, pyi);
                                }
                            }
#pragma unroll
                            for (int i = 0; i < TY; ++i) {
                                const int d = rr - NN - i;
                                const int ad = d < 0 ? -d : d;
                                if (ad >= 1 && ad <= NN) fma4(acc[J][i], wy[ad], c);
                            }
                        }
#pragma unroll
                        for (int i = 0; i < TY; ++i)
#pragma unroll
                            for (int i2 = 0; i2 < TY; ++i2) {
                                const int ad = i2 > i ? i2 - i : i - i2;
                                if (ad >= 1 && ad <= NN) fma4(acc[J][i], wy[ad], u[i2]);
                            }
                        // z taps: window = ZH chunks | own chunk | ZH chunks, point stride ST floats
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            float w[4 * (2 * ZH + 1)];
#pragma unroll
                            for (int k = 0; k < 2 * ZH; ++k) {
                                float4 t = lds128f(sb + hb[k] + i * pitch);
                                if constexpr (CPLX) {
                                    if (zphase) {
                                        const int wbits = (zwrap >> (2 * k)) & 3;
                                        if (wbits == 1) t = cmul4(t, pzr, -pzi);
                                        if (wbits == 2) t = cmul4(t, pzr, pzi);
                                    }
                                }
                                const int base = 4 * (k < ZH ? k : k + 1);
                                w[base] = t.x; w[base + 1] = t.y; w[base + 2] = t.z; w[base + 3] = t.w;
                            }
                            w[4 * ZH] = u[i].x; w[4 * ZH + 1] = u[i].y; w[4 * ZH + 2] = u[i].z; w[4 * ZH + 3] = u[i].w;
                            float4 &a = acc[J][i];
#pragma unroll
                            for (int j = 1; j <= NN; ++j) {
                                a.x = fmaf(wz[j], w[4 * ZH + 0 - j * ST] + w[4 * ZH + 0 + j * ST], a.x);
                                a.y = fmaf(wz[j], w[4 * ZH + 1 - j * ST] + w[4 * ZH + 1 + j * ST], a.y);
                                a.z = fmaf(wz[j], w[4 * ZH + 2 - j * ST] + w[4 * ZH + 2 + j * ST], a.z);
                                a.w = fmaf(wz[j], w[4 * ZH + 3 - j * ST] + w[4 * ZH + 3 + j * ST], a.w);
                            }
                        }
                    }
                } else if constexpr (CPLX) {
                    // complex128: the rows of the thread's column stream through one register
                    // pair (no copy of the own values is kept: at 168 registers that is what
                    // lets the loads run ahead; measured +8 % on cfg4, -9 % for float64)
                    // used only if the step completes an output plane
                    double *const o = obase + (long long)(m.y + (m.x & kXMask) - 2 * NN) * plane_d;
                    const bool store_now = (m.x & kOut) != 0;

                    // One own row of the incoming plane: its value c adds w_x[|d|] c to the outputs
                    // xl + d in flight (d = -NN: complete after this, stored and gone; d = +NN: born).
                    auto x_taps_row = [&](int i, const double2 c) {
                        double2 &lv = acc[(J + NN + 1) % NS][i];
                        fma2(lv, wx[NN], c);
                        if (store_now && (row_ok & (1u << i)))
                            __stcs(reinterpret_cast<double2 *>(o + i * rowd), lv);
#pragma unroll
                        for (int d = 1; d < NN; ++d) {
                            fma2(acc[(J + NS - d) % NS][i], wx[d], c);
                            fma2(acc[(J + d) % NS][i], wx[d], c);
                        }
                        acc[(J + NN) % NS][i] = mul2(wx[NN], c);
                    };

                    if (!(m.x & kCentre)) {
                        // ---- halo step (prologue / epilogue of a band segment): x taps only
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            double2 c = make_double2(0.0, 0.0);
                            if (!(m.x & kZero)) {
                                c = lds128(ub + (NN + i) * pitch);
                                if (CPLX && (PH & 1)) {
                                    // rows past a ragged tile end are wrapped rows: neighbours of the
                                    // last valid rows, so they carry the y Bloch factor
                                    if (yhi && r0 + NN + i >= nlo + nmid) c = cmul(c, g.ph_re[1], g.ph_im[1]);
                                    if (xphase && (m.x & (kWrapLo | kWrapHi)))
                                        c = cmul(c, g.ph_re[0], (m.x & kWrapLo) ? -g.ph_im[0] : g.ph_im[0]);
                                }
                            }
                            x_taps_row(i, c);
                        }
                    } else {
                        // ---- centre step: the TY + 2 NN rows of the thread's column stream through
                        // one register pair; a halo row feeds the y taps, an own row also the x taps,
                        // the diagonal (+ v_eff) and the z taps of its output
#pragma unroll
                        for (int rr = 0; rr < TY + 2 * NN; ++rr) {
                            double2 c = lds128(ub + rr * pitch);
                            if (CPLX && (PH & 1)) {
                                if (rr < NN) {
                                    if (ylo && r0 + rr < nlo) c = cmul(c, g.ph_re[1], -g.ph_im[1]);
                                } else if (yhi && r0 + rr >= nlo + nmid) {
                                    c = cmul(c, g.ph_re[1], g.ph_im[1]);
                                }
                            }
#pragma unroll
                            for (int i = 0; i < TY; ++i) {  // y taps into the other rows
                                const int d = rr - NN - i;
                                const int ad = d < 0 ? -d : d;
                                if (ad >= 1 && ad <= NN) fma2(acc[J][i], wy[ad], c);
                            }
                            if (rr >= NN && rr < NN + TY) {
                                const int i = rr - NN;
                                x_taps_row(i, c);
                                double2 &a = acc[J][i];
                                // diagonal (+ v_eff)
                                double d0 = wdiag;
                                if (HAS_V) d0 += lds64(sb + v_off + i * pitchv);
                                // z taps
                                {
                                    // chunk = one complex point; hz = L_NN .. L_1, R_1 .. R_NN
                                    double2 hz[2 * ZH];
#pragma unroll
                                    for (int k = 0; k < 2 * ZH; ++k) hz[k] = lds128(sb + hb[k] + i * pitch);
                                    if ((PH & 2) && zphase) {
#pragma unroll
                                        for (int k = 0; k < 2 * ZH; ++k) {
                                            const int wbits = (zwrap >> (2 * k)) & 3;
                                            if (wbits == 1) hz[k] = cmul(hz[k], g.ph_re[2], -g.ph_im[2]);
                                            if (wbits == 2) hz[k] = cmul(hz[k], g.ph_re[2], g.ph_im[2]);
                                        }
                                    }
                                    if constexpr (!EX) {
                                        a.x = fma(d0, c.x, a.x);
                                        a.y = fma(d0, c.y, a.y);
                                    }
                                    if constexpr (EX) {
                                        // a holds the backward x and y taps of this row; add the
                                        // backward z taps: eps += d |c|^2 + 2 Re conj(c) a
#pragma unroll
                                        for (int j = 1; j <= NN; ++j) fma2(a, wz[j], hz[NN - j]);
                                        if (row_ok & (1u << i)) {
                                            const double s2 = fma(c.x, c.x, c.y * c.y);
                                            ex_n[i % EXC] += s2;
                                            ex_e[i % EXC] = fma(c.x, a.x, fma(c.y, a.y, fma(0.5 * d0, s2, ex_e[i % EXC])));
                                        }
#pragma unroll
                                        for (int j = 1; j <= NN; ++j) fma2(a, wz[j], hz[NN + j - 1]);
                                        a.x = fma(d0, c.x, a.x);
                                        a.y = fma(d0, c.y, a.y);
                                    } else {
#pragma unroll
                                        for (int j = 1; j <= NN; ++j) {
                                            fma2(a, wz[j], hz[NN - j]);
                                            fma2(a, wz[j], hz[NN + j - 1]);
                                        }
                                    }
                                }
                            }
                        }
                    }

                } else {
                    // ---- own values of the incoming plane
                    if (!(m.x & kZero)) {
#pragma unroll
                        for (int i = 0; i < TY; ++i)
#pragma unroll
                            for (int t = 0; t < TC; ++t)
                                u[i * TC + t] = lds128(ub + (NN + i) * pitch + t * 16);
                        if constexpr ((PH & 1) != 0) {
                            // real Bloch factor -1: wrapped x planes, and own rows past a ragged tile
                            // end (wrapped rows: y neighbours of the last valid rows)
                            const bool xneg = xphase && (m.x & (kWrapLo | kWrapHi));
#pragma unroll
                            for (int i = 0; i < TY; ++i)
                                if (xneg != (yhi && r0 + NN + i >= nlo + nmid)) {
#pragma unroll
                                    for (int t = 0; t < TC; ++t)
                                        u[i * TC + t] = make_double2(-u[i * TC + t].x, -u[i * TC + t].y);
                                }
                        }
                    } else {
#pragma unroll
                        for (int p = 0; p < NP; ++p) u[p] = make_double2(0.0, 0.0);
                    }

                    // ---- x taps, oldest output first: it is complete after this and leaves
#pragma unroll
                    for (int p = 0; p < NP; ++p) fma2(acc[(J + NN + 1) % NS][p], wx[NN], u[p]);
                    if (m.x & kOut) {
                        double *o = obase + (long long)(m.y + (m.x & kXMask) - 2 * NN) * plane_d;
#pragma unroll
                        for (int i = 0; i < TY; ++i)
                            if (row_ok & (1u << i)) {
#pragma unroll
                                for (int t = 0; t < TC; ++t)
                                    __stcs(reinterpret_cast<double2 *>(o + i * rowd) + t,
                                           acc[(J + NN + 1) % NS][i * TC + t]);
                            }
                    }
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
#pragma unroll
                        for (int d = 1; d < NN; ++d) {  // outputs xl - d and xl + d
                            fma2(acc[(J + NS - d) % NS][p], wx[d], u[p]);
                            fma2(acc[(J + d) % NS][p], wx[d], u[p]);
                        }
                    }

                    if (m.x & kCentre) {
                        if constexpr (EX) {
                            // acc[J] holds the backward x taps B of this plane: eps += u (B + H_rest u),
                            // the second term once acc[J] is complete (below)
#pragma unroll
                            for (int i = 0; i < TY; ++i)
                                if (row_ok & (1u << i))
                                    ex_e[i % EXC] = fma(u[i].x, acc[J][i].x, fma(u[i].y, acc[J][i].y, ex_e[i % EXC]));
                        }
                        // ---- diagonal (+ v_eff), or the Jacobi form (1 - omega) phi + rhs_coef rhs
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            double d0 = wdiag, d1 = wdiag;
                            if (MODE == 1) {
                                const double2 vv = lds128(sb + v_off + i * pitchv);
                                d0 += vv.x;
                                d1 += vv.y;
                            }
                            acc[J][i].x = fma(d0, u[i].x, acc[J][i].x);
                            acc[J][i].y = fma(d1, u[i].y, acc[J][i].y);
                            if (MODE == 2) {
                                const double2 vv = lds128(sb + v_off + i * pitchv);
                                acc[J][i].x = fma(g.rhs_coef, vv.x, acc[J][i].x);
                                acc[J][i].y = fma(g.rhs_coef, vv.y, acc[J][i].y);
                            }
                        }
                        // ---- y taps: stream the TY + 6 rows of the thread's column through
#pragma unroll
                        for (int rr = 0; rr < TY + 2 * NN; ++rr) {
                            if (rr >= NN && rr < NN + TY) continue;  // own rows: already in u
                            double2 c[TC];
#pragma unroll
                            for (int t = 0; t < TC; ++t) c[t] = lds128(ub + rr * pitch + t * 16);
                            if constexpr ((PH & 1) != 0) {
                                // the own values above carry the x sign of a wrapped plane, but a centre
                                // plane is never wrapped: only the y wraps matter here
                                if ((rr < NN) ? (ylo && r0 + rr < nlo) : (yhi && r0 + rr >= nlo + nmid)) {
#pragma unroll
                                    for (int t = 0; t < TC; ++t) c[t] = make_double2(-c[t].x, -c[t].y);
                                }
                            }
#pragma unroll
                            for (int i = 0; i < TY; ++i) {
                                const int d = rr - NN - i;
                                const int ad = d < 0 ? -d : d;
                                if (ad >= 1 && ad <= NN) {
#pragma unroll
                                    for (int t = 0; t < TC; ++t) fma2(acc[J][i * TC + t], wy[ad], c[t]);
                                }
                            }
                        }
                        // own rows are y neighbours of each other
#pragma unroll
                        for (int i = 0; i < TY; ++i)
#pragma unroll
                            for (int i2 = 0; i2 < TY; ++i2) {
                                const int ad = i2 > i ? i2 - i : i - i2;
                                if (ad >= 1 && ad <= NN) {
#pragma unroll
                                    for (int t = 0; t < TC; ++t)
                                        fma2(acc[J][i * TC + t], wy[ad], u[i2 * TC + t]);
                                }
                            }
                        // ---- z taps
#pragma unroll
                        for (int i = 0; i < TY; ++i) {
                            {
                                double2 &a = acc[J][i];
                                const double2 o = u[i];
                                if constexpr (NN == 3) {
                                    // chunk = points (z, z+1); halo = z-3 | z-2,z-1 | z+2,z+3 | z+4.
                                    // The two 8-byte halo words come in two loads whose lanes
                                    // alternate (by groups of 8) between z-3 and z+4, so each half
                                    // warp touches 32 distinct banks (an 8-byte load at a 16-byte
                                    // lane stride would be a 2-way bank conflict).
                                    const double e0 = lds64(sb + off8a + i * pitch);
                                    const double e1 = lds64(sb + off8b + i * pitch);
                                    double l3 = swp ? e1 : e0;
                                    double r4 = swp ? e0 : e1;
                                    double2 l21 = lds128(sb + hb[1] + i * pitch);
                                    double2 r23 = lds128(sb + hb[2] + i * pitch);
                                    if constexpr ((PH & 2) != 0) {
                                        if (zphase) {  // wrapped halo chunks flip their sign
                                            if (zwrap & (3 << 0)) l3 = -l3;
                                            if (zwrap & (3 << 2)) l21 = make_double2(-l21.x, -l21.y);
                                            if (zwrap & (3 << 4)) r23 = make_double2(-r23.x, -r23.y);
                                            if (zwrap & (3 << 6)) r4 = -r4;
                                        }
                                    }
                                    a.x = fma(wz[1], l21.y, a.x);
                                    a.x = fma(wz[1], o.y, a.x);
                                    a.x = fma(wz[2], l21.x, a.x);
                                    a.x = fma(wz[2], r23.x, a.x);
                                    a.x = fma(wz[3], l3, a.x);
                                    a.x = fma(wz[3], r23.y, a.x);
                                    a.y = fma(wz[1], o.x, a.y);
                                    a.y = fma(wz[1], r23.x, a.y);
                                    a.y = fma(wz[2], l21.y, a.y);
                                    a.y = fma(wz[2], r23.y, a.y);
                                    a.y = fma(wz[3], l21.x, a.y);
                                    a.y = fma(wz[3], r4, a.y);
                                } else if constexpr (NN == 2) {
                                    // halo = z-2,z-1 | z+2,z+3: the two neighbouring chunks
                                    double2 l21 = lds128(sb + hb[0] + i * pitch);
                                    double2 r23 = lds128(sb + hb[1] + i * pitch);
                                    if constexpr ((PH & 2) != 0) {
                                        if (zphase) {
                                            if (zwrap & (3 << 0)) l21 = make_double2(-l21.x, -l21.y);
                                            if (zwrap & (3 << 2)) r23 = make_double2(-r23.x, -r23.y);
                                        }
                                    }
                                    a.x = fma(wz[1], l21.y, a.x);
                                    a.x = fma(wz[1], o.y, a.x);
                                    a.x = fma(wz[2], l21.x, a.x);
                                    a.x = fma(wz[2], r23.x, a.x);
                                    a.y = fma(wz[1], o.x, a.y);
                                    a.y = fma(wz[1], r23.x, a.y);
                                    a.y = fma(wz[2], l21.y, a.y);
                                    a.y = fma(wz[2], r23.y, a.y);
                                } else if constexpr (NN >= 4) {
                                    // general form: all halo chunks as 16-byte loads.  zl[p] = point
                                    // z - 2 ZH + p (left block, farthest chunk first), zr[p] = point
                                    // z + 2 + p (right block); own chunk = points z, z + 1.
                                    double zl[2 * ZH], zr[2 * ZH];
#pragma unroll
                                    for (int k = 0; k < ZH; ++k) {
                                        const double2 tl = lds128(sb + hb[k] + i * pitch);
                                        const double2 tr = lds128(sb + hb[ZH + k] + i * pitch);
                                        zl[2 * k] = tl.x;
                                        zl[2 * k + 1] = tl.y;
                                        zr[2 * k] = tr.x;
                                        zr[2 * k + 1] = tr.y;
                                    }
#pragma unroll
                                    for (int j = 1; j <= NN; ++j) {
                                        a.x = fma(wz[j], zl[2 * ZH - j], a.x);
                                        a.x = fma(wz[j], (j == 1) ? o.y : zr[j - 2 < 0 ? 0 : j - 2], a.x);
                                        a.y = fma(wz[j], (j == 1) ? o.x : zl[2 * ZH - (j - 1)], a.y);
                                        a.y = fma(wz[j], zr[j - 1], a.y);
                                    }
                                } else {
                                    // halo = z-1 | z+2: two 8-byte words, fetched pairwise as above
                                    const double e0 = lds64(sb + off8a + i * pitch);
                                    const double e1 = lds64(sb + off8b + i * pitch);
                                    double l1 = swp ? e1 : e0;
                                    double r2 = swp ? e0 : e1;
                                    if constexpr ((PH & 2) != 0) {
                                        if (zphase) {
                                            if (zwrap & (3 << 0)) l1 = -l1;
                                            if (zwrap & (3 << 2)) r2 = -r2;
                                        }
                                    }
                                    a.x = fma(wz[1], l1, a.x);
                                    a.x = fma(wz[1], o.y, a.x);
                                    a.y = fma(wz[1], o.x, a.y);
                                    a.y = fma(wz[1], r2, a.y);
                                }
                            }
                        }
                        if constexpr (EX) {
#pragma unroll
                            for (int i = 0; i < TY; ++i)
                                if (row_ok & (1u << i)) {
                                    ex_e[i % EXC] = fma(u[i].x, acc[J][i].x, fma(u[i].y, acc[J][i].y, ex_e[i % EXC]));
                                    ex_n[i % EXC] = fma(u[i].x, u[i].x, fma(u[i].y, u[i].y, ex_n[i % EXC]));
                                }
                        }
                    }

                }

                // ---- release the slot (the producer refills it once every compute warp has)
                __syncwarp();
                if (elect_one()) mbar_arrive(empty_bar + 8 * st);

                // ---- float64 / float32 paths: the output NN planes ahead is born
                if constexpr (F32) {
#pragma unroll
                    for (int p = 0; p < NP; ++p)
                        acc[(J + NN) % NS][p] = make_float4(wx[NN] * u[p].x, wx[NN] * u[p].y,
                                                            wx[NN] * u[p].z, wx[NN] * u[p].w);
                } else if constexpr (!CPLX) {
#pragma unroll
                    for (int p = 0; p < NP; ++p) acc[(J + NN) % NS][p] = mul2(wx[NN], u[p]);
                }
                if constexpr (EX) {
                    // end of a band segment: this warp's partial sums go out, fixed butterfly order
                    if (mn.y != m.y || q + 1 == nsteps) {
                        double se = 0.0, sn = 0.0;
#pragma unroll
                        for (int i = 0; i < EXC; ++i) {
                            se += ex_e[i];
                            sn += ex_n[i];
                            ex_e[i] = ex_n[i] = 0.0;
                        }
                        if (CPLX) se *= 2.0;  // the complex body accumulates half of eps
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) {
                            se += __shfl_xor_sync(0xffffffffu, se, o);
                            sn += __shfl_xor_sync(0xffffffffu, sn, o);
                        }
                        if ((tid & 31) == 0) {
                            double *w = aux.ws + 2 * ((((team * aux.maxseg + ex_seg) * cfg.nytiles + yt) *
                                                       (long long)nwarps) + (tid >> 5));
                            w[0] = se;
                            w[1] = sn;
                        }
                        ++ex_seg;
                    }
                }
                if (++st == (uint32_t)K) {
                    st = 0;
                    par ^= 1u;
                }
                m = mn;
            }
        }
    }
}

}  // namespace
