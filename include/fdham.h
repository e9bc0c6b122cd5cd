/*
 * fdham.h -- C ABI of libfdham: the batched finite-difference Kohn-Sham apply on one B200.
 *
 *     (H psi)_b[i] = sum_{d in x,y,z} (-1/2 / h_d^2) [ c_0 psi_b[i]
 *                        + sum_{j=1..nn} c_j ( psi^_b(i + j e_d) + psi^_b(i - j e_d) ) ]
 *                    + v_eff[i] psi_b[i]
 *
 * Operation defined by: the PAW Hamiltonian Eq. 6, first two terms "-1/2 nabla^2 + v~_KS(r)"
 * (section III.A); the Laplacian is the "finite difference (FD) ...
 * representation of kinetic energy operator on a uniform Cartesian grid" (section
 * III.B.1), i.e. "applying a finite-difference stencil to a uniform grid", the first C hot spot
 * the paper lists (section II.B).  Boundaries: zero ("potential go to zero on the
 * cell boundaries") or periodic carrying the Bloch factor of Eq. 13
 * (PAPER.md:225).  Bands are independent.  Stencil weights c_j are the standard
 * central weights of order 2*nn (nn = 3: -49/18, 3/2, -3/20, 1/90, BASELINE.json); all readings
 * taken where the paper is silent are listed in DESIGN.md.
 *
 * psi^ (fused halo handling): for a tap index p_d = i_d +- j outside [0, n_d)
 *     zero-BC axis  -> 0
 *     periodic axis -> psi[p - w n_d e_d] * exp(+2 pi i k_d w), w = +1 past the upper end, -1
 *                      before the lower end (the array holds the full Bloch function).
 *
 * Conventions common to all calls
 *   - every function returns FD_OK (0) or a negative fd_status; nothing throws, aborts,
 *     allocates inside an apply, or synchronises the device (the *_host variant excepted);
 *   - "device pointer" = memory of the plan's CUDA device; "host pointer" = ordinary CPU memory;
 *   - arrays are C-contiguous, z fastest: psi/out [nbands, nx, ny, nz], v_eff [nx, ny, nz];
 *     element = double (FD_F64) or interleaved (re, im) doubles (FD_C128); v_eff is double (float
 *     for the single-precision dtypes FD_F32 / FD_C64);
 *   - psi and v_eff are read-only; out is fully overwritten (no accumulate) and must not overlap
 *     psi or v_eff;  the caller owns all three; the library owns only the plan;
 *   - applies are enqueued on `cuda_stream` (a cudaStream_t cast to void*, NULL = legacy default
 *     stream) and return immediately; a plan is immutable (the diagnostic fd_plan_set_kernel
 *     excepted: call it before the plan is shared) and may be used from several streams;
 *   - the plan's device must be the calling thread's current CUDA device in every call that
 *     launches or copies (FD_ERR_INVALID otherwise); fd_create itself restores the caller's
 *     current device before it returns;
 *   - there is no CPU fallback: without a usable CUDA device fd_create fails with FD_ERR_CUDA.
 */
#ifndef FDHAM_H
#define FDHAM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define FD_API __attribute__((visibility("default")))
#else
#define FD_API
#endif

typedef struct fd_plan fd_plan; /* opaque, owned by the library */

enum { FD_BC_ZERO = 0, FD_BC_PERIODIC = 1 };
enum { FD_F64 = 0, FD_C128 = 1, FD_F32 = 2, FD_C64 = 3 };
enum {
    FD_OK = 0,
    FD_ERR_INVALID = -1,     /* NULL pointer, bad shape/h/nn/bc/dtype/nbands, misaligned pointer  */
    FD_ERR_UNSUPPORTED = -2, /* valid request this build cannot run                               */
    FD_ERR_ALIAS = -3,       /* out overlaps psi or v_eff                                         */
    FD_ERR_CUDA = -4,        /* CUDA runtime failure (no device, launch error, ...)               */
    FD_ERR_NOMEM = -5,       /* host or device allocation failed                                  */
    FD_ERR_SCRATCH = -6      /* batch needs more than FD_STATIC_SCRATCH_BYTES of built-in scratch */
};

/* Kernel families, for fd_plan_set_kernel / fd_plan_get_kernel (diagnostics and A/B timing). */
enum {
    FD_KERNEL_AUTO = 0,    /* pick the fastest supported kernel for the plan (default)            */
    FD_KERNEL_GENERIC = 1, /* one thread per grid point, any nn / shape / bc                      */
    FD_KERNEL_SWEEP = 2    /* TMA-staged y-z tiles + register sweep along x (nn = 1..3)            */
};

/*
 * fd_create -- build an immutable plan: stencil weights
 * w_d[j] = -1/2 c_j / h_d^2, merged diagonal, per-axis wrap phases exp(+-2 pi i k_d), kernel and
 * tile choice.  Host-side only apart from selecting `device`.
 *   plan       out: receives the plan; untouched on failure
 *   shape      host: nx, ny, nz = extents of the STORED arrays (>= 1)
 *   h          host: grid spacings, atomic units (Bohr), finite and > 0
 *   nn         stencil half width (order 2*nn), 1..6
 *   bc         host: FD_BC_ZERO | FD_BC_PERIODIC per axis; a periodic axis needs n_d >= nn
 *   k_reduced  host: Bloch vector in reduced coordinates, NULL = Gamma; must be 0 on zero-BC axes
 *   dtype      FD_F64 (requires 2 k_d integer on every axis: the Bloch factors are then +-1 and the
 *              data stay real, e.g. the zone-boundary point k = 1/2) or FD_C128; FD_F32 / FD_C64:
 *              the same in single precision: psi, out AND v_eff are float32 /
 *              interleaved float32 pairs, fp32 accumulation, fd_apply_kinetic / fd_apply_hamiltonian
 *              only (every other call returns FD_ERR_UNSUPPORTED; there is no fallback to another
 *              precision).  The bandwidth kernel takes nn <= 3, every axis >= 8, nz a multiple of 4
 *              (FD_F32) or 2 (FD_C64), FD_F32 at Gamma; other plans run on the generic kernel
 *   device     CUDA device ordinal
 * Errors: FD_ERR_INVALID for any violated constraint above, FD_ERR_UNSUPPORTED for nx > 65535 or
 * ny > 262140 (no kernel of this build launches such a grid), FD_ERR_CUDA if the device cannot be
 * used, FD_ERR_NOMEM.
 */
FD_API int fd_create(fd_plan **plan, const int32_t shape[3], const double h[3], int32_t nn,
              const int32_t bc[3], const double k_reduced[3], int32_t dtype, int32_t device);

/*
 * fd_create_scaled -- fd_create with `scale` in place of the -1/2 of Eq. 6: the plan's applies
 * compute out = scale lap_FD psi (+ v_eff psi), weights w_d[j] = scale c_j / h_d^2.  scale = 1 gives
 * the plain FD Laplacian of the Poisson problem (the paper's grid Poisson solvers, PAPER.md:248,
 * use the same stencil).  fd_create(...) == fd_create_scaled(..., -0.5).
 * Extra error: FD_ERR_INVALID for a non-finite scale.
 */
FD_API int fd_create_scaled(fd_plan **plan, const int32_t shape[3], const double h[3], int32_t nn,
                     const int32_t bc[3], const double k_reduced[3], int32_t dtype, int32_t device,
                     double scale);

/*
 * fd_apply_kinetic -- out = T psi = -1/2 lap_FD psi  (steps a2+a3+a5+a6 of SURVEY 8(a); Eq. 6
 * first term).
 *   psi, out   device pointers, [nbands,nx,ny,nz] of the plan's dtype, 16-byte aligned
 *   nbands     >= 0; 0 is a no-op returning FD_OK
 * Errors: FD_ERR_INVALID (NULL plan/pointer, nbands < 0, misaligned), FD_ERR_ALIAS,
 * FD_ERR_CUDA (launch failure, checked with cudaPeekAtLastError, no sync).
 */
FD_API int fd_apply_kinetic(const fd_plan *plan, const void *psi, void *out, int64_t nbands,
                     void *cuda_stream);

/*
 * fd_apply_hamiltonian -- out = T psi + v_eff psi (adds step a4: the local potential of Eq. 6,
 * one real array shared by all bands).
 *   v_eff      device pointer, [nx,ny,nz] of the plan's REAL type -- double for FD_F64 / FD_C128
 *              plans, float for FD_F32 / FD_C64 plans (hence const void *: a single-precision
 *              caller passes its float array without a cast through the wrong type) -- 16-byte
 *              aligned
 * Other arguments and errors as fd_apply_kinetic.
 */
FD_API int fd_apply_hamiltonian(const fd_plan *plan, const void *psi, const void *v_eff, void *out,
                         int64_t nbands, void *cuda_stream);

/*
 * fd_apply_hamiltonian_host -- the same apply for HOST buffers (end-to-end path): copies psi and
 * v_eff to the device, applies, copies H psi back, in band chunks that overlap H2D, kernel and
 * D2H on internal streams.  v_eff may be NULL (kinetic only).  Blocks until `out` is complete.
 * Buffers may be pageable or pinned (pinned = faster).  Creates and destroys a workspace per call
 * (FD_ERR_NOMEM if that fails); a caller that applies repeatedly keeps one with the _ws form:
 *
 * fd_workspace_create -- device staging buffers (3 ring slots of `chunk_bytes` in + out, 0 = 64 MiB,
 *   at least one band; plus one v_eff array) and the internal streams, for plans of this plan's
 *   grid and dtype on its device.  Owned by the caller until fd_workspace_destroy (NULL = no-op).
 * fd_apply_hamiltonian_host_ws -- fd_apply_hamiltonian_host on a workspace: no allocation, no
 *   stream creation in the call.  One call at a time per workspace.  FD_ERR_INVALID if the
 *   workspace does not match the plan; FD_ERR_ALIAS if out_host overlaps psi_host or v_eff_host.
 */
typedef struct fd_workspace fd_workspace;
FD_API int fd_apply_hamiltonian_host(const fd_plan *plan, const void *psi_host, const double *v_eff_host,
                              void *out_host, int64_t nbands);
FD_API int fd_workspace_create(fd_workspace **ws, const fd_plan *plan, int64_t chunk_bytes);
FD_API int fd_workspace_destroy(fd_workspace *ws);
FD_API int fd_apply_hamiltonian_host_ws(const fd_plan *plan, fd_workspace *ws, const void *psi_host,
                                 const double *v_eff_host, void *out_host, int64_t nbands);

/*
 * the eigensolver epilogue.  Every SCF step (subspace diagonalisation, then the
 * Davidson / RMM-DIIS step) and every RT-TDDFT step (Eq. 91)
 * needs, right after H psi, the band energies and the residuals.
 *
 * fd_apply_hamiltonian_expect -- out = H psi (v_eff == NULL: T psi) AND, from the same pass,
 *     eps[b]  = Re sum_i conj(psi_b[i]) (H psi)_b[i]     (H is Hermitian: the imaginary part is zero)
 *     norm[b] = sum_i |psi_b[i]|^2                         (plain grid sums; x h_x h_y h_z = integrals)
 *   eps, norm   device pointers, double [nbands]
 *   workspace   device pointer, 16-byte aligned, >= fd_expect_workspace_bytes(plan, nbands) bytes,
 *               owned by the caller, scratch (per-warp partial sums; reduced in a fixed order by a
 *               second small launch: results are bit-reproducible run to run, no atomics)
 *   Other arguments and errors as fd_apply_hamiltonian; FD_ERR_INVALID also for a short workspace,
 *   FD_ERR_ALIAS if out overlaps eps / norm / workspace.
 * fd_expect_workspace_bytes -- bytes needed for a batch of nbands (>= 0), or a negative fd_status.
 * fd_residual -- r_b = hpsi_b - (eps[b] / norm[b]) psi_b  (the residual R_b = H psi_b - eps_b psi_b
 *   for normalised psi).  r may be exactly hpsi (in place) but must not overlap psi.
 */
FD_API int64_t fd_expect_workspace_bytes(const fd_plan *plan, int64_t nbands);
FD_API int fd_apply_hamiltonian_expect(const fd_plan *plan, const void *psi, const double *v_eff, void *out,
                                double *eps, double *norm, int64_t nbands, void *workspace,
                                int64_t workspace_bytes, void *cuda_stream);
FD_API int fd_residual(const fd_plan *plan, const void *psi, const void *hpsi, const double *eps,
                const double *norm, void *r, int64_t nbands, void *cuda_stream);

/*
 * fd_apply_hamiltonian_expect_static -- fd_apply_hamiltonian_expect without a workspace argument,
 * for callers that cannot allocate device memory.  Who they are: a plug-in running under a host
 * application whose memory pool owns the device and which forbids cudaMalloc in plug-ins; code on a
 * latency path, where cudaMalloc / cudaFree would synchronise the whole device; code whose device
 * memory belongs to a caching allocator that cannot be reached from C.  Such a caller has nowhere
 * to get the workspace of fd_apply_hamiltonian_expect from, so the library brings its own: a fixed
 * array of FD_STATIC_SCRATCH_BYTES (4 MiB) that is part of the library image.  Every GPU on which
 * the library's code gets loaded holds that array from then until the process exits.
 *
 *   plan, psi, v_eff, out, eps, norm, nbands, cuda_stream: as fd_apply_hamiltonian_expect; the
 *   caller still owns and passes every input and output.  Results are bit-identical to
 *   fd_apply_hamiltonian_expect on the same arguments (same kernels, same order of additions).
 *
 * What the call does not do: it calls no cudaMalloc, cudaFree or other allocating routine, on any
 * call.  What the first call on each device does in addition: it looks up the device address of
 * the array (cudaGetSymbolAddress, with the plan's device current) and caches it; the runtime may
 * load the library's code on that device at that moment.  Make that first call outside any stream
 * capture.
 *
 * Limit: a batch whose partial sums need more than FD_STATIC_SCRATCH_BYTES (the figure
 * fd_expect_workspace_bytes(plan, nbands) reports) is refused with FD_ERR_SCRATCH before anything
 * is launched; split the batch, or use fd_apply_hamiltonian_expect with a workspace of your own.
 * For scale: 96^3 x 256 bands on the fused form needs about 0.22 MiB; the two-pass form (batches on
 * the generic kernel) needs 16 bytes per band and per 16384 grid values.
 *
 * Sharing: all calls on one device use the same array, on whatever stream and for whatever plan,
 * and the array keeps what the last call wrote (no call depends on it: every value read was stored
 * earlier in the same call).  Two calls that can overlap on the GPU -- different streams without
 * an event between them, or different host threads -- race on the array and give wrong eps / norm
 * (out is unaffected).  Calls on one stream are ordered and safe.
 * Other errors as fd_apply_hamiltonian_expect (FD_ERR_UNSUPPORTED for FD_F32 / FD_C64 plans,
 * FD_ERR_INVALID when the plan's device is not current, ...).
 */
#define FD_STATIC_SCRATCH_BYTES (4 * 1024 * 1024)
FD_API int fd_apply_hamiltonian_expect_static(const fd_plan *plan, const void *psi, const double *v_eff,
                                       void *out, double *eps, double *norm, int64_t nbands,
                                       void *cuda_stream);

/*
 * fd_jacobi_sweep: one weighted-Jacobi relaxation sweep for A phi = rhs with
 * A = scale lap_FD, the operator of a plan made by fd_create_scaled (scale = 1: the Poisson
 * operator; "multigrid ... Jacobi or Gauss-Seidel" Poisson solvers):
 *     out[i] = phi[i] + omega (rhs[i] - (A phi)[i]) / A_ii,   A_ii = scale c_0 sum_d 1/h_d^2
 * every point from the OLD phi.  phi, rhs, out: device pointers, double [nbands,nx,ny,nz], 16-byte
 * aligned; out must not overlap phi or rhs.  FD_F64 plans only (FD_ERR_UNSUPPORTED otherwise).
 */
FD_API int fd_jacobi_sweep(const fd_plan *plan, const double *phi, const double *rhs, double *out,
                    int64_t nbands, double omega, void *cuda_stream);

/*
 * fd_poisson_residual -- out = rhs - A phi for the plan's A = scale lap_FD (the residual of the
 * Poisson problem, same kernels and argument rules as fd_jacobi_sweep).
 */
FD_API int fd_poisson_residual(const fd_plan *plan, const double *phi, const double *rhs, double *out,
                        int64_t nbands, void *cuda_stream);

/*
 * grid transfer between a fine grid (spacing h) and the coarse grid of spacing
 * 2h ("interpolating from one uniform grid to another", the second C hot spot of PAPER.md:150;
 * multigrid).  The paper prints no weights; readings R13 / R14:
 *   1-D interpolation of order p: a fine point on a coarse point copies it; a fine point half way
 *     between two coarse points is sum_{j=1..p} b_j (c[lo - j + 1] + c[lo + j]) with the midpoint
 *     Lagrange weights b_j (p = 1: 1/2; p = 2: 9/16, -1/16; p = 3: 150/256, -25/256, 3/256);
 *     3-D = tensor product.  Restriction = the transpose / 8: per axis weight 1/2 on the fine point
 *     of the coarse point and b_j / 2 on the fine points at distance 2j - 1.
 *   Index map per axis: periodic n_f = 2 n_c, coarse I on fine 2I; zero-BC n_f = 2 n_c + 1, coarse
 *     I on fine 2I + 1 (stored points are interior points; the walls coincide).  Values outside
 *     [0, n) are wrapped (periodic) or 0 (zero BC).
 * fd_restrict:    coarse[nbands, nc] <- fine[nbands, nf];   fd_interpolate: fine <- coarse.
 *   shape_fine   host: nf per axis (even >= 2 on periodic axes, odd >= 3 on zero-BC axes)
 *   bc           host: FD_BC_* per axis;   p: 1..3 (4..6: FD_ERR_UNSUPPORTED)
 *   fine, coarse device pointers (current device), double, C-contiguous, 8-byte aligned, no overlap
 * Stateless (no plan); enqueued on cuda_stream; errors as the applies, FD_ERR_UNSUPPORTED also for
 * z rows too long for the kernels' tiles (fine nz > 682 for fd_interpolate, coarse nz > 2048).
 */
FD_API int fd_restrict(const int32_t shape_fine[3], const int32_t bc[3], int32_t p, const double *fine,
                double *coarse, int64_t nbands, void *cuda_stream);
FD_API int fd_interpolate(const int32_t shape_fine[3], const int32_t bc[3], int32_t p,
                   const double *coarse, double *fine, int64_t nbands, void *cuda_stream);

/*
 * the PAW non-local term: third term of the PAW Hamiltonian, Eq. 6
 * "sum_a sum_ii' |p~^a_i> Delta H^a_ii' <p~^a_i'|", and with Delta S the overlap
 * operator S~ = 1 + sum |p~> Delta S <p~| of Eq. 7; "overlaps between projector
 * functions and wave functions" is the third C hot spot the paper lists.
 *
 *     P_b[a,i]  = dv sum_{r in box_a} p~^a_i(r) psi^_b(r),        dv = h_x h_y h_z
 *     out_b(r') += conj(phase(r)) sum_{i,i'} p~^a_i(r) dO^a_ii' P_b[a,i']   for every atom a
 *
 * PAW data sets are not available here, so the library takes whatever localised functions the
 * caller supplies (synthetic in tests and bench).  Atom a owns a box of box_size[a]
 * grid points starting at index box_start[a] (may be negative / past the end); p~^a_i is a real
 * array over the box, [n_i][sx][sy][sz]; dO^a a real n_i x n_i matrix.  A box point outside [0,n)
 * on a periodic axis stands for its home-cell image and carries the Bloch factor of psi^ (as in
 * the stencil) when read and its conjugate when written; on a zero-BC axis it is dropped.
 *
 * fd_paw_create -- copy the projector data to the plan's device, resolve the boxes into index
 *   tables, colour the atoms so that boxes handled together are disjoint (results do not depend on
 *   scheduling; no atomics).  All array arguments are HOST pointers: box_start, box_size
 *   [natoms][3], nproj [natoms] (1..32 each), proj (concatenated per atom), dh / ds (concatenated
 *   [n_i][n_i] per atom; either may be NULL).  FD_ERR_UNSUPPORTED: a box longer than a periodic
 *   axis, more than 32 functions on an atom, grids of 2^31 points or more.
 * fd_paw_nproj_total -- sum_a n_i (row length of P), or a negative fd_status.
 * fd_paw_project   -- coef[nbands][sum n_i] = P (plan dtype; device pointer, 16-byte aligned).
 * fd_paw_add_nonlocal -- out += sum |p~> Delta H <p~|psi>  (coef: scratch of the same size as P;
 *   it holds P on return).
 * fd_apply_hamiltonian_paw -- out = -1/2 lap_FD psi + v_eff psi + the Delta H term: the complete
 *   H~ psi~ of Eq. 6 (v_eff == NULL: kinetic + non-local).
 * fd_apply_overlap -- out = psi + sum |p~> Delta S <p~|psi>  (Eq. 7).
 * fd_paw_expect -- out[b] += (1/dv) Re sum_a P_b[a,:]^H dO^a P_b[a,:] for the projections `coef` of
 *   fd_paw_project: the PAW part of the grid sum <psi_b|H~|psi_b> (which = 0, Delta H) or of
 *   <psi_b|S~|psi_b> (which = 1, Delta S).  ACCUMULATES into out (double [nbands], device): applied to
 *   the eps / norm of fd_apply_hamiltonian_expect it completes them to the PAW Rayleigh quotient
 *   eps_b / norm_b = <psi|H~|psi> / <psi|S~|psi>, and fd_residual(plan, S~psi, H~psi, eps, norm, r)
 *   is then the residual H~ psi - lambda S~ psi of the generalised eigenproblem.
 * FD_F64 plans with Bloch factors -1 (2 k_d integer) are supported: a box point that wraps such an
 * axis, and a box that starts an odd number of cells from the home cell along it, take the sign.
 * Errors as fd_apply_hamiltonian; FD_ERR_INVALID also when paw was built for a plan that differs
 * from `plan` in shape, spacing, boundaries, k, dtype or device (its index tables, Bloch factors and
 * dv are the creating plan's), or when the matrix the call needs was not given at fd_paw_create;
 * FD_ERR_ALIAS also when coef overlaps psi or out.
 */
typedef struct fd_paw fd_paw;
FD_API int fd_paw_create(fd_paw **paw, const fd_plan *plan, int32_t natoms, const int32_t *box_start,
                  const int32_t *box_size, const int32_t *nproj, const double *proj_host,
                  const double *dh_host, const double *ds_host);
FD_API int fd_paw_destroy(fd_paw *paw);
FD_API int32_t fd_paw_nproj_total(const fd_paw *paw);
FD_API int fd_paw_project(const fd_plan *plan, const fd_paw *paw, const void *psi, void *coef,
                   int64_t nbands, void *cuda_stream);
FD_API int fd_paw_add_nonlocal(const fd_plan *plan, const fd_paw *paw, const void *psi, void *out,
                        void *coef, int64_t nbands, void *cuda_stream);
FD_API int fd_apply_hamiltonian_paw(const fd_plan *plan, const fd_paw *paw, const void *psi,
                             const double *v_eff, void *out, void *coef, int64_t nbands,
                             void *cuda_stream);
FD_API int fd_apply_overlap(const fd_plan *plan, const fd_paw *paw, const void *psi, void *out,
                     void *coef, int64_t nbands, void *cuda_stream);
FD_API int fd_paw_expect(const fd_plan *plan, const fd_paw *paw, int32_t which, const void *coef, double *out,
                  int64_t nbands, void *cuda_stream);

/*
 * Multigrid V-cycle for lap_FD phi = rhs on the f3 kernels ("multigrid ... Jacobi" Poisson solvers,
 * PAPER.md:248; the grids of PAPER.md:93).  The textbook cycle, per level l (spacing 2^l h):
 *     nu1 weighted-Jacobi sweeps;  r = rhs - A phi;  rhs_{l+1} = R r,  phi_{l+1} = 0;  recurse
 *     (nu_coarse sweeps on the coarsest level);  phi += I phi_{l+1};  nu2 sweeps.
 * fd_mg_create builds the hierarchy (levels are added while every axis can be coarsened -- even on
 *   periodic, odd on zero-BC axes -- and keeps max(nn, 2) points, at most max_levels), one plan per
 *   level and the level buffers for up to max_nbands right-hand sides (3 arrays per coarse level, one
 *   on the finest); transfer order p = 1..3.  fd_mg_levels: number of levels.
 * fd_mg_vcycle: one cycle IN PLACE on phi [nbands, nx, ny, nz] (device, float64, 16-byte aligned;
 *   rhs likewise, no overlap); a sequence of kernel launches on cuda_stream, no synchronisation.
 *   On a non-default stream the sequence is captured into a CUDA graph the first time an argument
 *   set (phi, rhs, nbands, nu1, nu2, nu_coarse, omega) is seen and replayed afterwards (the coarse
 *   levels are launch bound); the four most recently used argument sets are kept, so a solver
 *   that alternates a few right-hand-side buffers re-captures none of them.  On a stream the
 *   caller is capturing already the launches join the caller's graph.  Calls on one fd_mg are
 *   serialised.
 *   A single-level hierarchy (a grid that cannot be coarsened) does nu_coarse sweeps.  Errors as fd_jacobi_sweep / fd_restrict;
 *   FD_ERR_INVALID for nbands > max_nbands.
 */
typedef struct fd_mg fd_mg;
FD_API int fd_mg_create(fd_mg **mg, const int32_t shape[3], const double h[3], int32_t nn,
                 const int32_t bc[3], int32_t p, int32_t max_levels, int64_t max_nbands, int32_t device);
FD_API int fd_mg_destroy(fd_mg *mg);
FD_API int32_t fd_mg_levels(const fd_mg *mg);
FD_API int fd_mg_vcycle(const fd_mg *mg, double *phi, const double *rhs, int64_t nbands, int32_t nu1,
                 int32_t nu2, int32_t nu_coarse, double omega, void *cuda_stream);
/* fd_mg_get_info: info[0..2] = finest shape; [3] = max_nbands; [4] = device; [5] = levels;
 *   [6] = graph captures so far; [7] = 1 if graph capture was given up for this hierarchy (direct
 *   launches).  Lets a binding check phi / rhs before passing raw pointers on. */
FD_API int fd_mg_get_info(const fd_mg *mg, int64_t info[8]);

/*
 * fd_peak_kernel -- micro-benchmark kernels behind the roofline denominators (
 * not on the hot path; timed by bench.py --peaks with CUDA events).  kind 0: read n doubles of a
 * (b: 1-double sink); 1: write n doubles to a; 2: copy n doubles a -> b; 3: n rounds of 8 independent
 * DFMA per thread on blocks x 256 threads (a: 1-double sink).  blocks = 0: 8 CTAs per SM.  Device
 * pointers on the current device, 16-byte aligned; n even.
 */
FD_API int fd_peak_kernel(int32_t kind, void *a, void *b, int64_t n, int32_t blocks, void *cuda_stream);

/* fd_destroy -- free the plan; NULL is a no-op.  The caller must have synchronised any stream
 * still running an apply of this plan. */
FD_API int fd_destroy(fd_plan *plan);

/* fd_strerror -- static, thread-safe description of a status code. */
FD_API const char *fd_strerror(int status);

/* Diagnostics (not on the hot path).
 * fd_plan_set_kernel: force a kernel family (FD_ERR_UNSUPPORTED if the plan cannot run it);
 *   with `param` != 0 overriding the family's tile parameter (sweep: y rows per CTA).
 * fd_plan_get_kernel: family of the plan (the sweep family hands batches that are far too small
 *   to fill its persistent CTAs to the generic kernel unless it was forced).
 * fd_plan_kernel_for: family an apply of `nbands` bands will launch.
 * fd_plan_launches: kernels launched by this plan so far (for bench.py's gpu_launches).
 * fd_plan_get_weights: the 3*(nn+1) doubles w_d[j] = -1/2 c_j / h_d^2 (d-major) the kernels use.
 * fd_plan_get_info: info[0..2] = nx, ny, nz; [3] = nn; [4] = dtype (FD_F64 ...); [5] = device;
 *   [6] = bc bits (x | y << 1 | z << 2); [7] = kernel family.  Lets a binding check the arrays it is
 *   handed against the plan before it passes raw pointers on. */
FD_API int fd_plan_set_kernel(fd_plan *plan, int32_t kernel, int32_t param);
FD_API int fd_plan_get_kernel(const fd_plan *plan);
FD_API int fd_plan_kernel_for(const fd_plan *plan, int64_t nbands);
FD_API int64_t fd_plan_launches(const fd_plan *plan);
FD_API int fd_plan_get_weights(const fd_plan *plan, double *w, int32_t capacity);
FD_API int fd_plan_get_info(const fd_plan *plan, int32_t info[8]);

#ifdef __cplusplus
}
#endif
#endif /* FDHAM_H */
