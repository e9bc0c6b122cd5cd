/*
 * oracle/fd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU statement of the finite-difference Kohn-Sham apply
 *
 *     (H psi)_b[i] = sum_{d in x,y,z} (-1/2 / h_d^2) * [ c_0 psi_b[i]
 *                        + sum_{j=1..nn} c_j ( psi^_b(i + j e_d) + psi^_b(i - j e_d) ) ]
 *                    + v_eff[i] * psi_b[i]
 *
 * which is the first two terms of the PAW Hamiltonian, Eq. 6 of the paper
 * (section III.A: "-1/2 nabla^2 + v~_KS(r) + ..."), with the Laplacian in its
 * "finite difference (FD) ... representation of kinetic energy operator on a uniform Cartesian
 * grid" (section III.B.1), the stencil the paper names as a C hot spot
 * (section II.B).  The paper prints no coefficients; reading R1 takes the
 * standard central weights of order 2*nn (BASELINE.json gives nn=3: -49/18, 3/2, -3/20, 1/90).
 *
 * Boundary handling psi^ (readings R3, R5):
 *   - zero-BC axis   : psi^ = 0 outside [0, n_d)  ("potential go to zero on the cell boundaries",
 *                      PAPER.md:250; FD mode's flexible boundary conditions);
 *   - periodic axis  : psi^(p) = psi[p - w n_d] * exp(+2 pi i k_d w), w = floor(p_d / n_d), i.e. the
 *                      array holds the full Bloch function exp(+i(k+G).r) of Eq. 13.
 *
 * Everything is double precision (complex double for FD_C128), one triple loop per band, no
 * blocking, no fusion, no reordering beyond the definition.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call this file.  It shares no code with
 * paper_2310_14776_b200/csrc/.
 *
 * Every function here is pinned by tests/test_oracle_*.py (closed forms, brute force, textbook
 * coefficient table); nothing is "parity unpinned".
 *
 * Build: see oracle/build.py  (gcc -O2 -fopenmp -shared -fPIC, no -ffast-math).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define FDO_MAX_NN 12

enum { FDO_BC_ZERO = 0, FDO_BC_PERIODIC = 1 };

static const double FDO_PI = 3.14159265358979323846264338327950288;

static double fdo_factorial(int n)
{
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

/* Central finite-difference weights for d^2/dx^2 of order 2*nn on a unit-spaced grid
 * (reading R1):
 *     c_j = 2 (-1)^{j+1} (nn!)^2 / ( j^2 (nn-j)! (nn+j)! ),  j = 1..nn
 *     c_0 = -2 sum_{j=1..nn} 1/j^2
 * Writes c[0..nn].  Returns 0, or -1 for nn outside 1..FDO_MAX_NN. */
int fd_oracle_coeffs(int nn, double *c)
{
    if (nn < 1 || nn > FDO_MAX_NN || !c) return -1;
    double c0 = 0.0;
    for (int j = 1; j <= nn; ++j) {
        double sign = (j % 2 == 1) ? 1.0 : -1.0;
        double num = 2.0 * sign * fdo_factorial(nn) * fdo_factorial(nn);
        double den = (double)j * (double)j * fdo_factorial(nn - j) * fdo_factorial(nn + j);
        c[j] = num / den;
        c0 += 1.0 / ((double)j * (double)j);
    }
    c[0] = -2.0 * c0;
    return 0;
}

/* floor division for possibly negative p */
static inline int64_t fdo_floordiv(int64_t p, int64_t n)
{
    int64_t q = p / n;
    if ((p % n != 0) && ((p < 0) != (n < 0))) --q;
    return q;
}

typedef struct {
    int64_t n[3];
    double h[3];
    int nn;
    int bc[3];
    double k[3];
    double c[FDO_MAX_NN + 1];
    double scale; /* prefactor of the FD Laplacian: -1/2 (kinetic operator, Eq. 6) unless the
                     caller of fd_oracle_apply_scaled asks for another one */
} fdo_geom;

static int fdo_fill_geom(fdo_geom *g, const int32_t shape[3], const double h[3], int nn,
                         const int32_t bc[3], const double *k_reduced)
{
    if (!shape || !h || !bc) return -1;
    if (fd_oracle_coeffs(nn, g->c) != 0) return -1;
    g->nn = nn;
    g->scale = -0.5;
    for (int d = 0; d < 3; ++d) {
        if (shape[d] < 1 || !(h[d] > 0.0)) return -1;
        if (bc[d] != FDO_BC_ZERO && bc[d] != FDO_BC_PERIODIC) return -1;
        g->n[d] = shape[d];
        g->h[d] = h[d];
        g->bc[d] = bc[d];
        g->k[d] = k_reduced ? k_reduced[d] : 0.0;
    }
    return 0;
}

/* psi^ for a real array at Gamma: value at index idx[] shifted by `shift` along axis d. */
static inline double fdo_hat_real(const fdo_geom *g, const double *psi, const int64_t idx[3], int d,
                                  int64_t shift)
{
    int64_t p[3] = { idx[0], idx[1], idx[2] };
    p[d] += shift;
    if (p[d] < 0 || p[d] >= g->n[d]) {
        if (g->bc[d] == FDO_BC_ZERO) return 0.0;
        int64_t w = fdo_floordiv(p[d], g->n[d]);
        p[d] -= w * g->n[d];
    }
    return psi[(p[0] * g->n[1] + p[1]) * g->n[2] + p[2]];
}

/* psi^ for a complex array carrying Bloch phases. */
static inline double complex fdo_hat_cplx(const fdo_geom *g, const double complex *psi,
                                          const int64_t idx[3], int d, int64_t shift)
{
    int64_t p[3] = { idx[0], idx[1], idx[2] };
    double complex phase = 1.0;
    p[d] += shift;
    if (p[d] < 0 || p[d] >= g->n[d]) {
        if (g->bc[d] == FDO_BC_ZERO) return 0.0;
        int64_t w = fdo_floordiv(p[d], g->n[d]);
        p[d] -= w * g->n[d];
        phase = cexp(I * (2.0 * FDO_PI * g->k[d] * (double)w));
    }
    return psi[(p[0] * g->n[1] + p[1]) * g->n[2] + p[2]] * phase;
}

static inline double fdo_point_real(const fdo_geom *g, const double *psi, const double *v,
                                    const int64_t idx[3])
{
    const int64_t lin = (idx[0] * g->n[1] + idx[1]) * g->n[2] + idx[2];
    double acc = 0.0;
    for (int d = 0; d < 3; ++d) {
        double s = g->c[0] * psi[lin];
        for (int j = 1; j <= g->nn; ++j)
            s += g->c[j] * (fdo_hat_real(g, psi, idx, d, +j) + fdo_hat_real(g, psi, idx, d, -j));
        acc += (g->scale / (g->h[d] * g->h[d])) * s;
    }
    if (v) acc += v[lin] * psi[lin];
    return acc;
}

static inline double complex fdo_point_cplx(const fdo_geom *g, const double complex *psi,
                                            const double *v, const int64_t idx[3])
{
    const int64_t lin = (idx[0] * g->n[1] + idx[1]) * g->n[2] + idx[2];
    double complex acc = 0.0;
    for (int d = 0; d < 3; ++d) {
        double complex s = g->c[0] * psi[lin];
        for (int j = 1; j <= g->nn; ++j)
            s += g->c[j] * (fdo_hat_cplx(g, psi, idx, d, +j) + fdo_hat_cplx(g, psi, idx, d, -j));
        acc += (g->scale / (g->h[d] * g->h[d])) * s;
    }
    if (v) acc += v[lin] * psi[lin];
    return acc;
}

/*
 * out[b, ix, iy, iz] = (H psi)_b[ix, iy, iz] for b in [0, nbands); v_eff == NULL gives the kinetic
 * term only.  is_complex: 0 -> psi/out are double, k must be NULL or all zero;
 *             1 -> psi/out are C99 double complex (interleaved re, im).
 * nthreads: OpenMP threads over bands (<= 0: library default).  Returns 0 / -1 (bad argument).
 */
int fd_oracle_apply(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                    const double *k_reduced, int32_t is_complex, const void *psi,
                    const double *v_eff, void *out, int64_t nbands, int32_t nthreads)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, k_reduced) != 0) return -1;
    if (!psi || !out || nbands < 0) return -1;
    if (!is_complex)
        for (int d = 0; d < 3; ++d)
            if (g.k[d] != 0.0) return -1;
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < nbands; ++b) {
        for (int64_t ix = 0; ix < g.n[0]; ++ix)
            for (int64_t iy = 0; iy < g.n[1]; ++iy)
                for (int64_t iz = 0; iz < g.n[2]; ++iz) {
                    const int64_t idx[3] = { ix, iy, iz };
                    const int64_t lin = (ix * g.n[1] + iy) * g.n[2] + iz;
                    if (is_complex) {
                        const double complex *pb = (const double complex *)psi + b * P;
                        ((double complex *)out)[b * P + lin] = fdo_point_cplx(&g, pb, v_eff, idx);
                    } else {
                        const double *pb = (const double *)psi + b * P;
                        ((double *)out)[b * P + lin] = fdo_point_real(&g, pb, v_eff, idx);
                    }
                }
    }
    return 0;
}

/* Same as fd_oracle_apply with `scale` in place of the -1/2 of Eq. 6: out = scale lap_FD psi
 * (+ v_eff psi).  scale = 1 is the plain FD Laplacian of the Poisson problem (PAPER.md:248 names
 * the solvers that use it). */
int fd_oracle_apply_scaled(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                    const double *k_reduced, int32_t is_complex, const void *psi,
                    const double *v_eff, void *out, int64_t nbands, int32_t nthreads, double scale)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, k_reduced) != 0) return -1;
    if (!isfinite(scale)) return -1;
    g.scale = scale;
    if (!psi || !out || nbands < 0) return -1;
    if (!is_complex)
        for (int d = 0; d < 3; ++d)
            if (g.k[d] != 0.0) return -1;
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < nbands; ++b) {
        for (int64_t ix = 0; ix < g.n[0]; ++ix)
            for (int64_t iy = 0; iy < g.n[1]; ++iy)
                for (int64_t iz = 0; iz < g.n[2]; ++iz) {
                    const int64_t idx[3] = { ix, iy, iz };
                    const int64_t lin = (ix * g.n[1] + iy) * g.n[2] + iz;
                    if (is_complex) {
                        const double complex *pb = (const double complex *)psi + b * P;
                        ((double complex *)out)[b * P + lin] = fdo_point_cplx(&g, pb, v_eff, idx);
                    } else {
                        const double *pb = (const double *)psi + b * P;
                        ((double *)out)[b * P + lin] = fdo_point_real(&g, pb, v_eff, idx);
                    }
                }
    }
    return 0;
}

/*
 * Same definition evaluated only at npoints sampled outputs: points[4*s + {0,1,2,3}] =
 * (band, ix, iy, iz); out[s] (double or double complex).  psi is the whole batch
 * [nbands, nx, ny, nz].  Used for full-size parity where the whole oracle would be too slow.
 */
int fd_oracle_points(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                     const double *k_reduced, int32_t is_complex, const void *psi,
                     const double *v_eff, int64_t nbands, const int64_t *points, int64_t npoints,
                     void *out)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, k_reduced) != 0) return -1;
    if (!psi || !out || !points || nbands < 0 || npoints < 0) return -1;
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
    for (int64_t s = 0; s < npoints; ++s) {
        const int64_t b = points[4 * s];
        const int64_t idx[3] = { points[4 * s + 1], points[4 * s + 2], points[4 * s + 3] };
        if (b < 0 || b >= nbands) return -1;
        for (int d = 0; d < 3; ++d)
            if (idx[d] < 0 || idx[d] >= g.n[d]) return -1;
        if (is_complex)
            ((double complex *)out)[s] =
                fdo_point_cplx(&g, (const double complex *)psi + b * P, v_eff, idx);
        else
            ((double *)out)[s] = fdo_point_real(&g, (const double *)psi + b * P, v_eff, idx);
    }
    return 0;
}

/*
 * Explicit dense matrix of H (P x P, row-major, complex double), assembled entry by entry from
 * the definition by SCATTERING each tap into M[row, column] -- it does not call the apply above,
 * so apply-vs-dense is a brute-force cross check (tests/test_oracle_dense.py).
 * Taps that wrap onto the same column (n_d <= 2 nn) add up.
 */
int fd_oracle_dense(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                    const double *k_reduced, const double *v_eff, double complex *M)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, k_reduced) != 0) return -1;
    if (!M) return -1;
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
    memset(M, 0, (size_t)P * (size_t)P * sizeof(double complex));
    for (int64_t ix = 0; ix < g.n[0]; ++ix)
        for (int64_t iy = 0; iy < g.n[1]; ++iy)
            for (int64_t iz = 0; iz < g.n[2]; ++iz) {
                const int64_t row = (ix * g.n[1] + iy) * g.n[2] + iz;
                if (v_eff) M[row * P + row] += v_eff[row];
                for (int d = 0; d < 3; ++d) {
                    const double pref = g.scale / (g.h[d] * g.h[d]);
                    M[row * P + row] += pref * g.c[0];
                    for (int j = 1; j <= g.nn; ++j)
                        for (int sgn = -1; sgn <= 1; sgn += 2) {
                            int64_t p[3] = { ix, iy, iz };
                            double complex phase = 1.0;
                            p[d] += sgn * j;
                            if (p[d] < 0 || p[d] >= g.n[d]) {
                                if (g.bc[d] == FDO_BC_ZERO) continue;
                                int64_t w = fdo_floordiv(p[d], g.n[d]);
                                p[d] -= w * g.n[d];
                                phase = cexp(I * (2.0 * FDO_PI * g.k[d] * (double)w));
                            }
                            const int64_t col = (p[0] * g.n[1] + p[1]) * g.n[2] + p[2];
                            M[row * P + col] += pref * g.c[j] * phase;
                        }
                }
            }
    return 0;
}

/* Number of OpenMP threads a parallel region would use now (for bench.py's "cores"). */
int fd_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* =================================================================================================
 * SURVEY 8(f) "next" rows.  Same rules as above: the plain definition, double precision, no
 * blocking.  Every function below is pinned by tests/test_oracle_next_*.py.
 * ============================================================================================== */

/*
 * f2 -- eigensolver epilogue (section III.B.3: subspace diagonalisation and the
 * iterative eigensolver step need <psi_b|H|psi_b> and the residual; Davidson / RMM-DIIS
 * PAPER.md:318; every RT-TDDFT step applies H to every band, Eq. 91).
 *
 *     eps[b]  = sum_i conj(psi_b[i]) (H psi)_b[i]        (plain grid sum in index order: multiply
 *     norm[b] = sum_i |psi_b[i]|^2                         by dv = h_x h_y h_z for the integral)
 *
 * H = scale lap_FD + v_eff (scale = -1/2 is Eq. 6).  eps is returned complex; H is Hermitian, so
 * its imaginary part is rounding noise (pinned).  out may be NULL; else it receives H psi.
 */
int fd_oracle_expect(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                     const double *k_reduced, int32_t is_complex, const void *psi,
                     const double *v_eff, void *out, int64_t nbands, double scale,
                     double complex *eps, double *norm)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, k_reduced) != 0) return -1;
    if (!isfinite(scale) || !psi || !eps || !norm || nbands < 0) return -1;
    g.scale = scale;
    if (!is_complex)
        for (int d = 0; d < 3; ++d)
            if (g.k[d] != 0.0) return -1;
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < nbands; ++b) {
        double complex e = 0.0;
        double nrm = 0.0;
        for (int64_t ix = 0; ix < g.n[0]; ++ix)
            for (int64_t iy = 0; iy < g.n[1]; ++iy)
                for (int64_t iz = 0; iz < g.n[2]; ++iz) {
                    const int64_t idx[3] = { ix, iy, iz };
                    const int64_t lin = (ix * g.n[1] + iy) * g.n[2] + iz;
                    if (is_complex) {
                        const double complex *pb = (const double complex *)psi + b * P;
                        const double complex hp = fdo_point_cplx(&g, pb, v_eff, idx);
                        if (out) ((double complex *)out)[b * P + lin] = hp;
                        e += conj(pb[lin]) * hp;
                        nrm += creal(pb[lin]) * creal(pb[lin]) + cimag(pb[lin]) * cimag(pb[lin]);
                    } else {
                        const double *pb = (const double *)psi + b * P;
                        const double hp = fdo_point_real(&g, pb, v_eff, idx);
                        if (out) ((double *)out)[b * P + lin] = hp;
                        e += pb[lin] * hp;
                        nrm += pb[lin] * pb[lin];
                    }
                }
        eps[b] = e;
        norm[b] = nrm;
    }
    return 0;
}

/* f2 -- residual of the eigensolvers: r_b[i] = hpsi_b[i] - lambda[b] psi_b[i] (real lambda; with
 * lambda[b] = Re eps[b] / norm[b] this is R_b = H psi_b - eps_b psi_b of SURVEY 8(f) f2). */
int fd_oracle_residual(int64_t npoints, int32_t is_complex, const void *psi, const void *hpsi,
                       const double *lambda, void *out, int64_t nbands)
{
    if (!psi || !hpsi || !lambda || !out || npoints < 0 || nbands < 0) return -1;
    for (int64_t b = 0; b < nbands; ++b)
        for (int64_t i = 0; i < npoints; ++i) {
            const int64_t q = b * npoints + i;
            if (is_complex)
                ((double complex *)out)[q] = ((const double complex *)hpsi)[q] -
                                             lambda[b] * ((const double complex *)psi)[q];
            else
                ((double *)out)[q] = ((const double *)hpsi)[q] - lambda[b] * ((const double *)psi)[q];
        }
    return 0;
}

/*
 * f3 -- one weighted-Jacobi relaxation sweep for  A phi = rhs,  A = scale lap_FD  (PAPER.md:248,
 * section III.B.4: "multigrid ... Jacobi or Gauss-Seidel" Poisson solvers on the same grids with
 * the same kind of stencil; scale = 1 is the Poisson operator itself):
 *
 *     out[i] = phi[i] + omega ( rhs[i] - (A phi)[i] ) / A_ii,    A_ii = scale c_0 sum_d 1/h_d^2
 *
 * All points are updated from the OLD phi (Jacobi, not Gauss-Seidel).  Real arrays, Gamma point.
 */
int fd_oracle_jacobi(const int32_t shape[3], const double h[3], int32_t nn, const int32_t bc[3],
                     const double *phi, const double *rhs, double *out, int64_t nbands,
                     double omega, double scale)
{
    fdo_geom g;
    if (fdo_fill_geom(&g, shape, h, nn, bc, NULL) != 0) return -1;
    if (!phi || !rhs || !out || nbands < 0 || !isfinite(scale) || scale == 0.0 || !isfinite(omega))
        return -1;
    g.scale = scale;
    double diag = 0.0;
    for (int d = 0; d < 3; ++d) diag += scale * g.c[0] / (g.h[d] * g.h[d]);
    const int64_t P = g.n[0] * g.n[1] * g.n[2];
    for (int64_t b = 0; b < nbands; ++b)
        for (int64_t ix = 0; ix < g.n[0]; ++ix)
            for (int64_t iy = 0; iy < g.n[1]; ++iy)
                for (int64_t iz = 0; iz < g.n[2]; ++iz) {
                    const int64_t idx[3] = { ix, iy, iz };
                    const int64_t lin = (ix * g.n[1] + iy) * g.n[2] + iz;
                    const double a_phi = fdo_point_real(&g, phi + b * P, NULL, idx);
                    out[b * P + lin] = phi[b * P + lin] + omega * (rhs[b * P + lin] - a_phi) / diag;
                }
    return 0;
}

/*
 * f3 -- grid transfer between a fine grid (spacing h) and the coarse grid of spacing 2h
 * ("interpolating from one uniform grid to another" is the second C hot spot;
 * multigrid).  The paper prints no weights; reading R13 takes the
 * textbook choice: polynomial (Lagrange) interpolation of degree 2p-1 through the 2p nearest
 * coarse points per axis, tensor product over the axes, and restriction = its transpose / 8.
 *
 * Index map per axis (reading R14, consistent with R3): coarse point I sits on fine point
 * 2I + off, off = 0 on a periodic axis (n_f = 2 n_c), off = 1 on a zero-BC axis (n_f = 2 n_c + 1:
 * stored points are the interior ones, x_i = (i+1) h, the walls at -1 and n are shared).
 * Values outside [0,n) are 0 (zero BC) or wrapped (periodic); real arrays, Gamma point.
 *
 * 1-D midpoint weights: nodes at t = +-(j - 1/2), j = 1..p (in units of the coarse spacing),
 * b_j = prod_{m != j} (0 - t_m)/(t_j - t_m) over all 2p nodes (Lagrange basis at t = 0).
 * p = 1: 1/2;  p = 2: 9/16, -1/16;  p = 3: 150/256, -25/256, 3/256.
 */
#define FDO_MAX_P 6

int fd_oracle_transfer_weights(int32_t p, double *b /* b[1..p]; b[0] unused = 0 */)
{
    if (p < 1 || p > FDO_MAX_P || !b) return -1;
    double t[2 * FDO_MAX_P];
    for (int m = 0; m < p; ++m) {
        t[2 * m] = (double)(m + 1) - 0.5;      /* +(j - 1/2) */
        t[2 * m + 1] = -((double)(m + 1) - 0.5); /* -(j - 1/2) */
    }
    b[0] = 0.0;
    for (int j = 1; j <= p; ++j) {
        const int me = 2 * (j - 1); /* node +(j - 1/2) */
        double w = 1.0;
        for (int m = 0; m < 2 * p; ++m)
            if (m != me) w *= (0.0 - t[m]) / (t[me] - t[m]);
        b[j] = w;
    }
    return 0;
}

typedef struct {
    int64_t n[3];
    int bc[3];
} fdo_grid;

/* value at (possibly out-of-range) index p[] of a real array on grid gr: 0 or wrapped */
static inline double fdo_grid_value(const fdo_grid *gr, const double *a, int64_t px, int64_t py,
                                    int64_t pz)
{
    int64_t p[3] = { px, py, pz };
    for (int d = 0; d < 3; ++d)
        if (p[d] < 0 || p[d] >= gr->n[d]) {
            if (gr->bc[d] == FDO_BC_ZERO) return 0.0;
            p[d] -= fdo_floordiv(p[d], gr->n[d]) * gr->n[d];
        }
    return a[(p[0] * gr->n[1] + p[1]) * gr->n[2] + p[2]];
}

static int fdo_transfer_grids(const int32_t shape_fine[3], const int32_t bc[3], fdo_grid *fine,
                              fdo_grid *coarse, int off[3])
{
    if (!shape_fine || !bc) return -1;
    for (int d = 0; d < 3; ++d) {
        if (bc[d] != FDO_BC_ZERO && bc[d] != FDO_BC_PERIODIC) return -1;
        fine->n[d] = shape_fine[d];
        fine->bc[d] = coarse->bc[d] = bc[d];
        if (bc[d] == FDO_BC_PERIODIC) {
            if (shape_fine[d] < 2 || (shape_fine[d] & 1)) return -1;
            coarse->n[d] = shape_fine[d] / 2;
            off[d] = 0;
        } else {
            if (shape_fine[d] < 3 || !(shape_fine[d] & 1)) return -1;
            coarse->n[d] = (shape_fine[d] - 1) / 2;
            off[d] = 1;
        }
    }
    return 0;
}

/* 1-D restriction weight of fine offset a from the coarse point: 1/2 at a = 0, b_j / 2 at
 * a = +-(2j - 1), 0 at the other (even) offsets. */
static inline double fdo_restrict_w(const double *b, int a)
{
    if (a == 0) return 0.5;
    const int aa = a < 0 ? -a : a;
    if (!(aa & 1)) return 0.0;
    return 0.5 * b[(aa + 1) / 2];
}

/* coarse[b, ci, cj, ck] = sum_{a,b',c} r_a r_b' r_c fine^[b, 2ci+off_x+a, 2cj+off_y+b', 2ck+off_z+c],
 * offsets -(2p-1) .. 2p-1.  shape_fine = fine extents; coarse extents follow from bc (above). */
int fd_oracle_restrict(const int32_t shape_fine[3], const int32_t bc[3], int32_t p,
                       const double *fine, double *coarse, int64_t nbands)
{
    fdo_grid gf, gc;
    int off[3];
    double b[FDO_MAX_P + 1];
    if (fdo_transfer_grids(shape_fine, bc, &gf, &gc, off) != 0) return -1;
    if (fd_oracle_transfer_weights(p, b) != 0 || !fine || !coarse || nbands < 0) return -1;
    const int64_t Pf = gf.n[0] * gf.n[1] * gf.n[2], Pc = gc.n[0] * gc.n[1] * gc.n[2];
    const int m = 2 * p - 1;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < nbands * gc.n[0]; ++q) {
        const int64_t bd = q / gc.n[0], ci = q % gc.n[0];
        for (int64_t cj = 0; cj < gc.n[1]; ++cj)
            for (int64_t ck = 0; ck < gc.n[2]; ++ck) {
                double s = 0.0;
                for (int ax = -m; ax <= m; ++ax)
                    for (int ay = -m; ay <= m; ++ay)
                        for (int az = -m; az <= m; ++az) {
                            const double w = fdo_restrict_w(b, ax) * fdo_restrict_w(b, ay) *
                                             fdo_restrict_w(b, az);
                            if (w == 0.0) continue;
                            s += w * fdo_grid_value(&gf, fine + bd * Pf, 2 * ci + off[0] + ax,
                                                    2 * cj + off[1] + ay, 2 * ck + off[2] + az);
                        }
                coarse[bd * Pc + (ci * gc.n[1] + cj) * gc.n[2] + ck] = s;
            }
    }
    return 0;
}

/* 1-D interpolation: fine index f, e = f - off.  e even -> the coarse point e/2 itself (weight 1);
 * e odd -> midpoint between coarse (e-1)/2 and (e+1)/2: sum_j b_j (c[lo - j + 1] + c[lo + j]).
 * Returns the number of taps written to (idx[], w[]). */
static inline int fdo_interp_taps(const double *b, int p, int64_t e, int64_t idx[2 * FDO_MAX_P],
                                  double w[2 * FDO_MAX_P])
{
    if ((e & 1) == 0) {
        idx[0] = e / 2; /* e >= -1 always: off <= 1 */
        w[0] = 1.0;
        return 1;
    }
    /* lower coarse neighbour; e = -1 (fine index 0 on a zero-BC axis) is the midpoint of coarse -1
     * (the wall) and coarse 0 */
    const int64_t lo = fdo_floordiv(e - 1, 2);
    int n = 0;
    for (int j = 1; j <= p; ++j) {
        idx[n] = lo - j + 1;
        w[n++] = b[j];
        idx[n] = lo + j;
        w[n++] = b[j];
    }
    return n;
}

/* fine[b, f_x, f_y, f_z] = tensor product of the 1-D interpolations of the coarse array.
 * shape_fine = fine extents (output); coarse extents follow from bc. */
int fd_oracle_interpolate(const int32_t shape_fine[3], const int32_t bc[3], int32_t p,
                          const double *coarse, double *fine, int64_t nbands)
{
    fdo_grid gf, gc;
    int off[3];
    double b[FDO_MAX_P + 1];
    if (fdo_transfer_grids(shape_fine, bc, &gf, &gc, off) != 0) return -1;
    if (fd_oracle_transfer_weights(p, b) != 0 || !fine || !coarse || nbands < 0) return -1;
    const int64_t Pf = gf.n[0] * gf.n[1] * gf.n[2], Pc = gc.n[0] * gc.n[1] * gc.n[2];
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < nbands * gf.n[0]; ++q) {
        const int64_t bd = q / gf.n[0], fx = q % gf.n[0];
        int64_t ix[2 * FDO_MAX_P], iy[2 * FDO_MAX_P], iz[2 * FDO_MAX_P];
        double wx[2 * FDO_MAX_P], wy[2 * FDO_MAX_P], wz[2 * FDO_MAX_P];
        const int nx = fdo_interp_taps(b, p, fx - off[0], ix, wx);
        for (int64_t fy = 0; fy < gf.n[1]; ++fy) {
            const int ny = fdo_interp_taps(b, p, fy - off[1], iy, wy);
            for (int64_t fz = 0; fz < gf.n[2]; ++fz) {
                const int nz = fdo_interp_taps(b, p, fz - off[2], iz, wz);
                double s = 0.0;
                for (int a = 0; a < nx; ++a)
                    for (int c = 0; c < ny; ++c)
                        for (int e = 0; e < nz; ++e)
                            s += wx[a] * wy[c] * wz[e] *
                                 fdo_grid_value(&gc, coarse + bd * Pc, ix[a], iy[c], iz[e]);
                fine[bd * Pf + (fx * gf.n[1] + fy) * gf.n[2] + fz] = s;
            }
        }
    }
    return 0;
}

/*
 * f4 -- the PAW non-local term, third term of Eq. 6, and with dO = Delta S the
 * overlap operator of Eq. 7; "overlaps between projector functions and wave
 * functions" is the third C hot spot:
 *
 *     P_b[a,i]   = dv sum_{r in box_a} p~^a_i(r) psi^_b(r)                 (projections, dv = h_x h_y h_z)
 *     out_b(r') += sum_a sum_{i,i'} p~^a_i(r) conj(phase(r)) dO^a_{i i'} P_b[a,i']
 *
 * PAW data sets are not available, so the projector functions are synthetic: atom a
 * owns a box of box_size[a] grid points starting at (possibly negative / past-the-end) index
 * box_start[a]; p~^a_i is a real array over the box; dO^a is a real n_i x n_i matrix.  A box point
 * r outside [0,n) on a periodic axis stands for the home point r' = r - w n with the Bloch factor
 * of psi^ (reading R5) when it is read and its conjugate when it is written (the projector of the
 * crystal is sum_R e^{ik.R} p~(r - R)); on a zero-BC axis the part of the box outside is dropped.
 * accumulate = 0: out = non-local term only; 1: added to what out holds (H psi, or psi for S psi).
 * proj, dmat: concatenated per atom, [n_i][sx][sy][sz] and [n_i][n_i] doubles.
 * coef (may be NULL) receives P_b[a,i], [nbands][sum_a n_i], dtype of psi.
 */
int fd_oracle_paw_apply(const int32_t shape[3], const double h[3], const int32_t bc[3],
                        const double *k_reduced, int32_t is_complex, int32_t natoms,
                        const int32_t *box_start, const int32_t *box_size, const int32_t *nproj,
                        const double *proj, const double *dmat, const void *psi, void *out,
                        void *coef, int64_t nbands, int32_t accumulate)
{
    if (!shape || !h || !bc || !psi || natoms < 0 || nbands < 0) return -1;
    if (natoms > 0 && (!box_start || !box_size || !nproj || !proj)) return -1;
    if (!out && !coef) return -1;
    if (out && natoms > 0 && !dmat) return -1;
    int64_t n[3];
    double kk[3];
    for (int d = 0; d < 3; ++d) {
        if (shape[d] < 1 || !(h[d] > 0.0)) return -1;
        n[d] = shape[d];
        kk[d] = k_reduced ? k_reduced[d] : 0.0;
        if (!is_complex && kk[d] != 0.0) return -1;
    }
    const double dv = h[0] * h[1] * h[2];
    const int64_t P = n[0] * n[1] * n[2];
    int64_t ntot = 0;
    for (int a = 0; a < natoms; ++a) ntot += nproj[a];
    if (out && !accumulate) memset(out, 0, (size_t)(nbands * P) * (is_complex ? 16 : 8));
    for (int64_t b = 0; b < nbands; ++b) {
        int64_t poff = 0, doff = 0, coff = 0;
        for (int a = 0; a < natoms; ++a) {
            const int32_t *s0 = box_start + 3 * a, *sz = box_size + 3 * a;
            const int ni = nproj[a];
            const int64_t nb = (int64_t)sz[0] * sz[1] * sz[2];
            double complex pc[64];
            if (ni < 0 || ni > 64 || sz[0] < 0 || sz[1] < 0 || sz[2] < 0) return -1;
            /* projections */
            for (int i = 0; i < ni; ++i) pc[i] = 0.0;
            for (int64_t rx = 0; rx < sz[0]; ++rx)
                for (int64_t ry = 0; ry < sz[1]; ++ry)
                    for (int64_t rz = 0; rz < sz[2]; ++rz) {
                        int64_t p[3] = { s0[0] + rx, s0[1] + ry, s0[2] + rz };
                        double complex phase = 1.0;
                        int dropped = 0;
                        for (int d = 0; d < 3; ++d)
                            if (p[d] < 0 || p[d] >= n[d]) {
                                if (bc[d] == FDO_BC_ZERO) { dropped = 1; break; }
                                const int64_t w = fdo_floordiv(p[d], n[d]);
                                p[d] -= w * n[d];
                                phase *= cexp(I * (2.0 * FDO_PI * kk[d] * (double)w));
                            }
                        if (dropped) continue;
                        const int64_t lin = (p[0] * n[1] + p[1]) * n[2] + p[2];
                        const double complex val =
                            (is_complex ? ((const double complex *)psi)[b * P + lin]
                                        : (double complex)((const double *)psi)[b * P + lin]) * phase;
                        const int64_t r = (rx * sz[1] + ry) * sz[2] + rz;
                        for (int i = 0; i < ni; ++i) pc[i] += proj[poff + i * nb + r] * val;
                    }
            for (int i = 0; i < ni; ++i) pc[i] *= dv;
            if (coef)
                for (int i = 0; i < ni; ++i) {
                    if (is_complex) ((double complex *)coef)[b * ntot + coff + i] = pc[i];
                    else ((double *)coef)[b * ntot + coff + i] = creal(pc[i]);
                }
            if (out) {
                /* d_i = sum_i' dO_ii' P_i' */
                double complex dc[64];
                for (int i = 0; i < ni; ++i) {
                    dc[i] = 0.0;
                    for (int i2 = 0; i2 < ni; ++i2) dc[i] += dmat[doff + i * ni + i2] * pc[i2];
                }
                for (int64_t rx = 0; rx < sz[0]; ++rx)
                    for (int64_t ry = 0; ry < sz[1]; ++ry)
                        for (int64_t rz = 0; rz < sz[2]; ++rz) {
                            int64_t p[3] = { s0[0] + rx, s0[1] + ry, s0[2] + rz };
                            double complex phase = 1.0;
                            int dropped = 0;
                            for (int d = 0; d < 3; ++d)
                                if (p[d] < 0 || p[d] >= n[d]) {
                                    if (bc[d] == FDO_BC_ZERO) { dropped = 1; break; }
                                    const int64_t w = fdo_floordiv(p[d], n[d]);
                                    p[d] -= w * n[d];
                                    phase *= cexp(I * (2.0 * FDO_PI * kk[d] * (double)w));
                                }
                            if (dropped) continue;
                            const int64_t lin = (p[0] * n[1] + p[1]) * n[2] + p[2];
                            const int64_t r = (rx * sz[1] + ry) * sz[2] + rz;
                            double complex s = 0.0;
                            for (int i = 0; i < ni; ++i) s += proj[poff + i * nb + r] * dc[i];
                            s *= conj(phase);
                            if (is_complex) ((double complex *)out)[b * P + lin] += s;
                            else ((double *)out)[b * P + lin] += creal(s);
                        }
            }
            poff += (int64_t)ni * nb;
            doff += (int64_t)ni * ni;
            coff += ni;
        }
    }
    return 0;
}
