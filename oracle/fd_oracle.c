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

/*
 * Same definition evaluated only at npoints sampled outputs: points[4*s + {0,1,2,3}] =
 * (band, ix, iy, iz); out[s] (double or double complex).  psi is the whole batch
 * [nbands, nx, ny, nz].  Used for full-size parity where the whole oracle would be too slow.
 */
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
