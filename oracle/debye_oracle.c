/* debye_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what libdebye computes: the Debye summation
 *
 *     I(q) = sum_k f_k(q) sum_j f_j(q) sin(q r_jk) / (q r_jk)            (Eq. 2)
 *
 * written out as the definition (the paper's GPU algorithm reaches exactly Eq. 2; nothing is approximated
 * except floating point).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this file.  It shares no code, header, table or helper with
 * paper_1306_2258_b200/csrc (no per-type-pair partial sums, no recurrences, no 1/q factoring, sqrt not
 * rsqrt, libm sin).
 *
 * Readings of the paper used here:
 *   R1  both sums run over all N atoms including j = k (Eq. 2 is the expansion of |sum|^2 in Eq. 1).
 *   R2  sin(x)/x at x = 0 is its limit, 1 (self terms, coincident atoms, q = 0).
 *   R7  "only values for j <= k are computed" means I = sum_k f_k^2 + 2 sum_{j<k} f_j f_k sinc.
 *   R8  form factors are real, sign unrestricted.
 *   R10 form factors are given per atom TYPE: f_j(q_m) = fftab[type[j]][m]  (north_star narrowing).
 *   R10w optional per-atom weights (the one-parameter family of the paper's per-atom form factors,
 *        PAPER.md:44, 82): f_j(q_m) = weight[j] * fftab[type[j]][m]; weight == NULL means 1.
 *   R10p the paper's own general case (the form factors "cannot be factored out of the equation, because the
 *        non-uniform density of the water layer atoms around the molecule creates an intractable number of possible f_k f_j
 *        combinations"; the GPU memory holds "all N positions of atoms and at least one set of QN associated form
 *        factors for a specific q value", i.e. a Q x N table): f_j(q_m) = ff[j][m], one table row per
 *        ATOM (oracle_debye_peratom).
 * Inputs are the same float32 / int32 bytes the GPU gets, promoted exactly to double.
 *
 * Pins (tests/test_oracle_pins.py): two-atom closed form, I(0) = (sum f)^2, Eq. (1) by spherical quadrature,
 * chain / lattice / triangle / tetrahedron closed forms, coincident atoms, low-q expansion, rotation /
 * translation / permutation invariance, scaling identities, full == sym.  oracle_debye_peratom (R10p): two-atom and
 * triangle closed forms with different atoms, I(0) = (sum f)^2, Eq. (1) quadrature with a different f on every atom,
 * reduction to the per-type and weighted oracles, separable rows, permutation, full == sym (test_peratom_oracle_pins).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double sinc(double u) { return u == 0.0 ? 1.0 : sin(u) / u; }

static double dist(const float *a, const float *b)
{
    double dx = (double)a[0] - (double)b[0];
    double dy = (double)a[1] - (double)b[1];
    double dz = (double)a[2] - (double)b[2];
    return sqrt(dx * dx + dy * dy + dz * dz);
}

/* Eq. (2) literally: for every q_m, the full N x N double loop including j == k.
 * I[m] = sum_k sum_j F[t_k][m] F[t_j][m] sinc(q_m r_jk);  Abs[m] (optional) = same with |.| on each term,
 * so callers can print the condition number Abs/I.  Single thread, no symmetry. */
void oracle_debye_full_w(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab,
                         int32_t T, const float *q, int32_t M, double *I, double *Abs);
void oracle_debye_full(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T,
                       const float *q, int32_t M, double *I, double *Abs)
{
    oracle_debye_full_w(xyz, type, NULL, N, fftab, T, q, M, I, Abs);
}
/* The same with per-atom weights (reading R10w): f_k(q_m) = weight[k] F[t_k][m]. */
void oracle_debye_full_w(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab,
                         int32_t T, const float *q, int32_t M, double *I, double *Abs)
{
    (void)T;
    for (int m = 0; m < M; ++m) {
        long double acc = 0.0L, aabs = 0.0L;
        double qm = (double)q[m];
        for (int k = 0; k < N; ++k) {
            double fk = (double)fftab[(size_t)type[k] * M + m] * (weight ? (double)weight[k] : 1.0);
            for (int j = 0; j < N; ++j) {
                double fj = (double)fftab[(size_t)type[j] * M + m] * (weight ? (double)weight[j] : 1.0);
                double term = fk * fj * sinc(qm * dist(xyz + 3 * k, xyz + 3 * j));
                acc += term;
                aabs += fabs(term);
            }
        }
        I[m] = (double)acc;
        if (Abs) Abs[m] = (double)aabs;
    }
}

/* Reading R7: I = sum_k f_k (f_k + 2 sum_{j>k} f_j sinc(q r_jk)), rows k in [row0, row1) only (a row slab
 * is what bench.py times; row0=0,row1=N gives the whole profile).  One double accumulator per (row, q),
 * rows combined in long double.  OpenMP over rows, cyclic static schedule; threads <= 0 means all cores.
 * Returns the number of threads used. */
int32_t oracle_debye_sym_w(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab,
                           int32_t T, const float *q, int32_t M, int32_t row0, int32_t row1, int32_t threads,
                           double *I, double *Abs);
int32_t oracle_debye_sym(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T,
                         const float *q, int32_t M, int32_t row0, int32_t row1, int32_t threads,
                         double *I, double *Abs)
{
    return oracle_debye_sym_w(xyz, type, NULL, N, fftab, T, q, M, row0, row1, threads, I, Abs);
}
/* The same with per-atom weights (reading R10w). */
int32_t oracle_debye_sym_w(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab,
                           int32_t T, const float *q, int32_t M, int32_t row0, int32_t row1, int32_t threads,
                           double *I, double *Abs)
{
    (void)T;
    int nthr = 1;
#ifdef _OPENMP
    nthr = threads > 0 ? threads : omp_get_max_threads();
#endif
    long double *tot = (long double *)calloc((size_t)nthr * 2 * M, sizeof(long double));
#pragma omp parallel num_threads(nthr)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        long double *ti = tot + (size_t)tid * 2 * M, *ta = ti + M;
        double *row = (double *)malloc(sizeof(double) * 2 * M), *rabs = row + M;
#pragma omp for schedule(static, 1)
        for (int k = row0; k < row1; ++k) {
            const float *fk = fftab + (size_t)type[k] * M;
            for (int m = 0; m < M; ++m) row[m] = rabs[m] = 0.0;
            for (int j = k + 1; j < N; ++j) {
                const float *fj = fftab + (size_t)type[j] * M;
                double r = dist(xyz + 3 * k, xyz + 3 * j);
                double wj = weight ? (double)weight[j] : 1.0;
                for (int m = 0; m < M; ++m) {
                    double t = wj * (double)fj[m] * sinc((double)q[m] * r);
                    row[m] += t;
                    rabs[m] += fabs(t);
                }
            }
            for (int m = 0; m < M; ++m) {
                double f = (double)fk[m] * (weight ? (double)weight[k] : 1.0);
                ti[m] += (long double)(f * f) + 2.0L * (long double)f * (long double)row[m];
                ta[m] += (long double)(f * f) + 2.0L * (long double)fabs(f) * (long double)rabs[m];
            }
        }
        free(row);
    }
    for (int m = 0; m < M; ++m) {
        long double a = 0.0L, b = 0.0L;
        for (int t = 0; t < nthr; ++t) { a += tot[(size_t)t * 2 * M + m]; b += tot[(size_t)t * 2 * M + M + m]; }
        I[m] = (double)a;
        if (Abs) Abs[m] = (double)b;
    }
    free(tot);
    return nthr;
}

/* Reading R10p: Eq. (2) with per-ATOM form factors ff[N][M], written as the definition over the full
 * N x N double loop including j == k when sym == 0, and as  sum_k f_k (f_k + 2 sum_{j>k} f_j sinc) with
 * OpenMP over rows when sym != 0.  No types, no weights: ff[j][m] is used as given. */
void oracle_debye_peratom(const float *xyz, const float *ff, int32_t N, const float *q, int32_t M, int32_t sym,
                          double *I, double *Abs)
{
    if (!sym) {
        for (int m = 0; m < M; ++m) {
            long double acc = 0.0L, aabs = 0.0L;
            for (int k = 0; k < N; ++k)
                for (int j = 0; j < N; ++j) {
                    double term = (double)ff[(size_t)k * M + m] * (double)ff[(size_t)j * M + m] *
                                  sinc((double)q[m] * dist(xyz + 3 * k, xyz + 3 * j));
                    acc += term;
                    aabs += fabs(term);
                }
            I[m] = (double)acc;
            if (Abs) Abs[m] = (double)aabs;
        }
        return;
    }
    for (int m = 0; m < M; ++m) {
        long double acc = 0.0L, aabs = 0.0L;
#pragma omp parallel for schedule(static, 1) reduction(+ : acc, aabs)
        for (int k = 0; k < N; ++k) {
            double fk = (double)ff[(size_t)k * M + m], row = 0.0, rabs = 0.0;
            for (int j = k + 1; j < N; ++j) {
                double t = (double)ff[(size_t)j * M + m] * sinc((double)q[m] * dist(xyz + 3 * k, xyz + 3 * j));
                row += t;
                rabs += fabs(t);
            }
            acc += (long double)(fk * fk) + 2.0L * (long double)fk * (long double)row;
            aabs += (long double)(fk * fk) + 2.0L * (long double)fabs(fk) * (long double)rabs;
        }
        I[m] = (double)acc;
        if (Abs) Abs[m] = (double)aabs;
    }
}

/* Eq. (1): I(q) = < | sum_j f_j exp(i q.r_j) |^2 >_Omega by brute-force quadrature over
 * the direction of q: Gauss-Legendre nodes in cos(theta) (passed in: mu[n], wmu[n], weights summing to 2)
 * times a 2n-point midpoint rule in phi.  Takes per-atom form factors f[N] at ONE q.  Small N only. */
double oracle_eq1_quadrature(const double *x, const double *f, int32_t N, double q, const double *mu,
                             const double *wmu, int32_t n)
{
    long double acc = 0.0L;
    int nphi = 2 * n;
    for (int a = 0; a < n; ++a) {
        double st = sqrt(1.0 - mu[a] * mu[a]);
        for (int b = 0; b < nphi; ++b) {
            double phi = 2.0 * M_PI * (b + 0.5) / nphi;
            double ux = st * cos(phi), uy = st * sin(phi), uz = mu[a];
            double re = 0.0, im = 0.0;
            for (int j = 0; j < N; ++j) {
                double ph = q * (ux * x[3 * j] + uy * x[3 * j + 1] + uz * x[3 * j + 2]);
                re += f[j] * cos(ph);
                im += f[j] * sin(ph);
            }
            acc += (long double)(wmu[a] * 0.5 / nphi) * (long double)(re * re + im * im);
        }
    }
    return (double)acc;
}
