/*
 * bench_cpu/tablemethod.c -- BENCH-ONLY CPU restatement of the paper's own method (second half).
 *
 * Not part of libtj, not part of the oracle: reached only from bench.py (the `cpu_table_method` leg) and from
 * tests/test_cpu_table_method.py, which checks it against the oracle.  It exists so that the paper's headline
 * "6-25x over recursion-based pipelines" (TT 25.3x and EE 6.7x at lmax = 4722 on 8 Apple-M3 cores,
 * PAPER.md:232-234) can be re-measured on the GPU box's own host cores, table method against the Schulten-Gordon
 * oracle, beside the GPU number.
 *
 * What it does, as the paper describes its CPU code:
 *   - tables: ln g(p) from Eq. 12, g(p) = (p - 1/2)/p g(p-1), g(0) = 1, then
 *     g and 1/g by exponentiation; 1/(J+1) precomputed;
 *   - driver: OpenMP dynamic over l1, thread-private scalars, row-major K, upper triangle, then the
 *     lower triangle from the symmetry of K/(2 l2+1);
 *   - l3 loop: l3 from |l1-l2| in steps of 2 (even J), the halved indices p = J/2,
 *     p1 = p - l1, p2 = p - l2, p3 = p - l3 advance by +1, +1, +1, -1 per step;
 *   - TT term (Eq. 10):  (j1 j2 j3;000)^2 = g(p1) g(p2) g(p3) / ((J+1) g(p));
 *   - EE term (Eq. 16, coefficients of Eqs. B14-B16, as read in DESIGN.md 2):
 *       (j1 j2 j3;0 -2 2)^2 = [ a^2 X^2 + 2 a b s sqrt(X^2 Y^2) + b^2 Y^2 ] / eta^2,   s = -1 for even J,
 *       X = (j1 j2 j3;000), Y = (j1 j2 j3+2;000), with (j1,j2,j3) = (l3,l1,l2) by the column permutation of Eq. 7
 *       (PAPER.md:119-123).
 * K = (2 l2+1)/(4 pi) sum_l3 (2 l3+1) W_l3 (symbol)^2   (Eqs. 3-4).
 */
#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int pmax;        /* tables hold p = 0..pmax */
    double *g;       /* g(p) */
    double *ginv;    /* 1/g(p) */
    double *invJ1;   /* 1/(J+1) for J = 0..2 pmax */
} tm_tables;

int tm_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void tm_free(tm_tables *t)
{
    if (!t) return;
    free(t->g); free(t->ginv); free(t->invJ1); free(t);
}

/* ln g by the recurrence, then exponentiate */
tm_tables *tm_build(int lmax)
{
    tm_tables *t = (tm_tables *)calloc(1, sizeof(tm_tables));
    if (!t) return NULL;
    t->pmax = 2 * lmax + 2;
    t->g = (double *)malloc(sizeof(double) * (size_t)(t->pmax + 1));
    t->ginv = (double *)malloc(sizeof(double) * (size_t)(t->pmax + 1));
    t->invJ1 = (double *)malloc(sizeof(double) * (size_t)(2 * t->pmax + 2));
    if (!t->g || !t->ginv || !t->invJ1) { tm_free(t); return NULL; }
    double lng = 0.0;
    t->g[0] = 1.0; t->ginv[0] = 1.0;
    for (int p = 1; p <= t->pmax; ++p) {
        lng += log(((double)p - 0.5) / (double)p);
        t->g[p] = exp(lng);
        t->ginv[p] = exp(-lng);
    }
    for (int J = 0; J <= 2 * t->pmax + 1; ++J) t->invJ1[J] = 1.0 / ((double)J + 1.0);
    return t;
}

/* (l1 l2 l3;000)^2 for even J from the tables, Eq. 10 */
static inline double x2_000(const tm_tables *t, int p, int p1, int p2, int p3)
{
    return t->g[p1] * t->g[p2] * t->g[p3] * t->ginv[p] * t->invJ1[2 * p];
}

/*
 * Rows l1 = rows[0..nrows) of K^TT and/or K^EE, all columns l2 = 0..lmax, written to TT/EE as [nrows][lmax+1]
 * (NULL: skip).  Windows W have l3max+1 entries.  With full = 1 the rows must be 0..lmax in order; then only
 * l2 >= l1 is computed and the lower triangle is filled from the symmetry.
 */
int tm_coupling_rows(const tm_tables *t, int lmax, int l3max, const double *Wtt, const double *Wpp, int nrows,
                     const int *rows, int full, double *TT, double *EE)
{
    const double inv4pi = 1.0 / (4.0 * 3.14159265358979323846264338327950288);
    const long N = (long)lmax + 1;
    if (!t || lmax < 0 || l3max < 0 || t->pmax < 2 * lmax + 2) return -1;
#pragma omp parallel for schedule(dynamic)
    for (int r = 0; r < nrows; ++r) {
        const int l1 = rows[r];
        for (int l2 = full ? l1 : 0; l2 <= lmax; ++l2) {
            const int lo = l1 > l2 ? l1 - l2 : l2 - l1;
            const int hi = l1 + l2 < l3max ? l1 + l2 : l3max;
            double stt = 0.0, see = 0.0;
            /* per-pair constants of Eqs. B14-B16 with (j2, j3) = (l1, l2) */
            const int pol = EE && l1 >= 2 && l2 >= 2;
            const double j2 = l1, j3 = l2;
            const double lam = sqrt(j2 * (j2 + 1.0) * (j3 + 1.0) * (j3 + 2.0));
            const double eta2 = (j2 - 1.0) * (j2 + 2.0) * (j3 - 1.0) * j3;
            /* halved indices at l3 = lo (J = l1 + l2 + lo is even) */
            int p = (l1 + l2 + lo) / 2, p1 = p - l1, p2 = p - l2, p3 = p - lo;
            for (int l3 = lo; l3 <= hi; l3 += 2, ++p, ++p1, ++p2, --p3) {
                const double w = 2.0 * l3 + 1.0;
                const double X2 = x2_000(t, p, p1, p2, p3);
                if (TT) stt += w * Wtt[l3] * X2;
                if (pol) {
                    /* Y = (l3, l1, l2+2; 000): J -> J+2, so p -> p+1, p1 -> p1+1... in the paper's (j1,j2,j3) = (l3,l1,l2):
                       p - j1 = p3 + 1, p - j2 = p1 + 1, p - (j3+2) = p2 - 1 (negative: Y lies outside the triangle) */
                    const double Y2 = p2 >= 1 ? x2_000(t, p + 1, p1 + 1, p2 - 1, p3 + 1) : 0.0;
                    const double J = 2.0 * p, J1 = -l3 + l1 + l2, J2 = l3 - l1 + l2, J3 = l3 + l1 - l2;
                    const double al = lam + (2.0 * lam / j2) * (1.0 - (J + 2.0) * (J1 + 1.0) / (2.0 * (j2 + 1.0) * (j3 + 1.0)));
                    const double be = J3 >= 1.0 ? sqrt((J + 2.0) * (J1 + 1.0) * (J2 + 1.0) * J3 * (J + 3.0) * (J1 + 2.0) *
                                                       (J2 + 2.0) * (J3 - 1.0)) / (2.0 * lam) : 0.0;
                    const double sym2 = (al * al * X2 - 2.0 * al * be * sqrt(X2 * Y2) + be * be * Y2) / eta2;
                    see += w * Wpp[l3] * sym2;
                }
            }
            const double f = (2.0 * l2 + 1.0) * inv4pi;
            if (TT) TT[(long)r * N + l2] = f * stt;
            if (EE) EE[(long)r * N + l2] = f * see;
        }
    }
    if (full) {   /* lower triangle from the symmetry of K/(2 l2+1) */
        for (long l1 = 0; l1 <= lmax; ++l1)
            for (long l2 = 0; l2 < l1; ++l2) {
                const double f = (2.0 * l2 + 1.0) / (2.0 * l1 + 1.0);
                if (TT) TT[l1 * N + l2] = TT[l2 * N + l1] * f;
                if (EE) EE[l1 * N + l2] = EE[l2 * N + l1] * f;
            }
    }
    return 0;
}
