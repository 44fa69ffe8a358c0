/*
 * sg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU oracle for the pseudo-C_ell mode-coupling
 * matrices of arxiv/paper_2602_15605.  It evaluates the DEFINITION
 * of each matrix,
 *
 *   K^{TT}_{l1 l2} = (2 l2+1)/(4 pi) sum_{l3} (2 l3+1) W^{TT}_{l3} (l1 l2 l3; 0 0 0)^2      PAPER.md:76-78 Eq. 3, :340 Eq. A1
 *   K^{TE}_{l1 l2} = ... W^{TP}_{l3} [even L] (l1 l2 l3;000) (l1 l2 l3;-2 2 0)              PAPER.md:344 Eq. A2
 *   K^{EE}_{l1 l2} = ... W^{PP}_{l3} [even L] (l1 l2 l3;-2 2 0)^2                            PAPER.md:80-84 Eq. 4, :348 Eq. A3
 *   K^{EB}_{l1 l2} = ... W^{PP}_{l3} [odd  L] (l1 l2 l3;-2 2 0)^2                            PAPER.md:352 Eq. A4
 *   K = (2 l2+1) Xi
 *
 * with every Wigner-3j symbol taken from the Schulten-Gordon three-term
 * recursion in j1 (the method the paper names as the standard one, PAPER.md:33,
 * :45, :224) -- NOT from the paper's lookup-table formalism, which is what the
 * CUDA path implements.  The two meet only at the final matrices.
 *
 * Nothing here is shared with, imported by, or generated from the CUDA path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * Pins (tests/test_oracle_*.py): exact Racah rationals for all l <= 30 and a few
 * high-l symbols, orthogonality, parity zeros, full-sky identity, flat-window
 * closed form; the spin-1 sums: exact Racah (-1,1,0) symbols, full-sky and flat-window closed forms,
 * brute-force exact-rational sums.  No function in this file is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOMEM (-2)

static const double PI = 3.14159265358979323846264338327950288;

/* A(j) of the Schulten-Gordon recursion (Schulten & Gordon 1975):
 *   A(j) = sqrt( (j^2-(j2-j3)^2) ((j2+j3+1)^2-j^2) (j^2-m1^2) ) */
static double sg_A(double j, double j2, double j3, double m1)
{
    double a = j * j - (j2 - j3) * (j2 - j3);
    double b = (j2 + j3 + 1.0) * (j2 + j3 + 1.0) - j * j;
    double c = j * j - m1 * m1;
    double prod = a * b * c;
    if (prod <= 0.0) return 0.0;
    /* three separate roots: the product a*b*c reaches ~1e27 at l ~ 3e4, still exact enough,
       but separate roots keep every factor an exactly representable integer */
    return sqrt(a) * sqrt(b) * sqrt(c);
}

/* B(j) = -(2j+1) [ j2(j2+1) m1 - j3(j3+1) m1 - j(j+1)(m3-m2) ] */
static double sg_B(double j, double j2, double j3, double m1, double m2, double m3)
{
    return -(2.0 * j + 1.0) * (j2 * (j2 + 1.0) * m1 - j3 * (j3 + 1.0) * m1 - j * (j + 1.0) * (m3 - m2));
}

/*
 * f(j) = ( j  j2  j3 ; m1 m2 m3 ), m1 = -m2-m3, for all j = jmin..jmax,
 *   jmin = max(|j2-j3|, |m1|), jmax = j2+j3.
 * Recursion:  j A(j+1) f(j+1) + B(j) f(j) + (j+1) A(j) f(j-1) = 0.
 * Forward sweep from jmin, backward sweep from jmax, matched where both are large,
 * normalised by sum_j (2j+1) f(j)^2 = 1, sign fixed by sgn f(jmax) = (-1)^(j2-j3-m1).
 *
 * out must hold jmax-jmin+1 doubles.  Returns 0, or ORACLE_EINVAL when the
 * arguments admit no symbol (|m2|>j2 or |m3|>j3): then *jmin_out > *jmax_out.
 */
int oracle_3j_family(int j2, int j3, int m2, int m3, double *out, int *jmin_out, int *jmax_out)
{
    int m1 = -m2 - m3;
    int am1 = m1 < 0 ? -m1 : m1;
    int dj = j2 > j3 ? j2 - j3 : j3 - j2;
    int jmin = dj > am1 ? dj : am1;
    int jmax = j2 + j3;
    if (j2 < 0 || j3 < 0 || abs(m2) > j2 || abs(m3) > j3 || jmin > jmax) {
        if (jmin_out) *jmin_out = 1;
        if (jmax_out) *jmax_out = 0;
        return ORACLE_EINVAL;
    }
    if (jmin_out) *jmin_out = jmin;
    if (jmax_out) *jmax_out = jmax;
    int n = jmax - jmin + 1;
    double dj2 = j2, dj3 = j3, dm1 = m1, dm2 = m2, dm3 = m3;

    /* sign convention: sgn f(jmax) = (-1)^(j2-j3-m1) */
    int e = j2 - j3 - m1;
    double sgn_top = (e % 2 == 0) ? 1.0 : -1.0;

    if (n == 1) {
        out[0] = sgn_top / sqrt(2.0 * jmin + 1.0);
        return ORACLE_OK;
    }

    double *fwd = (double *)malloc(sizeof(double) * (size_t)n);
    double *bwd = (double *)malloc(sizeof(double) * (size_t)n);
    double *Aj = (double *)malloc(sizeof(double) * (size_t)(n + 2)); /* Aj[k] = A(jmin+k), k=0..n */
    if (!fwd || !bwd || !Aj) { free(fwd); free(bwd); free(Aj); return ORACLE_ENOMEM; }
    for (int k = 0; k <= n; ++k) Aj[k] = sg_A((double)(jmin + k), dj2, dj3, dm1);
    /* A(jmin) = 0 and A(jmax+1) = 0 by construction of the range */
    Aj[0] = 0.0;
    Aj[n] = 0.0;

    const double BIG = 1e200, SMALL = 1e-200;

    /* ---- forward sweep ---- */
    fwd[0] = 1.0;
    if (jmin == 0) {
        /* degenerate start (needs j2 = j3, m1 = 0): the j=0 row of the recursion is 0 = 0;
           the ratio follows from the explicit j=0,1 symbols: f(1) = -(m3-m2)/A(1) f(0) */
        fwd[1] = -(dm3 - dm2) / Aj[1] * fwd[0];
    } else {
        double j = jmin;
        fwd[1] = -(sg_B(j, dj2, dj3, dm1, dm2, dm3) * fwd[0]) / (j * Aj[1]);
    }
    for (int k = 1; k < n - 1; ++k) {
        double j = jmin + k;
        double num = sg_B(j, dj2, dj3, dm1, dm2, dm3) * fwd[k] + (j + 1.0) * Aj[k] * fwd[k - 1];
        fwd[k + 1] = -num / (j * Aj[k + 1]);
        if (fabs(fwd[k + 1]) > BIG) {
            for (int q = 0; q <= k + 1; ++q) fwd[q] *= SMALL;
        }
    }

    /* ---- backward sweep ---- */
    bwd[n - 1] = 1.0;
    {
        double j = jmax;
        bwd[n - 2] = -(sg_B(j, dj2, dj3, dm1, dm2, dm3) * bwd[n - 1]) / ((j + 1.0) * Aj[n - 1]);
    }
    for (int k = n - 2; k >= 1; --k) {
        double j = jmin + k;
        double num = j * Aj[k + 1] * bwd[k + 1] + sg_B(j, dj2, dj3, dm1, dm2, dm3) * bwd[k];
        bwd[k - 1] = -num / ((j + 1.0) * Aj[k]);
        if (fabs(bwd[k - 1]) > BIG) {
            for (int q = k - 1; q < n; ++q) bwd[q] *= SMALL;
        }
    }

    /* ---- match where both sweeps are large ---- */
    double maxf = 0.0, maxb = 0.0;
    for (int k = 0; k < n; ++k) {
        if (fabs(fwd[k]) > maxf) maxf = fabs(fwd[k]);
        if (fabs(bwd[k]) > maxb) maxb = fabs(bwd[k]);
    }
    int kstar = 0;
    double best = -1.0;
    for (int k = 0; k < n; ++k) {
        double v = (fabs(fwd[k]) / maxf) * (fabs(bwd[k]) / maxb);
        if (v > best) { best = v; kstar = k; }
    }
    double lam = fwd[kstar] / bwd[kstar];
    for (int k = 0; k <= kstar; ++k) out[k] = fwd[k];
    for (int k = kstar + 1; k < n; ++k) out[k] = lam * bwd[k];

    /* ---- normalise: sum_j (2j+1) f^2 = 1 ---- */
    double norm = 0.0;
    for (int k = 0; k < n; ++k) norm += (2.0 * (jmin + k) + 1.0) * out[k] * out[k];
    double scale = 1.0 / sqrt(norm);
    /* ---- sign ---- */
    if ((out[n - 1] < 0.0 ? -1.0 : 1.0) != sgn_top) scale = -scale;
    for (int k = 0; k < n; ++k) out[k] *= scale;

    free(fwd); free(bwd); free(Aj);
    return ORACLE_OK;
}

/* Integer bookkeeping of the l3 sum for one pair:
 * l3 runs over |l1-l2| .. min(l1+l2, l3max) with (l1+l2+l3) % 2 == parity.
 * nterms may be 0; then lo > hi. */
int oracle_l3_range(int l1, int l2, int l3max, int parity, int *l3_lo, int *l3_hi, int *nterms)
{
    if (l1 < 0 || l2 < 0 || l3max < 0 || (parity != 0 && parity != 1)) return ORACLE_EINVAL;
    int lo = l1 > l2 ? l1 - l2 : l2 - l1;
    int hi = l1 + l2 < l3max ? l1 + l2 : l3max;
    /* lo has the parity of l1+l2, i.e. J even at l3 = lo */
    if (parity == 1) lo += 1;
    if (hi >= lo && ((l1 + l2 + hi) & 1) != parity) hi -= 1;
    int n = hi >= lo ? (hi - lo) / 2 + 1 : 0;
    if (l3_lo) *l3_lo = lo;
    if (l3_hi) *l3_hi = hi;
    if (nterms) *nterms = n;
    return ORACLE_OK;
}

/*
 * Coupling-matrix entries for a list of (l1,l2) pairs, straight from Eqs. A1-A4.
 *   W??[l], l = 0..l3max  (any of them may be NULL together with its outputs)
 *   TT, TE, EE, EB: npairs doubles each (NULL to skip).  BB == EE.
 * Entries of the polarised blocks with min(l1,l2) < 2 are 0 (the spin-2 symbol
 * does not exist for |m| > l).
 */
int oracle_coupling_pairs(int l3max, const double *Wtt, const double *Wtp, const double *Wpp,
                          long npairs, const int *l1s, const int *l2s,
                          double *TT, double *TE, double *EE, double *EB)
{
    if (l3max < 0 || npairs < 0) return ORACLE_EINVAL;
    if ((TT && !Wtt) || (TE && !Wtp) || ((EE || EB) && !Wpp)) return ORACLE_EINVAL;
    int status = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (long q = 0; q < npairs; ++q) {
        int l1 = l1s[q], l2 = l2s[q];
        if (l1 < 0 || l2 < 0) {
#pragma omp atomic write
            status = ORACLE_EINVAL;
            continue;
        }
        int n = l1 + l2 - abs(l1 - l2) + 1;
        double *f0 = (double *)malloc(sizeof(double) * (size_t)n);
        double *f2 = (double *)malloc(sizeof(double) * (size_t)n);
        if (!f0 || !f2) {
            free(f0); free(f2);
#pragma omp atomic write
            status = ORACLE_ENOMEM;
            continue;
        }
        int jmin, jmax;
        /* f0(l3) = (l3 l1 l2; 0 0 0) = (l1 l2 l3; 0 0 0)  (even permutation) */
        oracle_3j_family(l1, l2, 0, 0, f0, &jmin, &jmax);
        /* f2(l3) = (l3 l1 l2; 0 -2 2) = (l1 l2 l3; -2 2 0)  (Eq. 7) */
        int have2 = (l1 >= 2 && l2 >= 2);
        if (have2) {
            int jmin2, jmax2;
            oracle_3j_family(l1, l2, -2, 2, f2, &jmin2, &jmax2);
        } else {
            for (int k = 0; k < n; ++k) f2[k] = 0.0;
        }
        double stt = 0.0, ste = 0.0, see = 0.0, seb = 0.0;
        int hi = jmax < l3max ? jmax : l3max;
        for (int l3 = jmin; l3 <= hi; ++l3) {
            int k = l3 - jmin;
            double w = 2.0 * l3 + 1.0;
            int even = ((l1 + l2 + l3) & 1) == 0;
            if (Wtt) stt += w * Wtt[l3] * f0[k] * f0[k];
            if (even) {
                if (Wtp) ste += w * Wtp[l3] * f0[k] * f2[k];
                if (Wpp) see += w * Wpp[l3] * f2[k] * f2[k];
            } else {
                if (Wpp) seb += w * Wpp[l3] * f2[k] * f2[k];
            }
        }
        double pref = (2.0 * l2 + 1.0) / (4.0 * PI);
        if (TT) TT[q] = pref * stt;
        if (TE) TE[q] = pref * ste;
        if (EE) EE[q] = pref * see;
        if (EB) EB[q] = pref * seb;
        free(f0); free(f2);
    }
    return status;
}

/*
 * Spin-1 analogue of Eqs. A1-A4 for a list of (l1,l2) pairs: the same sums with the (0,-1,1) symbol the paper
 * lists for lensing / aberration weights (symbol formulas PAPER.md:362-392 Eqs. B1-B6) in
 * place of the spin-2 one.  The paper defines no weights for these, so the blocks are defined here
 * (reading 19) as
 *   K^{01}_{l1 l2}  = (2 l2+1)/(4 pi) sum_{l3, J even} (2 l3+1) W^{01}_{l3} (l1 l2 l3;000) (l1 l2 l3;-1 1 0)
 *   K^{11+}_{l1 l2} = (2 l2+1)/(4 pi) sum_{l3, J even} (2 l3+1) W^{11}_{l3} (l1 l2 l3;-1 1 0)^2
 *   K^{11-}_{l1 l2} = (2 l2+1)/(4 pi) sum_{l3, J odd } (2 l3+1) W^{11}_{l3} (l1 l2 l3;-1 1 0)^2
 * with (l1 l2 l3;-1 1 0) = (l3 l1 l2;0 -1 1) (Eq. 7) from the same Schulten-Gordon recursion.
 * Entries with min(l1,l2) < 1 are 0.  Outputs may be NULL.
 */
int oracle_coupling_spin1_pairs(int l3max, const double *W01, const double *W11, long npairs, const int *l1s,
                                const int *l2s, double *K01, double *K11p, double *K11m)
{
    if (l3max < 0 || npairs < 0) return ORACLE_EINVAL;
    if ((K01 && !W01) || ((K11p || K11m) && !W11)) return ORACLE_EINVAL;
    int status = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (long q = 0; q < npairs; ++q) {
        int l1 = l1s[q], l2 = l2s[q];
        if (l1 < 0 || l2 < 0) {
#pragma omp atomic write
            status = ORACLE_EINVAL;
            continue;
        }
        int n = l1 + l2 - abs(l1 - l2) + 1;
        double *f0 = (double *)malloc(sizeof(double) * (size_t)n);
        double *f1 = (double *)malloc(sizeof(double) * (size_t)n);
        if (!f0 || !f1) {
            free(f0); free(f1);
#pragma omp atomic write
            status = ORACLE_ENOMEM;
            continue;
        }
        int jmin, jmax;
        oracle_3j_family(l1, l2, 0, 0, f0, &jmin, &jmax);
        if (l1 >= 1 && l2 >= 1) {
            int jmin1, jmax1;
            oracle_3j_family(l1, l2, -1, 1, f1, &jmin1, &jmax1);   /* m1 = 0: same j range as f0 */
        } else {
            for (int k = 0; k < n; ++k) f1[k] = 0.0;
        }
        double s01 = 0.0, s11p = 0.0, s11m = 0.0;
        int hi = jmax < l3max ? jmax : l3max;
        for (int l3 = jmin; l3 <= hi; ++l3) {
            int k = l3 - jmin;
            double w = 2.0 * l3 + 1.0;
            if (((l1 + l2 + l3) & 1) == 0) {
                if (W01) s01 += w * W01[l3] * f0[k] * f1[k];
                if (W11) s11p += w * W11[l3] * f1[k] * f1[k];
            } else {
                if (W11) s11m += w * W11[l3] * f1[k] * f1[k];
            }
        }
        double pref = (2.0 * l2 + 1.0) / (4.0 * PI);
        if (K01) K01[q] = pref * s01;
        if (K11p) K11p[q] = pref * s11p;
        if (K11m) K11m[q] = pref * s11m;
        free(f0); free(f1);
    }
    return status;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
