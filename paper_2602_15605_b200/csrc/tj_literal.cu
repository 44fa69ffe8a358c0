// tj_literal.cu -- the paper's own evaluation, restated as ONE plain kernel: an ablation
// and a "prior art on this GPU" baseline, not part of the hot path.
//
// Design of the paper's GPU path: one independent work-item per (l1,l2) of the upper
// triangle, each running the serial l3 loop in steps of 2 with direct table lookups
// (PAPER.md:186), results mirrored into the lower triangle.  Per term:
//
//   TT  (Eq. 10):   X^2 = g(p-j1) g(p-j2) g(p-j3) / ((J+1) g(p)),  p = J/2
//   EE  (Eq. 16, with Eqs. B14-B16 at PAPER.md:435-447 as read in DESIGN.md 2, readings 3-5):
//       (j1 j2 j3;0 -2 2)^2 = eta^-2 ( alpha^2 X^2 + 2 alpha beta s(J) sqrt(X^2 Y^2) + beta^2 Y^2 ),  s(J) = -1,
//       Y = (j1 j2 j3+2;000),  (j1,j2,j3) = (l3,l1,l2)  [Eq. 7: (l1 l2 l3;-2 2 0) = (l3 l1 l2;0 -2 2)],
//       lambda^2 = j2(j2+1)(j3+1)(j3+2),  eta^2 = (j2-1)(j2+2)(j3-1)j3,
//       alpha = lambda + (2 lambda/j2) (1 - (J+2)(J1+1) / (2 (j2+1)(j3+1))),
//       beta  = (1/(2 lambda)) [ (J+2)(J1+1)(J2+1)J3 (J+3)(J1+2)(J2+2)(J3-1) ]^(1/2),
//       J1 = -j1+j2+j3, J2 = j1-j2+j3, J3 = j1+j2-j3.
//
// i.e. two table products, two square roots and a division-free but long coefficient chain per term -- the
// cost structure behind the paper's "EE ~ 5x TT".  The hot path (tj_sweep.cu) replaces
// all of it by one table product times a polynomial.  The only liberty taken here: the 1/g(p)
// and 1/(J+1) tables of PAPER.md:186 are the folded table h[p] = 1/((2p+1) g(p)) the library already holds.
#include "tj_internal.cuh"

namespace tj {
namespace {

constexpr int LIT_THREADS = 128;

__global__ void __launch_bounds__(LIT_THREADS) literal_kernel(const double *__restrict__ g, const double *__restrict__ h,
                                                              const double *__restrict__ wtt,
                                                              const double *__restrict__ wpp, double *TT, double *EE,
                                                              int lmax, int l3max)
{
    const int l1 = (int)blockIdx.y;
    const int l2 = (int)(blockIdx.x * LIT_THREADS + threadIdx.x);
    if (l2 < l1 || l2 > lmax) return;
    const int s = l1 + l2;
    const int hi = s < l3max ? s : l3max;
    const bool pol = EE != nullptr && l1 >= 2;
    // per-pair constants of Eqs. B14-B16 in (j2,j3) = (l1,l2)
    const double j2 = (double)l1, j3 = (double)l2;
    const double lam = sqrt(j2 * (j2 + 1.0) * (j3 + 1.0) * (j3 + 2.0));
    const double eta2 = (j2 - 1.0) * (j2 + 2.0) * (j3 - 1.0) * j3;
    const double inv_eta2 = pol ? 1.0 / eta2 : 0.0;
    const double c_al = pol ? 2.0 * lam / j2 : 0.0, c_in = 1.0 / (2.0 * (j2 + 1.0) * (j3 + 1.0));
    const double inv_2lam = 0.5 / lam;
    double stt = 0.0, see = 0.0;
    for (int l3 = l2 - l1; l3 <= hi; l3 += 2) {   // even J only: parity skipping
        const int J = s + l3, p = J >> 1;
        const double X2 = g[p - l3] * g[p - l1] * g[p - l2] * h[p];
        if (TT) stt = fma(wtt[l3], X2, stt);
        if (pol) {
            const double Y2 = g[p + 1 - l3] * g[p + 1 - l1] * g[p - 1 - l2] * h[p + 1];   // g[-1] = 0 closes J3 = 0
            const double dJ = (double)J, J1 = (double)(s - l3), J2 = (double)(l3 - l1 + l2), J3 = (double)(l3 + l1 - l2);
            const double al = lam + c_al * (1.0 - (dJ + 2.0) * (J1 + 1.0) * c_in);
            const double rad = (dJ + 2.0) * (J1 + 1.0) * (J2 + 1.0) * J3 * (dJ + 3.0) * (J1 + 2.0) * (J2 + 2.0) * (J3 - 1.0);
            const double be = J3 >= 1.0 ? inv_2lam * sqrt(rad) : 0.0;
            const double sym2 = (al * al * X2 - 2.0 * al * be * sqrt(X2 * Y2) + be * be * Y2) * inv_eta2;
            see = fma(wpp[l3], sym2, see);
        }
    }
    // K = (2 l2+1) Xi and its mirror; prefolded windows already carry (2 l3+1)/(4 pi)
    const long long N = (long long)lmax + 1;
    if (TT) {
        TT[(long long)l1 * N + l2] = stt * (double)(2 * l2 + 1);
        TT[(long long)l2 * N + l1] = stt * (double)(2 * l1 + 1);
    }
    if (EE) {
        EE[(long long)l1 * N + l2] = see * (double)(2 * l2 + 1);
        EE[(long long)l2 * N + l1] = see * (double)(2 * l1 + 1);
    }
}

}  // namespace

cudaError_t launch_literal(const Tables &T, const double *wtt, const double *wpp, double *TT, double *EE, int l3max,
                           cudaStream_t st)
{
    const int N = T.lmax + 1;
    dim3 grid((unsigned)((N + LIT_THREADS - 1) / LIT_THREADS), (unsigned)N, 1);
    literal_kernel<<<grid, LIT_THREADS, 0, st>>>(T.g, T.h, wtt, wpp, TT, EE, T.lmax, l3max);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace tj
