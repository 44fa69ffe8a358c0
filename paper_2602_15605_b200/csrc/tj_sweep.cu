// tj_sweep.cu -- the fused l3 sweep (steps a4 + a5 of the hot path).
//
// What one (l1,l2) pair accumulates (Eq. 10, Eqs. 13-16, B14-B17, A1-A4), with
// s = l1+l2, u_l = l(l+1), D_l = (l-1)l(l+1)(l+2), W'_X[l] = (2l+1) W_X[l]/(4 pi):
//
//   even step t (l3 = s-2t, t = 0..min(l1,l2)):
//       X^2 = h[s-t] g[t] g[l1-t] g[l2-t]                     (Eq. 10 with p=s-t, p1=l2-t, p2=l1-t, p3=t)
//       A2  = (u_l3 - u_l1 - u_l2 + 1)^2 - (2 u_l1 u_l2 + 1)   (= 2A; (l1 l2 l3;-2 2 0) = X A / sqrt(D_l1 D_l2))
//       S_TT += W'_TT[l3] X^2;   S_TE += W'_TP[l3] X^2 A2;   S_EE += W'_PP[l3] X^2 A2^2
//   odd step t (l3 = s-2t-1, t = 0..min(l1,l2)-1):
//       Z^2 = ginv[s-t] gB[t] gA[l1-t] gA[l2-t],  e = u_l3 - u_l1 - u_l2 + 2
//       S_EB += W'_PP[l3] Z^2 e^2
//   Xi_TT = S_TT,  Xi_TE = S_TE/(2 sqrt(D)),  Xi_EE = S_EE/(4D),  Xi_EB = S_EB/(4D),  D = D_l1 D_l2.
//
// Mapping to the machine.  A thread owns R pairs on ONE anti-diagonal,
// (l1,l2) = (a+i, c-i), so s, l3, h[s-t] g[t], the three W'[l3] and u_l3 are per-THREAD values per step,
// and the two per-pair table factors g[a+i-t], g[c-i-t] slide through two R-deep register rings:
// each step loads ONE new element per ring.  Lanes run along c: the per-row loads are warp broadcasts,
// everything else is consecutive doubles (no bank or sector conflicts).  Per even step a thread issues
// 8R+4 FP64 instructions against 8 loads.  Steps outside a pair's triangle (or beyond l3max) hit the zero
// guard bands of the tables / windows and add exact zeros, so the warp runs one branch-free t range.
#include "tj_internal.cuh"

namespace tj {
namespace {

__device__ __forceinline__ double ldg(const double *p) { return __ldg(p); }

// L1 prefetch of a table line the sweep will reach TJ_PF unrolled blocks from now (0 = off)
#ifndef TJ_PF
#define TJ_PF 0
#endif
#ifndef TJ_MINB
#define TJ_MINB 3
#endif
__device__ __forceinline__ void pf(const double *p)
{
#if TJ_PF > 0
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#endif
}

template <int R, int MASK>
__global__ void __launch_bounds__(SWEEP_THREADS, TJ_MINB) sweep_kernel(const __grid_constant__ SweepParams P)
{
    constexpr bool kTT = (MASK & M_TT) != 0, kTE = (MASK & M_TE) != 0, kEE = (MASK & M_EE) != 0,
                   kEB = (MASK & M_EB) != 0;
    constexpr bool kEven = kTT || kTE || kEE;
    constexpr bool kA2 = kTE || kEE;

    // ---- tile decode: binary search of blockIdx.x in the descending-band prefix ----
    const int tile = blockIdx.x;
    int lo = 0, hi = P.nbands;  // tile_start[lo] <= tile < tile_start[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(P.tile_start + mid) <= tile) lo = mid; else hi = mid;
    }
    const int band = P.nbands - 1 - lo;
    const int cb = tile - __ldg(P.tile_start + lo);
    const int a = band * R;
    const int c = a + cb * SWEEP_THREADS + (int)threadIdx.x;
    const int s = a + c;
    const int s_min = s - (int)(threadIdx.x & 31);  // warp-uniform: smallest s of the warp

    // a warp whose columns all lie beyond lmax has nothing to store
    if (s_min - a - (R - 1) > P.lmax) return;

    // ---- per-pair constants ----
    double c12[R], kk[R];
    if (kA2 || kEB) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double l1 = (double)(a + i), l2 = (double)(c - i);
            const double u1 = l1 * (l1 + 1.0), u2 = l2 * (l2 + 1.0);
            c12[i] = u1 + u2 - 2.0;                  // odd branch: e = u3 - c12
            kk[i] = __fma_rn(2.0 * u1, u2, 1.0);     // even branch: A2 = d1^2 - kk
        }
    }

    const int t_end = a + R - 1;  // last step any pair of the band can have (t <= min(l1,l2) <= l1)

    // =========================== odd-J branch: EB ===========================
    if (kEB) {
        double acc[R];
#pragma unroll
        for (int i = 0; i < R; ++i) acc[i] = 0.0;
        // l3 = s-2t-1 <= l3max  <=>  t >= (s-1-l3max)/2
        int tb = s_min - 1 - P.l3max;
        tb = tb > 0 ? (tb + 1) >> 1 : 0;
        if (tb <= t_end) {
            const int nblk = (t_end - tb + R) / R;
            double wa[R], wb[R];
            const double *pa = P.gA + (a - tb);
            const double *pb = P.gA + (c - R + 1 - tb);
            const double *ph = P.ginv + (s - tb);
            const double *pg = P.gB + tb;
            const double *pw = P.wpp + (s - 2 * tb - 1);
            const double *pu = P.u3 + (s - 2 * tb - 1);
#pragma unroll
            for (int k = 1; k < R; ++k) wa[k] = ldg(pa + k);                       // G[k] = gA[a-t0+k]
#pragma unroll
            for (int i = 0; i < R - 1; ++i) wb[(R - i) % R] = ldg(pb + (R - 1 - i));  // H[-i] = gA[c-t0-i]
            // software pipeline: the raw table values of substep u+1 are loaded while substep u computes
            double xa = ldg(pa), xb = ldg(pb), xh = ldg(ph), xg = ldg(pg), xw = ldg(pw), xu = ldg(pu);
            for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
                for (int u = 0; u < R; ++u) {
                    wa[(R - u) % R] = xa;
                    wb[(R + 1 - u) % R] = xb;
                    const double hg = __dmul_rn(xh, xg);
                    const double q3 = __dmul_rn(xw, hg);
                    const double c3 = xu;
                    xa = ldg(pa - (u + 1)); xb = ldg(pb - (u + 1)); xh = ldg(ph - (u + 1)); xg = ldg(pg + (u + 1));
                    xw = ldg(pw - 2 * (u + 1)); xu = ldg(pu - 2 * (u + 1));
                    // op-major order: consecutive FP64 instructions share c3 / q3 in one operand slot, so
                    // the register-file reuse cache serves it and no instruction needs 3 bank reads
                    double r[R], e[R];
#pragma unroll
                    for (int i = 0; i < R; ++i) r[i] = __dmul_rn(wa[(i - u + R) % R], wb[(2 * R - i - u) % R]);
#pragma unroll
                    for (int i = 0; i < R; ++i) e[i] = __dsub_rn(c3, c12[i]);
#pragma unroll
                    for (int i = 0; i < R; ++i) r[i] = __dmul_rn(r[i], e[i]);
#pragma unroll
                    for (int i = 0; i < R; ++i) r[i] = __dmul_rn(r[i], e[i]);
#pragma unroll
                    for (int i = 0; i < R; ++i) acc[i] = __fma_rn(r[i], q3, acc[i]);
                }
                pa -= R; pb -= R; ph -= R; pg += R; pw -= 2 * R; pu -= 2 * R;
            }
        }
        // epilogue: Xi_EB = S_EB / (4 D)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int l1 = a + i, l2 = c - i;
            if (l2 >= l1 && l2 <= P.lmax && (P.lcut < 0 || l2 - l1 <= P.lcut)) {
                const double sd = P.isd[l1] * P.isd[l2];
                const long long col = P.lcut < 0 ? (long long)l2 : (long long)(l2 - l1 + P.lcut);
                if (P.EB) P.EB[(long long)l1 * P.ld + col] = acc[i] * (0.25 * sd * sd);
            }
        }
    }

    // =========================== even-J branch: TT, TE, EE ===========================
    if (kEven) {
        double att[kTT ? R : 1], ate[kTE ? R : 1], aee[kEE ? R : 1];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            if (kTT) att[i] = 0.0;
            if (kTE) ate[i] = 0.0;
            if (kEE) aee[i] = 0.0;
        }
        if (kA2) {
#pragma unroll
            for (int i = 0; i < R; ++i) c12[i] += 1.0;   // even branch: d1 = d+1 = u3 - (u1+u2-1)
        }
        // l3 = s-2t <= l3max  <=>  t >= (s-l3max)/2
        int tb = s_min - P.l3max;
        tb = tb > 0 ? (tb + 1) >> 1 : 0;
        if (tb <= t_end) {
            const int nblk = (t_end - tb + R) / R;
            double wa[R], wb[R];
            const double *pa = P.g + (a - tb);
            const double *pb = P.g + (c - R + 1 - tb);
            const double *ph = P.h + (s - tb);
            const double *pg = P.g + tb;
            const double *pwtt = P.wtt + (s - 2 * tb);
            const double *pwtp = P.wtp + (s - 2 * tb);
            const double *pwpp = P.wpp + (s - 2 * tb);
            const double *pu = P.u3 + (s - 2 * tb);
#pragma unroll
            for (int k = 1; k < R; ++k) wa[k] = ldg(pa + k);
#pragma unroll
            for (int i = 0; i < R - 1; ++i) wb[(R - i) % R] = ldg(pb + (R - 1 - i));
            double xa = ldg(pa), xb = ldg(pb), xh = ldg(ph), xg = ldg(pg);
            double xtt = kTT ? ldg(pwtt) : 0.0, xtp = kTE ? ldg(pwtp) : 0.0, xpp = kEE ? ldg(pwpp) : 0.0;
            double xu = kA2 ? ldg(pu) : 0.0;
            for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
                for (int u = 0; u < R; ++u) {
                    wa[(R - u) % R] = xa;
                    wb[(R + 1 - u) % R] = xb;
                    const double hg = __dmul_rn(xh, xg);
                    double q0 = 0.0, q1 = 0.0, q2 = 0.0;
                    if (kTT) q0 = __dmul_rn(xtt, hg);
                    if (kTE) q1 = __dmul_rn(xtp, hg);
                    if (kEE) q2 = __dmul_rn(xpp, hg);
                    const double c3 = xu;
                    xa = ldg(pa - (u + 1)); xb = ldg(pb - (u + 1)); xh = ldg(ph - (u + 1)); xg = ldg(pg + (u + 1));
                    if (kTT) xtt = ldg(pwtt - 2 * (u + 1));
                    if (kTE) xtp = ldg(pwtp - 2 * (u + 1));
                    if (kEE) xpp = ldg(pwpp - 2 * (u + 1));
                    if (kA2) xu = ldg(pu - 2 * (u + 1));
                    // op-major order (see the odd branch): q0/q1/q2/c3 stay in the operand reuse cache
                    double r[R], A2[kA2 ? R : 1];
#pragma unroll
                    for (int i = 0; i < R; ++i) r[i] = __dmul_rn(wa[(i - u + R) % R], wb[(2 * R - i - u) % R]);
                    if (kA2) {
#pragma unroll
                        for (int i = 0; i < R; ++i) A2[i] = __dsub_rn(c3, c12[i]);
                    }
                    if (kTT) {
#pragma unroll
                        for (int i = 0; i < R; ++i) att[i] = __fma_rn(r[i], q0, att[i]);
                    }
                    if (kA2) {
#pragma unroll
                        for (int i = 0; i < R; ++i) A2[i] = __fma_rn(A2[i], A2[i], -kk[i]);
#pragma unroll
                        for (int i = 0; i < R; ++i) r[i] = __dmul_rn(r[i], A2[i]);
                        if (kTE) {
#pragma unroll
                            for (int i = 0; i < R; ++i) ate[i] = __fma_rn(r[i], q1, ate[i]);
                        }
                        if (kEE) {
#pragma unroll
                            for (int i = 0; i < R; ++i) r[i] = __dmul_rn(r[i], A2[i]);
#pragma unroll
                            for (int i = 0; i < R; ++i) aee[i] = __fma_rn(r[i], q2, aee[i]);
                        }
                    }
                }
                pa -= R; pb -= R; ph -= R; pg += R;
                pwtt -= 2 * R; pwtp -= 2 * R; pwpp -= 2 * R; pu -= 2 * R;
            }
        }
        // epilogue: Xi_TT = S_TT; Xi_TE = S_TE/(2 sqrt D); Xi_EE = S_EE/(4 D)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int l1 = a + i, l2 = c - i;
            if (l2 >= l1 && l2 <= P.lmax && (P.lcut < 0 || l2 - l1 <= P.lcut)) {
                const long long col = P.lcut < 0 ? (long long)l2 : (long long)(l2 - l1 + P.lcut);
                const long long idx = (long long)l1 * P.ld + col;
                if (kTT && P.TT) P.TT[idx] = att[i];
                if (kA2) {
                    const double sd = P.isd[l1] * P.isd[l2];
                    if (kTE && P.TE) P.TE[idx] = ate[i] * (0.5 * sd);
                    if (kEE && P.EE) P.EE[idx] = aee[i] * (0.25 * sd * sd);
                }
            }
        }
    }
}

template <int R, int MASK>
cudaError_t launch_one(const SweepParams &P, int total_tiles, cudaStream_t st)
{
    if (total_tiles <= 0) return cudaSuccess;
    sweep_kernel<R, MASK><<<total_tiles, SWEEP_THREADS, 0, st>>>(P);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_sweep(const SweepParams &P, int mask, int total_tiles, cudaStream_t st)
{
    switch (mask) {
        case M_TT: return launch_one<R_TT, M_TT>(P, total_tiles, st);
        case M_TE | M_EE | M_EB: return launch_one<R_POL, M_TE | M_EE | M_EB>(P, total_tiles, st);
        case M_TT | M_TE | M_EE | M_EB: return launch_one<R_POL, M_TT | M_TE | M_EE | M_EB>(P, total_tiles, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace tj
