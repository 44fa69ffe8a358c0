// tj_small.cu -- the whole hot path (a2-a6) in ONE launch, for small lmax.
//
// Below a few hundred multipoles a coupling call is a few microseconds of arithmetic, and the three launches of the
// general path (prepare -> staged sweep -> writer), its scratch allocation and the start-up latency of the bulk-copy
// pipeline cost ten times that (config 0, lmax = 256: 45-58 us).  Here every table the method needs fits in shared
// memory, so one kernel does everything: each CTA pre-folds the windows (step a2: W' = (2l+1) W / 4 pi) and copies
// the lookup tables (step a1's output) into its shared memory, every thread then sweeps the R pairs (a+i, c-i) of one
// anti-diagonal (step a4: they share s, l3, h[s-t] g[t] and the windows per step) and stores K = (2 l2+1) Xi and its
// mirror (2 l1+1) Xi directly (steps a5-a6).  No scratch, no tile list, no second pass.
//
// The arithmetic per entry is, operation for operation and in the same order of l3, that of tj_sweep.cu /
// tj_writer.cu, so results are bit-identical to the general path.  tests/test_zz_no_alloc.py holds the
// two against each other at the same sizes (tj_coupling_pol_static always runs the general path); the band-limited,
// row-block, batched and host-buffer tests of tests/test_gpu_parity.py compare general-path variants with
// general-path calls above LMAX_SMALL (or this kernel with itself below it), not the two with each other.
#include "tj_internal.cuh"

namespace tj {
namespace {

constexpr int SM_THREADS = 128;
// pairs per thread: 2 up to lmax = SM_LMAX_R2, 4 above.  A small problem is bound by its longest thread (one warp per
// scheduler, ~30 cycles of FP64 latency per dependent operation), a larger one by the instruction count (measured
// per call, all five blocks: lmax 256: 20.9 us with R = 2, 24.9 with R = 4; lmax 640: 124 vs 108 us).
constexpr int SM_LMAX_R2 = 400;
constexpr int SM_U = 4;      // steps per block: operands of U steps are loaded before their arithmetic starts
constexpr int SM_GL = 32;    // zero doubles below index 0 of every shared table (indices reach -2(R-1)-2U, windows -2(R+2U))
constexpr int SM_GH = 16;    // and above the last entry (h[s-t] reaches pmax + R/2)
static_assert(2 * (4 + 2 * SM_U) <= SM_GL, "low guard");

struct SmallParams {
    const double *g, *ginv, *h, *gA, *gB, *isd;   // the handle's tables (index 0)
    const double *Wtt, *Wtp, *Wpp;                // raw windows, nW entries (NULL: block not requested)
    double *TT, *TE, *EE, *BB, *EB;               // outputs, (lmax+1)^2 (NULL: not stored)
    int lmax, l3max, pmax, nW;
};

// One CTA: rows a..a+R-1 (a = blockIdx.y R), SM_THREADS columns, ONE parity of J (blockIdx.z = 1: odd J, the EB
// block; 0: even J, TT/TE/EE/BB) -- the two branches share nothing but the pair, and a small problem is bound by the
// length of its longest thread, so they run side by side.
template <int MASK, int R>
__global__ void __launch_bounds__(SM_THREADS) small_kernel(const __grid_constant__ SmallParams P)
{
    constexpr bool kTT = (MASK & M_TT) != 0, kPol = (MASK & (M_TE | M_EE | M_EB)) != 0;
    constexpr int U = SM_U;
    constexpr bool SWP = !kPol;    // TT alone: the products of block k+1 are formed while the chains of block k run
    extern __shared__ __align__(16) double sm[];
    const int np = SM_GL + P.pmax + 1 + SM_GH, nl = SM_GL + P.l3max + 1 + SM_GH;
    const bool odd = kPol && blockIdx.z == 1;
    const int a = (int)blockIdx.y * R;
    const int c = a + (int)(blockIdx.x * SM_THREADS + threadIdx.x);
    if (a + (int)(blockIdx.x * SM_THREADS) - (R - 1) > P.lmax) return;   // whole CTA beyond the last column

    // ---- shared tables.  even J: g, h, W'_TT, W'_TP, W'_PP;  odd J: gA (ring factors), gB, ginv, W'_PP ----
    double *sa = sm + SM_GL, *sb = sa + np, *sc = sb + np;   // ring table; step factor; 1/(J+1)g(p) resp. 1/g(p)
    double *sw0 = sc + np, *sw1 = sw0 + nl, *sw2 = sw1 + nl, *su = sw2 + nl;   // windows; u_l = l(l+1)
    // the tables come by bulk copy, guards included (the handle's tables carry zero guard bands of their own, and
    // np is even with index -SM_GL 16-byte aligned); the threads pre-fold the windows meanwhile
    __shared__ __align__(8) unsigned long long bar;
    const uint32_t bar_s = (uint32_t)__cvta_generic_to_shared(&bar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const uint32_t bytes = (uint32_t)np * 8u;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_s), "r"(bytes * (odd ? 3u : 2u)) : "memory");
        auto fetch = [&](double *dst, const double *src) {
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             (uint32_t)__cvta_generic_to_shared(dst - SM_GL)),
                         "l"(src - SM_GL), "r"(bytes), "r"(bar_s)
                         : "memory");
        };
        if (odd) { fetch(sa, P.gA); fetch(sb, P.gB); fetch(sc, P.ginv); }
        else { fetch(sa, P.g); fetch(sc, P.h); }
    }
    const double inv4pi = 0.079577471545947667884441881686257181;  // 1/(4 pi)
    constexpr int PF = 4;   // window entries per thread and pass: all loads of a pass are in flight together
    for (int l0 = -SM_GL + (int)threadIdx.x; l0 < P.l3max + 1 + SM_GH; l0 += PF * SM_THREADS) {
        double x0[PF], x1[PF], x2[PF];
#pragma unroll
        for (int k = 0; k < PF; ++k) {
            const int l = l0 + k * SM_THREADS;
            const bool in = l >= 0 && l < P.nW && l <= P.l3max;
            x0[k] = (in && (odd ? P.Wpp != nullptr : (kTT && P.Wtt != nullptr))) ? (odd ? P.Wpp[l] : P.Wtt[l]) : 0.0;
            x1[k] = (in && !odd && kPol && P.Wtp != nullptr) ? P.Wtp[l] : 0.0;
            x2[k] = (in && !odd && kPol && P.Wpp != nullptr) ? P.Wpp[l] : 0.0;
        }
#pragma unroll
        for (int k = 0; k < PF; ++k) {
            const int l = l0 + k * SM_THREADS;
            if (l >= P.l3max + 1 + SM_GH) break;
            const double f = __dmul_rn(2.0 * (double)l + 1.0, inv4pi);          // as prepare_kernel
            if (kPol) su[l] = (double)l * ((double)l + 1.0);
            const bool in = l >= 0 && l < P.nW && l <= P.l3max;                  // outside: +0.0, as prepare_kernel
            if (odd || kTT) sw0[l] = in ? __dmul_rn(f, x0[k]) : 0.0;
            if (!odd && kPol) { sw1[l] = in ? __dmul_rn(f, x1[k]) : 0.0; sw2[l] = in ? __dmul_rn(f, x2[k]) : 0.0; }
        }
    }
    __syncthreads();   // windows written, barrier initialised
    {
        uint32_t done;
        do {
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(done) : "r"(bar_s), "r"(0u) : "memory");
        } while (!done);
    }
    if (c - (R - 1) > P.lmax) return;   // no pair of this thread has l2 <= lmax
    if (!odd) sb = sa;                  // even J: the step factor g[t] comes from the same table as the ring factors

    const int s = a + c;
    const int t_end = a + R - 1;
    double c12[R], kk[R];
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const double l1 = (double)(a + i), l2 = (double)(c - i);
        const double u1 = l1 * (l1 + 1.0), u2 = l2 * (l2 + 1.0);
        c12[i] = odd ? u1 + u2 - 2.0 : u1 + u2 - 1.0;   // odd: e = u3 - c12; even: d1 = d+1 = u3 - c12
        kk[i] = __fma_rn(2.0 * u1, u2, 1.0);
    }
    double acc0[R], acc1[R], acc2[R];   // odd: S_EB in acc0;  even: S_TT, S_TE, S_EE
#pragma unroll
    for (int i = 0; i < R; ++i) { acc0[i] = 0.0; acc1[i] = 0.0; acc2[i] = 0.0; }

    // l3 = s-2t-par <= l3max.  Steps run in blocks of U: every operand of a block is loaded before its arithmetic
    // starts, and the arithmetic is operation-major over the U x R terms of the block (every level is U*R independent
    // instructions): one warp per scheduler is the common case here, and a dependent FP64 operation costs ~30 cycles,
    // so latency, not issue, is what counts.  Only the accumulations are ordered (in t).  With SWP (TT alone) the
    // products of block k+1 are formed while the accumulation chains of block k run (software pipelining by one
    // block: lmax = 256 10.6 -> 8.3 us; for the polarised blocks the second set of products costs more registers
    // than the overlap gains).  The walk is extended past t_end to whole blocks -- there the ring factors are the
    // zero guards and add exact zeros -- and SWP prepares one block more, which is never accumulated.
    const int par = odd ? 1 : 0;
    int tb = s - par - P.l3max;
    tb = tb > 0 ? (tb + 1) >> 1 : 0;
    if (SWP) {   // TT alone: two sets of block products (q0 = W' h g[t], r) alternate
        struct Prod { double q0[U], r[U][R]; };
        auto prepare = [&](int t0, Prod &B) {
            double vh[U], vg[U], vb[U][R];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int t = t0 + u;
                vh[u] = sc[s - t];
                vg[u] = sb[t];
                B.q0[u] = sw0[s - 2 * t];
#pragma unroll
                for (int i = 0; i < R; ++i) { B.r[u][i] = sa[a + i - t]; vb[u][i] = sa[c - i - t]; }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) vh[u] = __dmul_rn(vh[u], vg[u]);                      // hg
#pragma unroll
            for (int u = 0; u < U; ++u) B.q0[u] = __dmul_rn(B.q0[u], vh[u]);                  // q0
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) B.r[u][i] = __dmul_rn(B.r[u][i], vb[u][i]);       // r
        };
        auto accumulate = [&](const Prod &B) {
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) acc0[i] = __fma_rn(B.r[u][i], B.q0[u], acc0[i]);
        };
        Prod A, B;
        prepare(tb, A);
        for (int t0 = tb; t0 <= t_end; t0 += 2 * U) {
            prepare(t0 + U, B);
            accumulate(A);
            if (t0 + U > t_end) break;
            prepare(t0 + 2 * U, A);
            accumulate(B);
        }
    } else {
    for (int t0 = tb; t0 <= t_end; t0 += U) {
        double vh[U], vg[U], w0[U], w1[U], w2[U], c3[U], r[U][R], vb[U][R];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int t = t0 + u, l3 = s - 2 * t - par;
            vh[u] = sc[s - t];
            vg[u] = sb[t];
            w0[u] = (odd || kTT) ? sw0[l3] : 0.0;
            w1[u] = (!odd && kPol) ? sw1[l3] : 0.0;
            w2[u] = (!odd && kPol) ? sw2[l3] : 0.0;
            c3[u] = kPol ? su[l3] : 0.0;
#pragma unroll
            for (int i = 0; i < R; ++i) { r[u][i] = sa[a + i - t]; vb[u][i] = sa[c - i - t]; }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) vh[u] = __dmul_rn(vh[u], vg[u]);                      // hg
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int i = 0; i < R; ++i) r[u][i] = __dmul_rn(r[u][i], vb[u][i]);           // r
        if (odd) {
#pragma unroll
            for (int u = 0; u < U; ++u) w0[u] = __dmul_rn(w0[u], vh[u]);                  // q3
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) vb[u][i] = __dsub_rn(c3[u], c12[i]);          // e
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) r[u][i] = __dmul_rn(r[u][i], vb[u][i]);
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) r[u][i] = __dmul_rn(r[u][i], vb[u][i]);
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < R; ++i) acc0[i] = __fma_rn(r[u][i], w0[u], acc0[i]);
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (kTT) w0[u] = __dmul_rn(w0[u], vh[u]);                                 // q0, q1, q2
                if (kPol) { w1[u] = __dmul_rn(w1[u], vh[u]); w2[u] = __dmul_rn(w2[u], vh[u]); }
            }
            if (kTT) {
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) acc0[i] = __fma_rn(r[u][i], w0[u], acc0[i]);
            }
            if (kPol) {
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) vb[u][i] = __dsub_rn(c3[u], c12[i]);      // d1
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) vb[u][i] = __fma_rn(vb[u][i], vb[u][i], -kk[i]);   // A2
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) r[u][i] = __dmul_rn(r[u][i], vb[u][i]);   // rA
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) acc1[i] = __fma_rn(r[u][i], w1[u], acc1[i]);
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) r[u][i] = __dmul_rn(r[u][i], vb[u][i]);   // rAA
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int i = 0; i < R; ++i) acc2[i] = __fma_rn(r[u][i], w2[u], acc2[i]);
            }
        }
    }
    }

    // ---- scale, mirror, store (steps a5 + a6) ----
    const long long N = (long long)P.lmax + 1;
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int l1 = a + i, l2 = c - i;
        if (l2 < l1 || l2 > P.lmax) continue;
        const double w2c = (double)(2 * l2 + 1), w1c = (double)(2 * l1 + 1);
        const long long d = (long long)l1 * N + l2, m = (long long)l2 * N + l1;
        auto put = [&](double *M, double xi) {
            if (M == nullptr) return;
            M[d] = xi * w2c;
            if (l1 != l2) M[m] = xi * w1c;
        };
        const double sd = kPol ? P.isd[l1] * P.isd[l2] : 0.0;
        if (odd) {
            put(P.EB, acc0[i] * (0.25 * sd * sd));
        } else {
            if (kTT) put(P.TT, acc0[i]);
            if (kPol) {
                const double xee = acc2[i] * (0.25 * sd * sd);
                put(P.TE, acc1[i] * (0.5 * sd));
                put(P.EE, xee);
                put(P.BB, xee);
            }
        }
    }
}

template <int MASK, int R> cudaError_t launch_small_one(const SmallParams &P, cudaStream_t st)
{
    constexpr bool kPol = MASK != M_TT;
    const size_t smem = small_smem_bytes((P.pmax - 1) / 2, P.l3max);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(small_kernel<MASK, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((unsigned)((P.lmax + R - 1) / SM_THREADS + 1), (unsigned)num_bands(P.lmax, R), kPol ? 2 : 1);
    g_last_sweep = SweepGeometry{R, MASK, 0, 0, 0, 1, 2, 0, 0, (int)(grid.x * grid.y * grid.z)};
    small_kernel<MASK, R><<<grid, SM_THREADS, smem, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}
template <int MASK> cudaError_t launch_small_r(const SmallParams &P, cudaStream_t st)
{
    return P.lmax <= SM_LMAX_R2 ? launch_small_one<MASK, 2>(P, st) : launch_small_one<MASK, 4>(P, st);
}

}  // namespace

// shared memory one CTA of the single-launch path needs for the given sizes (bytes; the API compares it with the limit)
size_t small_smem_bytes(int lmax, int l3max)
{
    const size_t np = SM_GL + (size_t)(2 * lmax + 1) + 1 + SM_GH, nl = SM_GL + (size_t)l3max + 1 + SM_GH;
    return 8 * (3 * np + 4 * nl);
}

cudaError_t launch_small(const Tables &T, int mask, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                         double *TT, double *TE, double *EE, double *BB, double *EB, cudaStream_t st)
{
    SmallParams P;
    P.g = T.g; P.ginv = T.ginv; P.h = T.h; P.gA = T.gA; P.gB = T.gB; P.isd = T.isd;
    P.Wtt = d_Wtt; P.Wtp = d_Wtp; P.Wpp = d_Wpp;
    P.TT = TT; P.TE = TE; P.EE = EE; P.BB = BB; P.EB = EB;
    P.lmax = T.lmax; P.l3max = T.l3max; P.pmax = T.pmax; P.nW = nW;
    constexpr int POL = M_TE | M_EE | M_EB;
    switch (mask) {
        case M_TT: return launch_small_r<M_TT>(P, st);
        case POL: return launch_small_r<POL>(P, st);
        case M_TT | POL: return launch_small_r<M_TT | POL>(P, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace tj
