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
//   Xi_TT = S_TT,  Xi_TE = S_TE/(2 sqrt D),  Xi_EE = S_EE/(4D),  Xi_EB = S_EB/(4D),  D = D_l1 D_l2.
//
// Mapping to the machine.  A thread owns R pairs on ONE anti-diagonal,
// (l1,l2) = (a+i, c-i), so s, l3, h[s-t] g[t], the three W'[l3] and u_l3 are per-THREAD values per step,
// and the two per-pair table factors g[a+i-t], g[c-i-t] slide through two R-deep register rings: each
// step reads ONE new element per ring.  Lanes run along c.  Steps outside a pair's triangle (or beyond
// l3max) hit the zero guard bands of the tables / windows and add exact zeros, so a warp runs one
// branch-free t range.
//
// Where the per-step table values come from: shared memory, filled by the bulk-copy engine
// (cp.async.bulk + mbarrier), one private double-buffered pipeline PER WARP.  A warp walks its t range in
// STAGES of TS steps.  For one stage every value the warp will read is a contiguous slice of a table:
//
//     row ring      g [a - t]           TS          doubles   (broadcast)
//     step factor   g [t]               TS          doubles   (broadcast)
//     column ring   g [cw-R+1+j - t]    TS+31       doubles   (lane j)
//     1/(J+1)g(p)   h [a+cw+j - t]      TS+31       doubles
//     windows, u3   pairs (W'_TT, W'_TP)[a+cw+j - 2t] and (W'_PP, u)[a+cw+j - 2t]    2(TS-1)+32 pairs each
//                   (written as pairs by prepare_kernel; the TT-only sweep reads the plain W'_TT array)
//
// (odd-J branch: gA, gB, gA, ginv and the (W'_PP, u) pairs at l3 = s-2t-1).  Lane 0 asks the copy engine for
// the slices of stage k+2 as soon as the warp has finished stage k; the copies land while the warp computes
// stage k+1, and completion is signalled through the buffer's mbarrier (transaction bytes).  The inner
// loop then reads shared memory only: no L1 miss can stall it, an address is one 32-bit register plus an
// immediate, and warps are independent of each other -- a CTA is ONE warp (tj_internal.cuh), so that
// everything the producer computes derives from blockIdx and stays in the uniform datapath.
//
// Issue model (measured): with the FP64 pipe busy a scheduler issues one warp instruction
// per ~2 cycles whatever its type, so the time of this kernel is proportional to its instruction count.
// Hence: as many pairs per thread as registers allow (R = 12 for dense sweeps), 16-byte loads where two
// values sit side by side (window pairs; the step factor g[t] of two steps), long stages, and, with PIPE,
// the TE/EE accumulations of step t issued at the start of step t+1, when all their inputs are long ready
// (measured 0.5 % better than undeferred).
//
// Bulk copies need 16-byte aligned source, destination and size; table slices start at any double, so a slice
// whose first index is odd is fetched from the even index below it and the consumers add that parity `e` to
// their offsets.  Stages advance by TS (even), so `e` is fixed per array for the whole walk.
#include "tj_internal.cuh"

namespace tj {
namespace {

// steps per stage (a multiple of R, even): long stages amortise the stage turn-over (measured at lmax = 10^4 with
// 4-warp CTAs: TS = 24 148.8 ms, 48 143.4 ms, 96 141.7 ms; at lmax = 2000 96 is 1-1.6 % better than 48 as well, now
// that the last stage is cut at the band's last block)
constexpr int TS_DENSE = 96;      // dense polarised sweeps
constexpr int TS_SPIN1 = 96;      // spin-1 sweeps (measured at lmax = 10^4: 48: 100.24 ms per call, 96: 99.39 ms; lmax = 2000: 0.970 / 0.957 ms)
constexpr int TS_BAND = 64;       // band-limited sweeps (measured at config 4: 32: 0.3444 ms, 48: 0.3416, 64: 0.3417, 96: 0.3508)
constexpr bool PIPE_DENSE = true; // TE/EE accumulations of step t issued at the start of step t+1
constexpr int NBUF = 2;   // buffers per warp
constexpr int PAD = 2;    // doubles in front of each slice: the software-pipelined read of "step TS" lands here

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// capacities (doubles, all even) of the slices inside one stage buffer
template <int TS, int NW, bool PK, bool DIAG> struct Lay {
    static constexpr int CA = PAD + TS + 2;            // row ring / step factor
    static constexpr int CB = PAD + TS + 32 + 2;       // column ring / h
    static constexpr int CW = PAD + 2 * TS + 32 + 2;   // windows, u3
    // the diagonal tiling reads the step factor per lane (TS+31 values) and the column ring as a broadcast
    static constexpr int OA = 0, OG = OA + CA, OB = OG + (DIAG ? CB : CA), OH = OB + (DIAG ? CA : CB);
    static constexpr int OW0 = OH + CB;                // TT-only sweep: the plain W'_TT slices, one per window set
    // polarised sweeps read the windows as pairs (prepare_kernel): (W'_TT, W'_TP)[l] and (W'_PP, u_l)[l], one array
    // of 2*CW doubles per window set each, in the same region (the TT-only sweep keeps the plain W'_TT slot OW0)
    static constexpr int OPA = OH + CB, OPB = OPA + NW * 2 * CW;
    static constexpr int BUFD = PK ? OPB + NW * 2 * CW : OW0 + NW * CW;   // doubles per buffer
};

// one slice: n doubles starting at table index i0 (any parity) -> buffer offset off (+PAD)
__device__ __forceinline__ uint32_t slice(uint32_t buf, int off, const double *tab, int i0, int n, uint32_t bar)
{
    const int ie = i0 & ~1;                 // even index at or below i0 (two's complement: also for i0 < 0)
    const int cnt = (n + (i0 - ie) + 1) & ~1;
    bulk_g2s(buf + (uint32_t)(off + PAD) * 8u, tab + ie, (uint32_t)cnt * 8u, bar);
    return (uint32_t)cnt * 8u;
}
__device__ __forceinline__ int slice_bytes(int i0, int n)
{
    const int ie = i0 & ~1;
    return ((n + (i0 - ie) + 1) & ~1) * 8;
}

// SPIN = 2: the paper's blocks (above).  SPIN = 1: the same sweep with the (l1 l2 l3;-1 1 0) symbol
// (DESIGN.md 3 item 6):  even step: (-1 1 0) = X d / (2 sqrt(u1 u2)), d = u3-u1-u2, so the
// "TE" slot accumulates W' X^2 d and the "EE" slot W' X^2 d^2; odd step: (-1 1 0)^2 = Z^2 / (4 u1 u2), so the "EB"
// slot accumulates W' Z^2; P.isd then holds 1/sqrt(u_l) and the epilogue scales are the same expressions.
template <int R, int MASK, int TS, int MINB, bool PIPE, int NW, int SPIN, bool ROWS, bool DIAG>
__global__ void __launch_bounds__(SWEEP_THREADS, MINB * (128 / SWEEP_THREADS)) sweep_tma_kernel(const __grid_constant__ SweepParams P)
{
    constexpr bool kTT = (MASK & M_TT) != 0, kTE = (MASK & M_TE) != 0, kEE = (MASK & M_EE) != 0,
                   kEB = (MASK & M_EB) != 0;
    constexpr bool kEven = kTT || kTE || kEE;
    constexpr bool kA2 = kTE || kEE;
    constexpr bool kPk = MASK != M_TT;   // windows and u3 come as pairs (wA, wB)
    using L = Lay<TS, NW, kPk, DIAG>;
    constexpr int NWL = 2 * (TS - 1) + 32;   // l3 values one stage of a warp covers
    // diagonal tiling: the step factor g[t+j] is the per-lane slice and the column ring g[c-i-t] a broadcast
    constexpr int NG = DIAG ? TS + 31 : TS, NB = DIAG ? TS : TS + 31;
    constexpr int LG = DIAG ? 1 : 0, LB = DIAG ? 0 : 1;   // which of the two a lane offsets by its index
    static_assert(TS % R == 0 && TS % 2 == 0, "stage length: a multiple of R and even");
    static_assert(2 * (R + TS) + 8 <= GUARD_LO, "a warp reads down to index -2(R+TS) of a window: the low guard band must cover it");
    static_assert(R + 64 + 8 <= GUARD_HI, "columns up to lmax+R-1+31 and their sums a+c: the high guard band must cover them");
    static_assert(R % 2 == 0, "even R: every block of R steps starts at an even step, which aligns the paired loads of the step factor");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int NWARP = SWEEP_THREADS / 32;

    static_assert(!DIAG || (SWEEP_THREADS == 32 && NW == 1 && SPIN == 2 && !ROWS && !PIPE), "diagonal tiling: one warp, one window set, undeferred accumulation");
    const int lane = (int)(threadIdx.x & 31), warp = SWEEP_THREADS == 32 ? 0 : (int)(threadIdx.x >> 5);   // 0: keeps the warp's addresses CTA-uniform
    int a, cw;   // lane 0's first row and column
    if (DIAG) {
        // ---- diagonal tiling (band-limited calls, tj_internal.cuh): tile = (delta group, diagonal block) ----
        const int grp = (int)blockIdx.x / P.nd, n = (int)blockIdx.x - grp * P.nd;
        a = 32 * n - (R - 1);
        cw = a + diag_d0(R, grp);
    } else {
        // ---- tile decode: binary search of blockIdx.x in the descending-band prefix ----
        const int tile = (int)blockIdx.x + P.tile_off;
        int lo = 0, hi = P.nbands;
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (__ldg(P.tile_start + mid) <= tile) lo = mid; else hi = mid;
        }
        const int band = P.nbands - 1 - lo;
        const int cb = tile - __ldg(P.tile_start + lo);
        a = band * R;
        cw = (ROWS ? band_c_lo(R, band, P.row_lo) : a) + cb * SWEEP_THREADS + warp * 32;   // first column of the warp
    }
    // the thread's pairs are (al+i, c-i).  Dense tiling: lanes run along the column, every lane has the rows a..a+R-1.
    // Diagonal tiling: lane j is lane 0 shifted by (j, j), and walks the steps t+j while lane 0 walks t, so that every
    // lane has the same number of steps; all table offsets below are lane 0's, the per-lane shift is in the slices.
    const int c = cw + lane;
    const int al = DIAG ? a + lane : a;
    const int sw = a + cw;                               // smallest s of the warp (diagonal tiling: lane 0's s)

    // a warp whose columns all lie beyond lmax has nothing to store
    if (cw - (R - 1) > P.lmax) return;

    double *const wbuf = reinterpret_cast<double *>(smem_raw) + warp * (NBUF * L::BUFD);
    const uint32_t wbuf_s = smem_u32(wbuf);
    const uint32_t bar_s = smem_u32(smem_raw) + (uint32_t)(NWARP * NBUF * L::BUFD) * 8u + (uint32_t)warp * (NBUF * 8u);
    if (lane == 0) {
#pragma unroll
        for (int b = 0; b < NBUF; ++b) mbar_init(bar_s + 8u * b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    // ---- the warp's walk: odd-J stages first, then even-J stages ----
    const int t_end = a + R - 1;   // last step any pair of the band can have
    int tbo = sw - 1 - P.l3max;    // odd:  l3 = s-2t-1 <= l3max
    // first steps rounded down to even (an extra step adds exact zeros): the step factor g[t] is then read two steps
    // per 16-byte load.  The result is then passed through an empty asm statement, so that the compiler can NOT prove
    // its parity and pair the row-ring loads too: those go into fixed ring registers and a paired load costs two
    // register moves.
    // Diagonal tiling: lane j starts j steps after lane 0, so lane 0 may start below 0 (the guard band of g[t] adds
    // exact zeros there) but not below -32: then every lane starts at or below its own first step max(0, .).
    // Then the first step moves further down so that the walk is whole blocks of R steps ENDING at the last step
    // (leading steps have l3 > l3max, where the prefolded windows are 0): in the last block pair i is live in step
    // u iff i >= u (even: t = a+u <= l1 = a+i; odd: t = a-1+u <= l1-1), and it runs in triangular form (below).
    int tbe = sw - P.l3max;        // even: l3 = s-2t   <= l3max
    const int t_end_o = DIAG ? t_end - 1 : t_end;   // odd branch: its last step is l1-1
    if (DIAG) {
        tbo = max((tbo + 1) >> 1, -32);
        tbo = t_end_o + 1 - R * ((t_end_o - tbo + R) / R);
        tbe = max((tbe + 1) >> 1, -32);
        tbe = t_end + 1 - R * ((t_end - tbe + R) / R);
    } else {
        tbo = tbo > 0 ? ((tbo + 1) >> 1) & ~1 : 0;
        tbe = tbe > 0 ? ((tbe + 1) >> 1) & ~1 : 0;
        asm("" : "+r"(tbo), "+r"(tbe));   // opaque to the optimiser from here on (see above)
    }
    const int nso = (kEB && tbo <= t_end_o) ? (t_end_o - tbo + TS) / TS : 0;
    const int nse = (kEven && tbe <= t_end) ? (t_end - tbe + TS) / TS : 0;
    const int ntot = nso + nse;

    // producer (lane 0): ask for every slice of global stage index q
    auto issue = [&](int q) {
        const int b = q % NBUF;
        const uint32_t buf = wbuf_s + (uint32_t)(b * L::BUFD) * 8u;
        const uint32_t bar = bar_s + 8u * b;
        if (q < nso) {
            const int t0 = tbo + q * TS, tl = t0 + TS - 1;
            uint32_t bytes = slice_bytes(a - tl, TS) + slice_bytes(t0, NG) + slice_bytes(cw - R + 1 - tl, NB) +
                             slice_bytes(sw - tl, TS + 31) + NW * (2 * NWL * 8);
            mbar_expect_tx(bar, bytes);
            slice(buf, L::OA, P.gA, a - tl, TS, bar);
            slice(buf, L::OG, P.gB, t0, NG, bar);
            slice(buf, L::OB, P.gA, cw - R + 1 - tl, NB, bar);
            slice(buf, L::OH, P.ginv, sw - tl, TS + 31, bar);
#pragma unroll
            for (int w = 0; w < NW; ++w)   // pairs (W'_PP, u_l), l = l3lo .. l3lo+NWL-1: always 16-byte aligned
                bulk_g2s(buf + (uint32_t)(L::OPB + w * 2 * L::CW + 2 * PAD) * 8u,
                         P.wB + w * P.wstride + 2 * (long long)(sw - 2 * tl - 1), 2 * NWL * 8, bar);
        } else {
            const int t0 = tbe + (q - nso) * TS, tl = t0 + TS - 1;
            uint32_t bytes = slice_bytes(a - tl, TS) + slice_bytes(t0, NG) + slice_bytes(cw - R + 1 - tl, NB) +
                             slice_bytes(sw - tl, TS + 31) +
                             (kPk ? NW * 2 * (2 * NWL * 8) : NW * slice_bytes(sw - 2 * tl, NWL));
            mbar_expect_tx(bar, bytes);
            slice(buf, L::OA, P.g, a - tl, TS, bar);
            slice(buf, L::OG, P.g, t0, NG, bar);
            slice(buf, L::OB, P.g, cw - R + 1 - tl, NB, bar);
            slice(buf, L::OH, P.h, sw - tl, TS + 31, bar);
            if (kPk) {
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    const long long o = w * P.wstride + 2 * (long long)(sw - 2 * tl);
                    bulk_g2s(buf + (uint32_t)(L::OPA + w * 2 * L::CW + 2 * PAD) * 8u, P.wA + o, 2 * NWL * 8, bar);
                    bulk_g2s(buf + (uint32_t)(L::OPB + w * 2 * L::CW + 2 * PAD) * 8u, P.wB + o, 2 * NWL * 8, bar);
                }
            } else {
#pragma unroll
                for (int w = 0; w < NW; ++w)
                    slice(buf, L::OW0 + w * L::CW, P.wtt + w * P.wstride, sw - 2 * tl, NWL, bar);
            }
        }
    };
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NBUF; ++q)
            if (q < ntot) issue(q);
    }

    // ---- per-pair constants ----
    double c12[R], kk[R];
    if (kA2 || kEB) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double l1 = (double)(al + i), l2 = (double)(c - i);
            const double u1 = l1 * (l1 + 1.0), u2 = l2 * (l2 + 1.0);
            c12[i] = SPIN == 2 ? u1 + u2 - 2.0 : u1 + u2 - 1.0;   // odd branch: e = u3 - c12 (spin 1: unused)
            kk[i] = __fma_rn(2.0 * u1, u2, 1.0);     // even branch: A2 = d1^2 - kk (spin 1: unused)
        }
    }

    int q = 0;   // global stage index

    // =========================== odd-J branch: EB ===========================
    if (kEB) {
        double acc[NW][R];
#pragma unroll
        for (int w = 0; w < NW; ++w)
#pragma unroll
            for (int i = 0; i < R; ++i) acc[w][i] = 0.0;
        if (nso > 0) {
            double wa[R], wb[R];
            {   // ring start-up straight from global memory (once per warp)
                const double *pa = P.gA + (a - tbo);
                const double *pb = P.gA + (c - LG * lane - R + 1 - tbo);
#pragma unroll
                for (int k = 1; k < R; ++k) wa[k] = __ldg(pa + k);
#pragma unroll
                for (int i = 0; i < R - 1; ++i) wb[(R - i) % R] = __ldg(pb + (R - 1 - i));
            }
            // consumer offsets: parity of each slice's first index is the same in every stage (TS even)
            const int tl0 = tbo + TS - 1;
            const int oa = L::OA + PAD + ((a - tl0) & 1) + (TS - 1);
            const int og = L::OG + PAD + (tbo & 1) + LG * lane;
            const int ob = L::OB + PAD + ((cw - R + 1 - tl0) & 1) + (TS - 1) + LB * lane;
            const int oh = L::OH + PAD + ((sw - tl0) & 1) + (TS - 1) + lane;
            for (int k = 0; k < nso; ++k, ++q) {
                // blocks of R steps this stage really has (the last stage is cut at the band's last step)
                const int nblk = min(TS / R, (t_end_o - (tbo + k * TS) + R) / R);
                const int b = q % NBUF;
                mbar_wait(bar_s + 8u * b, (uint32_t)((q / NBUF) & 1));
                const double *sb = wbuf + b * L::BUFD;
                const double *pa = sb + oa, *pg = sb + og, *pb = sb + ob, *ph = sb + oh;
                // pairs (W'_PP, u_l) at l3 = s-2t-1: lane's element of step t0+j is 2(TS-1)+lane-2j
                const double2 *pB = reinterpret_cast<const double2 *>(sb + L::OPB + 2 * PAD) + 2 * (TS - 1) + LB * lane;
                double xa = pa[0], xb = pb[0], xh = ph[0];
                double2 xg2 = DIAG ? make_double2(pg[0], 0.0) : *reinterpret_cast<const double2 *>(pg);   // g[t] of steps 0, 1
                double xg = xg2.x;
                double xw[NW], xu;
                {
                    const double2 v0 = pB[0];
                    xw[0] = v0.x; xu = v0.y;
#pragma unroll
                    for (int w = 1; w < NW; ++w) xw[w] = pB[w * L::CW].x;
                }
                // blocks of R steps (tj_sweep_odd_block.inc); TRI: the last block of a diagonal-tiling walk
                const bool tri_last = DIAG && k == nso - 1;
                const int nfull = tri_last ? nblk - 1 : nblk;
#pragma unroll 1
                for (int blk = 0; blk < nfull; ++blk) {
                    constexpr bool TRI = false;
#include "tj_sweep_odd_block.inc"
                    pa -= R; pb -= R; ph -= R; pg += R; pB -= 2 * R;
                }
                if constexpr (DIAG) {
                    if (tri_last) {
                        constexpr bool TRI = true;
#include "tj_sweep_odd_block.inc"
                    }
                }
                __syncwarp();
                if (lane == 0 && q + NBUF < ntot) issue(q + NBUF);
            }
        }
        // epilogue: Xi_EB = S_EB / (4 D)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int l1 = al + i, l2 = c - i;
            if (l2 >= l1 && l2 <= P.lmax && (P.lcut < 0 || l2 - l1 <= P.lcut) && (!DIAG || l1 >= 0)) {
                const double sd = P.isd[l1] * P.isd[l2];
                // diagonal tiling: Xi goes to the transposed scratch [l2-l1][l1] (lanes = consecutive l1: coalesced)
                const long long idx = DIAG ? (long long)(l2 - l1) * P.ld + l1
                                           : (long long)l1 * P.ld + (P.lcut < 0 ? (long long)l2 : (long long)(l2 - l1 + P.lcut));
                if (P.EB && !ROWS) {
#pragma unroll
                    for (int w = 0; w < NW; ++w)
                        P.EB[w * P.ostride + idx] = acc[w][i] * (0.25 * sd * sd);
                }
                if (P.EB && ROWS) {
                    // row block: a block of full rows has no in-place triangle to mirror, so the final values are stored
                    // here: K = (2 l2+1) Xi at [l1][l2] and (2 l1+1) Xi at [l2][l1], where inside
                    const double v = acc[0][i] * (0.25 * sd * sd);
                    if (l1 >= P.row_lo && l1 < P.row_hi) P.EB[(long long)(l1 - P.row_lo) * P.ld + l2] = v * (double)(2 * l2 + 1);
                    if (l2 >= P.row_lo && l2 < P.row_hi && l2 != l1) P.EB[(long long)(l2 - P.row_lo) * P.ld + l1] = v * (double)(2 * l1 + 1);
                }
            }
        }
    }

    // =========================== even-J branch: TT, TE, EE ===========================
    if (kEven) {
        double att[NW][kTT ? R : 1], ate[NW][kTE ? R : 1], aee[NW][kEE ? R : 1];
#pragma unroll
        for (int w = 0; w < NW; ++w)
#pragma unroll
            for (int i = 0; i < R; ++i) {
                if (kTT) att[w][i] = 0.0;
                if (kTE) ate[w][i] = 0.0;
                if (kEE) aee[w][i] = 0.0;
            }
        if (kA2) {
#pragma unroll
            for (int i = 0; i < R; ++i) c12[i] += 1.0;   // even branch: d1 = d+1 = u3 - (u1+u2-1)
        }
        if (nse > 0) {
            double wa[R], wb[R];
            {
                const double *pa = P.g + (a - tbe);
                const double *pb = P.g + (c - LG * lane - R + 1 - tbe);
#pragma unroll
                for (int k = 1; k < R; ++k) wa[k] = __ldg(pa + k);
#pragma unroll
                for (int i = 0; i < R - 1; ++i) wb[(R - i) % R] = __ldg(pb + (R - 1 - i));
            }
            // PIPE: products of step t are accumulated at the start of step t+1 (see the loop body)
            double rA[kTE ? R : 1], rAA[kEE ? R : 1], p1[NW], p2[NW];
#pragma unroll
            for (int w = 0; w < NW; ++w) { p1[w] = 0.0; p2[w] = 0.0; }
#pragma unroll
            for (int i = 0; i < R; ++i) { if (kTE) rA[i] = 0.0; if (kEE) rAA[i] = 0.0; }
            const int tl0 = tbe + TS - 1;
            const int oa = L::OA + PAD + ((a - tl0) & 1) + (TS - 1);
            const int og = L::OG + PAD + (tbe & 1) + LG * lane;
            const int ob = L::OB + PAD + ((cw - R + 1 - tl0) & 1) + (TS - 1) + LB * lane;
            const int oh = L::OH + PAD + ((sw - tl0) & 1) + (TS - 1) + lane;
            const int ow = PAD + ((sw - 2 * tl0) & 1) + 2 * (TS - 1) + LB * lane;
            for (int k = 0; k < nse; ++k, ++q) {
                const int nblk = min(TS / R, (t_end - (tbe + k * TS) + R) / R);
                const int b = q % NBUF;
                mbar_wait(bar_s + 8u * b, (uint32_t)((q / NBUF) & 1));
                const double *sb = wbuf + b * L::BUFD;
                const double *pa = sb + oa, *pg = sb + og, *pb = sb + ob, *ph = sb + oh;
                const double *pwtt = sb + L::OW0 + ow;   // TT-only sweep: plain W'_TT
                // polarised sweeps: pairs (W'_TT, W'_TP) and (W'_PP, u_l) at l3 = s-2t
                const double2 *pA = reinterpret_cast<const double2 *>(sb + L::OPA + 2 * PAD) + 2 * (TS - 1) + LB * lane;
                const double2 *pB = reinterpret_cast<const double2 *>(sb + L::OPB + 2 * PAD) + 2 * (TS - 1) + LB * lane;
                double xa = pa[0], xb = pb[0], xh = ph[0];
                double2 xg2 = DIAG ? make_double2(pg[0], 0.0) : *reinterpret_cast<const double2 *>(pg);   // g[t] of steps 0, 1
                double xg = xg2.x;
                double xtt[NW], xtp[NW], xpp[NW], xu = 0.0;
                // windows (and u3) of the step whose pair element sits `off` pairs from the lane's stage origin
                auto load_w = [&](int off) {
                    if (kPk) {
#pragma unroll
                        for (int w = 0; w < NW; ++w) {
                            const double2 va = pA[w * L::CW + off], vb = pB[w * L::CW + off];
                            xtt[w] = va.x; xtp[w] = va.y; xpp[w] = vb.x;
                            if (w == 0) xu = vb.y;
                        }
                    } else {
#pragma unroll
                        for (int w = 0; w < NW; ++w) xtt[w] = pwtt[w * L::CW + off];
                    }
                };
#pragma unroll
                for (int w = 0; w < NW; ++w) { xtt[w] = 0.0; xtp[w] = 0.0; xpp[w] = 0.0; }
                load_w(0);
                const bool tri_last = DIAG && k == nse - 1;
                const int nfull = tri_last ? nblk - 1 : nblk;
#pragma unroll 1
                for (int blk = 0; blk < nfull; ++blk) {
                    constexpr bool TRI = false;
#include "tj_sweep_even_block.inc"
                    pa -= R; pb -= R; ph -= R; pg += R;
                    pwtt -= 2 * R; pA -= 2 * R; pB -= 2 * R;
                }
                if constexpr (DIAG) {
                    if (tri_last) {   // the last block of the walk: pairs i < u are finished
                        constexpr bool TRI = true;
#include "tj_sweep_even_block.inc"
                    }
                }
                __syncwarp();
                if (lane == 0 && q + NBUF < ntot) issue(q + NBUF);
            }
            if (PIPE) {
#pragma unroll
            for (int i = 0; i < R; ++i) {   // the last step's products
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    if (kTE) ate[w][i] = __fma_rn(rA[i], p1[w], ate[w][i]);
                    if (kEE) aee[w][i] = __fma_rn(rAA[i], p2[w], aee[w][i]);
                }
            }
            }
        }
        // epilogue: Xi_TT = S_TT; Xi_TE = S_TE/(2 sqrt D); Xi_EE = S_EE/(4 D)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int l1 = al + i, l2 = c - i;
            if (l2 >= l1 && l2 <= P.lmax && (P.lcut < 0 || l2 - l1 <= P.lcut) && (!DIAG || l1 >= 0)) {
                const long long idx = DIAG ? (long long)(l2 - l1) * P.ld + l1
                                           : (long long)l1 * P.ld + (P.lcut < 0 ? (long long)l2 : (long long)(l2 - l1 + P.lcut));
                const double sd = kA2 ? P.isd[l1] * P.isd[l2] : 0.0;
                if (!ROWS) {
#pragma unroll
                    for (int w = 0; w < NW; ++w) {
                        const long long iw = idx + w * P.ostride;
                        if (kTT && P.TT) P.TT[iw] = att[w][i];
                        if (kTE && P.TE) P.TE[iw] = ate[w][i] * (0.5 * sd);
                        if (kEE && P.EE) P.EE[iw] = aee[w][i] * (0.25 * sd * sd);
                    }
                } else {   // row block (see the odd branch)
                    const bool in1 = l1 >= P.row_lo && l1 < P.row_hi, in2 = l2 >= P.row_lo && l2 < P.row_hi && l2 != l1;
                    const long long i1 = (long long)(l1 - P.row_lo) * P.ld + l2, i2 = (long long)(l2 - P.row_lo) * P.ld + l1;
                    const double w2 = (double)(2 * l2 + 1), w1 = (double)(2 * l1 + 1);   // K = (2 l2+1) Xi; mirrored: (2 l1+1) Xi
                    if (kTT && P.TT) { const double v = att[0][i]; if (in1) P.TT[i1] = v * w2; if (in2) P.TT[i2] = v * w1; }
                    if (kTE && P.TE) { const double v = ate[0][i] * (0.5 * sd); if (in1) P.TE[i1] = v * w2; if (in2) P.TE[i2] = v * w1; }
                    if (kEE && P.EE) {
                        const double v = aee[0][i] * (0.25 * sd * sd);
                        if (in1) { P.EE[i1] = v * w2; if (P.BB) P.BB[i1] = v * w2; }   // BB beside EE
                        if (in2) { P.EE[i2] = v * w1; if (P.BB) P.BB[i2] = v * w1; }
                    }
                }
            }
        }
    }
}

template <int R, int MASK, int TS, int MINB, bool PIPE, int NW = 1, int SPIN = 2, bool ROWS = false, bool DIAG = false>
cudaError_t launch_one(const SweepParams &P, int total_tiles, cudaStream_t st)
{
    g_last_sweep = SweepGeometry{R, MASK, TS, MINB, PIPE ? 1 : 0, NW, SPIN, ROWS ? 1 : 0, DIAG ? 1 : 0, total_tiles};
    if (total_tiles <= 0) return cudaSuccess;
    constexpr int NWARP = SWEEP_THREADS / 32;
    constexpr size_t smem = (size_t)NWARP * NBUF * Lay<TS, NW, MASK != M_TT, DIAG>::BUFD * 8 + (size_t)NWARP * NBUF * 8;
    if (smem > 48 * 1024) {   // opt-in beyond the default limit (per device, so not cached; one-warp CTAs stay below it)
        cudaError_t e = cudaFuncSetAttribute(sweep_tma_kernel<R, MASK, TS, MINB, PIPE, NW, SPIN, ROWS, DIAG>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    sweep_tma_kernel<R, MASK, TS, MINB, PIPE, NW, SPIN, ROWS, DIAG><<<total_tiles, SWEEP_THREADS, smem, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace

thread_local SweepGeometry g_last_sweep = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
thread_local long long g_launch_count = 0;

// Geometry per request: dense sweeps are long (up to lmax steps per pair), so the per-step
// overhead (prefactors, table reads) is spread over R = 12 pairs at 2 CTAs/SM with stages of 96 (48) steps;
// band-limited sweeps have <= lcut/2+1 steps per pair, so they keep R = 8 and stages of TS_BAND = 64 steps (TT alone: 32).
// Multi-window batching (nw window sets in one sweep): the geometric part of a term (r, A2, rA, rAA) is
// computed once and each window set adds 3 FMAs (1 in the odd branch); the accumulators of nw sets take the
// registers that R = 12 pairs use otherwise, hence R = 8 for nw = 2 and R = 6 for nw = 3.
int sweep_R(int mask, bool banded, int nw, int lmax, bool rows, int spin)
{
    if (mask == M_TT && nw > 1) return R_TT_MULTI;
    if (nw == 2) return R_MULTI2;
    if (nw == 3) return R_MULTI3;
    if (mask == M_TT) return banded ? R_TT_BAND : lmax >= LMAX_LONG ? R_TT_LONG : R_TT;
    if (banded) return R_POL_BAND;
    return (!rows && spin == 2 && lmax < LMAX_MID) ? R_POL_MID : R_POL;
}

cudaError_t launch_sweep(const SweepParams &P, int mask, int nw, int spin, int total_tiles, cudaStream_t st)
{
    constexpr int POL = M_TE | M_EE | M_EB, ALL = M_TT | POL;
    const bool banded = P.lcut >= 0;
    if (P.rows) {   // row blocks (tj_coupling_rows): dense, one window set, spin 2
        if (banded || nw != 1 || spin != 2) return cudaErrorInvalidValue;
        switch (mask) {
            case M_TT: return P.lmax >= LMAX_LONG ? launch_one<R_TT_LONG, M_TT, 64, 2, false, 1, 2, true>(P, total_tiles, st)
                                                  : launch_one<R_TT, M_TT, 48, 3, false, 1, 2, true>(P, total_tiles, st);
            case POL: return launch_one<R_POL, POL, TS_DENSE, 2, PIPE_DENSE, 1, 2, true>(P, total_tiles, st);
            case ALL: return launch_one<R_POL, ALL, TS_DENSE, 2, PIPE_DENSE, 1, 2, true>(P, total_tiles, st);
            default: return cudaErrorInvalidValue;
        }
    }
    if (spin == 1) {   // dense, one window set; TT-only requests use the spin-independent TT sweep below
        if (banded || nw != 1) return cudaErrorInvalidValue;
        if (mask == ALL) return launch_one<R_POL, ALL, TS_SPIN1, 2, PIPE_DENSE, 1, 1>(P, total_tiles, st);
        if (mask == POL) return launch_one<R_POL, POL, TS_SPIN1, 2, PIPE_DENSE, 1, 1>(P, total_tiles, st);
    }
    if (nw == 2 && !banded && mask == ALL) return launch_one<R_MULTI2, ALL, 48, 2, true, 2>(P, total_tiles, st);
    if (nw == 3 && !banded && mask == ALL) return launch_one<R_MULTI3, ALL, 36, 2, true, 3>(P, total_tiles, st);
    if (nw == 4 && !banded && mask == M_TT) return launch_one<R_TT_MULTI, M_TT, 48, 2, false, 4>(P, total_tiles, st);
    if (nw == 2 && !banded && mask == M_TT) return launch_one<R_TT_MULTI, M_TT, 48, 2, false, 2>(P, total_tiles, st);
    if (nw != 1) return cudaErrorInvalidValue;
    switch (mask) {
        case M_TT:
            return banded ? launch_one<R_TT_BAND, M_TT, 32, 3, false, 1, 2, false, true>(P, total_tiles, st)
                          : (P.lmax >= LMAX_LONG ? launch_one<R_TT_LONG, M_TT, 64, 2, false>(P, total_tiles, st)
                                                 : launch_one<R_TT, M_TT, 48, 3, false>(P, total_tiles, st));
        case POL:
            return banded ? launch_one<R_POL_BAND, POL, TS_BAND, 3, false, 1, 2, false, true>(P, total_tiles, st)
                          : (P.lmax >= LMAX_MID ? launch_one<R_POL, POL, TS_DENSE, 2, PIPE_DENSE>(P, total_tiles, st)
                                                       : launch_one<R_POL_MID, POL, TS_DENSE, 2, PIPE_DENSE>(P, total_tiles, st));
        case ALL:
            return banded ? launch_one<R_POL_BAND, ALL, TS_BAND, 3, false, 1, 2, false, true>(P, total_tiles, st)
                          : (P.lmax >= LMAX_MID ? launch_one<R_POL, ALL, TS_DENSE, 2, PIPE_DENSE>(P, total_tiles, st)
                                                       : launch_one<R_POL_MID, ALL, TS_DENSE, 2, PIPE_DENSE>(P, total_tiles, st));
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace tj
