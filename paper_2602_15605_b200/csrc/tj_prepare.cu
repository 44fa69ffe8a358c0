// tj_prepare.cu -- per-call preparation kernel: window pre-fold (step a2) + tile schedule (step a3).
//
// a2: W'_X[l] = (2l+1) W_X[l] / (4 pi) for l = 0..nW-1, zero in the guard bands and for l > l3max
//     (Eq. 3: the (2 j3+1) W~ factor and the 1/(4 pi); the sum simply stops
//     where the window stops).
//     The polarised sweeps read the windows as PAIRS, wA[l] = (W'_TT, W'_TP)[l] and wB[l] = (W'_PP, u_l)[l]
//     (u_l = l(l+1) rides along because the sweep needs it at the same index), written here as well.
// a3: the upper triangle is cut into row bands of R rows; band `b` needs band_num_tiles(b) CTAs of
//     SWEEP_THREADS columns.  Work per CTA grows with the band's row index (the sweep has min(l1,l2)+1
//     steps), so bands are issued in DESCENDING row order: CTA k of the 1-D grid finds its band by a
//     binary search in the exclusive prefix tile_start[] built here (largest-first dispatch, the
//     hardware CTA scheduler is the dynamic queue; PAPER.md:236 "dynamic scheduling", :259 "linearized
//     triangular iteration").
#include "tj_internal.cuh"

namespace tj {
namespace {

constexpr int PREP_THREADS = 256;

__global__ void __launch_bounds__(PREP_THREADS)
prepare_kernel(const double *__restrict__ Wtt, const double *__restrict__ Wtp, const double *__restrict__ Wpp, int nW,
               double *wtt, double *wtp, double *wpp, double2 *wA, double2 *wB, const double *__restrict__ u3,
               int nl_alloc,
               int *tile_start, int lmax, int l3max_eff, int R, int banded, int row_lo, int row_hi)
{
    const double inv4pi = 0.079577471545947667884441881686257181;  // 1/(4 pi)
    // band-limited calls (diagonal tiling) never read beyond l3max + 2 (R + TS) + 64 < l3max + GUARD_HI
    const int lo = -GUARD_LO, hi = banded ? min(nl_alloc - GUARD_LO, l3max_eff + GUARD_HI) : nl_alloc - GUARD_LO;
    for (int l = lo + (int)(blockIdx.x * PREP_THREADS + threadIdx.x); l < hi; l += (int)(gridDim.x * PREP_THREADS)) {
        const bool in = (l >= 0 && l < nW && l <= l3max_eff);
        const double f = (2.0 * (double)l + 1.0) * inv4pi;
        if (wtt) wtt[l] = (in && Wtt) ? f * Wtt[l] : 0.0;
        if (wtp) wtp[l] = (in && Wtp) ? f * Wtp[l] : 0.0;
        if (wpp) wpp[l] = (in && Wpp) ? f * Wpp[l] : 0.0;
        // packed pairs for the polarised sweeps: one 16-byte shared-memory load per pair and step
        wA[l] = make_double2((in && Wtt) ? f * Wtt[l] : 0.0, (in && Wtp) ? f * Wtp[l] : 0.0);
        wB[l] = make_double2((in && Wpp) ? f * Wpp[l] : 0.0, u3[l]);
    }
    if (blockIdx.x != 0 || banded) return;   // the diagonal tiling decodes its tiles in closed form

    // ---- tile schedule: exclusive prefix over bands in descending order ----
    __shared__ int part[PREP_THREADS];
    const int nb = num_bands(lmax, R);
    const int chunk = (nb + PREP_THREADS - 1) / PREP_THREADS;
    const int k0 = threadIdx.x * chunk, k1 = min(nb, k0 + chunk);
    int sum = 0;
    for (int k = k0; k < k1; ++k) sum += band_num_tiles(lmax, l3max_eff, R, nb - 1 - k, banded != 0, row_lo, row_hi);
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int i = 0; i < PREP_THREADS; ++i) { int v = part[i]; part[i] = run; run += v; }
        tile_start[nb] = run;
    }
    __syncthreads();
    int run = part[threadIdx.x];
    for (int k = k0; k < k1; ++k) {
        tile_start[k] = run;
        run += band_num_tiles(lmax, l3max_eff, R, nb - 1 - k, banded != 0, row_lo, row_hi);
    }
}

}  // namespace

cudaError_t launch_prepare(const Tables &T, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                           double *wtt, double *wtp, double *wpp, double *wA, double *wB, int *tile_start, int R,
                           int l3max_eff, bool banded, int row_lo, int row_hi, cudaStream_t st)
{
    const int nl = banded ? min(T.nl_alloc, GUARD_LO + l3max_eff + GUARD_HI) : T.nl_alloc;
    int nb = (nl + PREP_THREADS - 1) / PREP_THREADS;
    if (nb > 64) nb = 64;
    prepare_kernel<<<nb, PREP_THREADS, 0, st>>>(d_Wtt, d_Wtp, d_Wpp, nW, wtt, wtp, wpp, (double2 *)wA, (double2 *)wB,
                                                 T.u3, T.nl_alloc, tile_start,
                                                 T.lmax, l3max_eff, R, banded ? 1 : 0, row_lo, row_hi);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace tj
