// tj_internal.cuh -- shared declarations of libtj (not part of the public ABI).
//
// Notation follows PAPER.md / DESIGN.md: lmax, l3max, s = l1+l2, step t (even: l3 = s-2t,
// odd: l3 = s-2t-1), p = J/2, g(p) of Eq. 11, u_l = l(l+1), D_l = (l-1)l(l+1)(l+2).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/tj.h"

namespace tj {

// ---- table layout -------------------------------------------------------------------------
// Every p-indexed table (g, ginv, h, gA, gB) and every l3-indexed array (prefolded windows, u3)
// is allocated as [GUARD_LO + n + GUARD_HI] doubles and addressed through a pointer to index 0,
// so out-of-triangle steps read exact zeros instead of branching ("guard bands").
constexpr int GUARD_LO = 256;
constexpr int GUARD_HI = 768;

// ---- sweep tile geometry -------------------------------------------------------
// A thread owns R pairs on ONE anti-diagonal: (l1, l2) = (a+i, c-i), i = 0..R-1, a = band*R.
// Lanes run along c, so a warp covers rows a..a+R-1 and a skewed window of 32+R-1 columns.
// columns c per CTA.  ONE warp per CTA: a warp is an independent worker anyway (own stage pipeline, no CTA barrier),
// and with a single warp everything its producer needs (tile, stage, slice addresses, byte counts) derives from
// blockIdx alone, so ptxas keeps it in the uniform datapath instead of broadcasting five registers per bulk copy
// (measured at config 3: 137.3 ms with 128 threads, 136.3 with 64, 133.5 with 32).
constexpr int SWEEP_THREADS = 32;
// (the geometry constants below are the measured optima)
constexpr int R_POL = 12;           // pairs per thread, fused TT+TE+EE(+EB) sweep, dense storage, lmax >= LMAX_MID
constexpr int R_POL_MID = 8;        // same at lmax < LMAX_MID: shorter sweeps, fewer tiles -- smaller tiles balance better
                                    // (measured per call at lmax = 2000: R = 12 1.288 ms, 10 1.249, 8 1.227, 6 1.283)
constexpr int LMAX_MID = 2600;
constexpr int R_POL_BAND = 8;       // same, band-limited (short sweeps)
constexpr int R_TT = 16;            // pairs per thread, TT-only sweep (short sweeps)
constexpr int R_TT_BAND = 16;       // same, band-limited
constexpr int R_TT_LONG = 32;       // same, dense sweeps at lmax >= LMAX_LONG (measured at lmax = 10^4: 24.9 -> 22.8 ms)
constexpr int LMAX_SMALL = 800;     // up to here dense single-window calls take the single-launch path (tj_small.cu);
                                    // measured crossover with the general path: all blocks 188 vs 207 us at 800, 317 vs 288 at 1000
constexpr int LMAX_LONG = 4096;     // from here on a dense sweep uses the long-sweep geometry (R_TT_LONG; 96-step stages)
constexpr int R_MULTI2 = 8;         // pairs per thread, 2 window sets per sweep (tj_coupling_multi)
constexpr int R_MULTI3 = 6;         // pairs per thread, 3 window sets per sweep
constexpr int R_TT_MULTI = 16;      // pairs per thread, TT-only sweep of 2 or 4 windows

// mask bits of the blocks one sweep computes
constexpr int M_TT = 1, M_TE = 2, M_EE = 4, M_EB = 8;

__host__ __device__ inline int num_bands(int lmax, int R) { return (lmax + R) / R; }  // ceil((lmax+1)/R)

// Columns c needed by row band `band` (rows a..a+R-1, a = band*R): c_lo .. c_hi inclusive.
// A call may be restricted to the full rows [row_lo, row_hi) of the matrices (tj_coupling_rows; the whole matrix is
// row_lo = 0, row_hi = lmax+1): a band that reaches into the block needs all its columns c >= a (upper part of those
// rows); a band entirely above the block contributes only the mirrored entries, i.e. the pairs whose l2 = c-i lies in
// the block; bands below the block contribute nothing.
__host__ __device__ inline int band_c_lo(int R, int band, int row_lo)
{
    int a = band * R;
    return (a + R - 1 >= row_lo) ? a : row_lo;
}
__host__ __device__ inline int band_c_hi(int lmax, int l3max, int R, int band, bool banded, int row_lo, int row_hi)
{
    int a = band * R;
    int hi = lmax + R - 1;
    if (banded) {
        long long alt = (long long)a + 2 * R - 2 + l3max;
        if (alt < hi) hi = (int)alt;
    }
    if (a + R - 1 < row_lo && row_hi + R - 2 < hi) hi = row_hi + R - 2;
    return hi;
}
__host__ __device__ inline int band_num_tiles(int lmax, int l3max, int R, int band, bool banded, int row_lo, int row_hi)
{
    if (band * R >= row_hi) return 0;
    int lo = band_c_lo(R, band, row_lo);
    int hi = band_c_hi(lmax, l3max, R, band, banded, row_lo, row_hi);
    return hi >= lo ? (hi - lo + SWEEP_THREADS) / SWEEP_THREADS : 0;
}

// ---- diagonal tiling of a band |l1-l2| <= dmax (band-limited calls) -----------------------------
// A warp tile is (delta group, diagonal block n): lane j of the warp owns the R pairs (a+j+i, a+j+d0-i), i = 0..R-1,
// a = 32 n - (R-1): all on ONE anti-diagonal per lane, delta = l2-l1 = d0-2i the same in every lane.  With l3 <= lcut
// a pair has floor((lcut-delta)/2)+1 even steps whatever its l1, so all 32 lanes of a warp (and all R pairs of a
// thread, up to R-1-i steps) have the same step count: no lane waits for another (the column-major tiling of the
// dense sweep loses ~16 of <= lcut/2 steps to the spread of s inside a warp).  Groups hold R deltas of one parity:
// group 2m+p covers delta = p + 2Rm + 2i', i' = 0..R-1; groups are issued in ascending delta = descending work.
__host__ __device__ inline int diag_d0(int R, int grp) { return (grp & 1) + 2 * R * (grp >> 1) + 2 * (R - 1); }
__host__ __device__ inline int diag_num_groups(int dmax, int R)
{
    const int n0 = dmax / 2 + 1, n1 = (dmax + 1) / 2;   // even / odd deltas in 0..dmax
    return (n0 + R - 1) / R + (n1 + R - 1) / R;
}
__host__ __device__ inline int diag_num_blocks(int lmax, int R) { return (lmax + R + 31) / 32; }

// the sweep instantiation a launch used (for the roofline label of bench.py, tj_profile_geometry)
struct SweepGeometry { int R, mask, TS, minb, pipe, nw, spin, rows, diag, tiles; };   // TS = 0: small_kernel (tj_small.cu)
extern thread_local SweepGeometry g_last_sweep;
// kernels launched by this thread's coupling calls since the library was loaded (tj_profile_launches)
extern thread_local long long g_launch_count;

struct Tables {
    int lmax, l3max, pmax;          // p-tables hold p = 0..pmax = 2*lmax+1
    int np_alloc;                   // doubles per p-table incl. guards
    int nl_alloc;                   // doubles per l-table incl. guards (index range -GUARD_LO .. 2*lmax+GUARD_HI)
    double *base;                   // one device allocation
    // pointers to index 0
    double *g, *ginv, *h, *gA, *gB; // p-indexed
    double *u3;                     // l-indexed: u3[l] = l(l+1)
    double *isd;                    // l-indexed: 1/sqrt(D_l), 0 for l < 2
    double *isu;                    // l-indexed: 1/sqrt(u_l), 0 for l < 1 (spin-1 blocks)
};

struct SweepParams {
    const double *g, *ginv, *h, *gA, *gB, *u3, *isd;
    const double *wtt, *wtp, *wpp;  // prefolded windows W'_X[l] = (2l+1) W_X[l] / (4 pi), pointer to l = 0
    const double *wA, *wB;          // the same as pairs: wA[2l..] = (W'_TT, W'_TP)[l], wB[2l..] = (W'_PP, u_l)[l]
    double *TT, *TE, *EE, *EB;      // raw Xi, upper triangle [l1*ld+l2]; band-limited calls: transposed scratch [delta*ld + l1];
                                    // row blocks: the final K, direct and mirrored entries
    double *BB;                     // row blocks: receives the EE values as well (NULL: none)
    const int *tile_start;          // [nbands+1] exclusive prefix of tiles per band, bands in DESCENDING order
    int lmax, l3max, nbands, lcut;  // lcut < 0: dense storage
    int row_lo, row_hi;             // full rows [row_lo, row_hi) are computed (whole matrix: 0, lmax+1)
    int rows;                       // 1: compact row-block outputs [(l1-row_lo)*ld + l2], direct AND mirrored entries stored
    int tile_off;                   // first tile of this launch in the descending-band prefix (row-chunked launches)
    int nd;                         // diagonal tiling: diagonal blocks per delta group (grid = groups * nd)
    long long ld;                   // row stride of the outputs
    long long wstride;              // multi-window: doubles between the prefolded arrays of consecutive window sets
    long long ostride;              // multi-window: doubles between the output matrices of consecutive window sets
};

struct WriterParams {
    double *M[5];                   // TT, TE, EE, EB, (BB copy of EE or NULL)
    int nmat;                       // entries of M that take part in the mirror (<= 4)
    double *bb;                     // if non-NULL: receives a copy of M[bb_src]
    int bb_src;
    int lmax, lcut;                 // lcut < 0: dense
    long long ld;
    int ntile;                      // tiles per side (ceil((lmax+1)/32))
    int tile_band;                  // banded: tiles (I,J) with J-I <= tile_band
    int I0, I1;                     // tile rows [I0, I1) of this launch (row-chunked launches; whole matrix: 0, ntile)
};

// band-limited calls: transposed Xi scratch -> banded storage (tj_writer.cu)
struct BandWriterParams {
    const double *X[4];             // Xi blocks, X[delta*ldT + l1] = Xi(l1, l1+delta), delta = 0..dmax
    double *M[4];                   // banded outputs, M[l1*ld + (l2-l1+lcut)]
    int nmat;
    double *bb;                     // if non-NULL: receives a copy of M[bb_src]
    int bb_src;
    int lmax, lcut, dmax;           // dmax = min(lcut, lmax)
    long long ldT, ld;              // ld = 2*lcut+1
};

// binned output (tj_binned.cu): one chunk of rows [r0, r1) of Xi per block -> accumulated into nbins x nbins
struct BinParams {
    const double *X[4];             // X[m][(l1-r0)*ld + l2] = Xi(l1,l2) for l2 >= l1
    double *B[4];                   // B[m][b*nbins + b']
    int nmat;
    const int *edges;               // device, nbins+1 ascending bin edges
    const double *P, *Q;            // device, lmax+1 weights each
    int nbins, r0, r1, lmax;
    long long ld;
    int split;                      // CTAs per bin pair (launch_bin_split(nbins)); > 1: partial sums go through `part`
    double *part;                   // split > 1: [nmat][nbins(nbins+1)/2][split][2] doubles of scratch
};
int launch_bin_split(int nbins);
cudaError_t launch_bin(const BinParams &P, cudaStream_t st);

// kernels / launchers (defined in the .cu files)
cudaError_t launch_build_tables(const Tables &T, cudaStream_t st);
cudaError_t launch_prepare(const Tables &T, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                           double *wtt, double *wtp, double *wpp, double *wA, double *wB, int *tile_start, int R,
                           int l3max_eff, bool banded, int row_lo, int row_hi, cudaStream_t st);
int sweep_R(int mask, bool banded, int nw, int lmax, bool rows, int spin);   // pairs per thread (= rows per band) of the sweep that serves `mask` for nw window sets
cudaError_t launch_sweep(const SweepParams &P, int mask, int nw, int spin, int total_tiles, cudaStream_t st);
cudaError_t launch_writer(const WriterParams &P, cudaStream_t st);
cudaError_t launch_band_writer(const BandWriterParams &P, cudaStream_t st);
// single-launch path for small lmax (tj_small.cu)
size_t small_smem_bytes(int lmax, int l3max);
cudaError_t launch_small(const Tables &T, int mask, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                         double *TT, double *TE, double *EE, double *BB, double *EB, cudaStream_t st);
cudaError_t launch_literal(const Tables &T, const double *wtt, const double *wpp, double *TT, double *EE, int l3max,
                           cudaStream_t st);   // paper-literal ablation kernel (tj_literal.cu)

}  // namespace tj
