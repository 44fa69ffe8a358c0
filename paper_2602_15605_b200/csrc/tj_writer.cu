// tj_writer.cu -- triangle -> full matrix writer (step a6), dense and banded.
//
// The sweep leaves Xi(l1,l2), l1 <= l2, in the upper triangle of each output.  Xi is symmetric
// (PAPER.md:236 as read in DESIGN.md reading #8) and K_{l1 l2} = (2 l2+1) Xi(l1,l2), so
//     M[l1][l2] = (2 l2+1) Xi,      M[l2][l1] = (2 l1+1) Xi.
// One CTA owns one 32x32 tile pair (I,J), I <= J, of every block: it reads the Xi tile once (coalesced along l2), scales
// it in place, and writes the mirrored tile through a shared-memory transpose so that both writes are
// full coalesced row segments.  Both products use the SAME Xi double, so (2 l1+1) M[l1][l2] and
// (2 l2+1) M[l2][l1] agree to the last rounding.  BB, when requested next to EE, is written from the
// same registers.
//
// Banded storage (step a7): address(l1,l2) = l1*ld + (l2-l1+lcut), valid for |l1-l2| <= lcut.  The band-limited
// sweep (diagonal tiling) leaves Xi in a transposed scratch X[delta][l1]; band_writer_kernel turns it into
// sector-aligned row segments of the band, direct and mirrored part alike, and writes 0.0 into the slots whose l2
// falls outside 0..lmax -- every slot of the outputs is written exactly once.
#include "tj_internal.cuh"

namespace tj {
namespace {

constexpr int WT = 32;          // tile edge
constexpr int WROWS = 8;        // rows per pass (blockDim.y)

__device__ __forceinline__ long long addr(int r, int c, long long ld, int lcut)
{
    return lcut < 0 ? (long long)r * ld + c : (long long)r * ld + (c - r + lcut);
}

__global__ void __launch_bounds__(WT * WROWS) writer_kernel(const __grid_constant__ WriterParams P)
{
    // one CTA handles its tile pair for ALL blocks: every thread has 4 x nmat independent loads in flight before
    // the first store (the kernel is a latency-bound copy; with one block per CTA it reached 0.70 of the copy peak)
    __shared__ double tile[4][WT][WT + 1];
    // tile pair decode: blockIdx.x enumerates (I, dJ) with J = I + dJ
    const int I = P.I0 + blockIdx.x / (P.tile_band + 1);
    const int J = I + blockIdx.x % (P.tile_band + 1);
    if (J >= P.ntile) return;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int N = P.lmax + 1;

    // ---- read the Xi tiles (rows l1 in I, cols l2 in J) ----
    const int l2 = J * WT + tx;
    double xi[4][WT / WROWS];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
        const double *M = P.M[m];
#pragma unroll
        for (int k = 0; k < WT; k += WROWS) {
            const int l1 = I * WT + ty + k;
            const bool ok = l1 < N && l2 < N && l2 >= l1 && (P.lcut < 0 || l2 - l1 <= P.lcut);
            xi[m][k / WROWS] = ok ? M[addr(l1, l2, P.ld, P.lcut)] : 0.0;
        }
    }
    // ---- scale in place, stage for the transpose ----
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
        double *M = P.M[m];
        double *bb = (P.bb != nullptr && m == P.bb_src) ? P.bb : nullptr;
#pragma unroll
        for (int k = 0; k < WT; k += WROWS) {
            const int l1 = I * WT + ty + k;
            const bool ok = l1 < N && l2 < N && l2 >= l1 && (P.lcut < 0 || l2 - l1 <= P.lcut);
            const double x = xi[m][k / WROWS];
            if (ok) {
                const long long ix = addr(l1, l2, P.ld, P.lcut);
                const double v = x * (double)(2 * l2 + 1);
                M[ix] = v;
                if (bb) bb[ix] = v;
            }
            tile[m][ty + k][tx] = x;
        }
    }
    __syncthreads();
    // ---- mirrored tiles: rows r = l2 in J, cols q = l1 in I; strictly lower triangle only ----
    const int q = I * WT + tx;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
        double *M = P.M[m];
        double *bb = (P.bb != nullptr && m == P.bb_src) ? P.bb : nullptr;
#pragma unroll
        for (int k = 0; k < WT; k += WROWS) {
            const int r = J * WT + ty + k;
            if (r < N && q < N && q < r && (P.lcut < 0 || r - q <= P.lcut)) {
                const double v = tile[m][tx][ty + k] * (double)(2 * q + 1);
                const long long ix = addr(r, q, P.ld, P.lcut);
                M[ix] = v;
                if (bb) bb[ix] = v;
            }
        }
    }
}

}  // namespace

// Band writer: transposed Xi scratch X[delta][l1] -> banded outputs M[r][j], j = l2-r+lcut in 0..2 lcut.
//   slot (r, j), d = j - lcut, l2 = r + d:   M = (2 l2+1) Xi(min(r,l2), max(r,l2)) = (2 l2+1) X[|d|][min(r, l2)]
// (direct part d >= 0: K_{r l2} = (2 l2+1) Xi(r,l2); mirrored part d < 0: K_{r l2} = (2 l2+1) Xi(l2,r)),
// and 0.0 where l2 falls outside 0..lmax: every slot of the outputs is written exactly once, by this kernel.
//
// Sector alignment.  A band row holds 2 lcut+1 doubles, so rows start on 8-byte boundaries only; a tile whose row
// segments begin at a fixed slot would begin and end inside 32-byte sectors that another CTA completes later, which
// costs a quarter of the write bandwidth (measured on the dense writer: 0.74 of the copy peak with rows of 10001
// doubles, 0.96 with rows of 10016).  The scratch is read-only here, so the tiles can be ragged instead: in row r the
// CTA of slot tile T writes the slots [32 T - s_r, 32 T - s_r + 32), s_r = (flat index of the row's first slot) mod 4 --
// 32 consecutive doubles that start on a sector boundary in every row.  Over the 32 rows of a CTA the slots span 35
// values of d; for each of them the 32 sources X[|d|][r0 + min(d,0) + 0..31] are consecutive doubles of the scratch,
// staged through shared memory and read back transposed.
__global__ void __launch_bounds__(WT * WROWS, 4) band_writer_kernel(const __grid_constant__ BandWriterParams P)
{
    // one CTA handles its tile for ALL blocks: every thread has 5 x nmat independent loads in flight before the first
    // store (measured at config 4: one block per CTA 0.128 ms, all blocks 0.100 ms; 4 CTAs/SM at 64 registers 0.100 ms,
    // 5 / 6 CTAs/SM with spills 0.111 / 0.151 ms; the round-1 form with fixed slot tiles 0.108 ms)
    constexpr int ND = WT + 3;                 // signed deltas a CTA's slots span
    constexpr int NK = (ND + WROWS - 1) / WROWS;
    __shared__ double sx[4][ND][WT + 1];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int r0 = (int)blockIdx.y * WT;
    const int W = 2 * P.lcut + 1;
    const int d_lo = (int)blockIdx.x * WT - 3 - P.lcut;   // signed delta of slot 32 T - 3
    double v[4][NK];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
        const double *X = P.X[m];
#pragma unroll
        for (int q = 0; q < NK; ++q) {
            const int k = ty + q * WROWS;
            const int d = d_lo + k, ad = d < 0 ? -d : d;
            const int l1 = r0 + tx + (d < 0 ? d : 0);       // row of Xi: min(r, l2) for r = r0 + tx
            const bool ok = k < ND && ad <= P.dmax && l1 >= 0 && l1 + ad <= P.lmax;
            v[m][q] = ok ? X[(long long)ad * P.ldT + l1] : 0.0;
        }
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
#pragma unroll
        for (int q = 0; q < NK; ++q)
            if (ty + q * WROWS < ND) sx[m][ty + q * WROWS][tx] = v[m][q];
    }
    __syncthreads();
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        if (m >= P.nmat) break;
        double *M = P.M[m];
        double *bb = (P.bb != nullptr && m == P.bb_src) ? P.bb : nullptr;
        const unsigned base4 = (unsigned)((reinterpret_cast<uintptr_t>(M) >> 3) & 3);   // the output's own offset in its sector
#pragma unroll
        for (int k = ty; k < WT; k += WROWS) {
            const int r = r0 + k;
            if (r > P.lmax) break;
            const long long f0 = (long long)r * W;
            const int s = (int)((f0 + base4) & 3);
            const int j = (int)blockIdx.x * WT - s + tx;    // slot
            if (j < 0 || j >= W) continue;
            const int d = j - P.lcut, l2 = r + d;
            // out of range: the source was staged as 0.0; 0.0 * (2 l2+1) would be -0.0 for l2 < 0, hence the select
            const double o = (l2 >= 0 && l2 <= P.lmax) ? sx[m][d - d_lo][k] * (double)(2 * l2 + 1) : 0.0;
            M[f0 + j] = o;
            if (bb) bb[f0 + j] = o;
        }
    }
}

cudaError_t launch_band_writer(const BandWriterParams &P, cudaStream_t st)
{
    if (P.nmat <= 0) return cudaSuccess;
    const int W = 2 * P.lcut + 1;
    dim3 grid((unsigned)((W + 3 + WT - 1) / WT), (unsigned)((P.lmax + WT) / WT), 1);
    band_writer_kernel<<<grid, dim3(WT, WROWS, 1), 0, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_writer(const WriterParams &P, cudaStream_t st)
{
    if (P.nmat <= 0 || P.I1 <= P.I0) return cudaSuccess;
    dim3 grid((unsigned)((P.I1 - P.I0) * (P.tile_band + 1)), 1, 1);
    dim3 block(WT, WROWS, 1);
    writer_kernel<<<grid, block, 0, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace tj
