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
// sweep (diagonal tiling) leaves Xi in a transposed scratch X[delta][l1]; band_writer_kernel turns 32x32 tiles of it
// into full row segments of the band, direct (column lcut+delta) and mirrored (column lcut-delta), and writes 0.0
// into the slots whose l2 falls outside 0..lmax -- every slot of the outputs is written exactly once.
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

// One CTA: deltas d0..d0+31 of ONE banded output, and
//   direct:  rows l1 = r0..r0+31:       M[l1][lcut+delta] = (2(l1+delta)+1) Xi(l1, l1+delta)   source X[delta][l1]
//   mirror:  rows r = r0+d0..r0+d0+31:  M[r][lcut-delta]  = (2(r-delta)+1)  Xi(r-delta, r)     source X[delta][r-delta]
// Both are 32 consecutive columns per row, and both sources are read as 32 consecutive doubles per delta and
// transposed through shared memory.  The mirror rows are shifted by d0 against the direct rows so that the two source
// tiles cover the same l1 range (r0-31..r0+31): the second read of an element comes from L2, not from HBM.
// (delta = 0: one slot, written by the direct part.)  Slots whose l2 falls outside 0..lmax get 0.0; CTAs of negative
// r0 (blockIdx.y below y0) only write the mirror-side zeros of the rows r < delta.  Every slot is written exactly once.
__global__ void __launch_bounds__(WT * WROWS) band_writer_kernel(const __grid_constant__ BandWriterParams P, int y0)
{
    __shared__ double td[WT][WT + 1], tm[WT][WT + 1];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int d0 = blockIdx.x * WT, r0 = ((int)blockIdx.y - y0) * WT, m = blockIdx.z;
    if (r0 < 0 && r0 + d0 + WT - 1 < 0) return;   // neither direct rows nor mirror rows
    const double *X = P.X[m];
    double *M = P.M[m];
    double *bb = (P.bb != nullptr && m == P.bb_src) ? P.bb : nullptr;
#pragma unroll
    for (int k = ty; k < WT; k += WROWS) {
        const int delta = d0 + k;
        const int l1d = r0 + tx, l1m = r0 - k + tx;
        const bool okd = delta <= P.dmax && l1d >= 0 && l1d + delta <= P.lmax;
        const bool okm = delta <= P.dmax && delta >= 1 && l1m >= 0 && l1m + delta <= P.lmax;
        td[k][tx] = okd ? X[(long long)delta * P.ldT + l1d] : 0.0;
        tm[k][tx] = okm ? X[(long long)delta * P.ldT + l1m] : 0.0;
    }
    __syncthreads();
    const int delta = d0 + tx;
    if (delta > P.lcut) return;
#pragma unroll
    for (int k = ty; k < WT; k += WROWS) {
        const int l1 = r0 + k;           // direct row
        if (l1 >= 0 && l1 <= P.lmax) {
            const double v = td[tx][k] * (double)(2 * (l1 + delta) + 1);   // out of range: 0.0 * positive = 0.0
            const long long ix = (long long)l1 * P.ld + P.lcut + delta;
            M[ix] = v;
            if (bb) bb[ix] = v;
        }
        const int r = r0 + d0 + k;       // mirror row; its source row of Xi is l1 = r - delta = r0 + k - tx
        if (delta >= 1 && r >= 0 && r <= P.lmax) {
            const int lm = r - delta;
            const double v = lm >= 0 ? tm[tx][k] * (double)(2 * lm + 1) : 0.0;
            const long long ix = (long long)r * P.ld + P.lcut - delta;
            M[ix] = v;
            if (bb) bb[ix] = v;
        }
    }
}

cudaError_t launch_band_writer(const BandWriterParams &P, cudaStream_t st)
{
    if (P.nmat <= 0) return cudaSuccess;
    const int y0 = (P.lcut + WT - 1) / WT;   // tiles of negative l1: the zeros of the rows r < delta
    dim3 grid((unsigned)(P.lcut / WT + 1), (unsigned)(y0 + (P.lmax + WT) / WT), (unsigned)P.nmat);
    band_writer_kernel<<<grid, dim3(WT, WROWS, 1), 0, st>>>(P, y0);
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
