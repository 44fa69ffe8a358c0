// tj_binned.cu -- binned output (reading 20): instead of the full matrices,
//
//     B^{XY}[b][b'] = sum_{l1 in bin b} sum_{l2 in bin b'} P[l1] K^{XY}[l1][l2] Q[l2],     K = (2 l2+1) Xi,
//
// for caller-supplied bins (edges[b] <= l < edges[b+1]) and per-l weights P, Q (e.g. the band-power operator and its
// inverse of a pseudo-C_l pipeline; the paper itself prints no binning operator).  The sweep leaves
// Xi(l1,l2), l1 <= l2, for a chunk of rows in scratch; this kernel takes the place of the mirrored writer: every Xi is
// read once and added to its two bins, (b(l1), b(l2)) with weight P[l1] Q[l2] (2 l2+1) and, for l2 > l1, the mirrored
// (b(l2), b(l1)) with weight P[l2] Q[l1] (2 l1+1) (Xi is symmetric).  The (lmax+1)^2 matrices are never
// written: 4 GB at lmax = 10^4 become nbins^2 numbers per block.
//
// Deterministic: a bin pair (b <= b') of one block is owned, for the chunk, by P.split CTAs that take the rows of the bin
// in turn (groups of BIN_TY rows, dealt cyclically: a partition fixed by the bin edges and P.split alone); the threads
// of a CTA add their terms in a fixed order and a fixed tree joins them.  With P.split = 1 that CTA adds its sum to
// the bin; otherwise every CTA stores its sum and bin_reduce_kernel adds the P.split partial sums in ascending order.
// The chunks follow each other on the stream.  P.split depends on the number of bins only (launch_bin_split): many
// narrow bins are one CTA each, as before; a few wide bins (one bin = the whole matrix in the extreme) would otherwise
// leave a handful of CTAs to stream the whole ~1 GiB chunk.
#include "tj_internal.cuh"

namespace tj {
namespace {

constexpr int BIN_TX = 32, BIN_TY = 8;

__global__ void __launch_bounds__(BIN_TX * BIN_TY) bin_kernel(const __grid_constant__ BinParams P)
{
    __shared__ double sd[BIN_TX * BIN_TY], sm[BIN_TX * BIN_TY];
    // bin pair: blockIdx.x = bp (bp+1)/2 + b, b <= bp
    const int idx = (int)blockIdx.x;
    int bp = (int)((sqrt(8.0 * (double)idx + 1.0) - 1.0) * 0.5);
    while ((long long)(bp + 1) * (bp + 2) / 2 <= idx) ++bp;
    while ((long long)bp * (bp + 1) / 2 > idx) --bp;
    const int b = idx - (int)((long long)bp * (bp + 1) / 2);
    const int m = (int)blockIdx.y;
    const int z = (int)blockIdx.z, S = P.split;
    const int i0 = max(P.edges[b], P.r0), i1 = min(P.edges[b + 1], P.r1);   // rows of the chunk in bin b
    const int j0 = P.edges[bp], j1 = P.edges[bp + 1];                        // columns in bin bp
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * BIN_TX + tx;
    double *part = S > 1 ? P.part + (((long long)m * gridDim.x + idx) * S + z) * 2 : nullptr;
    if (i0 >= i1 || j0 >= j1) {
        if (part && tid == 0) { part[0] = 0.0; part[1] = 0.0; }
        return;
    }
    const double *X = P.X[m];
    double d = 0.0, mi = 0.0;
    for (int l1 = i0 + ty + BIN_TY * z; l1 < i1; l1 += BIN_TY * S) {
        const double p1 = P.P[l1], q1w = P.Q[l1] * (double)(2 * l1 + 1);
        const double *row = X + (long long)(l1 - P.r0) * P.ld;
        for (int l2 = max(j0, l1) + tx; l2 < j1; l2 += BIN_TX) {   // upper triangle: l2 >= l1
            const double x = row[l2];
            d = fma(p1 * (x * (double)(2 * l2 + 1)), P.Q[l2], d);
            if (l2 > l1) mi = fma(P.P[l2] * x, q1w, mi);
        }
    }
    sd[tid] = d;
    sm[tid] = mi;
    __syncthreads();
    for (int s = BIN_TX * BIN_TY / 2; s > 0; s >>= 1) {
        if (tid < s) { sd[tid] += sd[tid + s]; sm[tid] += sm[tid + s]; }
        __syncthreads();
    }
    if (tid == 0 && part) {
        part[0] = sd[0];
        part[1] = sm[0];
    } else if (tid == 0) {
        double *B = P.B[m];
        if (b == bp) {
            B[(long long)b * P.nbins + b] += sd[0] + sm[0];
        } else {
            B[(long long)b * P.nbins + bp] += sd[0];
            B[(long long)bp * P.nbins + b] += sm[0];
        }
    }
}

// second pass of a split launch: one thread per (block, bin pair) adds the P.split partial sums in ascending order
__global__ void __launch_bounds__(128) bin_reduce_kernel(const __grid_constant__ BinParams P, int npairs)
{
    const int idx = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    const int m = (int)blockIdx.y;
    if (idx >= npairs) return;
    int bp = (int)((sqrt(8.0 * (double)idx + 1.0) - 1.0) * 0.5);
    while ((long long)(bp + 1) * (bp + 2) / 2 <= idx) ++bp;
    while ((long long)bp * (bp + 1) / 2 > idx) --bp;
    const int b = idx - (int)((long long)bp * (bp + 1) / 2);
    const double *part = P.part + ((long long)m * npairs + idx) * P.split * 2;
    double d = 0.0, mi = 0.0;
    for (int z = 0; z < P.split; ++z) { d += part[2 * z]; mi += part[2 * z + 1]; }
    double *B = P.B[m];
    if (b == bp) {
        B[(long long)b * P.nbins + b] += d + mi;
    } else {
        B[(long long)b * P.nbins + bp] += d;
        B[(long long)bp * P.nbins + b] += mi;
    }
}

}  // namespace

// CTAs per bin pair: enough that a launch fills the GPU a few times over (>= 4 x 148 CTAs per block; one bin: 592)
constexpr int BIN_SPLIT_MAX = 592;
int launch_bin_split(int nbins)
{
    const long long np = (long long)nbins * (nbins + 1) / 2;
    long long s = (BIN_SPLIT_MAX + np - 1) / np;
    return (int)(s < 1 ? 1 : s > BIN_SPLIT_MAX ? BIN_SPLIT_MAX : s);
}

cudaError_t launch_bin(const BinParams &P, cudaStream_t st)
{
    if (P.nmat <= 0 || P.nbins <= 0) return cudaSuccess;
    const long long np = (long long)P.nbins * (P.nbins + 1) / 2;
    if (np > 0x7fffffffLL) return cudaErrorInvalidValue;
    if (P.split < 1 || P.split > BIN_SPLIT_MAX || (P.split > 1 && !P.part)) return cudaErrorInvalidValue;
    bin_kernel<<<dim3((unsigned)np, (unsigned)P.nmat, (unsigned)P.split), dim3(BIN_TX, BIN_TY, 1), 0, st>>>(P);
    ++g_launch_count;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || P.split == 1) return e;
    bin_reduce_kernel<<<dim3((unsigned)((np + 127) / 128), (unsigned)P.nmat, 1), 128, 0, st>>>(P, (int)np);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace tj
