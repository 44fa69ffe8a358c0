// tj_tables.cu -- lookup-table build kernel (step a1).
//
// PAPER.md:166-186, Eqs. 11-12:  g(0) = 1,  g(p) = (p - 1/2)/p * g(p-1) = g(p-1) * (2p-1)/(2p).
// The paper builds ln g and exponentiates; g stays within [3e-3, 1] for p <= 3e4
// (g ~ (pi p)^(-1/2)), so here the product recurrence is carried directly, in
// double-double arithmetic and as a parallel scan, and every stored double is the faithfully rounded
// value of Eq. 11 (reading #10).
//
// Folded tables:  ginv = 1/g,  h = 1/((2p+1) g)  [Eq. 10's 1/(J+1) at J = 2p],
//                               gA = 2p g,   gB = (2p+1) g      [odd-J branch].
#include "tj_internal.cuh"

namespace tj {
namespace {

struct dd { double hi, lo; };

__device__ __forceinline__ dd two_sum(double a, double b)
{
    double s = a + b;
    double bb = s - a;
    double e = (a - (s - bb)) + (b - bb);
    return {s, e};
}
__device__ __forceinline__ dd quick_two_sum(double a, double b)
{
    double s = a + b;
    return {s, b - (s - a)};
}
__device__ __forceinline__ dd two_prod(double a, double b)
{
    double p = a * b;
    return {p, fma(a, b, -p)};
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b)
{
    dd p = two_prod(a.hi, b);
    p.lo = fma(a.lo, b, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    dd p = two_prod(a.hi, b.hi);
    p.lo += a.hi * b.lo + a.lo * b.hi;
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_div_d(dd a, double b)
{
    double q1 = a.hi / b;
    dd p = two_prod(q1, b);
    dd r = two_sum(a.hi, -p.hi);
    r.lo -= p.lo;
    r.lo += a.lo;
    double q2 = (r.hi + r.lo) / b;
    return quick_two_sum(q1, q2);
}
__device__ __forceinline__ dd dd_recip(dd a)
{
    double q1 = 1.0 / a.hi;
    // r = 1 - q1*a, exactly enough
    dd p = two_prod(q1, a.hi);
    double r = (1.0 - p.hi) - p.lo - q1 * a.lo;
    double q2 = r / a.hi;
    return quick_two_sum(q1, q2);
}

constexpr int TB_THREADS = 1024;

// One CTA.  Thread i owns the contiguous chunk p in [i*chunk, (i+1)*chunk).
//  1) local product of the ratios (2p-1)/(2p) over the chunk          (Eq. 12)
//  2) exclusive multiplicative scan of the chunk products across the CTA
//  3) re-walk the chunk from the scanned prefix, rounding and storing g and the folded tables.
__global__ void __launch_bounds__(TB_THREADS) build_tables_kernel(Tables T)
{
    __shared__ dd sc[TB_THREADS];
    const int n = T.pmax + 1;
    const int chunk = (n + TB_THREADS - 1) / TB_THREADS;
    const int tid = threadIdx.x;
    const int p0 = tid * chunk;
    const int p1 = min(n, p0 + chunk);

    dd loc = {1.0, 0.0};
    for (int p = max(p0, 1); p < p1; ++p) {
        loc = dd_mul_d(loc, (double)(2 * p - 1));
        loc = dd_div_d(loc, (double)(2 * p));
    }
    sc[tid] = loc;
    __syncthreads();
    // Hillis-Steele inclusive scan (multiplicative)
    for (int off = 1; off < TB_THREADS; off <<= 1) {
        dd v = sc[tid];
        if (tid >= off) v = dd_mul(sc[tid - off], v);
        __syncthreads();
        sc[tid] = v;
        __syncthreads();
    }
    dd run = (tid == 0) ? dd{1.0, 0.0} : sc[tid - 1];   // = g(p0 - 1) for p0 >= 1 (g(0) = 1)
    for (int p = p0; p < p1; ++p) {
        if (p >= 1) {
            run = dd_mul_d(run, (double)(2 * p - 1));
            run = dd_div_d(run, (double)(2 * p));
        }
        const double tp1 = (double)(2 * p + 1);
        dd gb = dd_mul_d(run, tp1);
        dd ga = dd_mul_d(run, (double)(2 * p));
        dd gi = dd_recip(run);
        dd hh = dd_recip(gb);
        T.g[p] = run.hi + run.lo;
        T.ginv[p] = gi.hi + gi.lo;
        T.h[p] = hh.hi + hh.lo;
        T.gA[p] = ga.hi + ga.lo;
        T.gB[p] = gb.hi + gb.lo;
    }
}

// l-indexed constants: u3[l] = l(l+1) over the whole guarded range (finite everywhere, exact integers),
// isd[l] = 1/sqrt((l-1) l (l+1) (l+2)) = 1/sqrt(u (u-2)), 0 for l < 2 and in the guards.
__global__ void build_ltables_kernel(Tables T)
{
    const int lo = -GUARD_LO, hi = T.nl_alloc - GUARD_LO;   // [lo, hi)
    for (int l = lo + (int)(blockIdx.x * blockDim.x + threadIdx.x); l < hi; l += (int)(gridDim.x * blockDim.x)) {
        double dl = (double)l;
        double u = dl * (dl + 1.0);
        T.u3[l] = u;
        T.isd[l] = (l >= 2 && l <= T.lmax) ? 1.0 / sqrt(u * (u - 2.0)) : 0.0;
        T.isu[l] = (l >= 1 && l <= T.lmax) ? 1.0 / sqrt(u) : 0.0;
    }
}

}  // namespace

cudaError_t launch_build_tables(const Tables &T, cudaStream_t st)
{
    // guards and the tail beyond pmax are zero: one memset of the whole allocation
    size_t bytes = sizeof(double) * ((size_t)5 * T.np_alloc + (size_t)3 * T.nl_alloc);
    cudaError_t e = cudaMemsetAsync(T.base, 0, bytes, st);
    if (e != cudaSuccess) return e;
    build_tables_kernel<<<1, TB_THREADS, 0, st>>>(T);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    int nb = (T.nl_alloc + 255) / 256;
    build_ltables_kernel<<<nb, 256, 0, st>>>(T);
    return cudaGetLastError();
}

}  // namespace tj
