// tj_api.cu -- the C ABI of libtj (include/tj.h): argument checks, stream-ordered scratch, launches.
#include <atomic>
#include <math.h>
#include <mutex>
#include <new>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "tj_internal.cuh"

using namespace tj;

namespace {

constexpr int WSET = 7;   // doubles of scratch per window set, in units of nl_alloc: wtt, wtp, wpp, wA (x2), wB (x2)

thread_local char g_errbuf[256] = "CUDA error";

int cuda_fail(cudaError_t e, const char *where)
{
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", where, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? TJ_ENOMEM : TJ_ECUDA;
}
#define TJ_CUDA(call, where)                                   \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return cuda_fail(e__, where);  \
    } while (0)

// keep freed scratch in the device's default mem pool instead of returning it to the OS after every call
// (per device: called from every tj_build_tables; setting the attribute again is harmless)
void tune_pool(int dev)
{
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) != cudaSuccess) return;
    unsigned long long thr = ~0ull;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
}

// Side streams and events of the host-buffer pipeline (run_coupling_rows_to_host).  They belong to a tables handle,
// i.e. to ONE device: created on first use, destroyed by tj_free_tables; the mutex serialises host-buffer calls that
// share a handle (each of them synchronises before it returns anyway).
constexpr int PIPE_MAX_CHUNKS = 24;
constexpr int PLAN_MAX_PARTS = 64;                  // devices that may share one matrix (tj_coupling_host_multi)
constexpr double HOST_COPY_RATE_DEFAULT = 54e9;     // bytes/s, contiguous device-to-host copy into pinned memory
constexpr double HOST_INSTR_RATE_DEFAULT = 1.6e13;  // FP64 thread-instructions/s of the dense sweep
struct HostPipe {
    std::mutex mu;
    cudaStream_t comp[2] = {nullptr, nullptr}, copy = nullptr;
    cudaEvent_t ev[PIPE_MAX_CHUNKS + 2];
    int nev = 0;
    bool have = false;
    // what the regime choice of run_coupling_rows_to_host assumes about the machine (tj_set_host_pipeline); the
    // defaults are the values measured on the B200 boxes this library was tuned on
    double copy_rate = HOST_COPY_RATE_DEFAULT, instr_rate = HOST_INSTR_RATE_DEFAULT;
    int last_regime = 0, last_chunks = 0;   // tj_host_pipeline_info
    cudaError_t ensure()
    {
        if (have) return cudaSuccess;
        cudaError_t e = cudaSuccess;
        for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaStreamCreateWithFlags(&comp[k], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking);
        for (int k = 0; k < PIPE_MAX_CHUNKS + 2 && e == cudaSuccess; ++k) {
            e = cudaEventCreateWithFlags(&ev[k], cudaEventDisableTiming);
            if (e == cudaSuccess) ++nev;
        }
        if (e != cudaSuccess) { destroy(); return e; }
        have = true;
        return cudaSuccess;
    }
    void destroy()
    {
        for (int k = 0; k < nev; ++k) cudaEventDestroy(ev[k]);
        nev = 0;
        for (int k = 0; k < 2; ++k) if (comp[k]) { cudaStreamDestroy(comp[k]); comp[k] = nullptr; }
        if (copy) { cudaStreamDestroy(copy); copy = nullptr; }
        have = false;
    }
};

// optional per-kernel timing of the most recent coupling call of this thread (tj_profile_*).  The events are kept per
// (thread, device): an event can only be recorded on a stream of the device it was created on, and one thread may
// drive several GPUs (one handle per device).  Profiling never decides a call's status: if an event cannot be created
// or recorded, the rest of that call goes unprofiled and the error is cleared from the runtime's last-error slot
// (the launchers end with cudaGetLastError(), which must report the LAUNCH).
std::atomic<int> g_profile{0};
constexpr int PROF_MAX_DEVICES = 64;
struct ProfEvents { cudaEvent_t ev[5]; bool have = false; };
struct ProfState {
    ProfEvents dev[PROF_MAX_DEVICES];
    int cur = -1;          // device of the call being profiled / of the last profiled call
    bool valid = false;    // all five events of the most recent call are recorded
    bool broken = false;   // an event call failed during the current call
};
thread_local ProfState g_prof;

void prof_record(int i, cudaStream_t st)
{
    if (!g_profile.load(std::memory_order_relaxed)) return;
    if (i == 0) {   // first event of a call: pick (and if need be create) the current device's events
        g_prof.broken = false;
        g_prof.valid = false;
        int d = -1;
        if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= PROF_MAX_DEVICES) {
            cudaGetLastError();
            g_prof.cur = -1;
            return;
        }
        g_prof.cur = d;
        ProfEvents &E = g_prof.dev[d];
        if (!E.have) {
            int made = 0;
            while (made < 5 && cudaEventCreate(&E.ev[made]) == cudaSuccess) ++made;
            if (made < 5) {
                cudaGetLastError();
                while (made > 0) cudaEventDestroy(E.ev[--made]);
                g_prof.broken = true;
                return;
            }
            E.have = true;
        }
    }
    if (g_prof.cur < 0 || g_prof.broken || !g_prof.dev[g_prof.cur].have) return;
    if (cudaEventRecord(g_prof.dev[g_prof.cur].ev[i], st) != cudaSuccess) {
        cudaGetLastError();
        g_prof.broken = true;
        g_prof.valid = false;
        return;
    }
    if (i == 4) g_prof.valid = true;
}

int total_tiles(int lmax, int l3max, int R, bool banded, int row_lo, int row_hi)
{
    long long n = 0;
    const int nb = num_bands(lmax, R);
    for (int b = 0; b < nb; ++b) n += band_num_tiles(lmax, l3max, R, b, banded, row_lo, row_hi);
    return n > 0x7fffffffLL ? -1 : (int)n;
}

// State of one coupling call between its pieces (coupling_begin / _sweep / _write / _end, below).
struct Call {
    const Tables *T = nullptr;
    bool banded = false;
    int lcut = -1, mask = 0, R = 0, l3max_eff = 0, nb = 0, ntiles = 0, ntile_w = 0;
    int nw = 1;                     // window sets per sweep (tj_coupling_multi: 2)
    int spin = 2;                   // 2: TT/TE/EE/EB; 1: K00/K01/K11+/K11- in the same slots (tj_coupling_spin1)
    int nW = 0;                     // entries per window
    int row_lo = 0, row_hi = 0;     // full rows [row_lo, row_hi) are computed (tj_coupling_rows; else 0, lmax+1)
    bool rows = false;              // row-block outputs
    long long N = 0, ld = 0;
    double *TT = nullptr, *TE = nullptr, *ee = nullptr, *EB = nullptr, *bb_copy = nullptr;
    unsigned char *scratch = nullptr;
    double *wtt = nullptr, *wtp = nullptr, *wpp = nullptr, *wA = nullptr, *wB = nullptr;
    int *tile_start = nullptr;
    // band-limited calls (diagonal tiling): the sweep leaves Xi in a transposed scratch xit[k][delta*ldT + l1]
    // (k-th requested block in the order TT, TE, EE, EB), the band writer scales / mirrors it into the outputs
    double *xit[4] = {nullptr, nullptr, nullptr, nullptr};
    long long ldT = 0;
    int dmax = 0;
    long long ostride = 0;          // doubles between the outputs of consecutive window sets (0: whole matrices, N * ld)
};

// Dense single-window spin-2 calls at small lmax take the single-launch path (tj_small.cu): below LMAX_SMALL the
// three launches and the scratch of the general path cost more than the arithmetic.
bool use_small_path(const Tables &T, int lcut, int nw, int spin)
{
    return lcut < 0 && nw == 1 && spin == 2 && T.lmax <= LMAX_SMALL && small_smem_bytes(T.lmax, T.l3max) <= 200 * 1024;
}

// One coupling call on device pointers.  lcut < 0: dense (l3max = handle's); else banded with l3 <= lcut.
int run_coupling(const tj_tables *tables, int lcut, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                 int nW, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st, int nw = 1,
                 int spin = 2);
int run_rows(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW, int row_lo,
             int row_hi, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st);
int run_coupling_rows_to_host(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                              int nW, double *const d_out[5], double *const h_out[5], cudaStream_t st, int part = 0,
                              int nparts = 1);
int chunk_plan(int lmax, int R, int nparts, int *bounds, int *owner);
int run_literal(const tj_tables *tables, const double *d_Wtt, const double *d_Wpp, int nW, double *d_TT, double *d_EE,
                cudaStream_t st);
int run_coupling_static(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                        double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st);
int run_binned(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW, int nbins,
               const int *h_edges, const double *d_P, const double *d_Q, double *d_TT, double *d_TE, double *d_EE,
               double *d_BB, double *d_EB, cudaStream_t st, int nw = 1);

}  // namespace

struct tj_tables {
    Tables T;
    int device = 0;     // the device the tables live on; every entry point checks that it is the current one
    HostPipe pipe;
};

namespace {
// TJ_EINVAL unless the handle's device is the calling thread's current device (streams, scratch and kernels of a call
// all belong to the current device: a handle built on another GPU cannot be used without cudaSetDevice)
int check_device(const tj_tables *tables)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return cuda_fail(cudaGetLastError(), "cudaGetDevice");
    return dev == tables->device ? TJ_OK : TJ_EINVAL;
}
}  // namespace

extern "C" {

const char *tj_strerror(int code)
{
    switch (code) {
        case TJ_OK: return "ok";
        case TJ_EINVAL: return "invalid argument";
        case TJ_ENOMEM: return "out of memory";
        case TJ_ECUDA: return g_errbuf;
        case TJ_ELIMIT: return "lmax exceeds TJ_STATIC_LMAX: the built-in scratch array of tj_coupling_pol_static is too small";
        default: return "unknown error code";
    }
}

int tj_build_tables(int lmax, int l3max, void *cuda_stream, tj_tables **out)
{
    if (!out) return TJ_EINVAL;
    *out = nullptr;
    if (lmax < 0 || l3max < 0 || lmax > 0x0fffffff / 4 || l3max > 2 * lmax) return TJ_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    tj_tables *h = new (std::nothrow) tj_tables;
    if (!h) return TJ_ENOMEM;
    Tables &T = h->T;
    T.lmax = lmax;
    T.l3max = l3max;
    T.pmax = 2 * lmax + 1;
    T.np_alloc = GUARD_LO + T.pmax + 1 + GUARD_HI;
    T.nl_alloc = GUARD_LO + 2 * lmax + 2 + GUARD_HI;   // even, like np_alloc: every table's index 0 is 16-byte aligned (bulk copies)
    size_t n = (size_t)5 * T.np_alloc + (size_t)3 * T.nl_alloc;
    cudaError_t e = cudaMalloc((void **)&T.base, n * sizeof(double));
    if (e != cudaSuccess) { delete h; return cuda_fail(e, "tj_build_tables/cudaMalloc"); }
    double *p = T.base + GUARD_LO;
    T.g = p;    p += T.np_alloc;
    T.ginv = p; p += T.np_alloc;
    T.h = p;    p += T.np_alloc;
    T.gA = p;   p += T.np_alloc;
    T.gB = p;   p += T.np_alloc;
    T.u3 = p;   p += T.nl_alloc;
    T.isd = p;  p += T.nl_alloc;
    T.isu = p;
    e = launch_build_tables(T, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetDevice(&h->device);
    if (e != cudaSuccess) { cudaFree(T.base); delete h; return cuda_fail(e, "tj_build_tables"); }
    tune_pool(h->device);
    *out = h;
    return TJ_OK;
}

void tj_free_tables(tj_tables *tables)
{
    if (!tables) return;
    tables->pipe.destroy();
    cudaFree(tables->T.base);
    delete tables;
}

int tj_tables_info(const tj_tables *tables, int *lmax, int *l3max, int *pmax)
{
    if (!tables) return TJ_EINVAL;
    if (lmax) *lmax = tables->T.lmax;
    if (l3max) *l3max = tables->T.l3max;
    if (pmax) *pmax = tables->T.pmax;
    return TJ_OK;
}

int tj_tables_copy(const tj_tables *tables, int which, double *h_dst, int count)
{
    if (!tables || !h_dst || count < 0) return TJ_EINVAL;
    const Tables &T = tables->T;
    const double *src = nullptr;
    int maxn = 0;
    switch (which) {
        case 0: src = T.g; maxn = T.pmax + 1; break;
        case 1: src = T.ginv; maxn = T.pmax + 1; break;
        case 2: src = T.h; maxn = T.pmax + 1; break;
        case 3: src = T.gA; maxn = T.pmax + 1; break;
        case 4: src = T.gB; maxn = T.pmax + 1; break;
        case 5: src = T.u3; maxn = T.lmax + 1; break;
        case 6: src = T.isd; maxn = T.lmax + 1; break;
        case 7: src = T.isu; maxn = T.lmax + 1; break;
        default: return TJ_EINVAL;
    }
    if (count > maxn) return TJ_EINVAL;
    { const int rcd = check_device(tables); if (rcd != TJ_OK) return rcd; }
    TJ_CUDA(cudaMemcpy(h_dst, src, sizeof(double) * (size_t)count, cudaMemcpyDeviceToHost), "tj_tables_copy");
    return TJ_OK;
}

int tj_coupling_tt(const tj_tables *tables, const double *d_Wtt, int nW, double *d_TT, void *cuda_stream)
{
    if (!tables || !d_Wtt || !d_TT) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    return run_coupling(tables, -1, d_Wtt, nullptr, nullptr, nW, d_TT, nullptr, nullptr, nullptr, nullptr,
                        (cudaStream_t)cuda_stream);
}

int tj_coupling_pol(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                    double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, void *cuda_stream)
{
    if (!tables) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    return run_coupling(tables, -1, d_Wtt, d_Wtp, d_Wpp, nW, d_TT, d_TE, d_EE, d_BB, d_EB, (cudaStream_t)cuda_stream);
}

int tj_coupling_pol_static(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                           double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, void *cuda_stream)
{
    if (!tables) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    return run_coupling_static(tables, d_Wtt, d_Wtp, d_Wpp, nW, d_TT, d_TE, d_EE, d_BB, d_EB, (cudaStream_t)cuda_stream);
}

int tj_coupling_band(const tj_tables *tables, int lcut, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                     double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, void *cuda_stream)
{
    if (!tables) return TJ_EINVAL;
    if (lcut < 0 || lcut > 2 * tables->T.lmax) return TJ_EINVAL;
    return run_coupling(tables, lcut, d_Wtt, d_Wtp, d_Wpp, lcut + 1, d_TT, d_TE, d_EE, d_BB, d_EB,
                        (cudaStream_t)cuda_stream);
}

int tj_coupling_multi(const tj_tables *tables, int nwin, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                      int nW, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, void *cuda_stream)
{
    if (!tables || nwin < 1) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t per = ((size_t)tables->T.lmax + 1) * ((size_t)tables->T.lmax + 1);
    // the batched sweep is instantiated for the full set of blocks; any other request runs one window set at a time
    const bool full = d_Wtt && d_Wtp && d_Wpp && d_TT && d_TE && (d_EE || d_BB) && d_EB;
    // TT alone (many temperature map pairs, covariance windows): four windows per sweep, then two, then one
    const bool tt_only = d_Wtt && d_TT && !d_TE && !d_EE && !d_BB && !d_EB;
    int w = 0;
    while (w < nwin) {
        // groups of three window sets per sweep; a remainder of 4 goes as 2 + 2, of 2 as one pair
        const int left = nwin - w;
        const int nw = tt_only ? (left >= 4 ? 4 : left >= 2 ? 2 : 1)
                               : !full ? 1 : (left == 4 || left == 2) ? 2 : left >= 3 ? 3 : 1;
        const size_t wi = (size_t)w * (size_t)nW, oi = (size_t)w * per;
        int rc = run_coupling(tables, -1, d_Wtt ? d_Wtt + wi : nullptr, d_Wtp ? d_Wtp + wi : nullptr,
                              d_Wpp ? d_Wpp + wi : nullptr, nW, d_TT ? d_TT + oi : nullptr, d_TE ? d_TE + oi : nullptr,
                              d_EE ? d_EE + oi : nullptr, d_BB ? d_BB + oi : nullptr, d_EB ? d_EB + oi : nullptr, st, nw);
        if (rc != TJ_OK) return rc;
        w += nw;
    }
    return TJ_OK;
}

int tj_coupling_spin1(const tj_tables *tables, const double *d_W00, const double *d_W01, const double *d_W11, int nW,
                      double *d_K00, double *d_K01, double *d_K11p, double *d_K11m, void *cuda_stream)
{
    if (!tables) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    // same sweep, spin-1 algebra: K00 rides in the TT slot, K01 in TE, K11+ in EE, K11- in EB
    return run_coupling(tables, -1, d_W00, d_W01, d_W11, nW, d_K00, d_K01, d_K11p, nullptr, d_K11m,
                        (cudaStream_t)cuda_stream, 1, 1);
}

int tj_coupling_rows(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                     int row_lo, int row_hi, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                     void *cuda_stream)
{
    if (!tables) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    if (row_lo < 0 || row_hi <= row_lo || row_hi > tables->T.lmax + 1) return TJ_EINVAL;
    return run_rows(tables, d_Wtt, d_Wtp, d_Wpp, nW, row_lo, row_hi, d_TT, d_TE, d_EE, d_BB, d_EB, (cudaStream_t)cuda_stream);
}

int tj_coupling_binned(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                       int nbins, const int *h_edges, const double *d_P, const double *d_Q, double *d_TT, double *d_TE,
                       double *d_EE, double *d_BB, double *d_EB, void *cuda_stream)
{
    if (!tables || !h_edges || !d_P || !d_Q || nbins < 1 || nbins > 46340) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    if (h_edges[0] < 0 || h_edges[nbins] > tables->T.lmax + 1) return TJ_EINVAL;
    for (int b = 0; b < nbins; ++b)
        if (h_edges[b + 1] < h_edges[b]) return TJ_EINVAL;
    return run_binned(tables, d_Wtt, d_Wtp, d_Wpp, nW, nbins, h_edges, d_P, d_Q, d_TT, d_TE, d_EE, d_BB, d_EB,
                      (cudaStream_t)cuda_stream);
}

int tj_coupling_binned_multi(const tj_tables *tables, int nwin, const double *d_Wtt, const double *d_Wtp,
                             const double *d_Wpp, int nW, int nbins, const int *h_edges, const double *d_P,
                             const double *d_Q, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                             void *cuda_stream)
{
    if (!tables || nwin < 1 || !h_edges || !d_P || !d_Q || nbins < 1 || nbins > 46340) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    if (h_edges[0] < 0 || h_edges[nbins] > tables->T.lmax + 1) return TJ_EINVAL;
    for (int b = 0; b < nbins; ++b)
        if (h_edges[b + 1] < h_edges[b]) return TJ_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nb2 = (size_t)nbins * (size_t)nbins;
    // grouping as tj_coupling_multi: the batched sweeps exist for the full set of blocks (3 or 2 window sets) and for TT
    // alone (4 or 2); any other request is binned one window set at a time
    const bool full = d_Wtt && d_Wtp && d_Wpp && d_TT && d_TE && (d_EE || d_BB) && d_EB;
    const bool tt_only = d_Wtt && d_TT && !d_TE && !d_EE && !d_BB && !d_EB;
    int w = 0;
    while (w < nwin) {
        const int left = nwin - w;
        const int nw = tt_only ? (left >= 4 ? 4 : left >= 2 ? 2 : 1)
                               : !full ? 1 : (left == 4 || left == 2) ? 2 : left >= 3 ? 3 : 1;
        const size_t wi = (size_t)w * (size_t)nW, oi = (size_t)w * nb2;
        int rc = run_binned(tables, d_Wtt ? d_Wtt + wi : nullptr, d_Wtp ? d_Wtp + wi : nullptr, d_Wpp ? d_Wpp + wi : nullptr,
                            nW, nbins, h_edges, d_P, d_Q, d_TT ? d_TT + oi : nullptr, d_TE ? d_TE + oi : nullptr,
                            d_EE ? d_EE + oi : nullptr, d_BB ? d_BB + oi : nullptr, d_EB ? d_EB + oi : nullptr, st, nw);
        if (rc != TJ_OK) return rc;
        w += nw;
    }
    return TJ_OK;
}

int tj_coupling_literal(const tj_tables *tables, const double *d_Wtt, const double *d_Wpp, int nW, double *d_TT,
                        double *d_EE, void *cuda_stream)
{
    if (!tables || (!d_TT && !d_EE)) return TJ_EINVAL;
    if (nW != tables->T.l3max + 1) return TJ_EINVAL;
    if ((d_TT && !d_Wtt) || (d_EE && !d_Wpp)) return TJ_EINVAL;
    if (tables->T.lmax > 65534) return TJ_EINVAL;   // grid.y = lmax+1
    return run_literal(tables, d_Wtt, d_Wpp, nW, d_TT, d_EE, (cudaStream_t)cuda_stream);
}

int tj_coupling_host(const tj_tables *tables, int band, int nW_or_lcut, const double *h_Wtt, const double *h_Wtp,
                     const double *h_Wpp, double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                     void *cuda_stream)
{
    if (!tables || nW_or_lcut < 0) return TJ_EINVAL;
    const Tables &T = tables->T;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int lcut = band ? nW_or_lcut : -1;
    const int nW = band ? nW_or_lcut + 1 : nW_or_lcut;
    if (!band && nW != T.l3max + 1) return TJ_EINVAL;
    if (band && lcut > 2 * T.lmax) return TJ_EINVAL;
    const size_t N = (size_t)T.lmax + 1;
    const size_t per = band ? N * (size_t)(2 * lcut + 1) : N * N;
    const double *hw[3] = {h_Wtt, h_Wtp, h_Wpp};
    double *ho[5] = {h_TT, h_TE, h_EE, h_BB, h_EB};
    // BB is a copy of EE: when both are requested compute one matrix and copy it out twice
    const bool bb_from_ee = (h_EE && h_BB);
    int nout = 0;
    for (int k = 0; k < 5; ++k) if (ho[k] && !(k == 3 && bb_from_ee)) ++nout;
    if (nout == 0) return TJ_EINVAL;
    { const int rcd = check_device(tables); if (rcd != TJ_OK) return rcd; }
    double *dw = nullptr, *dout = nullptr;
    TJ_CUDA(cudaMallocAsync((void **)&dw, sizeof(double) * 3 * (size_t)nW, st), "tj_coupling_host/alloc windows");
    cudaError_t e = cudaMallocAsync((void **)&dout, sizeof(double) * per * (size_t)nout, st);
    if (e != cudaSuccess) { cudaFreeAsync(dw, st); return cuda_fail(e, "tj_coupling_host/alloc outputs"); }
    const double *dwp[3] = {nullptr, nullptr, nullptr};
    for (int k = 0; k < 3; ++k) {
        if (!hw[k]) continue;
        dwp[k] = dw + (size_t)k * nW;
        e = cudaMemcpyAsync((void *)dwp[k], hw[k], sizeof(double) * (size_t)nW, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) break;
    }
    double *dop[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    int rc = TJ_OK;
    if (e == cudaSuccess) {
        int j = 0;
        for (int k = 0; k < 5; ++k)
            if (ho[k] && !(k == 3 && bb_from_ee)) dop[k] = dout + per * (size_t)(j++);
        // The chunked pipeline needs copies that are asynchronous to the host: into pageable memory every
        // cudaMemcpy(2D)Async blocks the issuing thread until the copy is done, so chunk k+1 would not even be enqueued
        // before copy k has finished and the pipeline would run as compute, copy, compute, copy.  With any pageable
        // output the call therefore computes first and then copies each matrix out in one piece.
        bool pageable = false;
        for (int k = 0; k < 5 && !pageable; ++k) {
            if (!ho[k]) continue;
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, ho[k]) != cudaSuccess) { cudaGetLastError(); pageable = true; }
            else pageable = (at.type == cudaMemoryTypeUnregistered);
        }
        if (!band && !use_small_path(T, -1, 1, 2) && !pageable) {
            // dense: sweep, writer and the copies to the host pipelined by row chunks
            rc = run_coupling_rows_to_host(tables, dwp[0], dwp[1], dwp[2], nW, dop, ho, st);
        } else {
            if (!band && !use_small_path(T, -1, 1, 2)) {
                HostPipe &pipe = const_cast<tj_tables *>(tables)->pipe;
                std::lock_guard<std::mutex> lock(pipe.mu);
                pipe.last_regime = 3;
                pipe.last_chunks = 1;
            }
            rc = run_coupling(tables, lcut, dwp[0], dwp[1], dwp[2], nW, dop[0], dop[1], dop[2], dop[3], dop[4], st);
            if (rc == TJ_OK) {
                for (int k = 0; k < 5 && e == cudaSuccess; ++k) {
                    const double *src = (k == 3 && bb_from_ee) ? dop[2] : dop[k];
                    if (ho[k]) e = cudaMemcpyAsync(ho[k], src, sizeof(double) * per, cudaMemcpyDeviceToHost, st);
                }
            }
        }
    }
    cudaFreeAsync(dout, st);
    cudaFreeAsync(dw, st);
    cudaError_t es = cudaStreamSynchronize(st);
    if (rc != TJ_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "tj_coupling_host/copies");
    if (es != cudaSuccess) return cuda_fail(es, "tj_coupling_host/sync");
    return TJ_OK;
}

int tj_chunk_plan(int lmax, int tt_only, int nparts, int *h_bounds, int *h_owner, int *nchunks)
{
    if (lmax < 0 || nparts < 1 || nparts > PLAN_MAX_PARTS || !h_bounds || !h_owner || !nchunks) return TJ_EINVAL;
    const int R = sweep_R(tt_only ? M_TT : (M_TT | M_TE | M_EE | M_EB), false, 1, lmax, false, 2);
    *nchunks = chunk_plan(lmax, R, nparts, h_bounds, h_owner);
    return TJ_OK;
}

}  // extern "C"

namespace {

// one device's share of a dense host-buffer call, enqueued but not waited for (tj_coupling_host_part / _multi)
struct PartCall {
    double *dw = nullptr, *dout = nullptr;
    cudaStream_t st = nullptr;
    int rc = TJ_OK;
};

// the handle's device must be current
void part_enqueue(PartCall &pc, const tj_tables *tables, int part, int nparts, int nW, const double *const hw[3],
                  double *const ho[5], cudaStream_t st)
{
    const Tables &T = tables->T;
    pc.st = st;
    pc.rc = check_device(tables);
    if (pc.rc != TJ_OK) return;
    const size_t N = (size_t)T.lmax + 1, per = N * N;
    const bool bb_from_ee = (ho[2] && ho[3]);
    int nout = 0;
    for (int k = 0; k < 5; ++k) if (ho[k] && !(k == 3 && bb_from_ee)) ++nout;
    cudaError_t e = cudaMallocAsync((void **)&pc.dw, sizeof(double) * 3 * (size_t)nW, st);
    if (e == cudaSuccess) e = cudaMallocAsync((void **)&pc.dout, sizeof(double) * per * (size_t)nout, st);
    const double *dwp[3] = {nullptr, nullptr, nullptr};
    for (int k = 0; k < 3 && e == cudaSuccess; ++k) {
        if (!hw[k]) continue;
        dwp[k] = pc.dw + (size_t)k * nW;
        e = cudaMemcpyAsync((void *)dwp[k], hw[k], sizeof(double) * (size_t)nW, cudaMemcpyHostToDevice, st);
    }
    if (e != cudaSuccess) { pc.rc = cuda_fail(e, "tj_coupling_host_part/set-up"); return; }
    double *dop[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    int j = 0;
    for (int k = 0; k < 5; ++k)
        if (ho[k] && !(k == 3 && bb_from_ee)) dop[k] = pc.dout + per * (size_t)(j++);
    pc.rc = run_coupling_rows_to_host(tables, dwp[0], dwp[1], dwp[2], nW, dop, ho, st, part, nparts);
}

// frees the part's device memory (stream-ordered) and waits for its stream; the handle's device must be current
void part_finish(PartCall &pc)
{
    if (pc.dout) cudaFreeAsync(pc.dout, pc.st);
    if (pc.dw) cudaFreeAsync(pc.dw, pc.st);
    pc.dout = pc.dw = nullptr;
    cudaError_t es = cudaStreamSynchronize(pc.st);
    if (pc.rc == TJ_OK && es != cudaSuccess) pc.rc = cuda_fail(es, "tj_coupling_host_part/sync");
}

int part_args_ok(const tj_tables *tables, int nW, double *const ho[5])
{
    if (!tables || nW != tables->T.l3max + 1) return 0;
    if (!ho[0] && !ho[1] && !ho[2] && !ho[3] && !ho[4]) return 0;
    return 1;
}

}  // namespace

extern "C" {

int tj_coupling_host_part(const tj_tables *tables, int part, int nparts, int nW, const double *h_Wtt, const double *h_Wtp,
                          const double *h_Wpp, double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                          void *cuda_stream)
{
    const double *hw[3] = {h_Wtt, h_Wtp, h_Wpp};
    double *ho[5] = {h_TT, h_TE, h_EE, h_BB, h_EB};
    if (nparts < 1 || nparts > PLAN_MAX_PARTS || part < 0 || part >= nparts || !part_args_ok(tables, nW, ho)) return TJ_EINVAL;
    PartCall pc;
    part_enqueue(pc, tables, part, nparts, nW, hw, ho, (cudaStream_t)cuda_stream);
    part_finish(pc);
    return pc.rc;
}

int tj_coupling_host_multi(tj_tables *const *tables, int ndev, int nW, const double *h_Wtt, const double *h_Wtp,
                           const double *h_Wpp, double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                           void *const *cuda_streams)
{
    const double *hw[3] = {h_Wtt, h_Wtp, h_Wpp};
    double *ho[5] = {h_TT, h_TE, h_EE, h_BB, h_EB};
    if (!tables || ndev < 1 || ndev > PLAN_MAX_PARTS) return TJ_EINVAL;
    for (int g = 0; g < ndev; ++g) {
        if (!part_args_ok(tables[g], nW, ho) || tables[g]->T.lmax != tables[0]->T.lmax) return TJ_EINVAL;
        for (int q = 0; q < g; ++q)
            if (tables[q] == tables[g]) return TJ_EINVAL;   // one handle per part: each owns the side streams of its share
    }
    int dev0 = -1;
    TJ_CUDA(cudaGetDevice(&dev0), "tj_coupling_host_multi/cudaGetDevice");
    PartCall pc[PLAN_MAX_PARTS];
    int rc = TJ_OK;
    // enqueue every device's share (nothing here waits for a GPU), then wait for them one by one
    for (int g = 0; g < ndev; ++g) {
        cudaError_t e = cudaSetDevice(tables[g]->device);
        if (e != cudaSuccess) { pc[g].rc = cuda_fail(e, "tj_coupling_host_multi/cudaSetDevice"); continue; }
        part_enqueue(pc[g], tables[g], g, ndev, nW, hw, ho, cuda_streams ? (cudaStream_t)cuda_streams[g] : nullptr);
    }
    for (int g = 0; g < ndev; ++g) {
        if (cudaSetDevice(tables[g]->device) == cudaSuccess) part_finish(pc[g]);
        if (rc == TJ_OK) rc = pc[g].rc;
    }
    cudaSetDevice(dev0);
    return rc;
}

int tj_set_host_pipeline(tj_tables *tables, double d2h_bytes_per_s, double fp64_instr_per_s)
{
    if (!tables || !(d2h_bytes_per_s >= 0.0) || !(fp64_instr_per_s >= 0.0)) return TJ_EINVAL;   // NaN fails both
    std::lock_guard<std::mutex> lock(tables->pipe.mu);
    tables->pipe.copy_rate = d2h_bytes_per_s > 0.0 ? d2h_bytes_per_s : HOST_COPY_RATE_DEFAULT;
    tables->pipe.instr_rate = fp64_instr_per_s > 0.0 ? fp64_instr_per_s : HOST_INSTR_RATE_DEFAULT;
    return TJ_OK;
}

int tj_host_pipeline_info(const tj_tables *tables, int *regime, int *nchunks)
{
    if (!tables) return TJ_EINVAL;
    HostPipe &pipe = const_cast<tj_tables *>(tables)->pipe;
    std::lock_guard<std::mutex> lock(pipe.mu);
    if (regime) *regime = pipe.last_regime;
    if (nchunks) *nchunks = pipe.last_chunks;
    return TJ_OK;
}

int tj_l3_range(int l1, int l2, int l3max, int parity, int *l3_lo, int *l3_hi, int *nterms)
{
    if (l1 < 0 || l2 < 0 || l3max < 0 || (parity != 0 && parity != 1)) return TJ_EINVAL;
    // expressed through the step indices the kernel walks (tj_sweep_counts): l3 = s-2t-parity
    int te_lo, te_hi, to_lo, to_hi;
    tj_sweep_counts(l1, l2, l3max, &te_lo, &te_hi, &to_lo, &to_hi);
    const int s = l1 + l2;
    const int t_lo = parity ? to_lo : te_lo, t_hi = parity ? to_hi : te_hi;
    int n = t_hi - t_lo + 1;
    int lo = s - 2 * t_hi - parity, hi = s - 2 * t_lo - parity;
    if (n <= 0) { n = 0; hi = lo - 2; }   // empty: hi < lo
    if (l3_lo) *l3_lo = lo;
    if (l3_hi) *l3_hi = hi;
    if (nterms) *nterms = n;
    return TJ_OK;
}

int tj_sweep_counts(int l1, int l2, int l3max, int *te_lo, int *te_hi, int *to_lo, int *to_hi)
{
    if (l1 < 0 || l2 < 0 || l3max < 0) return TJ_EINVAL;
    const int s = l1 + l2, mn = l1 < l2 ? l1 : l2;
    int a = s - l3max;          // even: s-2t <= l3max
    a = a > 0 ? (a + 1) >> 1 : 0;
    int b = s - 1 - l3max;      // odd:  s-2t-1 <= l3max
    b = b > 0 ? (b + 1) >> 1 : 0;
    if (te_lo) *te_lo = a;
    if (te_hi) *te_hi = mn;
    if (to_lo) *to_lo = b;
    if (to_hi) *to_hi = mn - 1;
    return TJ_OK;
}

int tj_profile_enable(int on)
{
    g_profile.store(on ? 1 : 0);
    return TJ_OK;
}

int tj_profile_get(double *h_ms3)
{
    if (!h_ms3) return TJ_EINVAL;
    if (g_prof.cur < 0 || !g_prof.valid || !g_prof.dev[g_prof.cur].have) return TJ_EINVAL;
    const cudaEvent_t *ev = g_prof.dev[g_prof.cur].ev;
    TJ_CUDA(cudaEventSynchronize(ev[4]), "tj_profile_get");
    float a = 0.f, b = 0.f, c = 0.f;
    TJ_CUDA(cudaEventElapsedTime(&a, ev[0], ev[1]), "tj_profile_get");
    TJ_CUDA(cudaEventElapsedTime(&b, ev[2], ev[3]), "tj_profile_get");
    TJ_CUDA(cudaEventElapsedTime(&c, ev[3], ev[4]), "tj_profile_get");
    h_ms3[0] = a; h_ms3[1] = b; h_ms3[2] = c;
    return TJ_OK;
}

int tj_profile_last_sweep(int *h_geo10)
{
    if (!h_geo10) return TJ_EINVAL;
    const SweepGeometry &G = g_last_sweep;
    const int v[10] = {G.R, G.mask, G.TS, G.minb, G.pipe, G.nw, G.spin, G.rows, G.diag, G.tiles};
    memcpy(h_geo10, v, sizeof(v));
    return G.R > 0 ? TJ_OK : TJ_EINVAL;
}

int tj_profile_launches(long long *h_count)
{
    if (!h_count) return TJ_EINVAL;
    *h_count = g_launch_count;
    return TJ_OK;
}

}  // extern "C"

namespace {

// ---- one coupling call, in pieces (the host-buffer path launches the middle two per row chunk) -------------
int coupling_begin(Call &C, const tj_tables *tables, int lcut, const double *d_Wtt, const double *d_Wtp,
                   const double *d_Wpp, int nW, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                   cudaStream_t st, int nw = 1, int spin = 2, int row_lo = -1, int row_hi = -1)
{
    const Tables &T = tables->T;
    { const int rcd = check_device(tables); if (rcd != TJ_OK) return rcd; }
    g_prof.valid = false;   // set again when this call has recorded all of its events
    C.T = &T;
    C.nw = nw;
    C.spin = spin;
    C.nW = nW;
    C.banded = lcut >= 0;
    C.lcut = lcut;
    // an output needs its window (TJ_EINVAL otherwise)
    if ((d_TT && !d_Wtt) || (d_TE && !d_Wtp) || ((d_EE || d_BB || d_EB) && !d_Wpp)) return TJ_EINVAL;
    if (!d_TT && !d_TE && !d_EE && !d_BB && !d_EB) return TJ_EINVAL;
    // EE target: EE if given, else BB takes the even spin-2 block directly
    C.TT = d_TT; C.TE = d_TE; C.EB = d_EB;
    C.ee = d_EE ? d_EE : d_BB;
    C.bb_copy = (d_EE && d_BB) ? d_BB : nullptr;
    // smallest instantiated sweep that covers the request
    if (!d_TE && !C.ee && !d_EB) C.mask = M_TT;
    else if (d_TT) C.mask = M_TT | M_TE | M_EE | M_EB;
    else C.mask = M_TE | M_EE | M_EB;
    C.R = sweep_R(C.mask, C.banded, nw, T.lmax, row_lo >= 0, spin);
    C.l3max_eff = C.banded ? lcut : T.l3max;
    C.N = (long long)T.lmax + 1;
    C.rows = row_lo >= 0;
    C.row_lo = C.rows ? row_lo : 0;
    C.row_hi = C.rows ? row_hi : T.lmax + 1;
    C.ld = C.banded ? (long long)(2 * lcut + 1) : C.N;
    C.dmax = C.banded ? (lcut < T.lmax ? lcut : T.lmax) : 0;
    C.ldT = (C.N + 15) & ~15LL;
    if (C.banded) {
        const long long n = (long long)diag_num_groups(C.dmax, C.R) * diag_num_blocks(T.lmax, C.R);
        C.ntiles = n > 0x7fffffffLL ? -1 : (int)n;
    } else {
        C.ntiles = total_tiles(T.lmax, C.l3max_eff, C.R, false, C.row_lo, C.row_hi);
    }
    if (C.ntiles < 0) return TJ_EINVAL;
    C.nb = num_bands(T.lmax, C.R);
    C.ntile_w = (int)((C.N + 31) / 32);

    // ---- stream-ordered scratch: 3 prefolded windows + tile prefix
    // per window set: three plain prefolded arrays + two arrays of pairs (7 nl_alloc doubles)
    const size_t wbytes = sizeof(double) * WSET * (size_t)T.nl_alloc * (size_t)nw;
    const size_t tbytes = sizeof(int) * (size_t)(C.nb + 1 + 1);
    const size_t tb_al = (tbytes + 127) & ~(size_t)127;
    int nxit = 0;
    if (C.banded) nxit = (C.TT ? 1 : 0) + (C.TE ? 1 : 0) + (C.ee ? 1 : 0) + (C.EB ? 1 : 0);
    const size_t xper = (size_t)(C.dmax + 1) * (size_t)C.ldT;   // doubles per transposed Xi block
    TJ_CUDA(cudaMallocAsync((void **)&C.scratch, wbytes + tb_al + sizeof(double) * xper * (size_t)nxit, st), "coupling/scratch");
    for (int k = 0; k < nxit; ++k) C.xit[k] = (double *)(C.scratch + wbytes + tb_al) + xper * (size_t)k;
    C.wtt = (double *)C.scratch + GUARD_LO;
    C.wtp = C.wtt + T.nl_alloc;
    C.wpp = C.wtp + T.nl_alloc;
    C.wA = C.wpp - GUARD_LO + T.nl_alloc + 2 * GUARD_LO;
    C.wB = C.wA + 2 * (size_t)T.nl_alloc;
    C.tile_start = (int *)(C.scratch + wbytes);

    prof_record(0, st);
    cudaError_t e = cudaSuccess;
    for (int w = 0; w < nw && e == cudaSuccess; ++w) {   // window set w: inputs [w][nW], prefolded arrays 3*nl_alloc apart
        const size_t wi = (size_t)w * (size_t)nW, wo = (size_t)w * WSET * (size_t)T.nl_alloc;
        e = launch_prepare(T, d_Wtt ? d_Wtt + wi : nullptr, d_Wtp ? d_Wtp + wi : nullptr, d_Wpp ? d_Wpp + wi : nullptr,
                           nW, C.wtt + wo, C.wtp + wo, C.wpp + wo, C.wA + wo, C.wB + wo, C.tile_start, C.R, C.l3max_eff,
                           C.banded, C.row_lo, C.row_hi, st);
    }
    prof_record(1, st);
    if (e != cudaSuccess) { cudaFreeAsync(C.scratch, st); C.scratch = nullptr; return cuda_fail(e, "coupling/prepare"); }
    return TJ_OK;
}

// tiles of the descending-band prefix that precede band b (= tiles of all bands > b); host copy of what
// prepare_kernel writes to tile_start[]
int tiles_above(const Call &C, int b)
{
    long long n = 0;
    for (int k = C.nb - 1; k > b; --k) n += band_num_tiles(C.T->lmax, C.l3max_eff, C.R, k, C.banded, C.row_lo, C.row_hi);
    return (int)n;
}

// sweep of the row bands [b0, b1)
cudaError_t coupling_sweep(const Call &C, int b0, int b1, cudaStream_t st)
{
    const Tables &T = *C.T;
    SweepParams P;
    P.g = T.g; P.ginv = T.ginv; P.h = T.h; P.gA = T.gA; P.gB = T.gB; P.u3 = T.u3;
    P.isd = C.spin == 1 ? T.isu : T.isd;
    P.wtt = C.wtt; P.wtp = C.wtp; P.wpp = C.wpp; P.wA = C.wA; P.wB = C.wB;
    // a block the instantiated sweep computes but the caller did not ask for has a NULL target and is not stored
    P.TT = C.TT; P.TE = C.TE; P.EE = C.ee; P.EB = C.EB;
    P.BB = C.rows ? C.bb_copy : nullptr;
    P.tile_start = C.tile_start;
    P.lmax = T.lmax; P.l3max = C.l3max_eff; P.nbands = C.nb; P.lcut = C.banded ? C.lcut : -1; P.ld = C.ld;
    P.nd = diag_num_blocks(T.lmax, C.R);
    if (C.banded) {   // diagonal tiling: Xi goes to the transposed scratch
        int k = 0;
        if (C.TT) P.TT = C.xit[k++];
        if (C.TE) P.TE = C.xit[k++];
        if (C.ee) P.EE = C.xit[k++];
        if (C.EB) P.EB = C.xit[k++];
        P.ld = C.ldT;
    }
    const bool all = (b0 == 0 && b1 == C.nb);
    P.tile_off = all ? 0 : tiles_above(C, b1 - 1);
    P.wstride = WSET * (long long)T.nl_alloc;
    P.row_lo = C.row_lo; P.row_hi = C.row_hi; P.rows = C.rows ? 1 : 0;
    P.ostride = C.ostride ? C.ostride : C.N * C.ld;
    const int n = all ? C.ntiles : tiles_above(C, b0 - 1) - P.tile_off;
    return launch_sweep(P, C.mask, C.nw, C.mask == M_TT ? 2 : C.spin, n, st);
}

// scale + mirror of the 32-row tile rows [I0, I1)
cudaError_t coupling_write(const Call &C, int I0, int I1, cudaStream_t st)
{
    if (C.banded) {
        BandWriterParams B;
        memset(&B, 0, sizeof(B));
        int n = 0;
        B.bb_src = -1;
        if (C.TT) { B.X[n] = C.xit[n]; B.M[n] = C.TT; ++n; }
        if (C.TE) { B.X[n] = C.xit[n]; B.M[n] = C.TE; ++n; }
        if (C.ee) { if (C.bb_copy) { B.bb = C.bb_copy; B.bb_src = n; } B.X[n] = C.xit[n]; B.M[n] = C.ee; ++n; }
        if (C.EB) { B.X[n] = C.xit[n]; B.M[n] = C.EB; ++n; }
        B.nmat = n;
        B.lmax = C.T->lmax; B.lcut = C.lcut; B.dmax = C.dmax; B.ldT = C.ldT; B.ld = C.ld;
        return launch_band_writer(B, st);
    }
    WriterParams W;
    memset(&W, 0, sizeof(W));
    int n = 0;
    W.bb = nullptr; W.bb_src = -1;
    if (C.TT) W.M[n++] = C.TT;
    if (C.TE) W.M[n++] = C.TE;
    if (C.ee) { if (C.bb_copy) { W.bb = C.bb_copy; W.bb_src = n; } W.M[n++] = C.ee; }
    if (C.EB) W.M[n++] = C.EB;
    W.nmat = n;
    W.lmax = C.T->lmax; W.lcut = -1; W.ld = C.ld;
    W.ntile = C.ntile_w;
    W.tile_band = W.ntile - 1;
    W.I0 = I0; W.I1 = I1;
    cudaError_t e = cudaSuccess;
    for (int w = 0; w < C.nw && e == cudaSuccess; ++w) {
        e = launch_writer(W, st);
        for (int k = 0; k < W.nmat; ++k) W.M[k] += C.N * C.ld;
        if (W.bb) W.bb += C.N * C.ld;
    }
    return e;
}

void coupling_end(Call &C, cudaStream_t st)
{
    if (C.scratch) cudaFreeAsync(C.scratch, st);
    C.scratch = nullptr;
}

int run_coupling(const tj_tables *tables, int lcut, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                 int nW, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st, int nw,
                 int spin)
{
    if (use_small_path(tables->T, lcut, nw, spin)) {
        // single-launch path (tj_small.cu): no scratch, no tile list
        { const int rcd = check_device(tables); if (rcd != TJ_OK) return rcd; }
        if ((d_TT && !d_Wtt) || (d_TE && !d_Wtp) || ((d_EE || d_BB || d_EB) && !d_Wpp)) return TJ_EINVAL;
        if (!d_TT && !d_TE && !d_EE && !d_BB && !d_EB) return TJ_EINVAL;
        const int mask = (!d_TE && !d_EE && !d_BB && !d_EB) ? M_TT : (d_TT ? M_TT : 0) | M_TE | M_EE | M_EB;
        g_prof.valid = false;
        prof_record(0, st); prof_record(1, st); prof_record(2, st);
        cudaError_t e = launch_small(tables->T, mask, d_Wtt, d_Wtp, d_Wpp, nW, d_TT, d_TE, d_EE, d_BB, d_EB, st);
        prof_record(3, st); prof_record(4, st);
        return e == cudaSuccess ? TJ_OK : cuda_fail(e, "coupling/small");
    }
    Call C;
    int rc = coupling_begin(C, tables, lcut, d_Wtt, d_Wtp, d_Wpp, nW, d_TT, d_TE, d_EE, d_BB, d_EB, st, nw, spin);
    if (rc != TJ_OK) return rc;
    prof_record(2, st);
    cudaError_t e = coupling_sweep(C, 0, C.nb, st);
    prof_record(3, st);
    if (e == cudaSuccess) e = coupling_write(C, 0, C.ntile_w, st);
    prof_record(4, st);
    if (e != cudaSuccess) rc = cuda_fail(e, "coupling");
    coupling_end(C, st);
    return rc;
}
// full rows [row_lo, row_hi) of every requested block, compact outputs (tj_coupling_rows)
int run_rows(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW, int row_lo,
             int row_hi, double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st)
{
    Call C;
    int rc = coupling_begin(C, tables, -1, d_Wtt, d_Wtp, d_Wpp, nW, d_TT, d_TE, d_EE, d_BB, d_EB, st, 1, 2, row_lo, row_hi);
    if (rc != TJ_OK) return rc;
    prof_record(2, st);
    cudaError_t e = coupling_sweep(C, 0, C.nb, st);
    prof_record(3, st);
    prof_record(4, st);
    if (e != cudaSuccess) rc = cuda_fail(e, "tj_coupling_rows");
    coupling_end(C, st);
    return rc;
}

// binned output (tj_binned.cu): the sweep runs over chunks of rows into Xi scratch, bin_kernel adds each chunk to the bins
// nw > 1 (tj_coupling_binned_multi): windows [nw][nW], outputs [nw][nbins^2]; the batched sweep leaves the nw Xi chunks
// of a block one after the other in its chunk buffer and every window set is binned from its own
int run_binned(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW, int nbins,
               const int *h_edges, const double *d_P, const double *d_Q, double *d_TT, double *d_TE, double *d_EE,
               double *d_BB, double *d_EB, cudaStream_t st, int nw)
{
    const Tables &T = tables->T;
    const long long N = (long long)T.lmax + 1;
    double *outs[4] = {d_TT, d_TE, d_EE ? d_EE : d_BB, d_EB};
    int nmat = 0;
    for (int k = 0; k < 4; ++k) nmat += outs[k] ? 1 : 0;
    if (nmat == 0) return TJ_EINVAL;
    if ((d_TT && !d_Wtt) || (d_TE && !d_Wtp) || ((d_EE || d_BB || d_EB) && !d_Wpp)) return TJ_EINVAL;
    // rows per chunk: whole row bands of the sweep, at most ~1 GiB of Xi scratch
    const int mask = (!d_TE && !outs[2] && !d_EB) ? M_TT : (d_TT ? M_TT : 0) | M_TE | M_EE | M_EB;
    const int R = sweep_R(mask, false, nw, T.lmax, false, 2);
    long long ch = ((1LL << 30) / (8 * N * nmat * nw)) / R * R;
    if (ch < R) ch = R;
    if (ch > N) ch = (N + R - 1) / R * R;
    const size_t xper = (size_t)ch * (size_t)N;
    const size_t ebytes = (sizeof(int) * (size_t)(nbins + 1) + 127) & ~(size_t)127;
    // a few wide bins: several CTAs per bin pair, their partial sums joined by a second pass (tj_binned.cu)
    const int split = launch_bin_split(nbins);
    const size_t pbytes = split > 1 ? (sizeof(double) * 2 * (size_t)split * (size_t)nmat * ((size_t)nbins * (nbins + 1) / 2) + 127) & ~(size_t)127 : 0;
    unsigned char *scr = nullptr;
    TJ_CUDA(cudaMallocAsync((void **)&scr, ebytes + pbytes + sizeof(double) * xper * (size_t)nmat * (size_t)nw, st), "tj_coupling_binned/scratch");
    int *d_edges = (int *)scr;
    double *xb = (double *)(scr + ebytes + pbytes);
    cudaError_t e = cudaMemcpyAsync(d_edges, h_edges, sizeof(int) * (size_t)(nbins + 1), cudaMemcpyHostToDevice, st);
    // the sweep's targets: one chunk buffer per requested block, in the order TT, TE, EE, EB
    double *bufs[4] = {nullptr, nullptr, nullptr, nullptr};
    {
        int k = 0;
        for (int m = 0; m < 4; ++m)
            if (outs[m]) bufs[m] = xb + xper * (size_t)nw * (size_t)(k++);
    }
    const size_t nb2 = (size_t)nbins * (size_t)nbins;
    Call C;
    int rc = TJ_OK;
    if (e == cudaSuccess) rc = coupling_begin(C, tables, -1, d_Wtt, d_Wtp, d_Wpp, nW, bufs[0], bufs[1], bufs[2], nullptr, bufs[3], st, nw);
    if (e == cudaSuccess && rc == TJ_OK) {
        C.ostride = (long long)xper;   // window set w of a block: its chunk buffer + w * xper
        BinParams B;
        memset(&B, 0, sizeof(B));
        double *bout[4] = {nullptr, nullptr, nullptr, nullptr};
        for (int m = 0; m < 4 && e == cudaSuccess; ++m) {
            if (!outs[m]) continue;
            bout[B.nmat++] = outs[m];
            e = cudaMemsetAsync(outs[m], 0, sizeof(double) * nb2 * (size_t)nw, st);
        }
        B.edges = d_edges; B.P = d_P; B.Q = d_Q; B.nbins = nbins; B.lmax = T.lmax; B.ld = N;
        B.split = split; B.part = split > 1 ? (double *)(scr + ebytes) : nullptr;
        prof_record(2, st);
        for (long long r0 = 0; r0 < N && e == cudaSuccess; r0 += ch) {
            const long long r1 = r0 + ch < N ? r0 + ch : N;
            // the sweep addresses Xi(l1,l2) as base[l1*N + l2]: shift the bases so that row r0 is row 0 of the chunk
            double **tgt[4] = {&C.TT, &C.TE, &C.ee, &C.EB};
            for (int m = 0; m < 4; ++m)
                if (outs[m]) *tgt[m] = bufs[m] - r0 * N;
            e = coupling_sweep(C, (int)(r0 / C.R), r1 == N ? C.nb : (int)(r1 / C.R), st);
            B.r0 = (int)r0; B.r1 = (int)r1;
            for (int w = 0; w < nw && e == cudaSuccess; ++w) {
                int k = 0;
                for (int m = 0; m < 4; ++m)
                    if (outs[m]) { B.X[k] = bufs[m] + (size_t)w * xper; B.B[k] = bout[k] + (size_t)w * nb2; ++k; }
                e = launch_bin(B, st);
            }
        }
        prof_record(3, st);
        if (e == cudaSuccess && d_EE && d_BB)
            e = cudaMemcpyAsync(d_BB, d_EE, sizeof(double) * nb2 * (size_t)nw, cudaMemcpyDeviceToDevice, st);
        prof_record(4, st);
        coupling_end(C, st);
    }
    cudaFreeAsync(scr, st);
    if (rc != TJ_OK) return rc;
    return e == cudaSuccess ? TJ_OK : cuda_fail(e, "tj_coupling_binned");
}

// ---- tj_coupling_pol_static: the dense call for callers that cannot allocate (include/tj.h) ------------------
// The scratch of a dense one-window call (WSET prefolded window arrays + the tile prefix) lives in this array
// instead of coming from cudaMallocAsync.  It is part of the module image: every device that loads libtj holds
// its own 2 MiB copy until the process ends.  Host code must never hand the NAME to a kernel -- on the host it
// stands for a shadow object, not for device memory; the device address comes from cudaGetSymbolAddress, asked once
// per device with that device current (static_scratch_ptr below).
static __device__ __align__(256) unsigned char g_static_scratch[TJ_STATIC_SCRATCH_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[STATIC_MAX_DEVICES];   // device address of g_static_scratch on device k (NULL: not asked yet)

// Device address of the array on `dev`, which must be the current device.  First use per device: one
// cudaGetSymbolAddress (it may load the module on that device, hence "before any stream capture" in tj.h).
int static_scratch_ptr(int dev, unsigned char **out)
{
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return TJ_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        unsigned char *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_static_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "tj_coupling_pol_static/cudaGetSymbolAddress");
        if (!ptr) return TJ_ECUDA;
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return TJ_OK;
}

// Same three kernels as the general path of run_coupling (prepare, staged sweep, mirrored writer), for the dense,
// one-window, spin-2 case only; the Call is filled here rather than by coupling_begin because that one allocates.
// Always the general path, whatever lmax: the single-launch kernel needs no scratch, but one code path keeps the
// contract simple (this is the variant of the scratch-using path, and its limit does not depend on a threshold).
int run_coupling_static(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                        double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB, cudaStream_t st)
{
    const Tables &T = tables->T;
    if ((d_TT && !d_Wtt) || (d_TE && !d_Wtp) || ((d_EE || d_BB || d_EB) && !d_Wpp)) return TJ_EINVAL;
    if (!d_TT && !d_TE && !d_EE && !d_BB && !d_EB) return TJ_EINVAL;
    if (T.lmax > TJ_STATIC_LMAX) return TJ_ELIMIT;
    { const int rcd = check_device(tables); if (rcd != TJ_OK) return rcd; }
    g_prof.valid = false;   // no events are recorded for this call

    Call C;
    C.T = &T;
    C.nW = nW;
    C.TT = d_TT; C.TE = d_TE; C.EB = d_EB;
    C.ee = d_EE ? d_EE : d_BB;
    C.bb_copy = (d_EE && d_BB) ? d_BB : nullptr;
    if (!d_TE && !C.ee && !d_EB) C.mask = M_TT;
    else if (d_TT) C.mask = M_TT | M_TE | M_EE | M_EB;
    else C.mask = M_TE | M_EE | M_EB;
    C.R = sweep_R(C.mask, false, 1, T.lmax, false, 2);
    C.l3max_eff = T.l3max;
    C.N = (long long)T.lmax + 1;
    C.row_lo = 0;
    C.row_hi = T.lmax + 1;
    C.ld = C.N;
    C.ntiles = total_tiles(T.lmax, C.l3max_eff, C.R, false, C.row_lo, C.row_hi);
    if (C.ntiles < 0) return TJ_EINVAL;
    C.nb = num_bands(T.lmax, C.R);
    C.ntile_w = (int)((C.N + 31) / 32);

    // layout of the array: [WSET * nl_alloc doubles: wtt, wtp, wpp, wA (pairs), wB (pairs)] [tile prefix, nb+1 ints]
    const size_t wbytes = sizeof(double) * WSET * (size_t)T.nl_alloc;
    const size_t tbytes = sizeof(int) * (size_t)(C.nb + 1 + 1);
    if (wbytes + tbytes > (size_t)TJ_STATIC_SCRATCH_BYTES) return TJ_ELIMIT;   // cannot happen for lmax <= TJ_STATIC_LMAX
    unsigned char *scr = nullptr;
    { const int rcs = static_scratch_ptr(tables->device, &scr); if (rcs != TJ_OK) return rcs; }
    C.wtt = (double *)scr + GUARD_LO;
    C.wtp = C.wtt + T.nl_alloc;
    C.wpp = C.wtp + T.nl_alloc;
    C.wA = C.wpp - GUARD_LO + T.nl_alloc + 2 * GUARD_LO;
    C.wB = C.wA + 2 * (size_t)T.nl_alloc;
    C.tile_start = (int *)(scr + wbytes);

    // prepare_kernel writes every element of the five window arrays (index -GUARD_LO .. nl_alloc-GUARD_LO-1, so the
    // guard bands too) and tile_start[0..nb]: nothing of an earlier call survives into what the sweep reads
    cudaError_t e = launch_prepare(T, d_Wtt, d_Wtp, d_Wpp, nW, C.wtt, C.wtp, C.wpp, C.wA, C.wB, C.tile_start, C.R,
                                   C.l3max_eff, false, C.row_lo, C.row_hi, st);
    if (e == cudaSuccess) e = coupling_sweep(C, 0, C.nb, st);
    if (e == cudaSuccess) e = coupling_write(C, 0, C.ntile_w, st);
    return e == cudaSuccess ? TJ_OK : cuda_fail(e, "tj_coupling_pol_static");
}

// paper-literal ablation (tj_literal.cu): prefold the windows, then one thread per pair
int run_literal(const tj_tables *tables, const double *d_Wtt, const double *d_Wpp, int nW, double *d_TT, double *d_EE,
                cudaStream_t st)
{
    Call C;
    int rc = coupling_begin(C, tables, -1, d_Wtt, nullptr, d_Wpp, nW, d_TT, nullptr, d_EE, nullptr, nullptr, st);
    if (rc != TJ_OK) return rc;
    cudaError_t e = launch_literal(*C.T, C.wtt, C.wpp, d_TT, d_EE, C.l3max_eff, st);
    if (e != cudaSuccess) rc = cuda_fail(e, "tj_coupling_literal");
    coupling_end(C, st);
    return rc;
}

// ---- dense call with HOST outputs, pipelined by row chunks ------------------------------------------------
// Full row l1 of a matrix is final once (i) the sweep and writer of its own row band have run (upper part
// and diagonal) and (ii) the writers of every band above it have run (they store the mirrored lower part).
// So the bands are processed in ASCENDING row chunks; after chunk k everything that chunk made final (see the
// copy loop) is copied to the host while chunk k+1 is computed.  Successive chunks alternate between two compute
// streams so that one chunk's last CTAs overlap the next chunk's first ones; within a chunk the tiles keep the
// descending (largest-first) order.
// Row chunks of a matrix shared by nparts devices (tj_chunk_plan): chunks of `rows` = a multiple of lcm(R, 32) rows, few
// enough that no device gets more than PIPE_MAX_CHUNKS of them, dealt to the devices by work -- the chunk with the most
// sweep steps (sum over its rows l1 of (l1+1)(N-l1)) first, each to the device with the least work so far, ties to the
// lower index.  bounds[0..n], owner[0..n-1]; returns n (<= PIPE_MAX_CHUNKS / 2 * nparts).
int chunk_plan(int lmax, int R, int nparts, int *bounds, int *owner)
{
    const long long N = (long long)lmax + 1;
    int L = R;
    while (L % 32) L += R;
    const long long units = (N + L - 1) / L;
    const long long cap = (long long)(PIPE_MAX_CHUNKS / 2) * nparts;   // 12 per device on average, never more than 24
    const long long rows = L * ((units + cap - 1) / cap);
    const int n = (int)((N + rows - 1) / rows);
    double work[PIPE_MAX_CHUNKS / 2 * PLAN_MAX_PARTS];
    for (int k = 0; k <= n; ++k) bounds[k] = (int)(k * rows < N ? k * rows : N);
    for (int k = 0; k < n; ++k) {
        double w = 0.0;
        for (long long l = bounds[k]; l < bounds[k + 1]; ++l) w += (double)(l + 1) * (double)(N - l);
        work[k] = w;
        owner[k] = -1;
    }
    double load[PLAN_MAX_PARTS] = {0.0};
    int count[PLAN_MAX_PARTS] = {0};
    for (int it = 0; it < n; ++it) {
        int best = -1;
        for (int k = 0; k < n; ++k)
            if (owner[k] < 0 && (best < 0 || work[k] > work[best])) best = k;
        int g = -1;
        for (int q = 0; q < nparts; ++q)
            if (count[q] < PIPE_MAX_CHUNKS && (g < 0 || load[q] < load[g])) g = q;
        owner[best] = g;
        load[g] += work[best];
        ++count[g];
    }
    return n;
}

int run_coupling_rows_to_host(const tj_tables *tables, const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                              int nW, double *const d_out[5], double *const h_out[5], cudaStream_t st, int part,
                              int nparts)
{
    HostPipe &pipe = const_cast<tj_tables *>(tables)->pipe;
    std::lock_guard<std::mutex> lock(pipe.mu);
    TJ_CUDA(pipe.ensure(), "host pipe");
    Call C;
    int rc = coupling_begin(C, tables, -1, d_Wtt, d_Wtp, d_Wpp, nW, d_out[0], d_out[1], d_out[2], d_out[3], d_out[4], st);
    if (rc != TJ_OK) return rc;

    // Which regime?  Device-to-host copies reach ~54 GB/s when contiguous and ~35 GB/s as pitched rectangles (measured on
    // this pool; the rates used below are the handle's, tj_set_host_pipeline).  A call whose copies take longer than its arithmetic even at the contiguous rate is
    // COPY-BOUND (config 2: 1.0 GB = 18.5 ms against 17.3 ms of compute): there every byte must move at the contiguous
    // rate and the copy engine must never wait, so whole rows go out, chunk after chunk, in many small chunks (a row
    // is final when its own chunk is done: its left part was mirrored there by the chunks above).  Otherwise the call
    // is COMPUTE-BOUND (config 3: 74 ms of copies behind 134 ms of compute) and what matters is a short tail: after
    // chunk k the L-shaped region it made final goes out (its rows from column r0 on, and columns [r0,r1) of all rows
    // below), so that the last rows, cheap to compute but as long as any other, are nearly all on the host already.
    int nmat_host = 0;
    for (int m = 0; m < 5; ++m) nmat_host += h_out[m] ? 1 : 0;
    const double copy_s = (double)nmat_host * (double)C.N * (double)C.N * 8.0 / pipe.copy_rate;
    const double n3 = (double)C.N * (double)C.N * (double)C.N / 6.0;   // even (and odd) steps of the upper triangle
    const double comp_s = (C.mask == M_TT ? 2.0 : 13.0) * n3 / pipe.instr_rate;
    // one part of several (tj_coupling_host_part / _multi): only the L-shaped regions are self-contained per chunk
    const bool rows_mode = nparts == 1 && copy_s > comp_s;
    // chunk ends as fractions of the rows.  Compute-bound: a first chunk of 20 % of the rows is 10 % of the work and
    // releases 36 % of the bytes (measured at config 3: 4 chunks 163 ms, 6 chunks 145 ms, these 10 chunks 135.4 ms;
    // device-buffer call 134.4 ms).  Copy-bound: 1 % first (the copy engine starts at once), then even steps; measured
    // at config 2 (floor: 1.0 GB at 54 GB/s = 18.5 ms): 8 chunks 25.9 ms, 13 chunks 22.2, 21 chunks 20.9, 24 chunks 20.5,
    // 32 chunks 22.1, 48 chunks 23.8 (the L-shaped scheme of the compute-bound case: 24.5 ms).
    static const double kFracL[] = {0.20, 0.35, 0.47, 0.57, 0.66, 0.74, 0.81, 0.88, 0.94, 1.0};
    double frac[PIPE_MAX_CHUNKS];
    int nfrac = 0;
    if (rows_mode) {
        frac[nfrac++] = 0.01;
        for (int k = 1; k <= 22; ++k) frac[nfrac++] = 0.01 + 0.98 * k / 22.0;
        frac[nfrac++] = 1.0;
    } else {
        for (double f : kFracL) frac[nfrac++] = f;
    }
    // chunk boundaries: multiples of lcm(R, 32) rows (whole row bands of the sweep, whole tile rows of the writer)
    int L = C.R;
    while (L % 32) L += C.R;
    int bound[PIPE_MAX_CHUNKS + 1];
    int nchunk = 0;
    bound[0] = 0;
    for (int k = 0; k < nfrac; ++k) {
        long long r = (k == nfrac - 1) ? C.N : (long long)(frac[k] * (double)C.N) / L * L;
        if (r > bound[nchunk]) bound[++nchunk] = (int)r;
    }
    // several parts: this part's chunks of the shared plan, in ascending row order (each with its own two bounds)
    int own_lo[PIPE_MAX_CHUNKS], own_hi[PIPE_MAX_CHUNKS];
    if (nparts > 1) {
        int pb[PIPE_MAX_CHUNKS / 2 * PLAN_MAX_PARTS + 1], po[PIPE_MAX_CHUNKS / 2 * PLAN_MAX_PARTS];
        const int n = chunk_plan(C.T->lmax, C.R, nparts, pb, po);
        nchunk = 0;
        for (int k = 0; k < n; ++k)
            if (po[k] == part) { own_lo[nchunk] = pb[k]; own_hi[nchunk] = pb[k + 1]; ++nchunk; }
    } else {
        for (int k = 0; k < nchunk; ++k) { own_lo[k] = bound[k]; own_hi[k] = bound[k + 1]; }
    }
    pipe.last_regime = nparts > 1 ? 4 : rows_mode ? 1 : 2;
    pipe.last_chunks = nchunk;
    cudaEvent_t *ev = pipe.ev;
    cudaEvent_t fork = ev[PIPE_MAX_CHUNKS], join = ev[PIPE_MAX_CHUNKS + 1];
    cudaError_t e = cudaEventRecord(fork, st);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaStreamWaitEvent(pipe.comp[k], fork, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe.copy, fork, 0);
    for (int k = 0; k < nchunk && e == cudaSuccess; ++k) {
        const int r0 = own_lo[k], r1 = own_hi[k];
        // successive chunks alternate between two compute streams: one chunk's last CTAs overlap the next one's first
        cudaStream_t cs = pipe.comp[k & 1];
        const int b1 = (r1 == C.N) ? C.nb : r1 / C.R;
        const int I1 = (r1 == C.N) ? C.ntile_w : r1 / 32;
        e = coupling_sweep(C, r0 / C.R, b1, cs);
        if (e == cudaSuccess) e = coupling_write(C, r0 / 32, I1, cs);
        if (e == cudaSuccess) e = cudaEventRecord(ev[k], cs);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe.copy, ev[k], 0);
        if (e == cudaSuccess && k > 0) e = cudaStreamWaitEvent(pipe.copy, ev[k - 1], 0);
        const size_t pitch = sizeof(double) * (size_t)C.N;
        for (int m = 0; m < 5 && e == cudaSuccess; ++m) {
            if (!h_out[m]) continue;
            const double *src = d_out[m] ? d_out[m] : d_out[2];   // BB without its own device matrix: the EE rows
            if (rows_mode) {
                const size_t o = (size_t)r0 * (size_t)C.N;
                e = cudaMemcpyAsync(h_out[m] + o, src + o, pitch * (size_t)(r1 - r0), cudaMemcpyDeviceToHost, pipe.copy);
                continue;
            }
            const size_t o1 = (size_t)r0 * (size_t)C.N + (size_t)r0;
            e = cudaMemcpy2DAsync(h_out[m] + o1, pitch, src + o1, pitch, sizeof(double) * (size_t)(C.N - r0),
                                  (size_t)(r1 - r0), cudaMemcpyDeviceToHost, pipe.copy);
            if (e == cudaSuccess && r1 < C.N) {
                const size_t o2 = (size_t)r1 * (size_t)C.N + (size_t)r0;
                e = cudaMemcpy2DAsync(h_out[m] + o2, pitch, src + o2, pitch, sizeof(double) * (size_t)(r1 - r0),
                                      (size_t)(C.N - r1), cudaMemcpyDeviceToHost, pipe.copy);
            }
        }
    }
    // join: the caller's stream continues after everything issued above.  If anything failed on the way, wait for
    // the whole device instead, so that no side stream still uses the scratch that is freed below.
    bool joined = e == cudaSuccess;
    for (int k = 0; k < 3 && joined; ++k) {
        cudaStream_t s = k < 2 ? pipe.comp[k] : pipe.copy;
        joined = cudaEventRecord(join, s) == cudaSuccess && cudaStreamWaitEvent(st, join, 0) == cudaSuccess;
    }
    if (!joined) cudaDeviceSynchronize();
    if (e != cudaSuccess) rc = cuda_fail(e, "coupling/host pipeline");
    coupling_end(C, st);
    return rc;
}

}  // namespace
