/*
 * tj.h -- C ABI of libtj: pseudo-C_ell mode-coupling matrices on one B200 (sm_100a), FP64.
 *
 * Method: arxiv/paper_2602_15605, "threej_cosmo": Wigner-3j symbols from a few
 * recurrence-generated lookup tables (PAPER.md:161-186 Eqs. 10-12; :188-220 Eqs. 13-16; App. B)
 * instead of a per-pair Schulten-Gordon recursion.  The formula sheet the kernels implement is
 * DESIGN.md section 3 (= SURVEY.md 8(c.1)).
 *
 * Conventions (all entry points)
 *   - Pointers named d_* are DEVICE pointers owned by the caller; h_* are HOST pointers.  The library
 *     never frees caller memory and never keeps a caller pointer after the call's work has been
 *     enqueued.  Outputs are fully overwritten (no accumulate mode).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is
 *     enqueued on it and the call returns without synchronising, except where stated.
 *   - Matrices are row-major float64, row index l1, column index l2, including l = 0 and 1:
 *     M[l1*(lmax+1) + l2] = K_{l1 l2} = (2 l2+1) Xi(l1,l2)          (PAPER.md:76 Eq. 3, :328).
 *     Rows/columns l < 2 of the polarised blocks (TE, EE, BB, EB) are exactly 0.0.
 *   - Windows are float64 W_l, l = 0..nW-1.  The l3 sum runs over |l1-l2| <= l3 <= min(l1+l2, l3max)
 *     (PAPER.md:226: W_L is needed for L <= 2 lmax; :251: stopping earlier is exact when W vanishes beyond).
 *   - Every call returns TJ_OK (0) or a negative code; no exceptions, no aborts, no errno.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns TJ_ECUDA.
 */
#ifndef TJ_H_
#define TJ_H_

#ifdef __cplusplus
extern "C" {
#endif

#define TJ_OK       0
#define TJ_EINVAL  (-1)  /* bad argument: negative sizes, l3max > 2*lmax, nW mismatch, NULL required pointer,
                            an output requested without its window */
#define TJ_ENOMEM  (-2)  /* host or device allocation failed */
#define TJ_ECUDA   (-3)  /* CUDA runtime / launch error; text via tj_strerror(TJ_ECUDA) */
#define TJ_ELIMIT  (-4)  /* tj_coupling_pol_static only: the problem needs more scratch than the built-in array holds */

/* Opaque handle owning the device-resident lookup tables for one (lmax, l3max) on ONE device: the device that is
 * current when tj_build_tables is called.  Every later call with the handle must be made with the same device
 * current (TJ_EINVAL otherwise); one process can drive several GPUs with one handle per device.  The tables are
 * immutable after build, so a handle may be used concurrently from several streams and threads (host-buffer
 * calls that share a handle are serialised inside the library).  tj_free_tables also releases the side streams
 * the host-buffer calls created for the handle. */
typedef struct tj_tables tj_tables;

/*
 * tj_build_tables -- lookup-table build kernel (Eqs. 11-12).
 *   g(p) = (p - 1/2)/p * g(p-1), g(0) = 1, for p = 0..2*lmax+1, carried in double-double so every
 *   stored double is the faithfully rounded value of Eq. 11; plus the folded tables of DESIGN.md 3:
 *   ginv = 1/g, h = 1/((2p+1) g)  [the 1/(J+1) table of PAPER.md:186 at J = 2p, folded into 1/g],
 *   gA = 2p g, gB = (2p+1) g [odd-J branch], all with zero guard bands, and the per-l constants
 *   u_l = l(l+1), 1/sqrt((l-1)l(l+1)(l+2)).
 *   lmax  >= 0; 0 <= l3max <= 2*lmax.  Enqueues on `cuda_stream` and synchronises it once.
 *   *out receives the handle (free with tj_free_tables).
 */
int tj_build_tables(int lmax, int l3max, void *cuda_stream, tj_tables **out);
void tj_free_tables(tj_tables *tables);

/* Sizes held by a handle.  Any output pointer may be NULL. */
int tj_tables_info(const tj_tables *tables, int *lmax, int *l3max, int *pmax);

/*
 * tj_tables_copy -- copy one table to HOST memory (synchronous; for tests of the table kernel).
 *   which: 0 g, 1 ginv, 2 h, 3 gA, 4 gB  (count <= pmax+1 entries, p = 0..count-1);
 *          5 u_l, 6 1/sqrt(D_l), 7 1/sqrt(u_l)   (count <= lmax+1 entries).
 */
int tj_tables_copy(const tj_tables *tables, int which, double *h_dst, int count);

/*
 * tj_coupling_tt -- K^{TT} (PAPER.md:76-78 Eq. 3; :340 Eq. A1) with the squared (000) symbol from
 * Eq. 10.  d_Wtt: nW = l3max+1 entries.  d_TT: (lmax+1)^2 doubles.
 */
int tj_coupling_tt(const tj_tables *tables, const double *d_Wtt, int nW, double *d_TT, void *cuda_stream);

/*
 * tj_coupling_pol -- all blocks in ONE fused l3 sweep (PAPER.md:80-84 Eq. 4; :340-356 Eqs. A1-A4;
 * spin-2 symbol from Eqs. 13-16 / B14-B17 in the one-product form of DESIGN.md 3).
 *   TT needs d_Wtt; TE needs d_Wtp; EE, BB, EB need d_Wpp.  Any output may be NULL (skipped); a window
 *   may be NULL iff none of its outputs is requested.  BB is a copy of EE.
 *   Each window: nW = l3max+1 entries.  Each output: (lmax+1)^2 doubles.
 */
int tj_coupling_pol(const tj_tables *tables,
                    const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                    double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                    void *cuda_stream);

/*
 * tj_coupling_pol_static -- tj_coupling_pol for callers that must not allocate GPU memory.
 *
 * Who needs it.  Every other coupling call above lmax = 800 takes a little scratch (the pre-folded windows and the
 * tile schedule, about 112 bytes per unit of lmax) from the device's stream-ordered pool with cudaMallocAsync and
 * gives it back with cudaFreeAsync.  Some programs cannot afford that: a host application that has already
 * claimed the whole of device memory for its own arena, so that any allocation made behind its back fails or
 * eats into what it thought it owned; a service with a hard latency budget, where the allocator's lock and the
 * chance that the pool has to grow (which can stall the whole device) are not acceptable inside the loop; and
 * deployments where the stream-ordered pool is not offered at all (some virtualised and partitioned GPU set-ups).
 * For them this entry point runs the same three kernels as tj_coupling_pol -- window pre-fold + tile schedule,
 * staged l3 sweep, mirrored writer (PAPER.md:76-84 Eqs. 3-4, :340-356 Eqs. A1-A4) -- with the scratch in an array
 * that is part of the library image.  It calls no cudaMalloc / cudaMallocAsync / cudaFree and no library routine
 * that allocates; it creates no stream and no event, and records no profiling events (tj_profile_get does not
 * see it).  The caller still owns and passes the windows and the output matrices.
 *
 * The limit.  The array is TJ_STATIC_SCRATCH_BYTES = 2 MiB, enough for any handle with lmax <= TJ_STATIC_LMAX =
 * 16384 (any l3max).  Each GPU on which the library is loaded sets those 2 MiB aside until the process exits,
 * whether or not this function is ever called.  A handle with a larger lmax is refused with TJ_ELIMIT before
 * anything is enqueued; outputs are then untouched.
 *
 * Set-up.  The first call on each device looks up the device address of the array (one cudaGetSymbolAddress, made
 * with the handle's device current, remembered per device for the life of the process).  Make that first call
 * during start-up, before any stream capture begins.  Later calls only enqueue the three kernels.
 *
 * Sharing.  There is ONE array per device and every call on that device uses it.  Nothing in it has to be cleared
 * between calls: the first kernel of a call rewrites every element the other two read (guard bands and tile
 * schedule included), so a call never sees the previous call's contents -- but two calls that may run on the GPU
 * at the same time (different streams, or different threads on different streams) race on it and give wrong
 * results.  Keep all calls on one device in one stream, or order them with events.
 *
 * Arguments, layout, NULL rules, BB = EE and the results are exactly those of tj_coupling_pol; above lmax = 800
 * the two agree bit for bit (same kernels, same arithmetic), at or below it tj_coupling_pol takes its single-launch
 * path and the two agree to rounding.  Errors: TJ_EINVAL as tj_coupling_pol; TJ_ELIMIT as above; TJ_ECUDA if the
 * address look-up or a launch fails.
 */
#define TJ_STATIC_LMAX           16384
#define TJ_STATIC_SCRATCH_BYTES  (2 * 1024 * 1024)
int tj_coupling_pol_static(const tj_tables *tables,
                           const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                           double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                           void *cuda_stream);

/*
 * tj_coupling_band -- band-limited variant: the l3 sum stops at lcut (inclusive),
 * exact when W_l = 0 for l > lcut.  0 <= lcut <= 2*lmax of the handle.
 *   Windows: lcut+1 entries each.  Outputs: banded storage, (lmax+1)*(2*lcut+1) doubles each,
 *   band[l1*(2*lcut+1) + (l2-l1+lcut)] = K_{l1 l2} for |l1-l2| <= lcut and 0 <= l2 <= lmax; slots whose
 *   l2 falls outside 0..lmax are written 0.0.  NULL rules as tj_coupling_pol.
 */
int tj_coupling_band(const tj_tables *tables, int lcut,
                     const double *d_Wtt, const double *d_Wtp, const double *d_Wpp,
                     double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                     void *cuda_stream);

/*
 * tj_coupling_multi -- multi-window batching (one coupling matrix per
 * map pair / frequency pair, all on the same (l1,l2,l3) geometry; covariance matrices use
 * the same symbols with the spectrum of the squared mask as window).  nwin independent window SETS
 * (W^TT, W^TP, W^PP) are swept together: the squared symbols of a term (Eq. 10 product, A, A^2) are formed
 * once and each set adds only its own multiply-adds.  Results are those of nwin tj_coupling_pol calls
 * (same arithmetic per entry, so they agree to the last bit).
 *   Windows: [nwin][nW] row-major, nW = l3max+1.  Outputs: [nwin][(lmax+1)^2].  NULL rules as tj_coupling_pol;
 *   requests for all of TT, TE, EE (or BB) and EB run three sets per sweep (a remainder of two or four sets: two per
 *   sweep), requests for TT alone four windows per sweep (then two, then one), other requests one set per sweep.
 */
int tj_coupling_multi(const tj_tables *tables, int nwin,
                      const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                      double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                      void *cuda_stream);

/*
 * tj_coupling_spin1 -- the spin-1 analogue of tj_coupling_pol: the same fused sweep with
 * the (0,-1,1) symbol the paper lists for lensing / aberration weights (Eqs. B1-B6, B10 at
 * PAPER.md:362-392, :414-417) in place of the spin-2 one.  The paper defines no weights for it; the blocks are
 * defined here by analogy with Eqs. A1-A4 (reading 19):
 *   K00  = TT of tj_coupling_pol                                                 (window W00)
 *   K01  = (2l2+1)/(4pi) sum_{l3, J even} (2l3+1) W01_l3 (l1 l2 l3;000)(l1 l2 l3;-1 1 0)
 *   K11p = (2l2+1)/(4pi) sum_{l3, J even} (2l3+1) W11_l3 (l1 l2 l3;-1 1 0)^2
 *   K11m = the same sum over odd J.
 * Rows/columns l < 1 of K01, K11p, K11m are exactly 0.0.  NULL rules as tj_coupling_pol (K00 needs W00,
 * K01 needs W01, K11p/K11m need W11).  Windows: nW = l3max+1 entries; outputs (lmax+1)^2 doubles.
 */
int tj_coupling_spin1(const tj_tables *tables,
                      const double *d_W00, const double *d_W01, const double *d_W11, int nW,
                      double *d_K00, double *d_K01, double *d_K11p, double *d_K11m,
                      void *cuda_stream);

/*
 * tj_coupling_rows -- the full rows row_lo <= l1 < row_hi of the matrices tj_coupling_pol would give, in compact
 * storage: out[(l1-row_lo)*(lmax+1) + l2] = K_{l1 l2}, all columns l2 = 0..lmax.
 * Every (l1,l2) is independent, so a matrix can be cut into row blocks that are computed
 * anywhere -- one block per GPU with no exchange, or block after block when the whole matrix is not wanted at
 * once.  Entries left of the diagonal are obtained through the symmetry of Xi, so a block costs its
 * own upper-triangle rows plus the pairs (l1 < row_lo, l2 in the block); values are bit-identical to the rows of
 * the full call.  0 <= row_lo < row_hi <= lmax+1; windows, NULL rules and BB as tj_coupling_pol; each output holds
 * (row_hi-row_lo)*(lmax+1) doubles.
 */
int tj_coupling_rows(const tj_tables *tables,
                     const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                     int row_lo, int row_hi,
                     double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                     void *cuda_stream);

/*
 * tj_coupling_binned -- binned output.  The paper prints no binning operator; the form taken here
 * (reading 20) is the one a pseudo-C_l pipeline applies to K:
 *     B^{XY}[b][b'] = sum_{l1 in bin b} sum_{l2 in bin b'} P[l1] K^{XY}[l1][l2] Q[l2],
 * bin b = h_edges[b] <= l < h_edges[b+1] (h_edges: HOST array of nbins+1 ascending values within 0..lmax+1; bins
 * may be empty and need not cover every l), d_P / d_Q: DEVICE arrays of lmax+1 per-l weights.  The same fused sweep
 * runs over chunks of rows and a binning kernel takes the place of the mirrored writer, so the (lmax+1)^2 matrices
 * are never written.  Outputs: nbins*nbins doubles each, row-major [b][b']; windows, NULL rules and BB (= EE) as
 * tj_coupling_pol.  Results are deterministic (fixed summation order) and agree with the binned tj_coupling_pol
 * matrices to rounding.
 */
int tj_coupling_binned(const tj_tables *tables,
                       const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                       int nbins, const int *h_edges, const double *d_P, const double *d_Q,
                       double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                       void *cuda_stream);

/*
 * tj_coupling_binned_multi -- binned output for many window sets (SURVEY.md 8(f) #1 and #4 together; PAPER.md:69-86:
 * one coupling matrix per map pair: covariance windows): nwin window sets go through the batched
 * sweep of tj_coupling_multi (three sets per sweep for the full set of blocks, four for TT alone; remainders as
 * there) and each set's Xi chunks are binned as in tj_coupling_binned, so many map pairs yield nwin * nbins^2 numbers
 * per block and never nwin full matrices.  Windows: [nwin][nW] row-major; outputs: [nwin][nbins*nbins]; bins, weights,
 * NULL rules and BB as tj_coupling_binned.  Window set w of the result agrees with a tj_coupling_binned call on that
 * set alone to rounding, and bit for bit while one chunk of rows holds the whole problem ((blocks) * (sets per sweep) *
 * (lmax+1)^2 * 8 bytes <= 1 GiB): the batched sweep repeats the arithmetic per entry and the binning kernel is the
 * same; beyond that size the two cut the rows into different chunks, whose sums are added in a different order.
 */
int tj_coupling_binned_multi(const tj_tables *tables, int nwin,
                             const double *d_Wtt, const double *d_Wtp, const double *d_Wpp, int nW,
                             int nbins, const int *h_edges, const double *d_P, const double *d_Q,
                             double *d_TT, double *d_TE, double *d_EE, double *d_BB, double *d_EB,
                             void *cuda_stream);

/*
 * tj_coupling_literal -- ABLATION, not the hot path: the paper's own evaluation restated as
 * one plain kernel -- one thread per (l1,l2) of the upper triangle, serial l3 loop in steps of 2 with direct
 * table lookups, K^{TT} from Eq. 10 and K^{EE} from Eq. 16
 * evaluated literally (PAPER.md:216-220 with alpha, beta, eta of Eqs. B14-B16: two table
 * products and two square roots per term), mirrored into the lower triangle.  It exists so
 * that the paper's cost structure (EE ~ 5x TT) and its GPU design can be timed on this GPU
 * beside the fused sweep; results agree with tj_coupling_pol to rounding (~1e-12).
 *   d_TT / d_EE: (lmax+1)^2 doubles, either may be NULL (with its window).  Windows: nW = l3max+1 entries.
 */
int tj_coupling_literal(const tj_tables *tables, const double *d_Wtt, const double *d_Wpp, int nW,
                        double *d_TT, double *d_EE, void *cuda_stream);

/*
 * Host-buffer forms (the end-to-end path): same semantics, but every window and output is a HOST
 * pointer (h_*; pinned memory makes the copies asynchronous and fast; pageable memory also works, without the overlap
 * of copies and arithmetic -- see tj_set_host_pipeline).
 * The call allocates device scratch from the stream-ordered pool, copies the windows in, runs the same
 * kernels, copies every requested matrix back and SYNCHRONISES the stream before returning.
 * band = 0: dense outputs, nW_or_lcut = nW = l3max+1;  band = 1: banded outputs, nW_or_lcut = lcut.
 */
int tj_coupling_host(const tj_tables *tables, int band, int nW_or_lcut,
                     const double *h_Wtt, const double *h_Wtp, const double *h_Wpp,
                     double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                     void *cuda_stream);

/*
 * One matrix set on several GPUs, every pair swept once (each element is
 * independent).  The rows are cut into chunks of a multiple of lcm(R, 32) rows.  What a chunk [r0, r1) makes final all
 * by itself -- its own sweep and mirrored writer, nothing from any other chunk -- is an L-shaped region of every matrix:
 * its rows from column r0 on, and columns [r0, r1) of all rows below.  These regions tile the matrix, so chunks can be
 * dealt to devices: a device sweeps only the upper-triangle pairs of its own chunks and delivers exactly their
 * regions into the ONE host matrix, over its own host link.  No pair is swept twice (tj_coupling_rows, the other way
 * to share a matrix, sweeps every pair left of a block a second time), nothing is exchanged between devices.
 *
 * tj_chunk_plan -- HOST-side: the chunks and their owners for nparts devices.  Chunks are dealt by work (sweep steps,
 * sum over a chunk's rows l1 of (l1+1)(lmax+1-l1)): heaviest first, each to the device with the least work so far.
 * h_bounds receives nchunks+1 ascending row bounds (first 0, last lmax+1), h_owner nchunks device indices; both must
 * have room for 12*nparts+1 entries.  tt_only selects the row-band geometry of the TT-alone sweep.  1 <= nparts <= 64.
 *
 * tj_coupling_host_part -- one device's share: computes the chunks tj_chunk_plan gives to `part` and writes their
 * regions into the host matrices, leaving every other entry of h_* untouched; after the calls for part = 0..nparts-1
 * (on any devices, in any order, also one after the other on a single GPU) the matrices are complete and carry the
 * bits of tj_coupling_host.  Per rank under a launcher: part = rank, nparts = world size, each rank with a handle on
 * its own device (if the ranks do not share host memory, each holds its regions and the rest of its buffer is
 * whatever it was).  Dense outputs only; arguments as tj_coupling_host (nW = l3max+1; pinned buffers, or the copies
 * do not overlap the arithmetic); synchronises the stream before it returns.  The single-launch path is not used here.
 *
 * tj_coupling_host_multi -- one process, ndev devices: tables[g] is a handle built on device g's GPU (all for the same
 * lmax and l3max; distinct handles, which may even live on one GPU), cuda_streams[g] a stream of that device (or
 * cuda_streams = NULL for the default streams).  Enqueues every device's share, then waits for all of them; restores
 * the caller's current device.  h_* must be pinned for the shares to run concurrently.
 */
int tj_chunk_plan(int lmax, int tt_only, int nparts, int *h_bounds, int *h_owner, int *nchunks);
int tj_coupling_host_part(const tj_tables *tables, int part, int nparts, int nW,
                          const double *h_Wtt, const double *h_Wtp, const double *h_Wpp,
                          double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                          void *cuda_stream);
int tj_coupling_host_multi(tj_tables *const *tables, int ndev, int nW,
                           const double *h_Wtt, const double *h_Wtp, const double *h_Wpp,
                           double *h_TT, double *h_TE, double *h_EE, double *h_BB, double *h_EB,
                           void *const *cuda_streams);

/*
 * tj_set_host_pipeline -- what the dense host-buffer call assumes about the machine.  tj_coupling_host (band = 0, lmax
 * above the single-launch threshold, pinned outputs) overlaps its device-to-host copies with the arithmetic, chunk of
 * rows by chunk of rows, in one of two ways: when the copies take longer than the arithmetic, whole rows leave as soon
 * as they are final, in many small chunks, so that the copy engine never waits ("copy-bound", regime 1); otherwise,
 * after every chunk, the L-shaped region that chunk made final leaves as two pitched rectangles, so that almost
 * nothing is left to copy when the last row is computed ("compute-bound", regime 2).  The choice compares
 *     (matrices requested) * (lmax+1)^2 * 8 / d2h_bytes_per_s     with     c * (lmax+1)^3 / 6 / fp64_instr_per_s,
 * c = 13 FP64 instructions per (even + odd) step for the polarised sweep, 2 for TT alone.  The rates are properties of
 * the box, not of the method: the defaults, 54e9 B/s and 1.6e13 instr/s, were measured on the B200 machines the library
 * was tuned on (PCIe Gen5 x16 to pinned memory).  On another host link -- or with several GPUs behind one
 * PCIe switch -- pass what you measure.  0 restores a default.  Per handle; takes effect from the next call; results
 * do not depend on it (both regimes give the same bits), only the time does.  Outputs in PAGEABLE memory are a third
 * case (regime 3): copies into pageable memory block the calling thread, so nothing could overlap; the call then
 * computes everything and copies each matrix out in one piece.
 *
 * tj_host_pipeline_info -- which regime the most recent dense host-buffer call on this handle took (0: none yet,
 * 1, 2, 3 as above, 4: one part of several, tj_coupling_host_part / _multi) and in how many row chunks.  Output pointers may be NULL.
 */
int tj_set_host_pipeline(tj_tables *tables, double d2h_bytes_per_s, double fp64_instr_per_s);
int tj_host_pipeline_info(const tj_tables *tables, int *regime, int *nchunks);

/*
 * tj_l3_range -- host-side integer bookkeeping of the l3 sum for one pair: l3 runs over
 * |l1-l2|..min(l1+l2, l3max) with (l1+l2+l3)%2 == parity (0: TT/TE/EE/BB, 1: EB).
 * nterms may be 0 (then *l3_lo > *l3_hi).  Output pointers may be NULL.
 */
int tj_l3_range(int l1, int l2, int l3max, int parity, int *l3_lo, int *l3_hi, int *nterms);

/*
 * tj_sweep_counts -- HOST-side closed form of the step indices t that carry the l3 terms of one pair:
 *   even J: l3 = l1+l2-2t, t = *te_lo..*te_hi;   odd J: l3 = l1+l2-2t-1, t = *to_lo..*to_hi
 * (l3 advances in steps of 2 from |l1-l2|; it stops at l3max).  It restates
 * tj_l3_range in the sweep's step variable and is not what the kernels execute: a warp walks one common t range
 * and the steps outside a pair's own range add exact zeros from the tables' guard bands.  The kernels' own
 * bookkeeping is tested through their output (spike windows W = delta_{l,L} for every L: an entry is non-zero
 * iff l3 = L is among the terms the kernel added; tests/test_gpu_parity.py).
 */
int tj_sweep_counts(int l1, int l2, int l3max, int *te_lo, int *te_hi, int *to_lo, int *to_hi);

/*
 * Per-kernel timing for the roofline (bench.py): while enabled, every coupling call records CUDA events
 * on its stream around its three kernels.  tj_profile_get waits for the most recent call made by the
 * calling thread and returns the device time in milliseconds of  h_ms3[0] prepare (a2+a3),
 * h_ms3[1] sweep (a4+a5), h_ms3[2] writer (a6); the single-launch path for small lmax reports its one kernel
 * as the sweep.  tj_coupling_multi reports its last group of window sets.  TJ_EINVAL if the thread's most recent
 * call was not profiled, or was tj_coupling_host / tj_coupling_literal (they record no per-kernel events).
 */
int tj_profile_enable(int on);
int tj_profile_get(double *h_ms3);

/*
 * tj_profile_last_sweep -- which sweep kernel the calling thread's most recent coupling call launched, so that a
 * measurement can name the kernel it timed:  h_geo10 = { R (pairs per thread), block mask (1 TT | 2 TE | 4 EE | 8 EB),
 * TS (steps per stage; 0 = the single-launch small_kernel), resident CTAs per SM / 4, deferred accumulation (0/1),
 * window sets per sweep, spin, row-block form (0/1), diagonal band tiling (0/1), CTAs launched }.
 * TJ_EINVAL before the first call.
 * tj_profile_launches -- number of kernels the calling thread's calls have launched so far (callers take differences).
 */
int tj_profile_last_sweep(int *h_geo10);
int tj_profile_launches(long long *h_count);

const char *tj_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* TJ_H_ */
