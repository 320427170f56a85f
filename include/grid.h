/* grid.h -- C ABI of the B200 convolutional gridder (libgridb200.so).
 *
 * The operation (section 2.2): "each visibility sample is treated as a Dirac delta,
 * convolved with some function, and then sampled onto the grid"; the gridding convolution function
 * (GCF) is read from a precomputed oversampled table selected per sample by "the
 * integer grid coordinates, the sub-grid coordinates for indexing the GCF, the w plane index"
 * (section 4); the GCF is separable, G_ij = Gu_i * Gv_j, and polarisation-independent
 * (PAPER.md:97-99, 178).  The two main entry points are the ones BASELINE.json:north_star fixes.
 * Exact semantics (quantiser, layouts, edge handling): DESIGN.md "Readings" R1-R24.
 *
 * Conventions
 *   - Every array argument is a DEVICE pointer owned by the caller, 16-byte aligned, unless it says
 *     HOST.  The library allocates no device memory; scratch space is the caller's workspace.
 *   - Return value 0 = success, negative = GRID_ERR_*; grid_last_error() gives a thread-local text.
 *   - All work is enqueued on `stream`; no call synchronises the host with the device.
 *   - A plan may be executed repeatedly; calls on one plan must not overlap in time.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails.
 */
#ifndef GRIDB200_GRID_H
#define GRIDB200_GRID_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GRID_OK                 0
#define GRID_ERR_INVALID_ARG   -1
#define GRID_ERR_UNSUPPORTED   -2   /* e.g. tap tables + batch buffers exceed shared memory */
#define GRID_ERR_CUDA          -3
#define GRID_ERR_STATE         -4   /* set_samples / set_workspace missing or too small */

typedef struct grid_plan grid_plan;           /* opaque, owned by the library */
typedef struct CUstream_st* grid_stream_t;    /* == cudaStream_t */

/* Create a plan for an N x N grid (BASELINE.json:north_star signature).
 *   grid_size  N, 1 <= N <= 32767, N >= support
 *   support    S >= 1, odd or even; footprint is S x S cells
 *   oversample O >= 1; taps tabulated at 1/O cell
 *   n_wplanes  >= 1, n_wplanes * oversample <= 65535
 *   n_pol      1, 2 or 4 complex polarisations per sample
 * Chooses the coarsening block (Cu x Cv), threads per CTA and batch length from a tuned table
 * keyed by (S, n_pol).  Returns NULL on error. */
grid_plan* grid_plan_create(int grid_size, int support, int oversample, int n_wplanes, int n_pol);

/* Number of samples of the next grid_execute calls (the execute signature carries no count).
 * n_vis >= 0; n_vis == 0 makes grid_execute a no-op (R23). */
int grid_plan_set_samples(grid_plan* plan, long long n_vis);

/* OPTIONAL performance hint: samples are ordered baseline-major, then time, then channel
 * (BASELINE.json:configs[0]), n_baselines*n_times*n_channels == n_vis.  It only changes the order in
 * which a chunk's samples are traversed (the sum is order-independent up to FP32 rounding, pin P11);
 * never the result beyond that.  Pass zeros to clear. */
int grid_plan_set_layout(grid_plan* plan, int n_baselines, int n_times, int n_channels);

/* Scratch memory the plan needs for the current n_vis, layout hint and sample order (quantised sample records +
 * counters; in cell order also the per-cell histogram and the ranks: grid_plan_set_sample_order).  Ask again after
 * grid_plan_set_samples, grid_plan_set_layout, grid_plan_set_sample_order or grid_plan_set_tuning. */
size_t grid_plan_workspace_bytes(const grid_plan* plan);
/* Caller-owned device scratch, >= grid_plan_workspace_bytes(), 256-byte aligned. */
int grid_plan_set_workspace(grid_plan* plan, void* dev_ptr, size_t bytes);

/* Grid all samples:  for every sample n whose S x S footprint lies inside the grid (others, and
 * samples with non-finite u, v or w, are skipped, R7):
 *     grid[j0+tj][i0+ti][p] += weights[n] * vis[n][p] * k[wp][sv][tj] * k[wp][su][ti]
 * with (i0,su) = Q(u_n), (j0,sv) = Q(v_n), wp = W(w_n) (R4, R5), FP32 arithmetic,
 * FP32 atomic accumulation (order nondeterministic).
 *   uvw          [n_vis][3] float32: u, v in cells from the centre cell floor(N/2); w in plane units
 *   vis          [n_vis][n_pol] complex64 (re, im interleaved), polarisation fastest
 *   weights      [n_vis] float32
 *   conv_kernel  [n_wplanes][oversample][support] complex64 separable taps (same table for u and v)
 *   grid         [N][N][n_pol] complex64, row = v, column = u; ACCUMULATED INTO, never zeroed
 * Steps: a1 quantise pass -- which for large inputs also sorts the samples by grid cell
 * (grid_plan_set_sample_order) --, then the gridding kernel (a2-a9). */
int grid_execute(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                 const float* conv_kernel, float* grid, grid_stream_t stream);

/* grid_execute without a caller-provided workspace and without any allocation: for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The workspace of the
 * call -- chunk queue and statistics, quantised records, chunk order, tap table copy; what grid_plan_set_workspace
 * otherwise supplies -- lives in ONE array of GRID_STATIC_SCRATCH_BYTES in the library's device image (every GPU that
 * loads the library holds it until the process exits).  Same arguments, same result and same kernels as
 * grid_execute; grid_plan_set_workspace need not have been called and is ignored.
 *   - Returns GRID_ERR_UNSUPPORTED, with the sizes in grid_last_error(), when grid_plan_workspace_bytes(plan) exceeds
 *     GRID_STATIC_SCRATCH_BYTES (20 MiB: about 1.2 million samples per call; fewer when the tap table has to be
 *     copied to global memory).  Grid larger inputs in several calls: the grid is accumulated into.
 *   - Calls no cudaMalloc / cudaFree or allocating library routine (one cudaGetSymbolAddress per device on first use).
 *   - The array is shared by every plan and every call on a device and keeps the last call's contents; the call
 *     clears the part that must start at zero (queue, statistics, order bins) on `stream` before use.  Two calls
 *     that overlap on the GPU (different streams, no ordering between them) RACE on it: serialise them. */
#define GRID_STATIC_SCRATCH_BYTES (20u << 20)
int grid_execute_static(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                        const float* conv_kernel, float* grid, grid_stream_t stream);

/* Compression, the step before the path ("merge adjacent visibilities with identical
 * oversampled position", done as a pre-process and reused for every major cycle; PAPER.md:91 lists what a
 * compressed sample carries).  Runs a1 and merges every run of consecutive samples with equal
 * (i0, su, j0, sv, wp) into one pre-weighted sample, in input order; skipped samples (R7) produce none.
 *   uvw, vis, weights   as for grid_execute (n_vis samples, grid_plan_set_samples)
 *   out_records  [>= n_vis] 8-byte records (opaque: cell, sub-offsets, plane), DEVICE, 16-byte aligned
 *   out_vis      [>= n_vis][n_pol] complex64: sum over the run of weights * vis (FP32, input order)
 *   out_count    DEVICE long long: number of compressed samples written
 * Needs the plan's workspace.  Supports 3..128 on grids of at least twice the padded support (the plans that run
 * the warp kernel, variant 3); GRID_ERR_UNSUPPORTED otherwise.  For supports that are not powers of two the
 * records are in the padded form described under grid_plan_set_tuning. */
int grid_compress(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                  void* out_records, float* out_vis, long long* out_count, grid_stream_t stream);

/* Grid n compressed samples produced by grid_compress (same plan, n <= the plan's n_vis):
 *     grid[j0+tj][i0+ti][p] += vis[k][p] * k[wp][sv][tj] * k[wp][su][ti]
 * i.e. steps a3-a9 of grid_execute on samples that are already quantised and pre-weighted -- the
 * input the paper's kernel takes.  n is a HOST value (read *out_count back first). */
int grid_execute_compressed(grid_plan* plan, const void* records, const float* vis, long long n,
                            const float* conv_kernel, float* grid, grid_stream_t stream);

/* Gridding with a dense (non-separable) GCF table (A-projection-like kernels; the paper
 * expects smaller gains there and does not measure it):
 *     grid[j0+tj][i0+ti][p] += weights[n] * vis[n][p] * conv_kernel_2d[wp][sv][su][tj][ti]
 *   conv_kernel_2d  [n_wplanes][oversample][oversample][support][support] complex64, DEVICE
 * Everything else as grid_execute (same Q, W, skipping rule, accumulation).  Power-of-two supports up to
 * 32 run on the coarsened kernel with the table read through L1/L2; other supports on a
 * one-atomic-per-update kernel (grid_last_error() says so after the call). */
int grid_execute_dense(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                       const float* conv_kernel_2d, float* grid, grid_stream_t stream);

/* The same with one dense table per polarisation (the coarsened kernel "assumed that the GCF is
 * polarization-independent ... cannot be directly applied to A-projection"; GCFs "dependent on
 * time, frequency, polarization"):
 *     grid[j0+tj][i0+ti][p] += weights[n] * vis[n][p] * conv_kernel_2d_pol[p][wp][sv][su][tj][ti]
 *   conv_kernel_2d_pol  [n_pol][n_wplanes][oversample][oversample][support][support] complex64, DEVICE
 * Same kernels as grid_execute_dense; a thread fetches the table values of each of its polarisations in turn. */
int grid_execute_dense_pol(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                           const float* conv_kernel_2d_pol, float* grid, grid_stream_t stream);

/* Degridding, the adjoint of grid_execute (the paper calls its own degridder preliminary
 * and does not measure it).  For every sample whose footprint lies inside the grid
 *     vis_out[n][p] = weights[n] * sum_{tj,ti} conj(k[wp][sv][tj] * k[wp][su][ti]) * grid[j0+tj][i0+ti][p]
 * with the same Q, W as grid_execute; skipped samples (R7) get zeros.  <grid_execute(V), G> equals
 * <V, grid_degrid(G)> (pin P7).  grid is read-only; vis_out [n_vis][n_pol] complex64 is overwritten.
 * Two kernels: for supports 3..128 the coarsened kernel run backwards -- owned grid values stay in registers
 * while the footprint covers them; otherwise (any support) a gather kernel bound by L2 bandwidth.
 * grid_plan_set_degrid_gather(plan, 1) forces the latter. */
int grid_degrid(grid_plan* plan, const float* uvw, const float* weights, const float* conv_kernel,
                const float* grid, float* vis_out, grid_stream_t stream);

/* on = 1: grid_degrid always uses the gather kernel (diagnostic / comparison); 0 = automatic (default). */
int grid_plan_set_degrid_gather(grid_plan* plan, int on);

/* Step a1 alone (the device pass that turns uvw into integer cell, sub-offset and plane index),
 * unpacked for inspection: out is int32 [n][6] = i0, j0, su, sv, wp, valid (invalid: -1 x5, 0).
 * Runs the same device function grid_execute uses.  n need not equal the plan's n_vis. */
int grid_quantise(grid_plan* plan, const float* uvw, long long n, int* out, grid_stream_t stream);

/* Override the tuned launch configuration (autotuning).  variant < 0 keeps the current kernel,
 * any other argument <= 0 keeps its current value (when the variant changes, threads_per_cta and ctas_per_sm fall
 * back to that variant's defaults unless given).
 * variant: 3 = warp-autonomous coarsened kernel with bin == support (default for supports 3..128 on grids of at
 *   least twice the padded support).  Supports that are not powers of two are zero-padded to the next power of
 *   two Sk (pin P14): every tap row exists in two copies, zeros behind the taps (footprint
 *   origin unchanged) and zeros in front (origin moved down by Sk - S), the second used only where the padded
 *   footprint would leave the grid; the result is the same sum, (Sk/S)^2 times the multiply-adds;
 * 1 = coarsened kernel with the paper's block-aligned, zero-padded bin (any support that fits a CTA; default for
 *   supports 1, 2 and for tiny grids);
 * 0 = naive scatter (one atomic per update; diagnostic baseline; never a default for supports 3..128).
 *   cu, cv            coarsening block per thread (u, v), each in {1,2,4,8}, cu*cv*n_pol <= 32
 *   threads_per_cta   multiple of 32, <= 1024
 *   batch             samples staged to shared memory per team per step
 *   chunk             samples a team grids before its final flush (1024)
 *   ctas_per_sm       persistent CTAs per SM
 * A block that is not instantiated for the plan's current polarisation split (grid_plan_set_pol_split)
 * resets the split to 1.  Returns GRID_ERR_UNSUPPORTED if the combination does not fit (shared
 * memory, registers). */
int grid_plan_set_tuning(grid_plan* plan, int variant, int cu, int cv, int threads_per_cta,
                         int batch, int chunk, int ctas_per_sm);

/* Order in which a chunk's samples are walked when the layout hint is set (the result is the same
 * sum in a different order, pin P11): mode -1 = choose per call from the mean hop between
 * consecutive samples measured by the quantise pass (default), 0 = input order (channel innermost,
 * odd time rows mirrored), 1 = time innermost over blocks of `time_block` time steps (power of two,
 * default 64; the padded kernel caps it at min(batch, 16); 0 keeps the current value).  PAPER.md:61, 107: the gain of register accumulation depends
 * on "the coordinates and ordering of the data". */
int grid_plan_set_traversal(grid_plan* plan, int mode, int time_block);

/* Order in which chunks enter the work queue (PAPER.md:103 fixes the chunks, not their order; the
 * result is the same sum): 1 = sorted by the coarse grid tile of the chunk's first sample, so that
 * chunks in flight together flush to neighbouring grid cells (three extra small launches per
 * grid_execute), 0 = input (baseline) order, -1 = sorted only when the grid exceeds 256 MB, i.e. twice
 * the L2 (default).  Variant 3 only; ignored otherwise. */
int grid_plan_set_chunk_order(grid_plan* plan, int mode);

/* Order in which grid_execute hands the samples to the gridding kernel (the result is the same sum in a different
 * order, pin P11; the gain of register accumulation depends on "the coordinates and ordering of the
 * data": an accumulator is flushed when its cell changes):
 *   1 = cell order: the a1 pass sorts the samples by the grid cell of their footprint origin (counting sort: per-cell
 *       histogram, prefix sum, scatter of 16-byte records that carry the sample's index, or for one polarisation the
 *       pre-weighted visibility; 5 launches instead of 1).  Consecutive samples then mostly share their cell and
 *       flushes become rare.  Needs the warp kernel (variant 3) and 4 bytes per grid cell + 20 bytes per sample
 *       more workspace (a sorted record has a 32-byte sector to itself): call grid_plan_workspace_bytes /
 *       grid_plan_set_workspace AFTER this call.  The layout hint, the traversal mode and the chunk order are then
 *       irrelevant.
 *   2 = cell order, kept: as 1, and the sorted records stay in the workspace -- the following grid_execute and
 *       grid_degrid calls on this plan skip the sort.  THE CALLER GUARANTEES that they pass the same uvw and weights
 *       (the paper's case: compression and quantisation are "done as a pre-process and reused for every major
 *       cycle"; only the visibilities change).  Any grid_plan_set_* call that changes samples,
 *       workspace, tuning or order, grid_compress and grid_execute_dense* drop the kept records; call
 *       grid_plan_set_sample_order(plan, 2) again after changing uvw or weights in place.  The workspace must not be
 *       shared with another plan meanwhile.
 *   0 = input order (chunks of the caller's baseline-major order, walked as grid_plan_set_traversal says).
 *  -1 = automatic (default): cell order when n_vis >= 2^20 and grid_size^2 <= 8 n_vis, unless the layout hint says
 *       the samples are single-channel tracks (they move a fraction of a cell per sample as they come);
 *       else input order.
 * Applies to grid_execute, grid_execute_dense* (coarsened kernel) and grid_degrid (whose results then go back to their
 * samples' places through the index in the record); grid_execute_static and grid_execute_compressed (its input is
 * already ordered by the caller) always use input order. */
int grid_plan_set_sample_order(grid_plan* plan, int mode);

/* Variant 3, n_pol = 4: spread the polarisations of one grid point over `lanes` adjacent threads
 * (1 or 2).  With 2, the two 16-byte atomics of a 32-byte grid point leave in one instruction and
 * cost the L2 one sector operation instead of two.  Set the block (cu, cv) first; returns
 * GRID_ERR_UNSUPPORTED if that combination is not instantiated. */
int grid_plan_set_pol_split(grid_plan* plan, int lanes);

/* Autotuning as the paper does it ("a small artificial data-set is synthesized and benchmarked with a
 * range of coarsening factors and work-group sizes, and the best combination is remembered ... separately for each
 * number of polarizations").
 *
 * grid_plan_autotune_candidates: HOST only, no device needed.  Writes up to max_candidates triples
 * (cu, cv, polarisation split) that are instantiated and fit this plan (shared memory, registers) into out[3*k..],
 * the plan's current block first; returns how many there are (<= 0: the plan does not run the warp kernel).
 *
 * grid_plan_autotune: synthesises n_samples samples on the device (0 = 1 << 20; tracks of a synthetic array
 * shaped by the layout hint if one is set, else single-channel tracks; counter-based generator seeded with
 * `seed`; random visibilities and weights, Kaiser-Bessel-like taps; where the plan grids in cell order the tracks
 * are confined to a part of the grid so that the set has the plan's samples per grid cell), grids them -- in the
 * plan's sample order -- with every candidate onto a
 * scratch grid of the plan's size (cudaMalloc'ed and freed here, like the inputs), times each with CUDA events on
 * `stream` (second of two runs) and installs the fastest (as grid_plan_set_tuning + grid_plan_set_pol_split
 * would).  Synchronises `stream`.  results, if not NULL, receives for every candidate, in the order of
 * grid_plan_autotune_candidates, the time in microseconds (< 0: failed) -- at most max_candidates entries.
 * Returns GRID_OK, GRID_ERR_CUDA (no device / out of memory) or GRID_ERR_UNSUPPORTED (not the warp kernel). */
int grid_plan_autotune_candidates(const grid_plan* plan, int* out, int max_candidates);
int grid_plan_autotune(grid_plan* plan, long long n_samples, unsigned int seed, float* results, int max_candidates,
                       grid_stream_t stream);

/* HOST out[20]: variant, cu, cv, bin_u, bin_v, team_threads, teams_per_cta, threads_per_cta, batch,
 * chunk, ctas_per_sm, smem_bytes, n_sm, traversal mode, time_block, chunk order mode,
 * polarisation split, warp groups per CTA, taps in global memory (0/1), sample order in effect (1 = cell order). */
int grid_plan_get_info(const grid_plan* plan, int* out);

/* Measurement hook: two caller-owned cudaEvent_t (passed as void*) that the following grid_execute
 * calls record on `stream` immediately before and after the gridding kernel (steps a2-a9; the
 * quantise pass a1 lies outside the pair).  NULL, NULL clears.  Nothing is synchronised. */
int grid_plan_set_kernel_events(grid_plan* plan, void* ev_start, void* ev_stop);

/* Checked build only (nvcc -DGRIDB200_CHECK, tests/test_gpu_checked_build.py; compute-sanitizer is closed on the
 * measurement pool): the warp kernel tests every global address it forms and every shared-memory slot it indexes
 * against its bounds, counts violations and suppresses the access.  HOST out[8] = violations since the last call
 * that reset the plan's queue: grid cell, sample index, raw slot, cooked slot, tap offset, degrid output index, 0, 0.
 * Synchronises `stream`.  The shipped library compiles the tests away and always reports zeros. */
int grid_plan_debug_counters(grid_plan* plan, unsigned int* out, grid_stream_t stream);

/* Kernel launches enqueued by the last grid_execute on this plan (for bench.py's gpu_launches). */
int grid_plan_last_launches(const grid_plan* plan);

void grid_plan_destroy(grid_plan* plan);

/* Thread-local description of the last error in this thread ("" if none). */
const char* grid_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GRIDB200_GRID_H */
