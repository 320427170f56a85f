// Host side of libgridb200.so: the C ABI of include/grid.h.  Product path only -- no CPU fallback,
// nothing from oracle/.
#include "../../include/grid.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cmath>
#include <new>

#include "grid_kernel.cuh"
#include "grid_warp_kernel.cuh"
#include "gridder_common.cuh"
#include "compress.cuh"
#include "degrid_kernel.cuh"
#include "quantise.cuh"
#include "cell_sort.cuh"

using namespace gridb200;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int round_up(int a, int b) { return (a + b - 1) / b * b; }

}  // namespace

struct grid_plan {
    int N, S, O, W, P;
    int Sk;                               // support the warp kernel runs with: S, or the next power of two (zero-padded taps)
    long long n_vis;
    int n_baselines, n_times, n_channels;
    void* workspace;
    size_t workspace_bytes;
    // tuning
    int variant, cu, cv, threads, batch, chunk, ctas_per_sm;
    int traversal, time_block;      // -1 auto / 0 channel-innermost / 1 time-innermost; Tc
    // derived
    int bin_u, bin_v, row_u, row_v, nbx, nby, team_threads, teams_per_cta, smem_bytes;
    int groups_per_cta, queue_teams;      // variant 3: warp groups per CTA; teams per queue entry (all variants)
    int dense;                            // internal (grid_execute_dense): non-separable table, read from global memory; 2: one per polarisation
    int taps_global;                      // variant 3: tap table read from global memory (too large for shared)
    int degrid_gather;                    // 1: grid_degrid always uses the gather kernel (diagnostic)
    int pol_split;                        // variant 3: lanes sharing one grid point's polarisations (1 or 2)
    int sort_chunks;                      // -1 auto (grid larger than L2), 0 off, 1 on
    int sample_order;                     // grid_plan_set_sample_order: -1 auto, 0 input order, 1 sorted by grid cell, 2 sorted and kept
    int order_kept;                       // mode 2: the workspace holds the sorted records of the current samples
    int n_sm, max_smem;
    int last_launches;
    int user_tuned;                       // set_tuning / set_pol_split was called: set_samples keeps the block
    cudaEvent_t ev_start, ev_stop;
};

namespace {

typedef void (*kernel_fn)(const GridParams);

template <int CU, int CV, int P>
kernel_fn pick() { return grid_coarsened_kernel<CU, CV, P>; }

// Instantiated coarsening blocks: near-square shapes only, Cu*Cv*P <= 32 accumulators.
kernel_fn lookup_kernel(int cu, int cv, int P) {
#define CASE(a, b, p) if (cu == a && cv == b && P == p) return pick<a, b, p>();
    CASE(1, 1, 1) CASE(2, 1, 1) CASE(2, 2, 1) CASE(4, 1, 1) CASE(4, 2, 1) CASE(4, 4, 1) CASE(8, 2, 1) CASE(8, 4, 1)
    CASE(1, 1, 2) CASE(2, 1, 2) CASE(2, 2, 2) CASE(4, 2, 2) CASE(4, 4, 2)
    CASE(1, 1, 4) CASE(2, 1, 4) CASE(2, 2, 4) CASE(4, 1, 4) CASE(4, 2, 4)
#undef CASE
    return nullptr;
}

// Variant 3 (grid_warp_kernel.cuh): kernel + the compile-time geometry the host needs.
struct WarpDesc {
    kernel_fn fn;
    int gt, tpg, team, max_threads;
    size_t (*group_bytes)(int);
};

template <int CU, int CV, int P, int LOGS, int PS, bool OK = (CU <= (1 << LOGS) && CV <= (1 << LOGS))>
struct WarpPick {
    static WarpDesc get() {
        using T = WarpKernelTraits<CU, CV, P, LOGS, PS>;
        return WarpDesc{grid_warp_kernel<CU, CV, P, LOGS, PS>, T::GT, T::TPG, T::TEAM, T::MAX_THREADS, &T::group_bytes};
    }
};
template <int CU, int CV, int P, int LOGS, int PS>
struct WarpPick<CU, CV, P, LOGS, PS, false> { static WarpDesc get() { return WarpDesc{nullptr, 0, 0, 0, 0, nullptr}; } };

template <int CU, int CV, int P, int PS>
WarpDesc pick_warp(int logs) {
    switch (logs) {
        case 2: return WarpPick<CU, CV, P, 2, PS>::get();
        case 3: return WarpPick<CU, CV, P, 3, PS>::get();
        case 4: return WarpPick<CU, CV, P, 4, PS>::get();
        case 5: return WarpPick<CU, CV, P, 5, PS>::get();
        // bins of 64 and 128 (tiles of 64 x 64): blocks of at least 8 points (teams of at most 512 threads)
        case 6: if constexpr (PS == 1 && CU * CV >= 8) return WarpPick<CU, CV, P, 6, PS>::get(); break;
        case 7: if constexpr (PS == 1 && CU * CV >= 8) return WarpPick<CU, CV, P, 7, PS>::get(); break;
    }
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

// Row-skip instantiations (grids far beyond the L2: DRAM-bound atomics), for the blocks such plans default to.
template <int CU, int CV, int P, int PS>
WarpDesc pick_warp_rs(int logs) {
#define RSCASE(l) case l: { using T = WarpKernelTraits<CU, CV, P, l, PS>; \
        return WarpDesc{grid_warp_kernel<CU, CV, P, l, PS, false, false, false, true>, T::GT, T::TPG, T::TEAM, T::MAX_THREADS, &T::group_bytes}; }
    switch (logs) { RSCASE(2) RSCASE(3) RSCASE(4) }
#undef RSCASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

WarpDesc lookup_warp(int cu, int cv, int P, int logs, int ps, bool row_skip = false) {
    if (row_skip) {
        if (cu == 2 && cv == 2 && P == 4 && ps == 2) { const WarpDesc d = pick_warp_rs<2, 2, 4, 2>(logs); if (d.fn) return d; }
        if (cu == 2 && cv == 2 && P == 4 && ps == 1) { const WarpDesc d = pick_warp_rs<2, 2, 4, 1>(logs); if (d.fn) return d; }
    }
#define CASE(a, b, p, s) if (cu == a && cv == b && P == p && ps == s) return pick_warp<a, b, p, s>(logs);
    // the blocks the autotuner chooses from (near-square shapes); 1x1 and 2x1 never won a sweep
    CASE(2, 2, 1, 1) CASE(4, 2, 1, 1) CASE(4, 4, 1, 1) CASE(8, 4, 1, 1)
    CASE(2, 2, 2, 1) CASE(4, 2, 2, 1) CASE(4, 4, 2, 1)
    CASE(2, 2, 4, 1) CASE(4, 2, 4, 1)
    CASE(2, 2, 4, 2) CASE(4, 2, 4, 2) CASE(4, 4, 4, 2)
#undef CASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

// Kernels that read the taps from global memory (table too large for shared memory): default blocks only.
template <int CU, int CV, int P>
WarpDesc pick_tg(int logs) {
#define TGBODY(l) if constexpr (CU <= (1 << l) && CV <= (1 << l)) { using T = WarpKernelTraits<CU, CV, P, l, 1>; \
        return WarpDesc{grid_warp_kernel<CU, CV, P, l, 1, false, true>, T::GT, T::TPG, T::TEAM, T::MAX_THREADS, &T::group_bytes}; }
#define TGCASE(l) case l: TGBODY(l) break;
    switch (logs) {
        TGCASE(2) TGCASE(3) TGCASE(4) TGCASE(5)
        case 6: if constexpr (CU * CV >= 8) { TGBODY(6) } break;
        case 7: if constexpr (CU * CV >= 8) { TGBODY(7) } break;
    }
#undef TGBODY
#undef TGCASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

WarpDesc lookup_warp_tg(int cu, int cv, int P, int logs) {
#define CASE(a, b, p) if (cu == a && cv == b && P == p) return pick_tg<a, b, p>(logs);
    CASE(2, 2, 1) CASE(4, 4, 1) CASE(8, 4, 1) CASE(2, 2, 2) CASE(4, 2, 2) CASE(2, 2, 4) CASE(4, 2, 4)
#undef CASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

// Dense (non-separable) GCF kernels: default blocks, S <= 32.  KIND 1: one table, 2: one table per polarisation.
template <int CU, int CV, int P, int KIND>
WarpDesc pick_dense(int logs) {
#define DCASE(l) case l: if constexpr (CU <= (1 << l) && CV <= (1 << l)) { using T = WarpKernelTraits<CU, CV, P, l, 1>; \
        return WarpDesc{grid_warp_kernel<CU, CV, P, l, 1, false, false, KIND>, T::GT, T::TPG, T::TEAM, T::MAX_THREADS, &T::group_bytes}; } break;
    switch (logs) { DCASE(2) DCASE(3) DCASE(4) DCASE(5) }
#undef DCASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

WarpDesc lookup_warp_dense(int cu, int cv, int P, int logs, int kind = 1) {
    if (kind == 2) {
#define CASE(a, b, p) if (cu == a && cv == b && P == p) return pick_dense<a, b, p, 2>(logs);
        CASE(2, 2, 2) CASE(4, 2, 2) CASE(2, 2, 4) CASE(4, 2, 4)
#undef CASE
        return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
    }
#define CASE(a, b, p) if (cu == a && cv == b && P == p) return pick_dense<a, b, p, 1>(logs);
    CASE(2, 2, 1) CASE(4, 4, 1) CASE(8, 4, 1) CASE(2, 2, 2) CASE(4, 2, 2) CASE(2, 2, 4) CASE(4, 2, 4)
#undef CASE
    return WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
}

// Dense GCF, any support: one thread per (sample, footprint row), one atomic per update (fallback).
template <int P>
__global__ void __launch_bounds__(256)
grid_scatter_dense_kernel(const CycRec* __restrict__ recs, const float2* __restrict__ vis, const float* __restrict__ weights,
                          const float2* __restrict__ kernel2d, float* __restrict__ grid, long long n_vis, int N, int S, int O,
                          long long pol_stride) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = g / S;
    const int tj = (int)(g - n * S);
    if (n >= n_vis) return;
    const CycRec rec = recs[n];
    if (rec.pos & 0x8000u) return;
    const int i0 = (int)(rec.pos & 0x7fffu), j0 = (int)(rec.pos >> 16);
    const uint32_t ru = rec.rows & 0xffffu, rv = rec.rows >> 16;
    const uint32_t su = ru - (ru / (uint32_t)O) * (uint32_t)O;
    const float2* k = kernel2d + ((size_t)rv * O + su) * S * S + (size_t)tj * S;
    const float w = weights[n];
    float* row = grid + ((size_t)(j0 + tj) * N + i0) * (2 * P);
    for (int ti = 0; ti < S; ++ti) {
#pragma unroll
        for (int q = 0; q < P; ++q) {
            const float2 gk = __ldg(k + (size_t)q * pol_stride + ti);       // pol_stride 0: one table for all polarisations
            float2 v = vis[n * P + q];
            v.x *= w; v.y *= w;
            red_add_v2(row + (size_t)(ti * P + q) * 2, gk.x * v.x - gk.y * v.y, gk.x * v.y + gk.y * v.x);
        }
    }
}

// Coarsened degridding kernels (grid_warp_kernel<..., DEGRID = true>): teams of at most one warp.
template <int CU, int CV, int P, bool TGF>
kernel_fn pick_degrid(int logs) {
    switch (logs) {
        case 2: if constexpr (!TGF && WarpKernelTraits<CU, CV, P, 2>::TEAM <= 32 && CU <= 4 && CV <= 4) return grid_warp_kernel<CU, CV, P, 2, 1, true, TGF>; break;
        case 3: if constexpr (!TGF && WarpKernelTraits<CU, CV, P, 3>::TEAM <= 32) return grid_warp_kernel<CU, CV, P, 3, 1, true, TGF>; break;
        case 4: if constexpr (WarpKernelTraits<CU, CV, P, 4>::TEAM <= 64) return grid_warp_kernel<CU, CV, P, 4, 1, true, TGF>; break;
        // teams of several warps (and tiles at S = 128): combined by atomics
        case 5: if constexpr (CU * CV >= 4) return grid_warp_kernel<CU, CV, P, 5, 1, true, TGF>; break;
        case 6: if constexpr (CU * CV >= 8) return grid_warp_kernel<CU, CV, P, 6, 1, true, TGF>; break;
        case 7: if constexpr (CU * CV >= 8) return grid_warp_kernel<CU, CV, P, 7, 1, true, TGF>; break;
    }
    return nullptr;
}

kernel_fn lookup_degrid(int cu, int cv, int P, int logs, bool tg = false) {
#define CASE(a, b, p) if (cu == a && cv == b && P == p) return tg ? pick_degrid<a, b, p, true>(logs) : pick_degrid<a, b, p, false>(logs);
    CASE(2, 2, 1) CASE(4, 2, 1) CASE(4, 4, 1) CASE(8, 4, 1)
    CASE(2, 2, 2) CASE(4, 2, 2) CASE(4, 4, 2)
    CASE(2, 2, 4) CASE(4, 2, 4)
#undef CASE
    return nullptr;
}

// multi-warp teams (and tiled bins) combine through atomics into a zeroed vis_out
bool degrid_needs_zeroed_output(int cu, int cv, int logs) {
    const int ts = (1 << logs) > 64 ? 64 : (1 << logs);
    return (ts / cu) * (ts / cv) > 32 || logs == 7;
}

int log2_exact(int v) {
    for (int l = 0; l < 31; ++l) if ((1 << l) == v) return l;
    return -1;
}

// Supports that are not powers of two run on the warp kernel with the tap rows zero-padded to the next power
// of two (pin P14: zero taps leave the grid unchanged).  Two padded copies of every row:
// zeros behind the taps (footprint origin unchanged), and zeros in front (origin moved down by the padding) for
// samples whose padded footprint would otherwise stick out of the grid's upper edge -- so the kernel needs no
// bounds test.  Needs N >= 2*Sk - S (a footprint cannot touch both edges).
int padded_support(int S, int N, int W, int O) {
    if (S < 3 || S > 128) return S;
    int sk = 4;
    while (sk < S) sk *= 2;
    if (sk == S) return S;
    if (N < 2 * sk - S || (long long)W * O * 2 > 65535) return S;
    return sk;
}
bool is_padded(const grid_plan* p) { return p->Sk != p->S; }
int tap_rows(const grid_plan* p) { return p->W * p->O * (is_padded(p) ? 2 : 1); }

bool cell_sort_on(const grid_plan* p);
// 16 bytes per sample; in cell order every record has a 32-byte sector of its own (kCellRecStride, cell_sort.cuh)
size_t records_bytes(const grid_plan* p) {
    return (size_t)((p->n_vis + 3) / 4 * 4) * sizeof(SampleRec) * (cell_sort_on(p) ? kCellRecStride : 1);
}

// workspace: [256 B counters][order bins][records][chunk order]
constexpr size_t kHeadBytes = 256 + 2 * kOrderBins * sizeof(uint32_t);
size_t order_capacity(const grid_plan* p) { return (size_t)(p->n_vis / 8 + 4096); }
size_t tap_table_bytes(const grid_plan* p);
size_t tap_table_offset(const grid_plan* p) {
    return kHeadBytes + records_bytes(p) + ((order_capacity(p) * sizeof(uint32_t) + 15) & ~(size_t)15);
}
size_t tap_table_bytes(const grid_plan* p) {
    return p->taps_global ? (size_t)tap_rows(p) * 2 * p->Sk * sizeof(float2) : 0;
}

// Cell order (cell_sort.cuh): grid_execute sorts the samples by grid cell in its a1 pass.  Automatic when the
// input is large enough for the extra launches to pay and the per-cell histogram is not much larger than the
// input itself (a sparse input on a huge grid would spend its time scanning empty cells).
constexpr long long kCellSortMinSamples = 1 << 20;
bool cell_sort_possible(const grid_plan* p) {
    return p->variant == 3 && p->n_vis > 0 && p->n_vis < 0x7fffffffLL;
}
bool cell_sort_on(const grid_plan* p) {
    if (p->sample_order == 0 || !cell_sort_possible(p)) return false;
    if (p->sample_order > 0) return true;
    // single-channel tracks (the paper's data) move a fraction of a cell per sample in input order:
    // nothing to gain (paper-shaped S = 32, P = 4: 6.07 ms in input order, 6.36 ms sorted)
    if (p->n_channels == 1 && (long long)p->n_baselines * p->n_times == p->n_vis) return false;
    return p->n_vis >= kCellSortMinSamples && (long long)p->N * p->N <= 8 * p->n_vis;
}
size_t cell_hist_entries(const grid_plan* p) {
    return ((size_t)p->N * p->N + 1 + kScanTile - 1) / kScanTile * kScanTile;
}
// [histogram / offsets][block sums][ranks]
size_t cell_sums_offset(const grid_plan* p) { return cell_hist_entries(p) * sizeof(uint32_t); }
size_t cell_ranks_offset(const grid_plan* p) {
    return cell_sums_offset(p) + (((cell_hist_entries(p) / kScanTile + 1) * sizeof(uint32_t) + 255) & ~(size_t)255);
}
size_t cell_sort_bytes(const grid_plan* p) {
    return cell_sort_on(p) ? cell_ranks_offset(p) + (size_t)((p->n_vis + 3) / 4 * 4) * sizeof(uint32_t) : 0;
}
size_t cell_sort_offset(const grid_plan* p) { return (tap_table_offset(p) + tap_table_bytes(p) + 255) & ~(size_t)255; }

// Derive bins, team shape and shared-memory footprint from the tuning; validate.
int derive(grid_plan* p) {
    if (p->variant == 0) {
        p->bin_u = p->bin_v = p->row_u = p->row_v = p->S;
        p->nbx = p->nby = p->S;
        p->team_threads = p->teams_per_cta = 0;
        p->smem_bytes = 0;
        return GRID_OK;
    }
    p->groups_per_cta = 0;
    if (p->variant == 3) {
        const int logs = log2_exact(p->Sk);
        if (logs < 2 || logs > 7)
            return fail(GRID_ERR_UNSUPPORTED, "variant 3 needs a support in [3, 128] (padded to a power of two) and a grid of "
                        "at least twice the padded support, got support %d on a grid of %d", p->S, p->N);
        WarpDesc d = lookup_warp(p->cu, p->cv, p->P, logs, p->pol_split);
        if (!d.fn)
            return fail(GRID_ERR_UNSUPPORTED, "coarsening block %dx%d (pol split %d) is not instantiated for %d pols, support %d",
                        p->cu, p->cv, p->pol_split, p->P, p->S);
        if (p->dense) {                                  // grid_execute_dense: no tap table on chip
            d = lookup_warp_dense(p->cu, p->cv, p->P, logs, p->dense);
            if (!d.fn || p->pol_split != 1)
                return fail(GRID_ERR_UNSUPPORTED, "dense GCF: block %dx%d is not instantiated for %d pols, support %d",
                            p->cu, p->cv, p->P, p->S);
        }
        // Tap table: in shared memory when it leaves at least half of it to the warp groups (and, for S = 32,
        // its offsets fit the record's 16 bits); otherwise read through L1/L2 from global memory (TG kernels).
        size_t taps = ((size_t)tap_rows(p) * 2 * p->Sk * sizeof(float2) + 15) & ~(size_t)15;
        p->taps_global = 0;
        if (p->dense) taps = 0;
        else if (taps > (size_t)p->max_smem / 2 || taps + d.group_bytes(p->batch) > (size_t)p->max_smem ||
            (logs == 5 && (long long)tap_rows(p) * 2 * p->Sk > 65535)) {
            const WarpDesc g = p->pol_split == 1 ? lookup_warp_tg(p->cu, p->cv, p->P, logs) : WarpDesc{nullptr, 0, 0, 0, 0, nullptr};
            if (!g.fn)
                return fail(GRID_ERR_UNSUPPORTED, "tap table (%zu B) needs the global-memory kernels, which are instantiated "
                            "for the default blocks with polarisation split 1 only (got %dx%d, split %d)",
                            taps, p->cu, p->cv, p->pol_split);
            d = g;
            taps = 0;
            p->taps_global = 1;
        }
        if (p->batch < 4 || (p->batch & (p->batch - 1)) != 0)
            return fail(GRID_ERR_UNSUPPORTED, "batch %d must be a power of two >= 4", p->batch);
        if (p->chunk < 1) return fail(GRID_ERR_UNSUPPORTED, "chunk %d must be positive", p->chunk);
        if (p->threads % 32 != 0 || p->threads < 32 || p->threads > 1024)
            return fail(GRID_ERR_UNSUPPORTED, "threads_per_cta %d must be a multiple of 32 in [32, 1024]", p->threads);
        int threads = p->threads < d.max_threads ? p->threads : d.max_threads;
        if (threads < d.gt)
            return fail(GRID_ERR_UNSUPPORTED, "a bin needs %d threads but the CTA may have %d", d.gt, threads);
        p->bin_u = p->bin_v = p->Sk;
        p->row_u = p->row_v = 2 * p->Sk;
        p->nbx = (p->Sk > 64 ? 64 : p->Sk) / p->cu;        // S = 128: a team covers a 64 x 64 tile of the bin
        p->nby = (p->Sk > 64 ? 64 : p->Sk) / p->cv;
        p->team_threads = d.team;
        int groups = threads / d.gt;
        if (d.gt > 32 && groups > 15) groups = 15;                 // one named barrier per group
        const size_t per_group = d.group_bytes(p->batch);
        if (taps + per_group > (size_t)p->max_smem)
            return fail(GRID_ERR_UNSUPPORTED, "tap tables (%zu B) + one group's buffers (%zu B) exceed %d B of shared memory",
                        taps, per_group, p->max_smem);
        const size_t fit = ((size_t)p->max_smem - taps) / per_group;
        if ((size_t)groups > fit) groups = (int)fit;
        p->groups_per_cta = groups;
        p->threads = groups * d.gt;
        p->teams_per_cta = groups * d.tpg;
        p->queue_teams = d.tpg;
        p->ctas_per_sm = 1;
        p->smem_bytes = (int)(taps + (size_t)groups * per_group);
        return GRID_OK;
    }
    if (!lookup_kernel(p->cu, p->cv, p->P))
        return fail(GRID_ERR_UNSUPPORTED, "coarsening block %dx%d is not instantiated for %d pols", p->cu, p->cv, p->P);
    // bin >= S + C - 1, multiple of the block
    p->bin_u = round_up(p->S + p->cu - 1, p->cu);
    p->bin_v = round_up(p->S + p->cv - 1, p->cv);
    p->row_u = p->bin_u + p->cu - 1;
    p->row_v = p->bin_v + p->cv - 1;
    p->nbx = p->bin_u / p->cu;
    p->nby = p->bin_v / p->cv;
    p->team_threads = p->nbx * p->nby;
    if (p->threads % 32 != 0 || p->threads < 32 || p->threads > 512)
        return fail(GRID_ERR_UNSUPPORTED, "threads_per_cta %d must be a multiple of 32 in [32, 512]", p->threads);
    if (p->team_threads > p->threads)
        return fail(GRID_ERR_UNSUPPORTED, "a bin needs %d threads but the CTA has %d (tiles across CTAs are not built yet)",
                    p->team_threads, p->threads);
    if (p->batch < 1 || (p->batch & (p->batch - 1)) != 0)
        return fail(GRID_ERR_UNSUPPORTED, "batch %d must be a power of two", p->batch);
    if (p->chunk < 1) return fail(GRID_ERR_UNSUPPORTED, "chunk %d must be positive", p->chunk);
    p->teams_per_cta = p->threads / p->team_threads;
    size_t taps = (size_t)p->W * p->O * p->row_u * sizeof(float2);
    if (p->cu != p->cv) taps += (size_t)p->W * p->O * p->row_v * sizeof(float2);
    taps = (taps + 15) & ~(size_t)15;
    const size_t per_team = (size_t)p->batch * (sizeof(SampleRec) + (size_t)p->P * sizeof(float2));
    if (taps + per_team > (size_t)p->max_smem)
        return fail(GRID_ERR_UNSUPPORTED, "tap tables (%zu B) + one batch buffer (%zu B) exceed %d B of shared memory",
                    taps, per_team, p->max_smem);
    // tiny bins: more teams than the batch buffers allow would not fit; idle the surplus threads
    const size_t fit = ((size_t)p->max_smem - taps) / per_team;
    if ((size_t)p->teams_per_cta > fit) p->teams_per_cta = (int)fit;
    const size_t stage = (size_t)p->teams_per_cta * per_team;
    p->smem_bytes = (int)(taps + stage);
    return GRID_OK;
}

void default_tuning(grid_plan* p) {
    p->variant = 1;
    p->threads = 256;
    p->batch = 64;
    p->chunk = 1024;
    p->ctas_per_sm = 2;
    p->traversal = -1;
    p->sort_chunks = -1;
    p->pol_split = 1;
    p->time_block = 64;
    // first guess per (S, P); refined by the autotune sweep -- see DESIGN.md
    if (p->P >= 4) {
        if (p->S >= 24) { p->cu = 4; p->cv = 2; }
        else if (p->S >= 12) { p->cu = 2; p->cv = 2; }
        else { p->cu = 2; p->cv = 1; }
    } else if (p->P == 2) {
        if (p->S >= 24) { p->cu = 4; p->cv = 4; }
        else { p->cu = 2; p->cv = 2; }
    } else {
        if (p->S >= 24) { p->cu = 8; p->cv = 4; }
        else if (p->S >= 12) { p->cu = 4; p->cv = 4; }
        else if (p->S >= 6) { p->cu = 4; p->cv = 2; }
        else { p->cu = 2; p->cv = 2; }
    }
    if (p->S < 4) { p->cu = 1; p->cv = 1; }
    // power-of-two supports: bin == support, no padding (grid_warp_kernel.cuh)
    const int logs = log2_exact(p->Sk);
    if (logs >= 2 && logs <= 7) {
        grid_plan trial = *p;
        trial.variant = 3;
        trial.threads = 1024;              // clipped to the kernel's register-limited maximum
        trial.batch = 32;
        trial.chunk = 256;
        // tuned per (S, P) on the BASELINE.json workloads
        const bool big_grid = (size_t)trial.N * trial.N * trial.P * sizeof(float2) > ((size_t)256 << 20);
        if (trial.P >= 4) {
            // grids beyond the L2 are bound by the atomic path: pair lanes so that one grid point
            // leaves as one 32-byte sector operation (grid_warp_kernel.cuh, PS)
            if (logs <= 3) { trial.cu = 2; trial.cv = 2; trial.pol_split = big_grid ? 2 : 1; }
            else if (logs == 4) { trial.cu = 4; trial.cv = 4; trial.pol_split = 2; }
            else { trial.cu = 4; trial.cv = 2; trial.pol_split = 1; }
        }
        else if (trial.P == 2) { trial.cu = (logs >= 3) ? 4 : 2; trial.cv = (logs >= 6) ? 4 : 2; }
        else if (logs == 2) { trial.cu = 2; trial.cv = 2; }
        else if (logs >= 5) { trial.cu = 8; trial.cv = 4; }
        else { trial.cu = 4; trial.cv = 4; }
        // Small inputs (fewer than ~4096 samples per SM; "low occupancy ... when the data is sparse") are
        // bound by the latency of a team's sequential walk, not by issue slots: small blocks spread a bin over more
        // threads (cfg0: 2x2 runs in 0.025 ms where 4x4 needs 0.054 ms).
        if (trial.n_vis >= 0 && trial.n_vis < 4096LL * trial.n_sm && logs <= 4) { trial.cu = 2; trial.cv = 2; }
        // Cell order (cell_sort.cuh): flushes are rare, so the block is chosen for the multiply-add loop alone and
        // lane pairing no longer pays (sweep of every instantiated block on the 11 large BASELINE.json workloads,
        // profiles/r2_cell_order.md); short chunks keep the CTAs in flight on neighbouring cells.
        if (cell_sort_on(&trial) && logs <= 5 && trial.P != 2) {
            trial.pol_split = 1;
            if (trial.P >= 4) {
                if (logs <= 3) { trial.cu = 2; trial.cv = 2; trial.pol_split = logs == 2 ? 2 : 1; }
                else { trial.cu = 4; trial.cv = 2; }
            } else {
                if (logs == 2) { trial.cu = 2; trial.cv = 2; }
                else if (logs == 3) { trial.cu = 4; trial.cv = 2; }
                else { trial.cu = 8; trial.cv = 4; }
            }
            if (logs <= 4) trial.chunk = 128;
        }
        // several teams share a warp at small supports: shrink the batch until all warps fit
        while (trial.batch > 8) {
            grid_plan probe = trial;
            if (derive(&probe) != GRID_OK) break;
            const WarpDesc d = lookup_warp(probe.cu, probe.cv, probe.P, logs, probe.pol_split);
            if (probe.threads >= d.max_threads - d.gt + 1) break;
            trial.batch /= 2;
        }
        if (derive(&trial) == GRID_OK) { *p = trial; return; }
        // tap table beyond shared memory: the global-memory kernels exist for split 1 and the default blocks
        trial.pol_split = 1;
        if (trial.P >= 4 && logs == 4) { trial.cu = 4; trial.cv = 2; }
        if (trial.P == 2) { trial.cu = 4; trial.cv = 2; }
        trial.batch = 32;
        if (derive(&trial) == GRID_OK) { *p = trial; return; }
    }
    // a bin must fit one CTA
    while (derive(p) != GRID_OK && p->threads < 512) p->threads *= 2;
    if (derive(p) != GRID_OK) {
        // supports whose bin exceeds a CTA (tiles across CTAs, are not built): smaller blocks,
        // and as the last resort the one-atomic-per-update kernel, which handles any support
        const int tries[4][2] = {{4, 2}, {2, 2}, {2, 1}, {1, 1}};
        for (int t = 0; t < 4 && derive(p) != GRID_OK; ++t) { p->cu = tries[t][0]; p->cv = tries[t][1]; p->threads = 512; }
        if (derive(p) != GRID_OK) {
            p->variant = 0; p->cu = p->cv = 1;
            snprintf(g_err, sizeof(g_err), "note: support %d on a grid of %d has no coarsened kernel; this plan uses the "
                     "one-atomic-per-update kernel (correct, slow)", p->S, p->N);
        } else {
            g_err[0] = 0;
        }
    }
}

long long ctas_hint(const grid_plan* p) { return (long long)p->n_sm * (p->groups_per_cta > 0 ? p->groups_per_cta : 1); }

QuantParams quant_params(const grid_plan* p) {
    QuantParams q;
    q.format = p->variant == 3 ? 2 : 0;
    q.c_centre = (double)p->O * (double)(p->N / 2) + 0.5;
    q.oversample = p->O;
    q.o_shift = -1;
    for (int k = 0; k < 16; ++k) if ((1 << k) == p->O) q.o_shift = k;
    q.shift = p->O - (p->O * p->S + 1) / 2;
    q.q_limit = (p->N - p->S + 1) * p->O;
    q.n_wplanes = p->W;
    q.pad = (p->variant == 3 && is_padded(p)) ? p->Sk - p->S : 0;
    q.sk = p->Sk;
    q.grid_size = p->N;
    const bool scatter = p->variant == 0;
    q.cu = scatter ? 1 : p->cu;
    q.cv = scatter ? 1 : p->cv;
    q.bin_u = p->bin_u; q.bin_v = p->bin_v; q.row_u = p->row_u; q.row_v = p->row_v;
    return q;
}

}  // namespace

// Autotuning: synthetic samples.  Tracks of a synthetic array: baseline b has a radius drawn
// log-uniformly up to 0.45 N and a random orientation; time step t turns it by 4 h / 256 per step (scaled to the
// hint's time count), channel c stretches it by up to 1.9x -- the structure of BASELINE.json's inputs, so that the
// footprint hops per sample as it does there.  Counter-based generator (one hash per value): no state.
__device__ __forceinline__ uint32_t tune_hash(uint32_t a, uint32_t b) {
    uint32_t x = a * 0x9E3779B1u ^ (b + 0x7F4A7C15u) * 0x85EBCA77u;
    x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
    return x;
}
__device__ __forceinline__ float tune_unit(uint32_t a, uint32_t b) { return (tune_hash(a, b) >> 8) * (1.0f / 16777216.0f); }

__global__ void __launch_bounds__(256)
tune_fill_kernel(float* __restrict__ uvw, float2* __restrict__ vis, float* __restrict__ weights, long long n, int P,
                 int N, int S, int W, int n_times, int n_chan, unsigned int seed, float extent) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const long long row = k / n_chan;
    const int c = (int)(k - row * n_chan), t = (int)(row % n_times);
    const uint32_t b = (uint32_t)(row / n_times);
    // extent < 1 (cell order): the tracks cover that fraction of the grid's width, so that the synthetic set has as
    // many samples per grid cell as the caller's input -- which is what decides how often a sorted walk moves
    const float rmax = fmaxf((0.45f * N - S) * extent, 2.f), rmin = fminf(0.02f * N * extent, rmax);
    const float r = rmin * __powf(rmax / rmin, tune_unit(seed, 3 * b));            // log-uniform radius
    const float th0 = 6.2831853f * tune_unit(seed, 3 * b + 1);
    const float th = th0 + 1.0471976f * (t - 0.5f * n_times) / (n_times > 1 ? n_times : 1);   // 60 degrees over the track
    const float f = n_chan > 1 ? 1.0f - 0.47f * (float)(n_chan - 1 - c) / (float)(n_chan - 1) : 1.0f;   // 0.9-1.7 GHz
    uvw[3 * k] = r * f * __cosf(th);
    uvw[3 * k + 1] = 0.5f * r * f * __sinf(th);                                   // declination -30 degrees: v compressed
    uvw[3 * k + 2] = W * tune_unit(seed, 3 * b + 2) * f;
    weights[k] = 0.5f + 0.5f * tune_unit(seed + 1, (uint32_t)k);
    for (int q = 0; q < P; ++q)
        vis[k * P + q] = make_float2(tune_unit(seed + 2, (uint32_t)(k * P + q)) - 0.5f, tune_unit(seed + 3, (uint32_t)(k * P + q)) - 0.5f);
}

__global__ void __launch_bounds__(256) tune_taps_kernel(float2* __restrict__ kern, int rows, int S) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= rows * S) return;
    const float d = (float)(k % S) - 0.5f * S + 0.5f;
    kern[k] = make_float2(__expf(-4.0f * d * d / (float)(S * S)), 1e-3f * d);
}

template <int P>
static void launch_degrid(int L, long long n, const CycRec* recs, const float* weights, const float2* kern,
                          const float2* grid, float2* out, int N, int S, cudaStream_t stream) {
    const unsigned blocks = (unsigned)((n * L + 255) / 256);
    if (L == 8) degrid_gather_kernel<P, 8><<<blocks, 256, 0, stream>>>(recs, weights, kern, grid, out, n, N, S);
    else if (L == 16) degrid_gather_kernel<P, 16><<<blocks, 256, 0, stream>>>(recs, weights, kern, grid, out, n, N, S);
    else degrid_gather_kernel<P, 32><<<blocks, 256, 0, stream>>>(recs, weights, kern, grid, out, n, N, S);
}

extern "C" {

const char* grid_last_error(void) { return g_err; }

grid_plan* grid_plan_create(int grid_size, int support, int oversample, int n_wplanes, int n_pol) {
    g_err[0] = 0;
    if (grid_size < 1 || grid_size > 32767 || support < 1 || support > grid_size || support > 128 ||
        oversample < 1 || n_wplanes < 1 || (long long)n_wplanes * oversample > 65535 ||
        !(n_pol == 1 || n_pol == 2 || n_pol == 4) ||
        (long long)(grid_size - support + 1) * oversample > 0x7fffffffLL) {
        fail(GRID_ERR_INVALID_ARG, "grid_plan_create: invalid argument (N=%d S=%d O=%d W=%d P=%d)",
             grid_size, support, oversample, n_wplanes, n_pol);
        return nullptr;
    }
    // Without a device the plan can still be created and inspected (host logic); every compute
    // entry point then fails with GRID_ERR_CUDA -- there is no CPU fallback.
    int dev = 0, n_sm = 148, max_smem = 227 * 1024;
    if (cudaGetDevice(&dev) == cudaSuccess) {
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    } else {
        (void)cudaGetLastError();
    }
    grid_plan* p = new (std::nothrow) grid_plan();
    if (!p) { fail(GRID_ERR_INVALID_ARG, "out of host memory"); return nullptr; }
    memset(p, 0, sizeof(*p));
    p->N = grid_size; p->S = support; p->O = oversample; p->W = n_wplanes; p->P = n_pol;
    p->Sk = padded_support(support, grid_size, n_wplanes, oversample);
    p->n_vis = -1;
    p->sample_order = -1;
    p->n_sm = n_sm;
    p->max_smem = max_smem - 1024;      // leave room for static shared memory
    default_tuning(p);
    if (derive(p) != GRID_OK) { delete p; return nullptr; }
    return p;
}

void grid_plan_destroy(grid_plan* plan) { delete plan; }

// the default block depends on the size of the input and on the order the samples are gridded in
static void retune(grid_plan* plan) {
    if (plan->user_tuned) return;
    grid_plan trial = *plan;
    default_tuning(&trial);
    trial.traversal = plan->traversal; trial.time_block = plan->time_block;     // set by their own calls
    trial.sort_chunks = plan->sort_chunks;
    if (derive(&trial) == GRID_OK) *plan = trial;
    g_err[0] = 0;
}

int grid_plan_set_samples(grid_plan* plan, long long n_vis) {
    if (!plan || n_vis < 0) return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_samples: invalid argument");
    plan->n_vis = n_vis;
    plan->order_kept = 0;
    retune(plan);
    return GRID_OK;
}

int grid_plan_set_layout(grid_plan* plan, int n_baselines, int n_times, int n_channels) {
    if (!plan || n_baselines < 0 || n_times < 0 || n_channels < 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_layout: invalid argument");
    plan->n_baselines = n_baselines; plan->n_times = n_times; plan->n_channels = n_channels;
    plan->order_kept = 0;
    retune(plan);                                    // the automatic sample order looks at the layout
    return GRID_OK;
}

size_t grid_plan_workspace_bytes(const grid_plan* plan) {
    if (!plan || plan->n_vis < 0) return 0;
    return cell_sort_on(plan) ? cell_sort_offset(plan) + cell_sort_bytes(plan) : tap_table_offset(plan) + tap_table_bytes(plan);
}

int grid_plan_set_workspace(grid_plan* plan, void* dev_ptr, size_t bytes) {
    if (!plan || (!dev_ptr && bytes) || ((uintptr_t)dev_ptr & 255) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_workspace: null or misaligned pointer");
    plan->workspace = dev_ptr;
    plan->workspace_bytes = bytes;
    plan->order_kept = 0;
    return GRID_OK;
}

int grid_plan_set_tuning(grid_plan* plan, int variant, int cu, int cv, int threads_per_cta, int batch,
                         int chunk, int ctas_per_sm) {
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_tuning: null plan");
    grid_plan trial = *plan;
    if (variant >= 0 && variant != trial.variant) {
        trial.variant = variant;
        // the other kernel's thread count does not carry over (variant 3 runs one CTA of up to 1024 threads per SM)
        if (threads_per_cta <= 0) trial.threads = variant == 3 ? 1024 : 256;
        if (ctas_per_sm <= 0) trial.ctas_per_sm = variant == 3 ? 1 : 2;
        if (variant != 3 && batch <= 0 && trial.batch < 16) trial.batch = 64;
    }
    if (cu > 0) trial.cu = cu;
    if (cv > 0) trial.cv = cv;
    if (threads_per_cta > 0) trial.threads = threads_per_cta;
    if (batch > 0) trial.batch = batch;
    if (chunk > 0) trial.chunk = chunk;
    if (ctas_per_sm > 0) trial.ctas_per_sm = ctas_per_sm;
    if (trial.variant < 0 || trial.variant > 3 || trial.variant == 2)
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_tuning: unknown variant %d", trial.variant);
    int rc = derive(&trial);
    if (rc != GRID_OK && trial.pol_split != 1 && (cu > 0 || cv > 0 || variant >= 0)) {
        trial.pol_split = 1;                // a block the current polarisation split does not offer
        rc = derive(&trial);
    }
    if (rc != GRID_OK) return rc;
    *plan = trial;
    plan->user_tuned = 1;
    plan->order_kept = 0;
    return GRID_OK;
}

static int execute_impl(grid_plan* plan, const float* uvw, const void* ext_recs, long long n_vis, const float* vis,
                        const float* weights, const float* conv_kernel, float* grid, cudaStream_t stream,
                        float* degrid_out = nullptr);

int grid_plan_autotune_candidates(const grid_plan* plan, int* out, int max_candidates) {
    if (!plan || !out || max_candidates < 1) return fail(GRID_ERR_INVALID_ARG, "grid_plan_autotune_candidates: invalid argument");
    if (plan->variant != 3) return 0;
    static const int blocks[][2] = {{2, 2}, {4, 2}, {4, 4}, {8, 4}};
    int n = 0;
    auto offer = [&](int cu, int cv, int ps) {
        if (n >= max_candidates) return;
        for (int k = 0; k < n; ++k) if (out[3 * k] == cu && out[3 * k + 1] == cv && out[3 * k + 2] == ps) return;
        grid_plan trial = *plan;
        trial.cu = cu; trial.cv = cv; trial.pol_split = ps; trial.threads = 1024;
        if (derive(&trial) != GRID_OK || trial.pol_split != ps) return;
        out[3 * n] = cu; out[3 * n + 1] = cv; out[3 * n + 2] = ps;
        ++n;
    };
    offer(plan->cu, plan->cv, plan->pol_split);                  // the current block first
    for (int ps = 1; ps <= (plan->P == 4 ? 2 : 1); ++ps)
        for (const auto& b : blocks) offer(b[0], b[1], ps);
    g_err[0] = 0;
    return n;
}

int grid_plan_autotune(grid_plan* plan, long long n_samples, unsigned int seed, float* results, int max_candidates,
                       grid_stream_t stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!plan || n_samples < 0) return fail(GRID_ERR_INVALID_ARG, "grid_plan_autotune: invalid argument");
    if (plan->variant != 3) return fail(GRID_ERR_UNSUPPORTED, "grid_plan_autotune: the plan does not run the warp kernel");
    int cand[3 * 32];
    const int n_cand = grid_plan_autotune_candidates(plan, cand, 32);
    if (n_cand <= 0) return fail(GRID_ERR_UNSUPPORTED, "grid_plan_autotune: no candidate block fits this plan");
    // shape of the synthetic data: the caller's layout if there is one, else single-channel tracks
    const bool hint = plan->n_baselines > 0 && plan->n_times > 0 && plan->n_channels > 0;
    const int n_times = hint ? plan->n_times : 256, n_chan = hint ? plan->n_channels : 1;
    long long n = n_samples > 0 ? n_samples : (1LL << 20);
    long long n_bl = n / ((long long)n_times * n_chan);
    if (n_bl < 1) n_bl = 1;
    n = n_bl * n_times * n_chan;
    if (n >= 0x7fffffffLL) return fail(GRID_ERR_INVALID_ARG, "grid_plan_autotune: too many samples");

    grid_plan t = *plan;                                         // a private plan: the caller's stays untouched until the end
    t.n_vis = n; t.n_baselines = (int)n_bl; t.n_times = n_times; t.n_channels = n_chan;
    // tune in the sample order the caller's plan will grid in (the synthetic set is smaller than the real input and
    // would not always get the same automatic choice)
    if (plan->n_vis > 0) t.sample_order = cell_sort_on(plan) ? 1 : 0;
    t.order_kept = 0;
    float extent = 1.f;
    if (cell_sort_on(&t) && plan->n_vis > n) extent = sqrtf((float)n / (float)plan->n_vis);
    t.ev_start = t.ev_stop = nullptr;
    const size_t grid_bytes = (size_t)plan->N * plan->N * plan->P * sizeof(float2);
    const size_t kern_bytes = (size_t)plan->W * plan->O * plan->S * sizeof(float2);
    float *d_uvw = nullptr, *d_w = nullptr, *d_grid = nullptr;
    float2 *d_vis = nullptr, *d_kern = nullptr;
    void* d_ws = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = GRID_OK, best = -1;
    float best_us = 0.f;
    auto cleanup = [&]() {
        cudaFree(d_uvw); cudaFree(d_w); cudaFree(d_grid); cudaFree(d_vis); cudaFree(d_kern); cudaFree(d_ws);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    };
    t.workspace_bytes = grid_plan_workspace_bytes(&t);
    if (cudaMalloc(&d_uvw, (size_t)n * 12) != cudaSuccess || cudaMalloc(&d_w, (size_t)n * 4) != cudaSuccess ||
        cudaMalloc(&d_vis, (size_t)n * plan->P * 8) != cudaSuccess || cudaMalloc(&d_kern, kern_bytes) != cudaSuccess ||
        cudaMalloc(&d_grid, grid_bytes) != cudaSuccess || cudaMalloc(&d_ws, t.workspace_bytes) != cudaSuccess ||
        cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        (void)cudaGetLastError();
        cleanup();
        return fail(GRID_ERR_CUDA, "grid_plan_autotune: no device, or out of device memory for the synthetic data set");
    }
    t.workspace = d_ws;
    tune_fill_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(d_uvw, d_vis, d_w, n, plan->P, plan->N, plan->S, plan->W,
                                                                     n_times, n_chan, seed, extent);
    tune_taps_kernel<<<(unsigned)(((long long)plan->W * plan->O * plan->S + 255) / 256), 256, 0, stream>>>(d_kern, plan->W * plan->O, plan->S);
    cudaMemsetAsync(d_grid, 0, grid_bytes, stream);
    for (int k = 0; k < n_cand && rc == GRID_OK; ++k) {
        grid_plan trial = t;
        trial.cu = cand[3 * k]; trial.cv = cand[3 * k + 1]; trial.pol_split = cand[3 * k + 2]; trial.threads = 1024;
        float us = -1.f;
        if (derive(&trial) == GRID_OK) {
            bool ok = true;
            for (int rep = 0; rep < 2 && ok; ++rep) {            // the second run is the measurement
                cudaEventRecord(e0, stream);
                ok = execute_impl(&trial, d_uvw, nullptr, n, reinterpret_cast<const float*>(d_vis), d_w,
                                  reinterpret_cast<const float*>(d_kern), d_grid, stream, nullptr) == GRID_OK;
                cudaEventRecord(e1, stream);
            }
            if (ok && cudaEventSynchronize(e1) == cudaSuccess) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                us = ms * 1e3f;
            } else if (cudaGetLastError() != cudaSuccess) {
                rc = fail(GRID_ERR_CUDA, "grid_plan_autotune: a candidate failed on the device");
            }
        }
        if (results && k < max_candidates) results[k] = us;
        if (us > 0.f && (best < 0 || us < best_us)) { best = k; best_us = us; }
    }
    cudaStreamSynchronize(stream);
    cleanup();
    if (rc != GRID_OK) return rc;
    if (best < 0) return fail(GRID_ERR_UNSUPPORTED, "grid_plan_autotune: no candidate ran");
    grid_plan tuned = *plan;
    tuned.cu = cand[3 * best]; tuned.cv = cand[3 * best + 1]; tuned.pol_split = cand[3 * best + 2]; tuned.threads = 1024;
    if (derive(&tuned) != GRID_OK) return GRID_ERR_UNSUPPORTED;
    *plan = tuned;
    plan->user_tuned = 1;
    g_err[0] = 0;
    return GRID_OK;
}

int grid_plan_get_info(const grid_plan* plan, int* out) {
    if (!plan || !out) return fail(GRID_ERR_INVALID_ARG, "grid_plan_get_info: null argument");
    const int v[20] = {plan->variant, plan->cu, plan->cv, plan->bin_u, plan->bin_v, plan->team_threads,
                       plan->teams_per_cta, plan->threads, plan->batch, plan->chunk, plan->ctas_per_sm,
                       plan->smem_bytes, plan->n_sm, plan->traversal, plan->time_block, plan->sort_chunks,
                       plan->pol_split, plan->groups_per_cta, plan->taps_global, cell_sort_on(plan) ? 1 : 0};
    memcpy(out, v, sizeof(v));
    return GRID_OK;
}

int grid_plan_set_traversal(grid_plan* plan, int mode, int time_block) {
    if (!plan || mode < -1 || mode > 1 || time_block < 0 || (time_block & (time_block - 1)) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_traversal: mode in {-1,0,1}, time_block a power of two or 0");
    plan->traversal = mode;
    if (time_block > 0) plan->time_block = time_block;
    return GRID_OK;
}

int grid_plan_set_pol_split(grid_plan* plan, int lanes) {
    if (!plan || (lanes != 1 && lanes != 2))
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_pol_split: lanes in {1,2}");
    grid_plan trial = *plan;
    trial.pol_split = lanes;
    trial.threads = 1024;
    const int rc = derive(&trial);
    if (rc != GRID_OK) return rc;
    *plan = trial;
    plan->user_tuned = 1;
    plan->order_kept = 0;
    return GRID_OK;
}

int grid_plan_set_degrid_gather(grid_plan* plan, int on) {
    if (!plan || (on != 0 && on != 1)) return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_degrid_gather: on in {0,1}");
    plan->degrid_gather = on;
    return GRID_OK;
}

int grid_plan_set_chunk_order(grid_plan* plan, int mode) {
    if (!plan || mode < -1 || mode > 1)
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_chunk_order: mode in {-1,0,1}");
    plan->sort_chunks = mode;
    return GRID_OK;
}

int grid_plan_set_sample_order(grid_plan* plan, int mode) {
    if (!plan || mode < -1 || mode > 2) return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_sample_order: mode must be -1, 0, 1 or 2");
    plan->order_kept = 0;
    if (mode >= 1 && plan->variant != 3)
        return fail(GRID_ERR_UNSUPPORTED, "grid_plan_set_sample_order: cell order needs the warp kernel (variant 3)");
    plan->sample_order = mode;
    retune(plan);
    return GRID_OK;
}

int grid_plan_last_launches(const grid_plan* plan) { return plan ? plan->last_launches : 0; }

int grid_plan_debug_counters(grid_plan* plan, unsigned int* out, grid_stream_t stream) {
    if (!plan || !out) return fail(GRID_ERR_INVALID_ARG, "grid_plan_debug_counters: null argument");
    memset(out, 0, 8 * sizeof(unsigned int));
    if (!plan->workspace) return GRID_OK;
    const unsigned int* src = reinterpret_cast<const unsigned int*>(plan->workspace) + kCheckBase;
    if (cudaMemcpyAsync(out, src, 8 * sizeof(unsigned int), cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
        return fail(GRID_ERR_CUDA, "grid_plan_debug_counters: %s", cudaGetErrorString(cudaGetLastError()));
    return GRID_OK;
}

int grid_plan_set_kernel_events(grid_plan* plan, void* ev_start, void* ev_stop) {
    if (!plan || ((ev_start == nullptr) != (ev_stop == nullptr)))
        return fail(GRID_ERR_INVALID_ARG, "grid_plan_set_kernel_events: pass two events or two NULLs");
    plan->ev_start = (cudaEvent_t)ev_start;
    plan->ev_stop = (cudaEvent_t)ev_stop;
    return GRID_OK;
}

int grid_quantise(grid_plan* plan, const float* uvw, long long n, int* out, grid_stream_t stream) {
    if (!plan || n < 0 || (n > 0 && (!uvw || !out)))
        return fail(GRID_ERR_INVALID_ARG, "grid_quantise: invalid argument");
    if (n == 0) return GRID_OK;
    const long long blocks = (n + 255) / 256;
    quantise_debug_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(uvw, out, n, quant_params(plan));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_quantise: %s", cudaGetErrorString(e));
    return GRID_OK;
}

// grid_execute proper.  ext_recs != NULL: the samples are already quantised and pre-weighted (compressed
// input): no a1 pass, no weights, records read from ext_recs; n_vis samples.
// degrid_out != NULL: run the DEGRID kernel (grid is read, degrid_out written; plan must be variant 3,
// pol split 1, team <= 32 -- the caller checks with lookup_degrid).
static int execute_impl(grid_plan* plan, const float* uvw, const void* ext_recs, long long n_vis, const float* vis,
                        const float* weights, const float* conv_kernel, float* grid, cudaStream_t stream,
                        float* degrid_out) {
    unsigned int* counters = reinterpret_cast<unsigned int*>(plan->workspace);
    SampleRec* recs = ext_recs ? reinterpret_cast<SampleRec*>(const_cast<void*>(ext_recs))
                               : reinterpret_cast<SampleRec*>(reinterpret_cast<unsigned char*>(plan->workspace) + kHeadBytes);
    uint32_t* bins = counters + 64;
    uint32_t* order = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned char*>(plan->workspace) + kHeadBytes + records_bytes(plan));

    // cell order: the a1 pass sorts the samples by grid cell (cell_sort.cuh); chunks are runs of the sorted records
    const bool sorted = !ext_recs && n_vis == plan->n_vis && cell_sort_on(plan);
    // the layout hint is used only if it is consistent with the sample count
    const bool have_layout = !sorted && !ext_recs && plan->n_channels > 0 && plan->n_times > 0 && plan->n_baselines > 0 &&
                             (long long)plan->n_baselines * plan->n_times * plan->n_channels == n_vis;
    const int n_chan = have_layout ? plan->n_channels : 0, n_times = have_layout ? plan->n_times : 0;
    float* hop_stats = reinterpret_cast<float*>(counters + 2);

    if (plan->variant == 3 && n_vis >= 0x7fffffffLL)
        return fail(GRID_ERR_UNSUPPORTED, "grid_execute: the warp kernel indexes samples with 31 bits (n_vis = %lld)", n_vis);
    // reset the chunk queue and the hop statistics, then a1: quantise pass
    if (cudaMemsetAsync(counters, 0, kHeadBytes, stream) != cudaSuccess)
        return fail(GRID_ERR_CUDA, "grid_execute: %s", cudaGetErrorString(cudaGetLastError()));
    // mode 2: the caller guarantees the same uvw and weights as in the call that sorted them -- the records are reused
    const bool keep = sorted && plan->sample_order == 2;
    if (sorted && keep && plan->order_kept) {
    } else if (sorted) {
        unsigned char* scratch = reinterpret_cast<unsigned char*>(plan->workspace) + cell_sort_offset(plan);
        uint32_t* hist = reinterpret_cast<uint32_t*>(scratch);
        uint32_t* sums = reinterpret_cast<uint32_t*>(scratch + cell_sums_offset(plan));
        uint32_t* ranks = reinterpret_cast<uint32_t*>(scratch + cell_ranks_offset(plan));
        const size_t entries = cell_hist_entries(plan);
        const unsigned scan_blocks = (unsigned)(entries / kScanTile);
        if (cudaMemsetAsync(hist, 0, entries * sizeof(uint32_t), stream) != cudaSuccess)
            return fail(GRID_ERR_CUDA, "grid_execute: %s", cudaGetErrorString(cudaGetLastError()));
        const unsigned blocks = (unsigned)(((n_vis + 3) / 4 + 255) / 256);
        const QuantParams qp = quant_params(plan);
        cell_count_kernel<<<blocks, 256, 0, stream>>>(uvw, n_vis, qp, hist, ranks);
        cell_scan_reduce_kernel<<<scan_blocks, 256, 0, stream>>>(hist, sums);
        cell_scan_sums_kernel<<<1, 1024, 0, stream>>>(sums, (int)scan_blocks);
        cell_scan_apply_kernel<<<scan_blocks, 256, 0, stream>>>(hist, sums);
        if (plan->P == 1 && !degrid_out && !keep)  // degridding needs the sample's index (where its result goes), kept records too
            cell_scatter_kernel<true><<<blocks, 256, 0, stream>>>(uvw, weights, reinterpret_cast<const float2*>(vis), n_vis, qp,
                                                                  hist, ranks, reinterpret_cast<uint4*>(recs));
        else
            cell_scatter_kernel<false><<<blocks, 256, 0, stream>>>(uvw, weights, nullptr, n_vis, qp, hist, ranks,
                                                                   reinterpret_cast<uint4*>(recs));
        plan->last_launches += 5;
        plan->order_kept = keep ? 1 : 0;
    } else if (!ext_recs) {
        const long long threads = (n_vis + 3) / 4;
        const long long blocks = (threads + 255) / 256;
        quantise_kernel<<<(unsigned)blocks, 256, 0, stream>>>(uvw, recs, n_vis, quant_params(plan), hop_stats,
                                                             n_chan, n_times, (float)(plan->bin_u + plan->bin_v), weights);
        plan->last_launches++;
    }

    GridParams gp;
    memset(&gp, 0, sizeof(gp));
    gp.recs = recs;
    gp.vis = reinterpret_cast<const float2*>(vis);
    gp.weights = weights;
    gp.kern = reinterpret_cast<const float2*>(conv_kernel);
    gp.grid = grid;
    gp.vis_out = reinterpret_cast<float2*>(degrid_out);
    gp.counters = counters;
    gp.rec16 = (plan->variant == 3 && !ext_recs) ? 1 : 0;
    gp.sorted = !sorted ? 0 : (plan->P == 1 && !degrid_out && !keep) ? 1 : 2;   // 1: records carry weight * vis, 2: {weight, index}
    gp.sorted_stride = kCellRecStride;
    gp.n_vis = n_vis;
    gp.N = plan->N; gp.S = plan->variant == 3 ? plan->Sk : plan->S;
    gp.n_rows = plan->variant == 3 ? tap_rows(plan) : plan->W * plan->O;
    gp.tap_pad = plan->variant == 3 ? plan->Sk - plan->S : 0;
    gp.dense_pol_stride = plan->dense == 2 ? (long long)plan->W * plan->O * plan->O * plan->S * plan->S : 0;
    gp.oversample = plan->O;
    gp.bin_u = plan->bin_u; gp.bin_v = plan->bin_v; gp.row_u = plan->row_u; gp.row_v = plan->row_v;
    gp.nbx = plan->nbx; gp.nby = plan->nby;
    gp.team_threads = plan->team_threads; gp.teams_per_cta = plan->teams_per_cta;
    gp.batch = plan->batch; gp.chunk = plan->chunk;

    if (plan->variant == 0) {
        if (plan->ev_start) cudaEventRecord(plan->ev_start, stream);
        const long long total = n_vis * plan->S;
        const long long blocks = (total + 255) / 256;
        if (blocks > 0x7fffffffLL) return fail(GRID_ERR_UNSUPPORTED, "grid_execute: too many samples for the scatter variant");
        if (plan->P == 1) grid_scatter_kernel<1><<<(unsigned)blocks, 256, 0, stream>>>(gp);
        else if (plan->P == 2) grid_scatter_kernel<2><<<(unsigned)blocks, 256, 0, stream>>>(gp);
        else grid_scatter_kernel<4><<<(unsigned)blocks, 256, 0, stream>>>(gp);
        plan->last_launches++;
    } else {
        int shift = 0;
        while ((1 << shift) < plan->batch) ++shift;
        gp.batch_shift = shift;
        // adaptive chunk length for small inputs: keep every SM busy
        const int qt = plan->variant == 3 ? plan->queue_teams : plan->teams_per_cta;   // teams per queue entry
        const int queues = plan->variant == 3 ? plan->groups_per_cta : 1;               // queue consumers per CTA
        long long want_groups = (long long)plan->n_sm * plan->ctas_per_sm * queues * 4;
        long long per_group = (long long)qt * plan->chunk;
        if ((n_vis + per_group - 1) / per_group < want_groups) {
            long long chunk = n_vis / (want_groups * qt);
            chunk = (chunk + plan->batch - 1) / plan->batch * plan->batch;
            if (chunk < plan->batch) chunk = plan->batch;
            if (chunk < gp.chunk) gp.chunk = (int)chunk;
            per_group = (long long)qt * gp.chunk;
        }
        gp.n_groups_a = (n_vis + per_group - 1) / per_group;
        gp.groups_per_cta = plan->groups_per_cta;
        // time-innermost decomposition: chunk = tc time steps x all channels of one baseline
        gp.hop_stats = hop_stats;
        gp.force_mode = have_layout ? plan->traversal : 0;
        gp.n_chan = n_chan; gp.n_times = n_times;
        // the padded kernel stages whole columns per batch (tc <= batch); the warp kernel does not care
        int tc = plan->time_block;
        if (plan->variant != 3) {
            if (tc > plan->batch) tc = plan->batch;
            if (tc > 16) tc = 16;          // its chunks are whole (baseline, time block) slabs: keep them small
            // small inputs: shorter time blocks until every team has a chunk
            while (have_layout && tc > 4 &&
                   (long long)plan->n_baselines * ((n_times + tc - 1) / tc) < want_groups * qt / 4) tc /= 2;
        }
        if (have_layout) {
            while (tc > 1 && tc / 2 >= n_times) tc /= 2;
            int tshift = 0;
            while ((1 << tshift) < tc) ++tshift;
            gp.tc = tc;
            gp.cb_shift = shift > tshift ? shift - tshift : 0;
            gp.n_tblocks = (n_times + tc - 1) / tc;
            gp.n_cblocks = 1;
            gp.chunk_cols = n_chan;
            if (plan->variant == 3) {      // chunk = tc time steps x chunk_cols channels ~ gp.chunk samples
                int cols = gp.chunk / tc;
                if (cols < 1) cols = 1;
                if (cols > n_chan) cols = n_chan;
                gp.chunk_cols = cols;
                gp.n_cblocks = (n_chan + cols - 1) / cols;
            }
            gp.n_chunks_b = (long long)plan->n_baselines * gp.n_tblocks * gp.n_cblocks;
            gp.n_groups_b = (gp.n_chunks_b + qt - 1) / qt;
        } else {
            gp.tc = 1; gp.n_tblocks = 1;
        }
        if (plan->variant == 3 && plan->Sk == 128) {              // 2 x 2 tiles per bin: four queue entries per chunk group
            gp.n_groups_a *= 4;
            gp.n_groups_b *= 4;
        }
        const long long max_groups = gp.n_groups_a > gp.n_groups_b ? gp.n_groups_a : gp.n_groups_b;
        const int logs = log2_exact(plan->variant == 3 ? plan->Sk : plan->S);
        if (plan->variant == 3 && plan->taps_global && !plan->dense) {   // a4: row-doubled table in global memory
            float2* gt = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(plan->workspace) + tap_table_offset(plan));
            const long long n_elems = (long long)tap_rows(plan) * 2 * plan->Sk;
            tap_table_kernel<<<(unsigned)((n_elems + 255) / 256), 256, 0, stream>>>(gp.kern, gt, n_elems, plan->Sk, plan->Sk - plan->S);
            gp.gtaps = gt;
            plan->last_launches++;
        }
        kernel_fn fn = plan->dense ? lookup_warp_dense(plan->cu, plan->cv, plan->P, logs, plan->dense).fn
                     : degrid_out ? lookup_degrid(plan->cu, plan->cv, plan->P, logs, plan->taps_global != 0)
                     : (plan->variant == 3 && plan->taps_global) ? lookup_warp_tg(plan->cu, plan->cv, plan->P, logs).fn
                     : plan->variant == 3 ? lookup_warp(plan->cu, plan->cv, plan->P, logs, plan->pol_split,
                                                        (size_t)plan->N * plan->N * plan->P * sizeof(float2) > ((size_t)1 << 30)).fn
                                          : lookup_kernel(plan->cu, plan->cv, plan->P);
        // a9 locality: sort the chunk ids by grid tile when the grid does not fit the L2
        if (plan->variant == 3) {
            const long long chunks_a = (n_vis + gp.chunk - 1) / gp.chunk;
            const long long max_chunks = chunks_a > gp.n_chunks_b ? chunks_a : gp.n_chunks_b;
            const size_t grid_bytes = (size_t)plan->N * plan->N * plan->P * sizeof(float2);
            const bool want = !sorted && (plan->sort_chunks > 0 || (plan->sort_chunks < 0 && grid_bytes > ((size_t)256 << 20)));
            const bool worth = plan->sort_chunks > 0 || max_chunks >= 4LL * ctas_hint(plan);   // auto: only when chunks queue up
            if (want && worth && max_chunks <= (long long)order_capacity(plan)) {
                int ts = 0;
                while ((plan->N >> ts) > 32) ++ts;
                gp.tile_shift = ts;
                const unsigned blocks = (unsigned)((max_chunks + 255) / 256);
                chunk_histogram_kernel<<<blocks, 256, 0, stream>>>(gp, bins);
                chunk_scan_kernel<<<1, kOrderBins, 0, stream>>>(bins);
                chunk_scatter_kernel<<<blocks, 256, 0, stream>>>(gp, bins, order);
                gp.order = order;
                plan->last_launches += 3;
            }
        }
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, plan->smem_bytes);
        if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_execute: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        if (plan->ev_start) cudaEventRecord(plan->ev_start, stream);
        long long ctas = (long long)plan->n_sm * plan->ctas_per_sm;
        const long long need = (max_groups + queues - 1) / queues;
        if (ctas > need) ctas = need;
        fn<<<(unsigned)ctas, plan->threads, plan->smem_bytes, stream>>>(gp);
        plan->last_launches++;
    }
    if (plan->ev_stop) cudaEventRecord(plan->ev_stop, stream);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_execute: launch failed: %s", cudaGetErrorString(e));
    return GRID_OK;
}

int grid_execute(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                 const float* conv_kernel, float* grid, grid_stream_t stream) {
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_execute: null plan");
    plan->last_launches = 0;
    if (plan->n_vis < 0) return fail(GRID_ERR_STATE, "grid_execute: call grid_plan_set_samples first");
    if (plan->n_vis == 0) return GRID_OK;                              // R23
    if (!uvw || !vis || !weights || !conv_kernel || !grid)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute: null array argument");
    if ((((uintptr_t)uvw | (uintptr_t)vis | (uintptr_t)weights | (uintptr_t)conv_kernel | (uintptr_t)grid) & 15) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute: array arguments must be 16-byte aligned");
    if (!plan->workspace || plan->workspace_bytes < grid_plan_workspace_bytes(plan))
        return fail(GRID_ERR_STATE, "grid_execute: workspace missing or smaller than grid_plan_workspace_bytes()");
    return execute_impl(plan, uvw, nullptr, plan->n_vis, vis, weights, conv_kernel, grid, (cudaStream_t)stream);
}

// ---- grid_execute_static: the call's workspace in the library's own device image (no allocation anywhere).
// In host code `g_static_scratch` is a host-side stand-in for the symbol, NOT a device address: the device address
// is asked for once per device (cudaGetSymbolAddress, with that device current) and that pointer goes to the kernels.
static __device__ __align__(256) unsigned char g_static_scratch[GRID_STATIC_SCRATCH_BYTES];

static int static_scratch_pointer(void** out) {
    constexpr int kMaxDevices = 64;
    static void* ptrs[kMaxDevices] = {nullptr};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        (void)cudaGetLastError();
        return fail(GRID_ERR_CUDA, "grid_execute_static: no current CUDA device (the gridder has no CPU fallback)");
    }
    if (!ptrs[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return fail(GRID_ERR_CUDA, "grid_execute_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        }
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return GRID_OK;
}

int grid_execute_static(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                        const float* conv_kernel, float* grid, grid_stream_t stream) {
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_execute_static: null plan");
    plan->last_launches = 0;
    if (plan->n_vis < 0) return fail(GRID_ERR_STATE, "grid_execute_static: call grid_plan_set_samples first");
    if (plan->n_vis == 0) return GRID_OK;                              // R23
    if (!uvw || !vis || !weights || !conv_kernel || !grid)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_static: null array argument");
    if ((((uintptr_t)uvw | (uintptr_t)vis | (uintptr_t)weights | (uintptr_t)conv_kernel | (uintptr_t)grid) & 15) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_static: array arguments must be 16-byte aligned");
    grid_plan call = *plan;                          // the caller's plan keeps its own workspace, if it has one
    call.sample_order = 0;                           // input order: the sort's histogram of the grid would not fit
    const size_t need = grid_plan_workspace_bytes(&call);
    if (need > (size_t)GRID_STATIC_SCRATCH_BYTES)
        return fail(GRID_ERR_UNSUPPORTED, "grid_execute_static: %lld samples need %zu bytes of workspace, the static scratch array "
                    "holds %u (about 1.2 million samples per call): grid the input in several calls, or use grid_execute "
                    "with grid_plan_set_workspace", plan->n_vis, need, (unsigned)GRID_STATIC_SCRATCH_BYTES);
    void* scratch = nullptr;
    const int rc0 = static_scratch_pointer(&scratch);
    if (rc0 != GRID_OK) return rc0;
    call.workspace = scratch;
    call.workspace_bytes = GRID_STATIC_SCRATCH_BYTES;
    // execute_impl clears the head of the workspace (queue counter, hop statistics, chunk-order bins) on `stream`
    // before the first kernel; records, chunk order and tap table are fully rewritten before they are read.
    const int rc = execute_impl(&call, uvw, nullptr, plan->n_vis, vis, weights, conv_kernel, grid, (cudaStream_t)stream);
    plan->last_launches = call.last_launches;
    return rc;
}

int grid_compress(grid_plan* plan, const float* uvw, const float* vis, const float* weights, void* out_records,
                  float* out_vis, long long* out_count, grid_stream_t stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_compress: null plan");
    plan->last_launches = 0;
    plan->order_kept = 0;                            // the records of this call overwrite the workspace
    if (plan->n_vis < 0) return fail(GRID_ERR_STATE, "grid_compress: call grid_plan_set_samples first");
    if (plan->variant != 3) return fail(GRID_ERR_UNSUPPORTED, "grid_compress: power-of-two supports (variant 3) only");
    if (!out_count) return fail(GRID_ERR_INVALID_ARG, "grid_compress: null out_count");
    if (plan->n_vis == 0) {
        if (cudaMemsetAsync(out_count, 0, sizeof(long long), stream) != cudaSuccess)
            return fail(GRID_ERR_CUDA, "grid_compress: %s", cudaGetErrorString(cudaGetLastError()));
        return GRID_OK;
    }
    if (!uvw || !vis || !weights || !out_records || !out_vis)
        return fail(GRID_ERR_INVALID_ARG, "grid_compress: null array argument");
    if (!plan->workspace || plan->workspace_bytes < grid_plan_workspace_bytes(plan))
        return fail(GRID_ERR_STATE, "grid_compress: workspace missing or smaller than grid_plan_workspace_bytes()");
    const long long n = plan->n_vis;
    const long long nb = (n + kCompressBlock - 1) / kCompressBlock;
    if (nb > 0x7fffffffLL) return fail(GRID_ERR_UNSUPPORTED, "grid_compress: too many samples");
    unsigned int* counters = reinterpret_cast<unsigned int*>(plan->workspace);
    unsigned char* rbase = reinterpret_cast<unsigned char*>(plan->workspace) + kHeadBytes;
    CycRec* recs = reinterpret_cast<CycRec*>(rbase);                               // 8 B per sample ...
    uint32_t* block_counts = reinterpret_cast<uint32_t*>(rbase + (size_t)((n + 3) / 4 * 4) * sizeof(CycRec));   // ... the rest of the 16 B
    if (cudaMemsetAsync(counters, 0, kHeadBytes, stream) != cudaSuccess)
        return fail(GRID_ERR_CUDA, "grid_compress: %s", cudaGetErrorString(cudaGetLastError()));
    QuantParams qp = quant_params(plan);
    qp.format = 1;                                   // compact 8-byte records: what compression compares and emits
    quantise_kernel<<<(unsigned)(((n + 3) / 4 + 255) / 256), 256, 0, stream>>>(
        uvw, reinterpret_cast<SampleRec*>(recs), n, qp, reinterpret_cast<float*>(counters + 2), 0, 0, 0.f);
    compress_count_kernel<<<(unsigned)nb, kCompressBlock, 0, stream>>>(recs, n, block_counts);
    compress_scan_kernel<<<1, 1024, 0, stream>>>(block_counts, (int)nb, out_count);
    const float2* v2 = reinterpret_cast<const float2*>(vis);
    CycRec* orec = reinterpret_cast<CycRec*>(out_records);
    float2* ovis = reinterpret_cast<float2*>(out_vis);
    if (plan->P == 1) compress_emit_kernel<1><<<(unsigned)nb, kCompressBlock, 0, stream>>>(recs, v2, weights, n, block_counts, orec, ovis);
    else if (plan->P == 2) compress_emit_kernel<2><<<(unsigned)nb, kCompressBlock, 0, stream>>>(recs, v2, weights, n, block_counts, orec, ovis);
    else compress_emit_kernel<4><<<(unsigned)nb, kCompressBlock, 0, stream>>>(recs, v2, weights, n, block_counts, orec, ovis);
    plan->last_launches = 4;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_compress: launch failed: %s", cudaGetErrorString(e));
    return GRID_OK;
}

int grid_degrid(grid_plan* plan, const float* uvw, const float* weights, const float* conv_kernel,
                const float* grid, float* vis_out, grid_stream_t stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_degrid: null plan");
    plan->last_launches = 0;
    if (plan->n_vis < 0) return fail(GRID_ERR_STATE, "grid_degrid: call grid_plan_set_samples first");
    if (plan->n_vis == 0) return GRID_OK;
    if (!uvw || !weights || !conv_kernel || !grid || !vis_out)
        return fail(GRID_ERR_INVALID_ARG, "grid_degrid: null array argument");
    if ((((uintptr_t)uvw | (uintptr_t)weights | (uintptr_t)conv_kernel | (uintptr_t)grid | (uintptr_t)vis_out) & 15) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_degrid: array arguments must be 16-byte aligned");
    if (!plan->workspace || plan->workspace_bytes < grid_plan_workspace_bytes(plan))
        return fail(GRID_ERR_STATE, "grid_degrid: workspace missing or smaller than grid_plan_workspace_bytes()");
    // the coarsened, register-resident kernel where the plan offers one; the gather kernel otherwise
    if (plan->variant == 3 && plan->degrid_gather == 0) {
        grid_plan tmp = *plan;                       // same plan with polarisation split 1 (shuffle reduction per team)
        tmp.pol_split = 1;
        tmp.threads = 1024;
        const int logs = log2_exact(plan->Sk);
        const int tries[3][2] = {{plan->cu, plan->cv}, {4, 2}, {2, 2}};
        for (int t = 0; t < 3; ++t) {
            tmp.cu = tries[t][0]; tmp.cv = tries[t][1];
            if (derive(&tmp) == GRID_OK && tmp.taps_global == plan->taps_global &&      // same workspace layout
                lookup_degrid(tmp.cu, tmp.cv, tmp.P, logs, tmp.taps_global != 0)) {
                if (degrid_needs_zeroed_output(tmp.cu, tmp.cv, logs) &&
                    cudaMemsetAsync(vis_out, 0, (size_t)plan->n_vis * plan->P * sizeof(float2), stream) != cudaSuccess)
                    return fail(GRID_ERR_CUDA, "grid_degrid: %s", cudaGetErrorString(cudaGetLastError()));
                const int rc = execute_impl(&tmp, uvw, nullptr, plan->n_vis, nullptr, weights, conv_kernel,
                                            const_cast<float*>(grid), stream, vis_out);
                plan->last_launches = tmp.last_launches;
                plan->order_kept = tmp.order_kept;   // gridding and degridding share the kept records
                return rc;
            }
        }
        g_err[0] = 0;                                // no coarsened kernel for this shape: gather below
    }
    const long long n = plan->n_vis;
    plan->order_kept = 0;                            // the gather kernel's records overwrite the workspace
    if (n * 32 / 256 + 1 > 0x7fffffffLL) return fail(GRID_ERR_UNSUPPORTED, "grid_degrid: too many samples");
    unsigned int* counters = reinterpret_cast<unsigned int*>(plan->workspace);
    CycRec* recs = reinterpret_cast<CycRec*>(reinterpret_cast<unsigned char*>(plan->workspace) + kHeadBytes);
    if (cudaMemsetAsync(counters, 0, 256, stream) != cudaSuccess)
        return fail(GRID_ERR_CUDA, "grid_degrid: %s", cudaGetErrorString(cudaGetLastError()));
    QuantParams qp = quant_params(plan);
    qp.format = 1;                                   // compact records (cell, tap rows) for every support
    qp.pad = 0;                                      // this kernel walks the real support
    quantise_kernel<<<(unsigned)(((n + 3) / 4 + 255) / 256), 256, 0, stream>>>(
        uvw, reinterpret_cast<SampleRec*>(recs), n, qp, reinterpret_cast<float*>(counters + 2), 0, 0, 0.f);
    const int L = plan->S <= 8 ? 8 : (plan->S <= 16 ? 16 : 32);
    const float2* k2 = reinterpret_cast<const float2*>(conv_kernel);
    const float2* g2 = reinterpret_cast<const float2*>(grid);
    float2* o2 = reinterpret_cast<float2*>(vis_out);
    if (plan->ev_start) cudaEventRecord(plan->ev_start, stream);
    if (plan->P == 1) launch_degrid<1>(L, n, recs, weights, k2, g2, o2, plan->N, plan->S, stream);
    else if (plan->P == 2) launch_degrid<2>(L, n, recs, weights, k2, g2, o2, plan->N, plan->S, stream);
    else launch_degrid<4>(L, n, recs, weights, k2, g2, o2, plan->N, plan->S, stream);
    if (plan->ev_stop) cudaEventRecord(plan->ev_stop, stream);
    plan->last_launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_degrid: launch failed: %s", cudaGetErrorString(e));
    return GRID_OK;
}

static int execute_dense_impl(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                              const float* conv_kernel_2d, float* grid, grid_stream_t stream_, bool per_pol) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!plan) return fail(GRID_ERR_INVALID_ARG, "grid_execute_dense: null plan");
    plan->last_launches = 0;
    plan->order_kept = 0;                            // the records of this call overwrite the workspace
    if (plan->n_vis < 0) return fail(GRID_ERR_STATE, "grid_execute_dense: call grid_plan_set_samples first");
    if (plan->n_vis == 0) return GRID_OK;
    if (!uvw || !vis || !weights || !conv_kernel_2d || !grid)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_dense: null array argument");
    if ((((uintptr_t)uvw | (uintptr_t)vis | (uintptr_t)weights | (uintptr_t)conv_kernel_2d | (uintptr_t)grid) & 15) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_dense: array arguments must be 16-byte aligned");
    if (!plan->workspace || plan->workspace_bytes < grid_plan_workspace_bytes(plan))
        return fail(GRID_ERR_STATE, "grid_execute_dense: workspace missing or smaller than grid_plan_workspace_bytes()");
    const long long table_elems = (long long)plan->W * plan->O * plan->O * plan->S * plan->S;
    if (table_elems * (per_pol ? plan->P : 1) > 0x7fffffffLL)
        return fail(GRID_ERR_UNSUPPORTED, "grid_execute_dense: table beyond 2^31 elements");
    const int logs = log2_exact(plan->S);
    if (logs >= 2 && logs <= 5) {                    // coarsened kernel with the default block of this (S, P); powers of two only
        grid_plan tmp = *plan;
        tmp.variant = 3; tmp.dense = (per_pol && tmp.P > 1) ? 2 : 1; tmp.pol_split = 1; tmp.threads = 1024; tmp.batch = 32; tmp.chunk = 256;
        if (tmp.P == 1) { tmp.cu = logs == 2 ? 2 : (logs == 5 ? 8 : 4); tmp.cv = logs == 2 ? 2 : 4; }
        else if (tmp.P == 2) { tmp.cu = logs == 2 ? 2 : 4; tmp.cv = 2; }
        else { tmp.cu = logs <= 3 ? 2 : 4; tmp.cv = 2; }
        if (!cell_sort_on(plan)) tmp.sample_order = 0;   // cell order only where the caller's workspace provides for it
        if (derive(&tmp) == GRID_OK) {               // uses a subset of the plan's workspace (no tap table copy)
            const int rc = execute_impl(&tmp, uvw, nullptr, plan->n_vis, vis, weights, conv_kernel_2d, grid, stream);
            plan->last_launches = tmp.last_launches;
            return rc;
        }
        g_err[0] = 0;
    }
    // any other support: one atomic per update
    snprintf(g_err, sizeof(g_err), "note: grid_execute_dense: support %d runs on the one-atomic-per-update kernel "
             "(the coarsened dense kernel covers powers of two up to 32)", plan->S);
    const long long n = plan->n_vis;
    if (n * plan->S / 256 + 1 > 0x7fffffffLL) return fail(GRID_ERR_UNSUPPORTED, "grid_execute_dense: too many samples");
    unsigned int* counters = reinterpret_cast<unsigned int*>(plan->workspace);
    CycRec* recs = reinterpret_cast<CycRec*>(reinterpret_cast<unsigned char*>(plan->workspace) + kHeadBytes);
    if (cudaMemsetAsync(counters, 0, 256, stream) != cudaSuccess)
        return fail(GRID_ERR_CUDA, "grid_execute_dense: %s", cudaGetErrorString(cudaGetLastError()));
    QuantParams qp = quant_params(plan);
    qp.format = 1;
    qp.pad = 0;
    quantise_kernel<<<(unsigned)(((n + 3) / 4 + 255) / 256), 256, 0, stream>>>(
        uvw, reinterpret_cast<SampleRec*>(recs), n, qp, reinterpret_cast<float*>(counters + 2), 0, 0, 0.f);
    const unsigned blocks = (unsigned)((n * plan->S + 255) / 256);
    const float2* v2 = reinterpret_cast<const float2*>(vis);
    const float2* k2 = reinterpret_cast<const float2*>(conv_kernel_2d);
    const long long ps = per_pol ? table_elems : 0;
    if (plan->P == 1) grid_scatter_dense_kernel<1><<<blocks, 256, 0, stream>>>(recs, v2, weights, k2, grid, n, plan->N, plan->S, plan->O, ps);
    else if (plan->P == 2) grid_scatter_dense_kernel<2><<<blocks, 256, 0, stream>>>(recs, v2, weights, k2, grid, n, plan->N, plan->S, plan->O, ps);
    else grid_scatter_dense_kernel<4><<<blocks, 256, 0, stream>>>(recs, v2, weights, k2, grid, n, plan->N, plan->S, plan->O, ps);
    plan->last_launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GRID_ERR_CUDA, "grid_execute_dense: launch failed: %s", cudaGetErrorString(e));
    return GRID_OK;
}

int grid_execute_dense(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                       const float* conv_kernel_2d, float* grid, grid_stream_t stream) {
    return execute_dense_impl(plan, uvw, vis, weights, conv_kernel_2d, grid, stream, false);
}

int grid_execute_dense_pol(grid_plan* plan, const float* uvw, const float* vis, const float* weights,
                           const float* conv_kernel_2d_pol, float* grid, grid_stream_t stream) {
    return execute_dense_impl(plan, uvw, vis, weights, conv_kernel_2d_pol, grid, stream, true);
}

int grid_execute_compressed(grid_plan* plan, const void* records, const float* vis, long long n,
                            const float* conv_kernel, float* grid, grid_stream_t stream) {
    if (!plan || n < 0) return fail(GRID_ERR_INVALID_ARG, "grid_execute_compressed: invalid argument");
    plan->last_launches = 0;
    if (plan->variant != 3) return fail(GRID_ERR_UNSUPPORTED, "grid_execute_compressed: power-of-two supports (variant 3) only");
    if (plan->n_vis < 0 || n > plan->n_vis)
        return fail(GRID_ERR_STATE, "grid_execute_compressed: set_samples must cover the uncompressed count (workspace size)");
    if (n == 0) return GRID_OK;
    if (!records || !vis || !conv_kernel || !grid)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_compressed: null array argument");
    if ((((uintptr_t)records | (uintptr_t)vis | (uintptr_t)conv_kernel | (uintptr_t)grid) & 15) != 0)
        return fail(GRID_ERR_INVALID_ARG, "grid_execute_compressed: array arguments must be 16-byte aligned");
    if (!plan->workspace || plan->workspace_bytes < grid_plan_workspace_bytes(plan))
        return fail(GRID_ERR_STATE, "grid_execute_compressed: workspace missing or too small");
    return execute_impl(plan, nullptr, records, n, vis, nullptr, conv_kernel, grid, (cudaStream_t)stream);
}

}  // extern "C"
