// Step a9, locality: the order in which chunks enter the queue.
//
// The paper hands out fixed-size chunks of baseline-ordered samples; which chunk a
// work-group takes next does not change the result.  On B200 the atomic flushes of a grid that does
// not fit the 126 MB L2 cost DRAM sector fetches (round 1, before this ordering existed: 35 GB of DRAM traffic
// per launch for cfg3's 2.1 GB grid; with it 8-12 GB, profiles/r2_ncu_full_cfg3.txt), because the ~7000 chunks in
// flight lie all over the uv plane.
// These three small kernels sort the chunk ids by the coarse grid tile of the chunk's first sample
// (counting sort: histogram, scan, scatter), so that chunks in flight together touch a few
// neighbouring tiles.  Inputs are the quantised records written by the a1 pass.
#pragma once
#include "gridder_common.cuh"

namespace gridb200 {

static constexpr int kOrderBins = 1024;          // 32 x 32 tiles

// The traversal mode the gridding kernel will use (same rule, same inputs: decided on the device from
// the hop statistics of the quantise pass).
__device__ __forceinline__ int pick_mode(const GridParams& gp) {
    int mode = gp.force_mode;
    if (mode < 0) {
        mode = 0;
        if (gp.n_chan > 1) {                    // one channel: input order already is time-innermost
            const float hc = __ldg(gp.hop_stats), ht = __ldg(gp.hop_stats + 1);
            const float cost0 = ((gp.n_chan - 1) * hc + ht) / gp.n_chan;     // mean hop per sample
            const float cost1 = ((gp.tc - 1) * ht + hc) / gp.tc;
            mode = cost1 < cost0 ? 1 : 0;
        }
    }
    return mode;
}

__device__ __forceinline__ long long chunk_count(const GridParams& gp, int mode) {
    return mode ? gp.n_chunks_b : (gp.n_vis + gp.chunk - 1) / gp.chunk;
}

// First sample of chunk c (input order; the serpentine mirror does not matter for a tile key).
__device__ __forceinline__ long long chunk_first_sample(const GridParams& gp, int mode, long long c) {
    if (mode == 0) return c * gp.chunk;
    const long long per_bl = (long long)gp.n_tblocks * gp.n_cblocks;
    const long long bl = c / per_bl;
    const int rem = (int)(c - bl * per_bl);
    const int tb = rem / gp.n_cblocks, cc = rem - tb * gp.n_cblocks;
    return (bl * gp.n_times + (long long)tb * gp.tc) * gp.n_chan + (long long)cc * gp.chunk_cols;
}

__device__ __forceinline__ uint32_t chunk_tile(const GridParams& gp, int mode, long long c) {
    // records are 8 bytes (CycRec) or, with the weight attached, 16: the origin is the first word either way
    const uint32_t* words = reinterpret_cast<const uint32_t*>(gp.recs);
    const uint32_t pos = __ldg(words + (size_t)chunk_first_sample(gp, mode, c) * (gp.rec16 ? 4 : 2));
    const uint32_t tx = (pos & 0x7fffu) >> gp.tile_shift, ty = (pos >> 16) >> gp.tile_shift;
    return ty * 32u + ((ty & 1u) ? 31u - tx : tx);            // boustrophedon over tile rows
}

// bins: [0, kOrderBins) counts -> offsets, [kOrderBins, 2*kOrderBins) scatter cursors (zeroed by the host)
__global__ void __launch_bounds__(256) chunk_histogram_kernel(const GridParams gp, uint32_t* bins) {
    const int mode = pick_mode(gp);
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= chunk_count(gp, mode)) return;
    atomicAdd(&bins[chunk_tile(gp, mode, c)], 1u);
}

__global__ void __launch_bounds__(kOrderBins) chunk_scan_kernel(uint32_t* bins) {
    __shared__ uint32_t s[kOrderBins];
    const int t = threadIdx.x;
    const uint32_t mine = bins[t];
    s[t] = mine;
    __syncthreads();
    for (int o = 1; o < kOrderBins; o <<= 1) {
        const uint32_t v = t >= o ? s[t - o] : 0u;
        __syncthreads();
        s[t] += v;
        __syncthreads();
    }
    bins[t] = s[t] - mine;                                   // exclusive prefix
}

__global__ void __launch_bounds__(256) chunk_scatter_kernel(const GridParams gp, uint32_t* bins, uint32_t* order) {
    const int mode = pick_mode(gp);
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= chunk_count(gp, mode)) return;
    const uint32_t tile = chunk_tile(gp, mode, c);
    const uint32_t at = bins[tile] + atomicAdd(&bins[kOrderBins + tile], 1u);
    order[at] = (uint32_t)c;
}

}  // namespace gridb200
