// The step before the path: compression.
//
// "Adjacent visibilities with identical oversampled position" (and w-plane) are merged into one
// pre-weighted sample before gridding; the paper does this offline and reports its rates per compressed
// sample.  Here it is a device pass over the quantised records of the a1 pass:
//   head(n)  = valid(n) and (n == 0 or not valid(n-1) or record(n) != record(n-1))
//   out[k]   = record of the k-th head, vis = sum over its run of weight * vis   (FP32, input order)
// Samples that a1 marks as skipped (R7) produce no output.  Three launches: heads per 1024-sample
// block, exclusive scan of the block counts, emit.
#pragma once
#include "gridder_common.cuh"

namespace gridb200 {

static constexpr int kCompressBlock = 1024;

__device__ __forceinline__ bool compress_is_head(const CycRec* recs, long long n) {
    const CycRec r = recs[n];
    if (r.pos & 0x8000u) return false;                       // skipped sample
    if (n == 0) return true;
    const CycRec p = recs[n - 1];
    return (p.pos & 0x8000u) != 0 || p.pos != r.pos || p.rows != r.rows;
}

__global__ void __launch_bounds__(kCompressBlock)
compress_count_kernel(const CycRec* __restrict__ recs, long long n, uint32_t* __restrict__ block_counts) {
    const long long i = (long long)blockIdx.x * kCompressBlock + threadIdx.x;
    const int head = (i < n && compress_is_head(recs, i)) ? 1 : 0;
    const int c = __syncthreads_count(head);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = (uint32_t)c;
}

// exclusive scan of block_counts[nb] in place (one CTA), total -> *out_count
__global__ void __launch_bounds__(1024)
compress_scan_kernel(uint32_t* block_counts, int nb, long long* out_count) {
    __shared__ uint32_t s[1024];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + threadIdx.x;
        const uint32_t mine = i < nb ? block_counts[i] : 0u;
        s[threadIdx.x] = mine;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const uint32_t v = threadIdx.x >= o ? s[threadIdx.x - o] : 0u;
            __syncthreads();
            s[threadIdx.x] += v;
            __syncthreads();
        }
        if (i < nb) block_counts[i] = carry + s[threadIdx.x] - mine;
        __syncthreads();
        if (threadIdx.x == 1023) carry += s[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out_count = (long long)carry;
}

template <int P>
__global__ void __launch_bounds__(kCompressBlock)
compress_emit_kernel(const CycRec* __restrict__ recs, const float2* __restrict__ vis, const float* __restrict__ weights,
                     long long n, const uint32_t* __restrict__ block_offsets, CycRec* __restrict__ out_recs,
                     float2* __restrict__ out_vis) {
    __shared__ uint32_t warp_counts[kCompressBlock / 32];
    const long long i = (long long)blockIdx.x * kCompressBlock + threadIdx.x;
    const bool head = i < n && compress_is_head(recs, i);
    const uint32_t ballot = __ballot_sync(0xffffffffu, head);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) warp_counts[warp] = __popc(ballot);
    __syncthreads();
    uint32_t before = 0;
    for (int w = 0; w < warp; ++w) before += warp_counts[w];
    if (!head) return;
    const long long k = (long long)block_offsets[blockIdx.x] + before + __popc(ballot & ((1u << lane) - 1u));
    const CycRec r = recs[i];
    float2 acc[P];
#pragma unroll
    for (int q = 0; q < P; ++q) acc[q] = make_float2(0.f, 0.f);
    long long m = i;
    do {                                                     // the run: following samples with the same record
        const float w = weights[m];
#pragma unroll
        for (int q = 0; q < P; ++q) {
            const float2 v = vis[m * P + q];
            acc[q].x = fmaf(w, v.x, acc[q].x);
            acc[q].y = fmaf(w, v.y, acc[q].y);
        }
        ++m;
    } while (m < n && recs[m].pos == r.pos && recs[m].rows == r.rows);
    out_recs[k] = r;
#pragma unroll
    for (int q = 0; q < P; ++q) out_vis[k * P + q] = acc[q];
}

}  // namespace gridb200
