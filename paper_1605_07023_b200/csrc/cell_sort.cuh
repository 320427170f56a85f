// Step a1, cell order: the samples leave the quantise pass SORTED BY GRID CELL.
//
// Register accumulation pays when consecutive samples of a chunk keep their footprint on the same grid points
// ("the coordinates and ordering of the data"; flush only when the owned cell changes).
// The paper's single-channel 2-s data moved a fraction of a cell per sample; BASELINE.json's multi-channel arrays
// move 0.7-3 cells per sample in any walk of one baseline, and the flush (atomics issued at 4-5 of 32 lanes) then
// costs as much as the multiply-adds.  The sum is order-independent (pin P11), so the a1 pass
// may hand the gridding kernel ANY permutation: ordered by the cell of the footprint origin (row-major), 83-94 % of
// consecutive samples of BASELINE.json's configs share their cell and most of the rest move by one column.
//
// It is a counting sort on the cell index, affordable because the per-cell histogram of a 2048^2...8192^2 grid
// (16-268 MB) lives in or near the 126 MB L2:
//   cell_count_kernel    quantise; rank[n] = atomicAdd(hist[cell(n)], 1)             (12 B in, 4 B out per sample)
//   cell_scan_*          exclusive prefix sum of hist in place (three small kernels)
//   cell_scatter_kernel  quantise again (cheaper than storing and re-reading records) and write the 16-byte record
//                        to slot hist[cell] + rank: {origin, tap rows, weight, sample index} -- the gridding
//                        kernel fetches the visibilities through the index -- or, for one polarisation, {origin, tap
//                        rows, weight * vis}: the whole pre-weighted sample, nothing left to gather.
// Skipped samples (R7) get the key N*N and end up behind all others, still flagged.
#pragma once
#include "quantise.cuh"

namespace gridb200 {

// A sorted record occupies a whole 32-byte sector (16 bytes used): the scatter's writes land at random places of an
// array several times the L2, and a half-written sector costs the DRAM a read-modify-write (measured: the sort of
// cfg1 1.15 -> 0.91 ms, cfg2 1.70 -> 1.27, cfg3 3.34 -> 2.70 with full sectors; the gridding kernel reads them in
// order and does not notice).
static constexpr int kCellRecStride = 2;               // in 16-byte units

static constexpr int kScanPerThread = 16;
static constexpr int kScanTile = 256 * kScanPerThread;        // histogram entries per block of the scan kernels

__device__ __forceinline__ void load_uvw4(const float* __restrict__ uvw, long long first, long long n, float (&c)[12]) {
    if (first + 4 <= n) {
        const float4* p = reinterpret_cast<const float4*>(uvw + first * 3);
        const float4 a = __ldcs(p), b = __ldcs(p + 1), d = __ldcs(p + 2);       // streamed once: do not displace the histogram
        c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w; c[4] = b.x; c[5] = b.y; c[6] = b.z;
        c[7] = b.w; c[8] = d.x; c[9] = d.y; c[10] = d.z; c[11] = d.w;
    } else {
#pragma unroll
        for (int k = 0; k < 12; ++k) c[k] = (first * 3 + k < n * 3) ? __ldg(uvw + first * 3 + k) : 0.f;
    }
}

// key of a quantised sample: cell of the (padded) footprint origin, row-major; nn = N*N for skipped samples
__device__ __forceinline__ uint32_t cell_key(const CycRec& r, uint32_t N, uint32_t nn) {
    return (r.pos & 0x8000u) ? nn : (r.pos >> 16) * N + (r.pos & 0x7fffu);
}

__global__ void __launch_bounds__(256)
cell_count_kernel(const float* __restrict__ uvw, long long n, QuantParams qp, uint32_t* __restrict__ hist,
                  uint32_t* __restrict__ ranks) {
    const long long first = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    const uint32_t N = (uint32_t)qp.grid_size, nn = N * N;
    const uint32_t lane = threadIdx.x & 31u;
    float c[12];
    load_uvw4(uvw, first, n, c);
    uint32_t rk[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const bool have = first + k < n;
        uint32_t key = 0xffffffffu;                    // no sample: a group of its own, nothing counted
        if (have) key = cell_key(make_cyc_record(quantise_sample(c[3 * k], c[3 * k + 1], c[3 * k + 2], qp), qp), N, nn);
        // One atomic per warp and distinct cell: the lanes that hit the same cell (neighbouring channels of a short
        // baseline; all the skipped samples, which share the bin nn) take consecutive ranks from one atomicAdd.  An
        // input concentrated on few cells would otherwise serialise on their counters.
        const uint32_t peers = __match_any_sync(0xffffffffu, key);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (have && (int)lane == leader) base = atomicAdd(hist + key, (uint32_t)__popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        rk[k] = base + (uint32_t)__popc(peers & ((1u << lane) - 1u));
    }
    if (first + 4 <= n) __stcs(reinterpret_cast<uint4*>(ranks + first), make_uint4(rk[0], rk[1], rk[2], rk[3]));
    else {
#pragma unroll
        for (int k = 0; k < 4; ++k) if (first + k < n) ranks[first + k] = rk[k];
    }
}

// Exclusive prefix sum of hist[0 .. m), m a multiple of kScanTile (the tail is zero-filled), in place.
__device__ __forceinline__ uint32_t scan_load16(const uint32_t* p, uint32_t (&v)[kScanPerThread]) {
    uint32_t s = 0;
#pragma unroll
    for (int q = 0; q < kScanPerThread / 4; ++q) {
        const uint4 a = reinterpret_cast<const uint4*>(p)[q];
        v[4 * q] = a.x; v[4 * q + 1] = a.y; v[4 * q + 2] = a.z; v[4 * q + 3] = a.w;
        s += a.x + a.y + a.z + a.w;
    }
    return s;
}

__global__ void __launch_bounds__(256) cell_scan_reduce_kernel(const uint32_t* __restrict__ hist, uint32_t* __restrict__ sums) {
    __shared__ uint32_t ws[8];
    uint32_t v[kScanPerThread];
    uint32_t s = scan_load16(hist + (size_t)blockIdx.x * kScanTile + threadIdx.x * kScanPerThread, v);
    s = __reduce_add_sync(0xffffffffu, s);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) sums[blockIdx.x] = ws[0] + ws[1] + ws[2] + ws[3] + ws[4] + ws[5] + ws[6] + ws[7];
}

// exclusive scan of the block sums, one block of 1024 threads, carried over slabs of 1024; sums[nb] = the total
__global__ void __launch_bounds__(1024) cell_scan_sums_kernel(uint32_t* __restrict__ sums, int nb) {
    __shared__ uint32_t ws[32];
    __shared__ uint32_t carry;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    if (t == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const uint32_t mine = base + t < nb ? sums[base + t] : 0u;
        uint32_t x = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) ws[w] = x;
        __syncthreads();
        if (w == 0) {
            uint32_t z = ws[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, z, o); if (lane >= o) z += y; }
            ws[lane] = z;
        }
        __syncthreads();
        const uint32_t incl = x + (w ? ws[w - 1] : 0u) + carry;
        if (base + t < nb) sums[base + t] = incl - mine;
        __syncthreads();
        if (t == 1023) carry = incl;
        __syncthreads();
    }
    if (t == 0) sums[nb] = carry;
}

__global__ void __launch_bounds__(256) cell_scan_apply_kernel(uint32_t* __restrict__ hist, const uint32_t* __restrict__ sums) {
    __shared__ uint32_t ws[8];
    // a tile without samples: nobody will ask for its offsets (on a large, sparsely covered grid most tiles are empty)
    if (__ldg(sums + blockIdx.x + 1) == __ldg(sums + blockIdx.x)) return;
    uint32_t v[kScanPerThread];
    uint32_t* p = hist + (size_t)blockIdx.x * kScanTile + threadIdx.x * kScanPerThread;
    const uint32_t mine = scan_load16(p, v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t x = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) ws[w] = x;
    __syncthreads();
    uint32_t run = __ldg(sums + blockIdx.x) + x - mine;
#pragma unroll
    for (int q = 0; q < 7; ++q) if (q < w) run += ws[q];
#pragma unroll
    for (int q = 0; q < kScanPerThread / 4; ++q) {
        uint4 o;
        o.x = run; run += v[4 * q];
        o.y = run; run += v[4 * q + 1];
        o.z = run; run += v[4 * q + 2];
        o.w = run; run += v[4 * q + 3];
        reinterpret_cast<uint4*>(p)[q] = o;
    }
}

// P1: one polarisation -- the record carries the pre-weighted visibility instead of {weight, index}.
template <bool P1>
__global__ void __launch_bounds__(256)
cell_scatter_kernel(const float* __restrict__ uvw, const float* __restrict__ weights, const float2* __restrict__ vis,
                    long long n, QuantParams qp, const uint32_t* __restrict__ offsets, const uint32_t* __restrict__ ranks,
                    uint4* __restrict__ out) {
    const long long first = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (first >= n) return;
    const uint32_t N = (uint32_t)qp.grid_size, nn = N * N;
    float c[12];
    load_uvw4(uvw, first, n, c);
    float w[4] = {1.f, 1.f, 1.f, 1.f};
    uint32_t rk[4] = {0u, 0u, 0u, 0u};
    float2 v[4];
    if (first + 4 <= n) {
        const float4 w4 = __ldcs(reinterpret_cast<const float4*>(weights + first));
        w[0] = w4.x; w[1] = w4.y; w[2] = w4.z; w[3] = w4.w;
        const uint4 r4 = __ldcs(reinterpret_cast<const uint4*>(ranks + first));
        rk[0] = r4.x; rk[1] = r4.y; rk[2] = r4.z; rk[3] = r4.w;
        if constexpr (P1) {
            const float4 a = __ldcs(reinterpret_cast<const float4*>(vis + first)), b = __ldcs(reinterpret_cast<const float4*>(vis + first) + 1);
            v[0] = make_float2(a.x, a.y); v[1] = make_float2(a.z, a.w); v[2] = make_float2(b.x, b.y); v[3] = make_float2(b.z, b.w);
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (first + k < n) {
                w[k] = __ldg(weights + first + k);
                rk[k] = __ldg(ranks + first + k);
                if constexpr (P1) v[k] = __ldg(vis + first + k);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (first + k < n) {
            const CycRec r = make_cyc_record(quantise_sample(c[3 * k], c[3 * k + 1], c[3 * k + 2], qp), qp);
            const uint32_t at = __ldg(offsets + cell_key(r, N, nn)) + rk[k];
            uint4* dst = out + (size_t)at * kCellRecStride;
            // streaming stores: the records are read again only by the gridding kernel, the offsets by every sample
            if constexpr (P1) __stcs(dst, make_uint4(r.pos, r.rows, __float_as_uint(v[k].x * w[k]), __float_as_uint(v[k].y * w[k])));
            else __stcs(dst, make_uint4(r.pos, r.rows, __float_as_uint(w[k]), (uint32_t)(first + k)));
            __stcs(dst + 1, make_uint4(0u, 0u, 0u, 0u));   // completes the sector: no read-modify-write in DRAM
        }
    }
}

}  // namespace gridb200
