// Steps a2-a9: the gridding kernel.  Romein's work distribution (Fig. 1) with the
// paper's thread coarsening (Fig. 2): a *team* of (Bu/Cu)*(Bv/Cv) threads covers one
// bin; each thread owns the Cu x Cv block of grid points with a fixed position modulo the bin, keeps
// their sums in registers while consecutive samples overlap, and flushes them with vector atomic adds
// when its block moves.  The bounding box is aligned to blocks, the tap rows
// are zero-padded, the GCF is rebuilt from separable taps in registers
// (PAPER.md:97-99), samples arrive in fixed-size chunks staged through shared memory
// (PAPER.md:91, 103).  New here: several teams per CTA (bins of small supports need < 32 threads),
// persistent CTAs pulling chunk groups from a queue, non-power-of-two bins.
#pragma once
#include "gridder_common.cuh"

namespace gridb200 {

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
    asm volatile("red.relaxed.gpu.global.add.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void red_add_v2(float* addr, float a, float b) {
    asm volatile("red.relaxed.gpu.global.add.v2.f32 [%0], {%1, %2};"
                 :: "l"(addr), "f"(a), "f"(b) : "memory");
}

__device__ __forceinline__ bool any_nonzero(const float2* v, int n) {
    uint32_t bits = 0;
    for (int k = 0; k < n; ++k) bits |= __float_as_uint(v[k].x) | __float_as_uint(v[k].y);
    return (bits << 1) != 0;          // ignores the sign of zero
}

// a8: add the thread's block to the grid and clear it.  `cell` = x | y << 16 of the block's first
// grid point.  Cells of the padded box that fall outside the grid only ever hold zeros (or garbage
// from 0*Inf); they are dropped by the bounds test.
template <int CU, int CV, int P>
__device__ __forceinline__ void flush_block(float2 (&acc)[CV][CU][P], uint32_t cell, float* grid, int N) {
    const int x = (int)(cell & 0xffffu), y = (int)(cell >> 16);
#pragma unroll
    for (int r = 0; r < CV; ++r) {
        if (y + r >= N) continue;
        float* row = grid + ((size_t)(y + r) * N + x) * (2 * P);
        if constexpr (P == 1 && (CU % 2) == 0) {
#pragma unroll
            for (int c = 0; c < CU; c += 2) {
                // x is a multiple of CU, N*P*8 keeps rows 16-byte aligned when N is even
                if (x + c + 1 < N && ((N & 1) == 0)) {
                    if (any_nonzero(&acc[r][c][0], 2))
                        red_add_v4(row + 2 * c, acc[r][c][0].x, acc[r][c][0].y, acc[r][c + 1][0].x,
                                   acc[r][c + 1][0].y);
                } else {
                    if (x + c < N && any_nonzero(&acc[r][c][0], 1))
                        red_add_v2(row + 2 * c, acc[r][c][0].x, acc[r][c][0].y);
                    if (x + c + 1 < N && any_nonzero(&acc[r][c + 1][0], 1))
                        red_add_v2(row + 2 * (c + 1), acc[r][c + 1][0].x, acc[r][c + 1][0].y);
                }
                acc[r][c][0] = make_float2(0.f, 0.f);
                acc[r][c + 1][0] = make_float2(0.f, 0.f);
            }
        } else {
#pragma unroll
            for (int c = 0; c < CU; ++c) {
                if (x + c < N && any_nonzero(&acc[r][c][0], P)) {
                    float* p = row + 2 * P * c;
                    if constexpr (P % 2 == 0) {
#pragma unroll
                        for (int q = 0; q < P; q += 2)
                            red_add_v4(p + 2 * q, acc[r][c][q].x, acc[r][c][q].y, acc[r][c][q + 1].x,
                                       acc[r][c][q + 1].y);
                    } else {
#pragma unroll
                        for (int q = 0; q < P; ++q) red_add_v2(p + 2 * q, acc[r][c][q].x, acc[r][c][q].y);
                    }
                }
#pragma unroll
                for (int q = 0; q < P; ++q) acc[r][c][q] = make_float2(0.f, 0.f);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < CV; ++r)
#pragma unroll
        for (int c = 0; c < CU; ++c)
#pragma unroll
            for (int q = 0; q < P; ++q) acc[r][c][q] = make_float2(0.f, 0.f);
}

// Shared memory: [u taps: n_rows*Lu float2][v taps: n_rows*Lv float2 (only if Cu != Cv)]
//                [records: teams*batch uint4][pre-weighted vis: teams*batch*P float2][queue slot]
template <int CU, int CV, int P>
__global__ void __launch_bounds__(512, 1)
grid_coarsened_kernel(const GridParams gp) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* taps_u = reinterpret_cast<float2*>(smem_raw);
    float2* taps_v = (CU == CV) ? taps_u : taps_u + (size_t)gp.n_rows * gp.row_u;
    size_t off = (size_t)gp.n_rows * gp.row_u * sizeof(float2);
    if (CU != CV) off += (size_t)gp.n_rows * gp.row_v * sizeof(float2);
    off = (off + 15) & ~(size_t)15;
    SampleRec* srec = reinterpret_cast<SampleRec*>(smem_raw + off);
    float2* svis = reinterpret_cast<float2*>(smem_raw + off + (size_t)gp.teams_per_cta * gp.batch * sizeof(SampleRec));
    __shared__ unsigned int s_group;

    const int tid = threadIdx.x;
    // a4: zero-padded separable tap rows: Cu-1 zeros, S taps, zeros up to Lu
    for (int k = tid; k < gp.n_rows * gp.row_u; k += blockDim.x) {
        const int r = k / gp.row_u, t = k - r * gp.row_u - (CU - 1);
        taps_u[k] = (t >= 0 && t < gp.S) ? __ldg(gp.kern + (size_t)r * gp.S + t) : make_float2(0.f, 0.f);
    }
    if (CU != CV) {
        for (int k = tid; k < gp.n_rows * gp.row_v; k += blockDim.x) {
            const int r = k / gp.row_v, t = k - r * gp.row_v - (CV - 1);
            taps_v[k] = (t >= 0 && t < gp.S) ? __ldg(gp.kern + (size_t)r * gp.S + t) : make_float2(0.f, 0.f);
        }
    }

    // a5: ownership.  team = bin instance, (bx, by) = block position inside the bin.
    const int team = tid / gp.team_threads;
    const int lt = tid - team * gp.team_threads;
    const bool active = team < gp.teams_per_cta;
    const int by = lt / gp.nbx;
    const int bxc = (lt - by * gp.nbx) * CU, byc = by * CV;
    const SampleRec* my_rec = srec + (size_t)team * gp.batch;
    const float2* my_vis = svis + (size_t)team * gp.batch * P;

    float2 acc[CV][CU][P];
#pragma unroll
    for (int r = 0; r < CV; ++r)
#pragma unroll
        for (int c = 0; c < CU; ++c)
#pragma unroll
            for (int q = 0; q < P; ++q) acc[r][c][q] = make_float2(0.f, 0.f);

    // Traversal order inside a chunk (the sum is order-independent, pin P11):
    //   mode 0: input order (channel innermost), odd time rows mirrored when the layout is known;
    //   mode 1: a chunk is Tc time steps x all channels of one baseline, walked time-innermost,
    //           serpentine.  Picked per call from the mean hop measured by the quantise pass.
    int mode = gp.force_mode;
    if (mode < 0) {
        mode = 0;
        if (gp.n_chan > 0) {
            const float hc = __ldg(gp.hop_stats), ht = __ldg(gp.hop_stats + 1);
            const float cost0 = ((gp.n_chan - 1) * hc + ht) / gp.n_chan;     // mean hop per sample
            const float cost1 = ((gp.tc - 1) * ht + hc) / gp.tc;
            mode = cost1 < cost0 ? 1 : 0;
        }
    }
    const long long n_groups = mode ? gp.n_groups_b : gp.n_groups_a;
    const int n_batches = mode ? (gp.n_chan + (1 << gp.cb_shift) - 1) >> gp.cb_shift
                               : (gp.chunk + gp.batch - 1) / gp.batch;
    const int stage_total = gp.teams_per_cta * gp.batch;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_group = atomicAdd(gp.counters, 1u);          // a9: chunk-group queue
        __syncthreads();
        const long long group = s_group;
        if (group >= n_groups) break;
        uint32_t cur = kInvalidRec;                                  // block currently in registers

        for (int b = 0; b < n_batches; ++b) {
            __syncthreads();
            // a2 + a3: stage one batch per team, pre-weighting the visibilities
            for (int kk = tid; kk < stage_total; kk += blockDim.x) {
                const int t = kk >> gp.batch_shift, s = kk & (gp.batch - 1);
                const long long chunk_id = group * gp.teams_per_cta + t;
                long long g = -1;
                int k = kk;                                          // shared-memory slot = traversal position
                if (mode == 0) {
                    const int in_chunk = b * gp.batch + s;
                    long long a = chunk_id * gp.chunk + in_chunk;
                    if (in_chunk < gp.chunk && a < gp.n_vis) {
                        if (gp.n_chan > 0) {                         // mirror odd time rows (serpentine)
                            const long long row = a / gp.n_chan;
                            const int col = (int)(a - row * gp.n_chan);
                            if (row & 1) a = row * gp.n_chan + (gp.n_chan - 1 - col);
                        }
                        g = a;
                    }
                } else if (chunk_id < gp.n_chunks_b) {
                    // thread s -> (time ti, channel ci): consecutive threads read consecutive channels
                    const int ti = s >> gp.cb_shift, ci = s & ((1 << gp.cb_shift) - 1);
                    const int col = (b << gp.cb_shift) + ci;
                    const long long bl = chunk_id / gp.n_tblocks;
                    const int tb = (int)(chunk_id - bl * gp.n_tblocks);
                    const int tabs = tb * gp.tc + ti;
                    const int tt = (col & 1) ? gp.tc - 1 - ti : ti;
                    k = (t << gp.batch_shift) + ci * gp.tc + tt;
                    if (col < gp.n_chan && tabs < gp.n_times)
                        g = (bl * gp.n_times + tabs) * (long long)gp.n_chan + col;
                }
                SampleRec rec;
                rec.x = kInvalidRec; rec.y = rec.z = rec.w = 0;
                if (g >= 0) rec = __ldg(gp.recs + g);
                srec[k] = rec;
                if (rec.x != kInvalidRec) {
                    const float w = __ldg(gp.weights + g);
                    if constexpr (P % 2 == 0) {
                        const float4* src = reinterpret_cast<const float4*>(gp.vis + g * P);
                        float4* dst = reinterpret_cast<float4*>(svis + (size_t)k * P);
#pragma unroll
                        for (int q = 0; q < P / 2; ++q) {
                            float4 v = __ldg(src + q);
                            v.x *= w; v.y *= w; v.z *= w; v.w *= w;
                            dst[q] = v;
                        }
                    } else {
#pragma unroll
                        for (int q = 0; q < P; ++q) {
                            float2 v = __ldg(gp.vis + g * P + q);
                            v.x *= w; v.y *= w;
                            svis[(size_t)k * P + q] = v;
                        }
                    }
                }
            }
            __syncthreads();
            if (!active) continue;

            // hot loop over the staged samples of this team's chunk
            for (int s = 0; s < gp.batch; ++s) {
                const SampleRec rec = my_rec[s];
                if (rec.x == kInvalidRec) continue;
                int relx = bxc - (int)(rec.y & 0xffffu);
                int rely = byc - (int)(rec.y >> 16);
                if (relx < 0) relx += gp.bin_u;
                if (rely < 0) rely += gp.bin_v;
                // first grid point of my block inside the aligned bounding box (never wraps)
                const uint32_t cell = rec.x + (uint32_t)relx + ((uint32_t)rely << 16);
                if (cell != cur) {                                   // a8: my block moved
                    if (cur != kInvalidRec) flush_block<CU, CV, P>(acc, cur, gp.grid, gp.N);
                    cur = cell;
                }
                const float2* tu = taps_u + rec.z + relx;
                const float2* tv = taps_v + rec.w + rely;
                float2 gu[CU], gv[CV], v[P];
#pragma unroll
                for (int c = 0; c < CU; ++c) gu[c] = tu[c];
#pragma unroll
                for (int r = 0; r < CV; ++r) gv[r] = tv[r];
#pragma unroll
                for (int q = 0; q < P; ++q) v[q] = my_vis[s * P + q];
#pragma unroll
                for (int r = 0; r < CV; ++r) {
#pragma unroll
                    for (int c = 0; c < CU; ++c) {
                        // a6: G_ij = Gv_j * Gu_i
                        const float gr = gv[r].x * gu[c].x - gv[r].y * gu[c].y;
                        const float gi = gv[r].x * gu[c].y + gv[r].y * gu[c].x;
#pragma unroll
                        for (int q = 0; q < P; ++q) {                // a7: 4 FFMA = 8 flops per update
                            acc[r][c][q].x = fmaf(gr, v[q].x, acc[r][c][q].x);
                            acc[r][c][q].x = fmaf(-gi, v[q].y, acc[r][c][q].x);
                            acc[r][c][q].y = fmaf(gr, v[q].y, acc[r][c][q].y);
                            acc[r][c][q].y = fmaf(gi, v[q].x, acc[r][c][q].y);
                        }
                    }
                }
            }
        }
        if (active && cur != kInvalidRec) flush_block<CU, CV, P>(acc, cur, gp.grid, gp.N);
    }
}

// Diagnostic baseline (variant 0): one thread per (sample, tap row), one atomic per cell and
// polarisation pair -- the "naive implementation" of PAPER.md:53.  Uses records made with Cu=Cv=1.
template <int P>
__global__ void __launch_bounds__(256)
grid_scatter_kernel(const GridParams gp) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = g / gp.S;
    const int tj = (int)(g - n * gp.S);
    if (n >= gp.n_vis) return;
    const SampleRec rec = __ldg(gp.recs + n);
    if (rec.x == kInvalidRec) return;
    const int i0 = (int)(rec.x & 0xffffu), j0 = (int)(rec.x >> 16);
    const float w = __ldg(gp.weights + n);
    float2 v[P];
#pragma unroll
    for (int q = 0; q < P; ++q) {
        v[q] = __ldg(gp.vis + n * P + q);
        v[q].x *= w; v[q].y *= w;
    }
    const float2 kv = __ldg(gp.kern + rec.w + tj);
    float* row = gp.grid + ((size_t)(j0 + tj) * gp.N + i0) * (2 * P);
    for (int ti = 0; ti < gp.S; ++ti) {
        const float2 ku = __ldg(gp.kern + rec.z + ti);
        const float gr = kv.x * ku.x - kv.y * ku.y, gi = kv.x * ku.y + kv.y * ku.x;
#pragma unroll
        for (int q = 0; q < P; ++q) {
            const float re = gr * v[q].x - gi * v[q].y, im = gr * v[q].y + gi * v[q].x;
            red_add_v2(row + (size_t)(ti * P + q) * 2, re, im);
        }
    }
}

}  // namespace gridb200
