// Steps a2-a9, power-of-two supports: the gridding kernel with bin == support ("each thread owns a
// coarsened C x C block of grid positions taken modulo the support", BASELINE.json:north_star).
//
// Romein's ownership: a thread is responsible for all grid points with a fixed position
// modulo the bin and keeps the one inside the current footprint in a register accumulator.  Thread
// coarsening: each thread owns Cu x Cv positions.  Differences from the paper's
// layout, made because its aligned, zero-padded bounding box wastes 36-56 % of the
// FMAs at supports 8-16 (the paper's own caveat for small GCFs):
//   * bin = S exactly, no padding: the Cu (Cv) positions of a thread are spread S/Cu (S/Cv) apart, so
//     every owned position is an independent Romein column/row and none ever wraps;
//   * the "did my points move" test is one AND of a per-sample bit mask (which
//     positions changed cell between consecutive samples, computed once per sample while staging)
//     with a per-thread constant -- amortised over the whole block like the paper's per-block test;
//   * tap rows are stored three times over (k[t mod S], t < 3S) so that the Cu tap loads of a thread
//     are one address plus compile-time offsets: m+n loads, m*n products.
// Skipped samples (R7) take part in the walk with zero visibilities; their coordinates are clamped.
#pragma once
#include "gridder_common.cuh"
#include "grid_kernel.cuh"

namespace gridb200 {

// Traversal position (batch b, slot k) of a chunk -> global sample index, or -1 past the end.
struct ChunkGeom {
    int mode;              // 0: contiguous run, odd time rows mirrored; 1: time-innermost block
    long long base;        // mode 0: first position; mode 1: first sample of (baseline, time block)
    int len;               // mode 0: positions in the chunk
    int h;                 // mode 1: time steps in this block (<= tc)
};

__device__ __forceinline__ int batch_count(const GridParams& gp, const ChunkGeom& cg, int b) {
    if (cg.mode == 0) {
        const int left = cg.len - b * gp.batch;
        return left < 0 ? 0 : (left < gp.batch ? left : gp.batch);
    }
    int cols = gp.n_chan - (b << gp.cb_shift);
    if (cols > (1 << gp.cb_shift)) cols = 1 << gp.cb_shift;
    return cols < 0 ? 0 : cols * cg.h;
}

__device__ __forceinline__ long long slot_to_sample(const GridParams& gp, const ChunkGeom& cg, int b, int k) {
    if (cg.mode == 0) {
        long long a = cg.base + (long long)b * gp.batch + k;
        if (gp.n_chan > 0) {                         // serpentine over time rows
            const long long row = a / gp.n_chan;
            const int col = (int)(a - row * gp.n_chan);
            if (row & 1) a = row * gp.n_chan + (gp.n_chan - 1 - col);
        }
        return a;
    }
    const int ci = k / cg.h, tt = k - ci * cg.h;
    const int col = (b << gp.cb_shift) + ci;
    const int ti = (col & 1) ? cg.h - 1 - tt : tt;
    return cg.base + (long long)ti * gp.n_chan + col;
}

// Bit mask of the bin positions whose grid point changes when the footprint origin goes from
// `from` to `to` (one axis).  All positions if it jumps by a whole support or more.
template <int LOGS>
__device__ __forceinline__ uint32_t moved_mask(int from, int to) {
    constexpr int S = 1 << LOGS;
    constexpr uint32_t ALL = 0xffffffffu >> (32 - S);
    const int d = to - from;
    if (d == 0) return 0u;
    const int ad = d < 0 ? -d : d;
    if (ad >= S) return ALL;
    const int start = (d > 0 ? from : to) & (S - 1);        // positions start .. start+ad-1 (cyclic)
    const uint32_t run = (1u << ad) - 1u;
    uint32_t m = run << start;
    if constexpr (S < 32) m |= m >> S; else m |= (start ? run >> (32 - start) : 0u);
    return m & ALL;
}

// One grid point (all polarisations): if `hit`, atomically add the accumulators and zero them.
template <int P>
__device__ __forceinline__ void flush_cell(float2 (&a)[P], float* p, uint32_t hit) {
    if constexpr (P == 4) {
        asm volatile(
            "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %9, 0;\n\t"
            "@q red.relaxed.gpu.global.add.v4.f32 [%8], {%0, %1, %2, %3};\n\t"
            "@q red.relaxed.gpu.global.add.v4.f32 [%8+16], {%4, %5, %6, %7};\n\t"
            "@q mov.f32 %0, 0f00000000;\n\t@q mov.f32 %1, 0f00000000;\n\t"
            "@q mov.f32 %2, 0f00000000;\n\t@q mov.f32 %3, 0f00000000;\n\t"
            "@q mov.f32 %4, 0f00000000;\n\t@q mov.f32 %5, 0f00000000;\n\t"
            "@q mov.f32 %6, 0f00000000;\n\t@q mov.f32 %7, 0f00000000;\n\t}"
            : "+f"(a[0].x), "+f"(a[0].y), "+f"(a[1].x), "+f"(a[1].y), "+f"(a[2].x), "+f"(a[2].y),
              "+f"(a[3].x), "+f"(a[3].y)
            : "l"(p), "r"(hit) : "memory");
    } else if constexpr (P == 2) {
        asm volatile(
            "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %5, 0;\n\t"
            "@q red.relaxed.gpu.global.add.v4.f32 [%4], {%0, %1, %2, %3};\n\t"
            "@q mov.f32 %0, 0f00000000;\n\t@q mov.f32 %1, 0f00000000;\n\t"
            "@q mov.f32 %2, 0f00000000;\n\t@q mov.f32 %3, 0f00000000;\n\t}"
            : "+f"(a[0].x), "+f"(a[0].y), "+f"(a[1].x), "+f"(a[1].y)
            : "l"(p), "r"(hit) : "memory");
    } else {
        static_assert(P == 1, "1, 2 or 4 polarisations");
        asm volatile(
            "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
            "@q red.relaxed.gpu.global.add.v2.f32 [%2], {%0, %1};\n\t"
            "@q mov.f32 %0, 0f00000000;\n\t@q mov.f32 %1, 0f00000000;\n\t}"
            : "+f"(a[0].x), "+f"(a[0].y)
            : "l"(p), "r"(hit) : "memory");
    }
}

template <int CU, int CV, int P, int LOGS>
__global__ void __launch_bounds__(512, 1)
grid_cyclic_kernel(const GridParams gp) {
    constexpr int S = 1 << LOGS;
    constexpr int DU = S / CU, DV = S / CV;          // spacing of a thread's owned positions
    constexpr int TEAM = DU * DV;                     // threads per bin
    constexpr int ROW = 3 * S;                        // tripled tap row
    static_assert(CU <= S && CV <= S, "block larger than the support");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* taps = reinterpret_cast<float2*>(smem_raw);
    size_t off = ((size_t)gp.n_rows * ROW * sizeof(float2) + 15) & ~(size_t)15;
    uint4* srec = reinterpret_cast<uint4*>(smem_raw + off);
    float2* svis = reinterpret_cast<float2*>(smem_raw + off + (size_t)gp.teams_per_cta * gp.batch * sizeof(uint4));
    __shared__ unsigned int s_group;

    const int tid = threadIdx.x;
    for (int k = tid; k < gp.n_rows * ROW; k += blockDim.x) {          // a4
        const int r = k / ROW, t = (k - r * ROW) & (S - 1);
        taps[k] = __ldg(gp.kern + (size_t)r * S + t);
    }

    // a5: ownership
    const int team = tid / TEAM, lt = tid - team * TEAM;
    const bool active = team < gp.teams_per_cta;
    const int r0 = lt % DU, s0 = lt / DU;
    uint32_t MX = 0, MY = 0;
#pragma unroll
    for (int a = 0; a < CU; ++a) MX |= 1u << (r0 + a * DU);
#pragma unroll
    for (int b = 0; b < CV; ++b) MY |= 1u << (s0 + b * DV);
    const uint4* my_rec = srec + (size_t)team * gp.batch;
    const float2* my_vis = svis + (size_t)team * gp.batch * P;
    const float2* my_tu = taps + r0;
    const float2* my_tv = taps + s0;
    const CycRec* recs = reinterpret_cast<const CycRec*>(gp.recs);

    float2 acc[CV][CU][P];
#pragma unroll
    for (int b = 0; b < CV; ++b)
#pragma unroll
        for (int a = 0; a < CU; ++a)
#pragma unroll
            for (int q = 0; q < P; ++q) acc[b][a][q] = make_float2(0.f, 0.f);

    // a8: atomically add the owned points selected by (mx, my) to the grid and clear them.  The
    // points are where the positions were for the PREVIOUS sample (origin i0p, j0p).
    auto flush = [&](uint32_t prevpos, uint32_t mx, uint32_t my) {
        const int i0p = (int)(prevpos & 0x7fffu), j0p = (int)(prevpos >> 16);
        int xa[CU], yb[CV];
#pragma unroll
        for (int a = 0; a < CU; ++a) xa[a] = i0p + ((r0 + a * DU - i0p) & (S - 1));
#pragma unroll
        for (int b = 0; b < CV; ++b) yb[b] = j0p + ((s0 + b * DV - j0p) & (S - 1));
#pragma unroll
        for (int b = 0; b < CV; ++b) {
#pragma unroll
            for (int a = 0; a < CU; ++a) {
                // predicated, in place (no branch, no temporaries: cf. the register-pressure note PAPER.md:93-95)
                const uint32_t hit = ((mx >> (r0 + a * DU)) | (my >> (s0 + b * DV))) & 1u;
                const uint32_t cellidx = (uint32_t)(yb[b] * gp.N + xa[a]);          // < 2^30
                float* p = gp.grid + (size_t)cellidx * (2 * P);
                flush_cell<P>(acc[b][a], p, hit);
            }
        }
    };

    int mode = gp.force_mode;
    if (mode < 0) {
        mode = 0;
        if (gp.n_chan > 0) {
            const float hc = __ldg(gp.hop_stats), ht = __ldg(gp.hop_stats + 1);
            const float cost0 = ((gp.n_chan - 1) * hc + ht) / gp.n_chan;
            const float cost1 = ((gp.tc - 1) * ht + hc) / gp.tc;
            mode = cost1 < cost0 ? 1 : 0;
        }
    }
    const long long n_groups = mode ? gp.n_groups_b : gp.n_groups_a;
    const int n_batches = mode ? (gp.n_chan + (1 << gp.cb_shift) - 1) >> gp.cb_shift
                               : (gp.chunk + gp.batch - 1) / gp.batch;
    const int stage_total = gp.teams_per_cta * gp.batch;

    auto chunk_geom = [&](long long chunk_id) {
        ChunkGeom cg;
        cg.mode = mode; cg.len = 0; cg.h = 1; cg.base = 0;
        if (mode == 0) {
            cg.base = chunk_id * gp.chunk;
            const long long left = gp.n_vis - cg.base;
            cg.len = left <= 0 ? 0 : (left < gp.chunk ? (int)left : gp.chunk);
        } else if (chunk_id < gp.n_chunks_b) {
            const long long bl = chunk_id / gp.n_tblocks;
            const int tb = (int)(chunk_id - bl * gp.n_tblocks);
            cg.h = gp.n_times - tb * gp.tc < gp.tc ? gp.n_times - tb * gp.tc : gp.tc;
            cg.base = (bl * gp.n_times + (long long)tb * gp.tc) * gp.n_chan;
        } else {
            cg.h = 0;
        }
        return cg;
    };

    for (;;) {
        __syncthreads();
        if (tid == 0) s_group = atomicAdd(gp.counters, 1u);          // a9
        __syncthreads();
        const long long group = s_group;
        if (group >= n_groups) break;
        const ChunkGeom my_cg = chunk_geom(group * gp.teams_per_cta + (active ? team : 0));
        uint32_t prevpos = 0;
        bool started = false;

        for (int b = 0; b < n_batches; ++b) {
            __syncthreads();
            // a2 + a3: stage a batch per team: pre-weighted visibilities, tap offsets, moved masks
            for (int kk = tid; kk < stage_total; kk += blockDim.x) {
                const int t = kk >> gp.batch_shift, k = kk & (gp.batch - 1);
                const ChunkGeom cg = chunk_geom(group * gp.teams_per_cta + t);
                const int cnt = (cg.mode == 1 && cg.h == 0) ? 0 : batch_count(gp, cg, b);
                if (k >= cnt) continue;
                const long long g = slot_to_sample(gp, cg, b, k);
                const uint2 raw = __ldg(reinterpret_cast<const uint2*>(recs + g));
                CycRec rec;
                rec.pos = raw.x; rec.rows = raw.y;
                uint32_t mx = 0, my = 0;
                if (k > 0 || b > 0) {
                    const long long gprev = k > 0 ? slot_to_sample(gp, cg, b, k - 1)
                                                  : slot_to_sample(gp, cg, b - 1, batch_count(gp, cg, b - 1) - 1);
                    const uint32_t pp = __ldg(&recs[gprev].pos);
                    mx = moved_mask<LOGS>((int)(pp & 0x7fffu), (int)(rec.pos & 0x7fffu));
                    my = moved_mask<LOGS>((int)(pp >> 16), (int)(rec.pos >> 16));
                }
                const int i0 = (int)(rec.pos & 0x7fffu), j0 = (int)(rec.pos >> 16);
                uint4 c;
                c.x = rec.pos & 0xffff7fffu;
                c.y = (uint32_t)((rec.rows & 0xffffu) * ROW + S - (i0 & (S - 1))) |
                      ((uint32_t)((rec.rows >> 16) * ROW + S - (j0 & (S - 1))) << 16);
                c.z = mx; c.w = my;
                srec[kk] = c;
                const bool valid = (rec.pos & 0x8000u) == 0;
                const float w = valid ? __ldg(gp.weights + g) : 0.f;
#pragma unroll
                for (int q = 0; q < P; ++q) {
                    float2 v = make_float2(0.f, 0.f);
                    if (valid) { v = __ldg(gp.vis + g * P + q); v.x *= w; v.y *= w; }
                    svis[(size_t)kk * P + q] = v;
                }
            }
            __syncthreads();
            if (!active) continue;
            const int cnt = (my_cg.mode == 1 && my_cg.h == 0) ? 0 : batch_count(gp, my_cg, b);

            for (int s = 0; s < cnt; ++s) {
                const uint4 c = my_rec[s];
                if ((c.z & MX) | (c.w & MY)) flush(prevpos, c.z, c.w);       // my points moved
                prevpos = c.x;
                started = true;
                const float2* tu = my_tu + (c.y & 0xffffu);
                const float2* tv = my_tv + (c.y >> 16);
                float2 gu[CU], gv[CV], v[P];
#pragma unroll
                for (int a = 0; a < CU; ++a) gu[a] = tu[a * DU];
#pragma unroll
                for (int bb = 0; bb < CV; ++bb) gv[bb] = tv[bb * DV];
#pragma unroll
                for (int q = 0; q < P; ++q) v[q] = my_vis[s * P + q];
#pragma unroll
                for (int bb = 0; bb < CV; ++bb) {
#pragma unroll
                    for (int a = 0; a < CU; ++a) {
                        const float gr = gv[bb].x * gu[a].x - gv[bb].y * gu[a].y;       // a6
                        const float gi = gv[bb].x * gu[a].y + gv[bb].y * gu[a].x;
#pragma unroll
                        for (int q = 0; q < P; ++q) {                                    // a7
                            acc[bb][a][q].x = fmaf(gr, v[q].x, acc[bb][a][q].x);
                            acc[bb][a][q].x = fmaf(-gi, v[q].y, acc[bb][a][q].x);
                            acc[bb][a][q].y = fmaf(gr, v[q].y, acc[bb][a][q].y);
                            acc[bb][a][q].y = fmaf(gi, v[q].x, acc[bb][a][q].y);
                        }
                    }
                }
            }
        }
        if (active && started) flush(prevpos, 0xffffffffu, 0xffffffffu);
    }
}

}  // namespace gridb200
