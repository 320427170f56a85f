// Steps a2-a9, power-of-two supports: the warp-autonomous gridding kernel (variant 3).
//
// Work distribution is Romein's: a thread is responsible for all grid points with a
// fixed position modulo the bin and keeps the one inside the current footprint in a register
// accumulator, flushing it with an atomic add when it changes.  Thread coarsening:
// each thread owns Cu x Cv positions, so tap loads, the "did my points move" test and the loop
// overhead are paid once per block of Cu*Cv*P accumulators.  The bin equals the support (no zero
// padding: the paper's aligned, padded box wastes 36-56 % of the FMAs at S = 8-16, its own caveat for
// small GCFs) and the Cu (Cv) positions of a thread are S/Cu (S/Cv) apart, so every
// owned position is an independent Romein column/row and never wraps.
//
// What is new relative to the paper's kernel, and why (B200 measurements in
// DESIGN.md section 6):
//   * on sm_100a integer/logic instructions cost 1.5-2 issue cycles against 1 for an FFMA, so the
//     flush path decides the rate once samples hop by a cell or more (BASELINE.json's data: 0.6
//     columns + 0.5 rows per sample).  The flush is therefore organised by moved COLUMN and moved ROW
//     of the bin: a one-cell move makes the owning threads execute Cv (or Cu) cell bodies, not
//     Cu*Cv, and the grid coordinates of the owned points are kept in registers and updated only
//     for the points that moved (no per-flush recomputation);
//   * a team never spans more than it must: a *group* is max(1, team/32) warps; groups share
//     nothing but the tap table, take chunks from the queue on their own and
//     synchronise only among their own warps -- no CTA-wide barrier in steady state;
//   * batches are staged by cp.async (LDGSTS) into a two-stage raw ring, then "cooked" in shared
//     memory by the group's own lanes (pre-weighting PAPER.md:91, tap offsets, moved masks) while the
//     next batch is in flight.
#pragma once
#include <type_traits>
#include "gridder_common.cuh"
#include "grid_kernel.cuh"             // red_add_v2 / red_add_v4
#include "chunk_order.cuh"

namespace gridb200 {

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

// Row-doubled copy of the tap table in global memory (TG kernels): t[r][k] = kern[r][k mod S], k < 2S.
__global__ void __launch_bounds__(256) tap_table_kernel(const float2* __restrict__ kern, float2* __restrict__ out,
                                                        long long n_elems, int S) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_elems) return;
    const long long r = k / (2 * S);
    const int t = (int)(k - r * 2 * S) & (S - 1);
    out[k] = __ldg(kern + r * S + t);
}

// The same for a 64-wide bin (S = 64): 64-bit mask.
__device__ __forceinline__ uint64_t moved_mask64(int from, int to) {
    const int d = to - from;
    if (d == 0) return 0ull;
    const int ad = d < 0 ? -d : d;
    if (ad >= 64) return ~0ull;
    const int start = (d > 0 ? from : to) & 63;
    const uint64_t run = (1ull << ad) - 1ull;
    uint64_t m = run << start;
    if (start) m |= run >> (64 - start);
    return m;
}

// S = 128 is split into 2 x 2 tiles of 64 x 64 bin positions, one team per tile ("one
// work-group per tile"; every tile reads the chunk's samples again).  Moved positions of the 64-wide
// window starting at bin position `lo`.
__device__ __forceinline__ uint64_t moved_mask_window128(int from, int to, int lo) {
    const int d = to - from;
    if (d == 0) return 0ull;
    const int ad = d < 0 ? -d : d;
    if (ad >= 128) return ~0ull;
    const int rel = (((d > 0 ? from : to) - lo) & 127);          // run [rel, rel + ad) in window coordinates, cyclic mod 128
    const unsigned __int128 run = (((unsigned __int128)1) << ad) - 1;
    unsigned __int128 m = run << rel;
    if (rel) m |= run >> (128 - rel);
    return (uint64_t)m;
}

struct WarpChunk {            // traversal geometry of one chunk (one team), 32 bytes in shared memory
    long long base;           // mode 0: first position; mode 1: first sample of (baseline, time block)
    int len;                  // mode 0: positions in the chunk; mode 1: channels in the chunk
    int h;                    // mode 1: time steps in this block (0: empty chunk)
    int col0, rowpar;         // mode 0 with layout: column of `base` and parity of its time row;
                              // mode 1: first channel of the chunk
    int tile, pad1;           // S = 128: which 64 x 64 tile of the bin this team covers (x + 2 y)
};

__device__ __forceinline__ void cp_async_4(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_8(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// PS ("polarisation split"): the P polarisations of a grid point are divided over PS adjacent lanes,
// each holding PT = P/PS of them.  With P = 4, PS = 2 the two 16-byte atomics that make up one
// 32-byte grid point come from neighbouring lanes of ONE instruction and reach the L2 as one sector
// operation instead of two -- the L2's atomic sector rate is the second bound of this kernel.
template <int CU, int CV, int P, int LOGS, int PS = 1>
struct WarpKernelTraits {
    static_assert(P % PS == 0, "polarisations must divide evenly over the split");
    static constexpr int S = 1 << LOGS;
    static constexpr int PT = P / PS;                     // polarisations per thread
    static constexpr int TS = S > 64 ? 64 : S;            // side of the part of the bin one team covers (tile)
    static constexpr int NT = (S / TS) * (S / TS);        // tiles per bin (1, or 4 at S = 128)
    static constexpr int DU = TS / CU, DV = TS / CV;     // spacing of a thread's owned positions
    static constexpr int TEAM = DU * DV * PS;             // threads per tile
    static constexpr int GW = TEAM > 32 ? TEAM / 32 : 1;  // warps per group
    static constexpr int GT = GW * 32;                    // threads per group
    static constexpr int TPG = TEAM >= 32 ? 1 : 32 / TEAM;    // teams (chunks in flight) per group
    static constexpr int ACC = 2 * CU * CV * PT;
    static constexpr int MAX_THREADS = ACC >= 48 ? 512 : (ACC >= 24 ? 768 : 1024);
    // shared memory of one group for a batch of B samples per team
    static constexpr bool W64 = TS == 64;                 // 64-bit moved masks live in a second 16-byte record
    __host__ __device__ static constexpr size_t cooked_bytes(int B) { return ((size_t)TPG * (B + 1) * (16 + (W64 ? 16 : 0) + 8 * P) + 15) & ~(size_t)15; }   // team stride B + 1 slots: see BP
    __host__ __device__ static constexpr size_t raw_bytes(int B) { return (size_t)TPG * B * (8 + 4 + 8 * P); }
    __host__ __device__ static constexpr size_t ctrl_bytes() { return 2 * TPG * sizeof(WarpChunk) + 2 * TPG * 4 + 16; }
    __host__ __device__ static constexpr size_t group_bytes(int B) {
        return (cooked_bytes(B) + 2 * raw_bytes(B) + ctrl_bytes() + 15) & ~(size_t)15;
    }
};

// DEGRID: the same ownership, staging and traversal run backwards: the
// registers hold the VALUES of the owned grid points (loaded when the footprint moves onto a new point,
// where gridding flushes), every sample takes sum conj(G_ij) * value over the owned points, a shuffle
// tree adds the team's partial sums and one lane stores weight * sum to vis_out.  No atomics.
// TG: the tap table does not fit shared memory (many w-planes: the paper uses 1229 per slice,
// PAPER.md:113) -- taps are read through L1/L2 from a row-doubled copy in global memory (gp.gtaps),
// as the paper's kernel does (Table 1 "unified cache").
// DENSE: gp.kern is a non-separable table [W][O][O][S][S]
// (plane, v sub-offset, u sub-offset, row, column); a thread fetches the Cu*Cv values of its points from
// global memory (L1/L2) instead of Cu+Cv taps, and no GCF product is formed.  S <= 32.
template <int CU, int CV, int P, int LOGS, int PS = 1, bool DEGRID = false, bool TG = false, bool DENSE = false>
__global__ void __launch_bounds__((WarpKernelTraits<CU, CV, P, LOGS, PS>::MAX_THREADS), 1)
grid_warp_kernel(const GridParams gp) {
    using T = WarpKernelTraits<CU, CV, P, LOGS, PS>;
    constexpr int PT = T::PT;
    constexpr int S = T::S, DU = T::DU, DV = T::DV, TEAM = T::TEAM, GW = T::GW, GT = T::GT, TPG = T::TPG;
    constexpr int TS = T::TS, NT = T::NT;
    static_assert(NT == 1 || TPG == 1, "tiled bins: one team per group");
    constexpr int ROW = 2 * S;                         // doubled tap row k[t mod S], t < 2S: offsets reach 2S-1
    constexpr bool W64 = T::W64;                       // S = 64: {pos, tap rows, -, -} + a mask record {mx, my} of 64 bits each
    constexpr bool WIDE = S == 32 || (DENSE && S < 32); // record format: masks in two words
    static_assert(!DENSE || (S <= 32 && !DEGRID && !TG), "dense tables: S <= 32, gridding only");
    using mask_t = typename std::conditional<W64, uint64_t, uint32_t>::type;
    static_assert(CU <= TS && CV <= TS, "block larger than the support");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* staps = reinterpret_cast<float2*>(smem_raw);
    const size_t taps_bytes = (TG || DENSE) ? 0 : ((size_t)gp.n_rows * ROW * sizeof(float2) + 15) & ~(size_t)15;
    const int B = gp.batch, bshift = gp.batch_shift;
    const int slots = TPG * B;

    const int tid = threadIdx.x;
    const int group = tid / GT, lg = tid - group * GT;
    unsigned char* gbase = smem_raw + taps_bytes + (size_t)group * T::group_bytes(B);
    // Cooked arrays: the teams of a group are B + 1 slots apart, so that the same sample slot of two teams
    // falls into different banks (a stride of B slots is a multiple of 128 bytes: every record and
    // visibility load of the hot loop was a 2-way bank conflict, 34 % of all shared wavefronts on cfg1).
    // The extra slot is also the slack the hot loop's read-ahead of the next record needs.
    const int BP = B + 1;
    const int cslots = TPG * BP;
    uint4* crec = reinterpret_cast<uint4*>(gbase);                                       // cooked records
    uint4* cmask = reinterpret_cast<uint4*>(gbase + (size_t)cslots * 16);                // W64 only (16-byte records first)
    float2* cvis = reinterpret_cast<float2*>(gbase + (size_t)cslots * (W64 ? 32 : 16)); // cooked vis
    unsigned char* rbase = gbase + T::cooked_bytes(B);
    const size_t rstage = T::raw_bytes(B);
    // raw stage layout: vis [slots][P] float2, rec [slots] 8 B, weights [slots] float
    WarpChunk* geom = reinterpret_cast<WarpChunk*>(rbase + 2 * rstage);                  // [2][TPG]
    uint32_t* last_pos = reinterpret_cast<uint32_t*>(geom + 2 * TPG);                    // [2][TPG]
    uint32_t* ctrl = last_pos + 2 * TPG;

    if constexpr (!TG && !DENSE) {
        for (int k = tid; k < gp.n_rows * ROW; k += blockDim.x) {      // a4
            const int r = k / ROW, t = (k - r * ROW) & (S - 1);
            staps[k] = __ldg(gp.kern + (size_t)r * S + t);
        }
    }
    __syncthreads();
    if (group >= gp.groups_per_cta) return;            // surplus threads (CTA not a multiple of GT)

    auto group_sync = [&]() {
        if constexpr (GW == 1) __syncwarp();
        else asm volatile("bar.sync %0, %1;" :: "r"(group + 1), "r"(GT) : "memory");
    };

    // a5: ownership
    const int tg = (TPG > 1) ? lg / TEAM : 0;          // my team within the group
    const int lt = lg - tg * TEAM;
    const int half = lt % PS, ct = lt / PS;            // my share of the polarisations; my block owner index
    const int r0 = ct % DU, s0 = ct / DU;
    mask_t MX = 0, MY = 0;
#pragma unroll
    for (int a = 0; a < CU; ++a) MX |= mask_t(1) << (r0 + a * DU);
#pragma unroll
    for (int b = 0; b < CV; ++b) MY |= mask_t(1) << (s0 + b * DV);
    const uint32_t MXY = (uint32_t)MX | ((uint32_t)MY << 16);      // S <= 16: both masks in one word
    const uint4* my_mask = cmask + (size_t)tg * BP;
    const uint4* my_rec = crec + (size_t)tg * BP;
    const float2* my_vis = cvis + (size_t)tg * BP * P + (DEGRID ? 0 : half * PT);   // DEGRID: {weight, sample code}
    const unsigned char* my_tu;
    const unsigned char* my_tv;
    if constexpr (TG) {
        my_tu = reinterpret_cast<const unsigned char*>(gp.gtaps + r0);
        my_tv = reinterpret_cast<const unsigned char*>(gp.gtaps + s0);
    } else {
        my_tu = reinterpret_cast<const unsigned char*>(staps + r0);
        my_tv = reinterpret_cast<const unsigned char*>(staps + s0);
    }
    const CycRec* recs = reinterpret_cast<const CycRec*>(gp.recs);

    float2 acc[CV][CU][PT];
#pragma unroll
    for (int b = 0; b < CV; ++b)
#pragma unroll
        for (int a = 0; a < CU; ++a)
#pragma unroll
            for (int q = 0; q < PT; ++q) acc[b][a][q] = make_float2(0.f, 0.f);
    int cx[CU];                     // x of the grid point currently held for owned column a
    uint32_t ry[CV];                // y * N of the grid point currently held for owned row b
#pragma unroll
    for (int a = 0; a < CU; ++a) cx[a] = 0;
#pragma unroll
    for (int b = 0; b < CV; ++b) ry[b] = 0;

    // the grid pointer lives in registers: reloading it from the constant bank inside the divergent
    // flush sections showed up as long-scoreboard stalls (profiles/)
    float* gridp = gp.grid;
    asm volatile("" : "+l"(gridp));

    // Clearing a flushed point: 2*PT moves from a zero the compiler cannot see (gp.fzero, constant bank).  With a
    // literal 0.f ptxas rebuilds four uniform zero registers inside every flush body.  Measured and not kept
    // (profiles/r2_flush_experiments.md): clearing by LDS.128 of zeros (fewer issue slots, but the shared-memory
    // pipe is the second limit of this kernel), clearing by FFMAs of hidden zeros (ptxas folds or hoists them).
    auto clear_point = [&](float2 (&v)[PT]) {
#pragma unroll
        for (int q = 0; q < PT; ++q) v[q] = make_float2(gp.fzero, gp.fzero);
    };

    // DEGRID: fetch the value of a grid point my team now covers
    auto load_point = [&](float2 (&v)[PT], uint32_t cell) {
        const float* p = gridp + (size_t)cell * (2 * P) + half * (2 * PT);
        if constexpr (PT == 4) {
            const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
            v[0] = make_float2(a.x, a.y); v[1] = make_float2(a.z, a.w);
            v[2] = make_float2(b.x, b.y); v[3] = make_float2(b.z, b.w);
        } else if constexpr (PT == 2) {
            const float4 a = *reinterpret_cast<const float4*>(p);
            v[0] = make_float2(a.x, a.y); v[1] = make_float2(a.z, a.w);
        } else {
            v[0] = *reinterpret_cast<const float2*>(p);
        }
    };

    // a8: one grid point, all polarisations: atomic add, then clear
    auto flush_point = [&](float2 (&v)[PT], uint32_t cell) {
        float* p = gridp + (size_t)cell * (2 * P) + half * (2 * PT);
        if constexpr (PT == 4) {
            red_add_v4(p, v[0].x, v[0].y, v[1].x, v[1].y);
            red_add_v4(p + 4, v[2].x, v[2].y, v[3].x, v[3].y);
        } else if constexpr (PT == 2) {
            red_add_v4(p, v[0].x, v[0].y, v[1].x, v[1].y);
        } else {
            red_add_v2(p, v[0].x, v[0].y);
        }
        clear_point(v);
    };

    // Same, but the atomic adds are predicated: used in the row pass for points whose column has
    // just been flushed (their accumulators are zero; skipping saves the L2 traffic, not a branch).
    auto flush_point_if = [&](float2 (&v)[PT], uint32_t cell, uint32_t skip) {
        float* p = gridp + (size_t)cell * (2 * P) + half * (2 * PT);
        if constexpr (PT == 4) {
            asm volatile("{\n\t.reg .pred q;\n\tsetp.eq.u32 q, %9, 0;\n\t"
                         "@q red.relaxed.gpu.global.add.v4.f32 [%8], {%0, %1, %2, %3};\n\t"
                         "@q red.relaxed.gpu.global.add.v4.f32 [%8+16], {%4, %5, %6, %7};\n\t}"
                         :: "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y),
                            "f"(v[3].x), "f"(v[3].y), "l"(p), "r"(skip) : "memory");
        } else if constexpr (PT == 2) {
            asm volatile("{\n\t.reg .pred q;\n\tsetp.eq.u32 q, %5, 0;\n\t"
                         "@q red.relaxed.gpu.global.add.v4.f32 [%4], {%0, %1, %2, %3};\n\t}"
                         :: "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "l"(p), "r"(skip) : "memory");
        } else {
            asm volatile("{\n\t.reg .pred q;\n\tsetp.eq.u32 q, %3, 0;\n\t"
                         "@q red.relaxed.gpu.global.add.v2.f32 [%2], {%0, %1};\n\t}"
                         :: "f"(v[0].x), "f"(v[0].y), "l"(p), "r"(skip) : "memory");
        }
        clear_point(v);
    };

    const int mode = pick_mode(gp);
    const long long n_groups = mode ? gp.n_groups_b : gp.n_groups_a;
    const int n_batches = mode ? (gp.chunk_cols * gp.tc + B - 1) >> bshift
                               : (gp.chunk + B - 1) >> bshift;

    // a9: take the next chunk group from the queue; lanes t < TPG work out their team's geometry
    auto fetch = [&](int par) -> long long {
        uint32_t v = 0;
        if constexpr (GW == 1) {
            if (lg == 0) v = atomicAdd(gp.counters, 1u);
            v = __shfl_sync(0xffffffffu, v, 0);
        } else {
            if (lg == 0) ctrl[0] = atomicAdd(gp.counters, 1u);
            group_sync();
            v = ctrl[0];
        }
        const long long g = v;
        if (g < n_groups && lg < TPG) {
            long long chunk_id = (g / NT) * TPG + lg;      // tiled bins: NT consecutive queue entries share a chunk
            bool have = true;
            if (gp.order) {                            // locality-sorted queue (chunk_order.cuh)
                have = chunk_id < chunk_count(gp, mode);
                if (have) chunk_id = __ldg(gp.order + chunk_id);
            }
            WarpChunk cg;
            cg.base = 0; cg.len = 0; cg.h = 0; cg.col0 = 0; cg.rowpar = 0; cg.tile = (int)(g % NT); cg.pad1 = 0;
            if (!have) {
            } else if (mode == 0) {
                cg.base = chunk_id * gp.chunk;
                const long long left = gp.n_vis - cg.base;
                cg.len = left <= 0 ? 0 : (left < gp.chunk ? (int)left : gp.chunk);
                if (gp.n_chan > 0) {
                    const long long row = cg.base / gp.n_chan;
                    cg.col0 = (int)(cg.base - row * gp.n_chan);
                    cg.rowpar = (int)(row & 1);
                }
            } else if (chunk_id < gp.n_chunks_b) {
                // chunk = (baseline, block of tc time steps, block of chunk_cols channels)
                const long long per_bl = (long long)gp.n_tblocks * gp.n_cblocks;
                const long long bl = chunk_id / per_bl;
                const int rem = (int)(chunk_id - bl * per_bl);
                const int tb = rem / gp.n_cblocks, cc = rem - tb * gp.n_cblocks;
                cg.h = gp.n_times - tb * gp.tc < gp.tc ? gp.n_times - tb * gp.tc : gp.tc;
                cg.base = (bl * gp.n_times + (long long)tb * gp.tc) * gp.n_chan;
                cg.col0 = cc * gp.chunk_cols;
                cg.len = gp.n_chan - cg.col0 < gp.chunk_cols ? gp.n_chan - cg.col0 : gp.chunk_cols;
            }
            geom[par * TPG + lg] = cg;
        }
        group_sync();
        return g;
    };

    auto count_of = [&](const WarpChunk& cg, int b) -> int {
        if (mode == 0) {
            const int left = cg.len - (b << bshift);
            return left < 0 ? 0 : (left < B ? left : B);
        }
        const int left = cg.len * cg.h - (b << bshift);        // columns of h time steps, walked one after another
        return left < 0 ? 0 : (left < B ? left : B);
    };

    auto sample_of = [&](const WarpChunk& cg, int b, int k) -> long long {
        if (mode == 0) {
            const int off = (b << bshift) + k;
            long long a = cg.base + off;
            if (gp.n_chan > 0) {                        // serpentine over time rows
                const uint32_t col = (uint32_t)(cg.col0 + off);
                const uint32_t radd = col / (uint32_t)gp.n_chan;
                const int colr = (int)(col - radd * (uint32_t)gp.n_chan);
                if ((cg.rowpar + radd) & 1u) a += gp.n_chan - 1 - 2 * colr;
            }
            return a;
        }
        const int q = (b << bshift) + k;
        const int ci = (int)((uint32_t)q / (uint32_t)cg.h), tt = q - ci * cg.h;
        const int col = cg.col0 + ci;
        const int ti = (col & 1) ? cg.h - 1 - tt : tt;
        return cg.base + (long long)ti * gp.n_chan + col;
    };

    // DEGRID: sample indices are kept as 31-bit offsets from here (a mirrored time row of the
    // channel-innermost walk reaches back to the start of its row, before the chunk's first position)
    auto out_base = [&](const WarpChunk& cg) -> long long { return mode == 0 ? cg.base - cg.col0 : cg.base; };

    // a3: start the copies of batch b of the chunk group `par` into raw stage `st`
    auto issue = [&](int par, int b, int st) {
        unsigned char* rs = rbase + (size_t)st * rstage;
        float2* rvis = reinterpret_cast<float2*>(rs);
        CycRec* rrec = reinterpret_cast<CycRec*>(rs + (size_t)slots * 8 * P);
        float* rw = reinterpret_cast<float*>(rs + (size_t)slots * (8 * P + 8));
        for (int kk = lg; kk < slots; kk += GT) {
            const int t = kk >> bshift, k = kk & (B - 1);
            const WarpChunk cg = geom[par * TPG + t];
            if (k >= count_of(cg, b)) continue;
            const long long g = sample_of(cg, b, k);
            cp_async_8(rrec + kk, recs + g);
            if (gp.weights) cp_async_4(rw + kk, gp.weights + g);       // null: pre-weighted (compressed) input
            if constexpr (DEGRID) {
            } else if constexpr (P == 1) cp_async_8(rvis + kk, gp.vis + g);
            else {
#pragma unroll
                for (int q = 0; q < P; q += 2) cp_async_16(rvis + (size_t)kk * P + q, gp.vis + g * P + q);
            }
        }
        cp_async_commit();
    };

    // a2: raw stage -> cooked records (tap offsets, moved masks) and pre-weighted visibilities
    auto cook = [&](int par, int b, int st) {
        const unsigned char* rs = rbase + (size_t)st * rstage;
        const float2* rvis = reinterpret_cast<const float2*>(rs);
        const CycRec* rrec = reinterpret_cast<const CycRec*>(rs + (size_t)slots * 8 * P);
        const float* rw = reinterpret_cast<const float*>(rs + (size_t)slots * (8 * P + 8));
        for (int kk = lg; kk < slots; kk += GT) {
            const int t = kk >> bshift, k = kk & (B - 1);
            const WarpChunk cg = geom[par * TPG + t];
            const int cnt = count_of(cg, b);
            uint4 c = make_uint4(0u, 0u, 0u, 0u);
            float w = 0.f;
            bool valid = false;
            const int ck = t * BP + k;                 // slot in the cooked arrays
            if constexpr (W64) cmask[ck] = make_uint4(0u, 0u, 0u, 0u);
            if (k < cnt) {
                const CycRec rec = rrec[kk];
                mask_t mx = 0, my = 0;
                if (k > 0 || b > 0) {
                    const uint32_t pp = k > 0 ? rrec[kk - 1].pos : last_pos[((b - 1) & 1) * TPG + t];
                    if constexpr (NT > 1) {
                        mx = moved_mask_window128((int)(pp & 0x7fffu), (int)(rec.pos & 0x7fffu), (cg.tile & 1) * TS);
                        my = moved_mask_window128((int)(pp >> 16), (int)(rec.pos >> 16), (cg.tile >> 1) * TS);
                    } else if constexpr (W64) {
                        mx = moved_mask64((int)(pp & 0x7fffu), (int)(rec.pos & 0x7fffu));
                        my = moved_mask64((int)(pp >> 16), (int)(rec.pos >> 16));
                    } else {
                        mx = moved_mask<LOGS>((int)(pp & 0x7fffu), (int)(rec.pos & 0x7fffu));
                        my = moved_mask<LOGS>((int)(pp >> 16), (int)(rec.pos >> 16));
                    }
                }
                if (k == cnt - 1) last_pos[(b & 1) * TPG + t] = rec.pos;
                const int i0 = (int)(rec.pos & 0x7fffu), j0 = (int)(rec.pos >> 16);
                const uint32_t xo = (rec.rows & 0xffffu) * ROW + S - (i0 & (S - 1));
                const uint32_t yo = (rec.rows >> 16) * ROW + S - (j0 & (S - 1));
                c.x = rec.pos & 0xffff7fffu;
                if constexpr (DENSE) {
                    // table row ((wp*O + sv)*O + su), in elements of S*S
                    const uint32_t ru = rec.rows & 0xffffu, rv = rec.rows >> 16;
                    const uint32_t su = ru - (ru / (uint32_t)gp.oversample) * (uint32_t)gp.oversample;
                    c.y = (rv * (uint32_t)gp.oversample + su) * (uint32_t)(S * S);
                    c.z = mx; c.w = my;
                } else if constexpr (W64) {
                    c.y = rec.rows;
                    cmask[ck] = make_uint4((uint32_t)mx, (uint32_t)((uint64_t)mx >> 32), (uint32_t)my, (uint32_t)((uint64_t)my >> 32));
                }
                else if constexpr (WIDE && TG) { c.y = rec.rows; c.z = mx; c.w = my; }     // offsets exceed 16 bits
                else if constexpr (WIDE) { c.y = xo | (yo << 16); c.z = mx; c.w = my; }
                else { c.y = xo * 8u; c.z = yo * 8u; c.w = mx | (my << 16); }
                valid = (rec.pos & 0x8000u) == 0;
                if (valid) w = gp.weights ? rw[kk] : 1.f;
            }
            crec[ck] = c;
            if constexpr (DEGRID) {
                // where the result goes: offset from the chunk base, bit 31 = skipped sample, all ones = no sample
                uint32_t code = 0xffffffffu;
                if (k < cnt) code = (uint32_t)(sample_of(cg, b, k) - out_base(cg)) | (valid ? 0u : 0x80000000u);
                cvis[(size_t)ck * P] = make_float2(w, __uint_as_float(code));
            } else {
#pragma unroll
                for (int q = 0; q < P; ++q) {
                    float2 v = make_float2(0.f, 0.f);
                    if (valid) { v = rvis[(size_t)kk * P + q]; v.x *= w; v.y *= w; }
                    cvis[(size_t)ck * P + q] = v;
                }
            }
        }
    };

    int par = 0;
    long long cur = fetch(par);
    if (cur < n_groups) issue(par, 0, 0);
    int st = 0;                                        // raw stage holding the next batch to cook
    while (cur < n_groups) {
        const WarpChunk my_cg = geom[par * TPG + tg];
        // first owned column / row position (inside my tile of the bin when the bin is tiled)
        const int px0 = r0 + (NT > 1 ? (my_cg.tile & 1) * TS : 0), py0 = s0 + (NT > 1 ? (my_cg.tile >> 1) * TS : 0);
        bool live = false;
        long long next = cur;
        int next_par = par;
        for (int b = 0; b < n_batches; ++b) {
            cp_async_wait_all();
            group_sync();                              // raw batch visible; previous hot loop done
            cook(par, b, st);
            group_sync();                              // cooked batch visible; raw stage consumed
            if (b + 1 < n_batches) {
                issue(par, b + 1, st ^ 1);
            } else {                                   // prefetch the first batch of the next group
                next_par = par ^ 1;
                next = fetch(next_par);
                if (next < n_groups) issue(next_par, 0, st ^ 1);
            }
            st ^= 1;

            int cnt = count_of(my_cg, b);
            if (b == 0 && cnt > 0) {                   // first sample of the chunk: take position
                live = true;
                const uint32_t p0 = my_rec[0].x;
                const int i0 = (int)(p0 & 0x7fffu), j0 = (int)(p0 >> 16);
#pragma unroll
                for (int a = 0; a < CU; ++a) cx[a] = i0 + ((px0 + a * DU - i0) & (S - 1));
#pragma unroll
                for (int bb = 0; bb < CV; ++bb) ry[bb] = (uint32_t)(j0 + ((py0 + bb * DV - j0) & (S - 1))) * (uint32_t)gp.N;
                if constexpr (DEGRID) {
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                        for (int a = 0; a < CU; ++a) load_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
                }
            }
            if constexpr (TPG > 1) cnt = __reduce_max_sync(0xffffffffu, cnt);

            const uint4* rp = my_rec;
            const float2* vp = my_vis;
            uint4 c = *rp;
            for (int s = 0; s < cnt; ++s) {
                // (the next record is loaded into the same registers once this one's fields have been consumed,
                //  below: no register rotation at the loop head; one slot of slack follows the batch)
                bool moved;
                mask_t mx_all = 0, my_all = 0;             // this sample's moved masks
                if constexpr (W64) {
                    const uint4 m = my_mask[s];
                    mx_all = (uint64_t)m.x | ((uint64_t)m.y << 32);
                    my_all = (uint64_t)m.z | ((uint64_t)m.w << 32);
                    moved = ((mx_all & MX) | (my_all & MY)) != 0;
                } else if constexpr (WIDE) {
                    mx_all = c.z; my_all = c.w;
                    moved = ((c.z & MX) | (c.w & MY)) != 0;
                } else {
                    mx_all = c.w; my_all = c.w >> 16;
                    moved = (c.w & MXY) != 0;
                }
                if (moved) {                           // a5/a8: some of my points moved
                    const int i0 = (int)(c.x & 0x7fffu), j0 = (int)(c.x >> 16);
                    const mask_t mxs = mx_all >> r0;
                    const mask_t mys = my_all >> s0;
                    if constexpr (DEGRID) {
                        // positions first, then the values of every point that changed (a point whose
                        // column AND row moved is fetched twice; harmless)
#pragma unroll
                        for (int a = 0; a < CU; ++a)
                            if (mxs & (mask_t(1) << (a * DU))) cx[a] = i0 + ((px0 + a * DU - i0) & (S - 1));
#pragma unroll
                        for (int bb = 0; bb < CV; ++bb)
                            if (mys & (mask_t(1) << (bb * DV))) ry[bb] = (uint32_t)(j0 + ((py0 + bb * DV - j0) & (S - 1))) * (uint32_t)gp.N;
#pragma unroll
                        for (int a = 0; a < CU; ++a) {
                            if (mxs & (mask_t(1) << (a * DU))) {
#pragma unroll
                                for (int bb = 0; bb < CV; ++bb) load_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
                            }
                        }
#pragma unroll
                        for (int bb = 0; bb < CV; ++bb) {
                            if (mys & (mask_t(1) << (bb * DV))) {
#pragma unroll
                                for (int a = 0; a < CU; ++a) load_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
                            }
                        }
                    } else {
#pragma unroll
                    for (int a = 0; a < CU; ++a) {
                        if (mxs & (mask_t(1) << (a * DU))) {  // owned column a left the footprint
#pragma unroll
                            for (int bb = 0; bb < CV; ++bb) flush_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
                            cx[a] = i0 + ((px0 + a * DU - i0) & (S - 1));
                        }
                    }
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb) {
                        if (mys & (mask_t(1) << (bb * DV))) { // owned row bb left the footprint
#pragma unroll
                            for (int a = 0; a < CU; ++a)
                                flush_point_if(acc[bb][a], ry[bb] + (uint32_t)cx[a], (mxs & (mask_t(1) << (a * DU))) ? 1u : 0u);
                            ry[bb] = (uint32_t)(j0 + ((py0 + bb * DV - j0) & (S - 1))) * (uint32_t)gp.N;
                        }
                    }
                    }
                }
                if constexpr (DENSE) {
                    const int mi = (px0 - (int)(c.x & 0x7fffu)) & (S - 1), mj = (py0 - (int)(c.x >> 16)) & (S - 1);
                    const float2* kb = gp.kern + c.y;
                    c = *++rp;                         // next sample's record
                    float2 g2[CV][CU], v[PT];
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                        for (int a = 0; a < CU; ++a)
                            g2[bb][a] = __ldg(kb + ((mj + bb * DV) & (S - 1)) * S + ((mi + a * DU) & (S - 1)));
#pragma unroll
                    for (int q = 0; q < PT; ++q) v[q] = vp[q];
                    vp += P;
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                        for (int a = 0; a < CU; ++a)
#pragma unroll
                            for (int q = 0; q < PT; ++q) {                                   // a7
                                acc[bb][a][q].x = fmaf(g2[bb][a].x, v[q].x, acc[bb][a][q].x);
                                acc[bb][a][q].x = fmaf(-g2[bb][a].y, v[q].y, acc[bb][a][q].x);
                                acc[bb][a][q].y = fmaf(g2[bb][a].x, v[q].y, acc[bb][a][q].y);
                                acc[bb][a][q].y = fmaf(g2[bb][a].y, v[q].x, acc[bb][a][q].y);
                            }
                    continue;
                }
                const float2* tu;
                const float2* tv;
                if constexpr (W64 || (WIDE && TG)) {
                    tu = reinterpret_cast<const float2*>(my_tu) + (size_t)(c.y & 0xffffu) * ROW + (S - ((c.x & 0x7fffu) & (S - 1))) + (px0 - r0);
                    tv = reinterpret_cast<const float2*>(my_tv) + (size_t)(c.y >> 16) * ROW + (S - ((c.x >> 16) & (S - 1))) + (py0 - s0);
                } else if constexpr (WIDE) {
                    tu = reinterpret_cast<const float2*>(my_tu) + (c.y & 0xffffu);
                    tv = reinterpret_cast<const float2*>(my_tv) + (c.y >> 16);
                } else {
                    tu = reinterpret_cast<const float2*>(my_tu + c.y);
                    tv = reinterpret_cast<const float2*>(my_tv + c.z);
                }
                c = *++rp;                             // next sample's record
                float2 gu[CU], gv[CV], v[PT];
#pragma unroll
                for (int a = 0; a < CU; ++a) gu[a] = tu[a * DU];
#pragma unroll
                for (int bb = 0; bb < CV; ++bb) gv[bb] = tv[bb * DV];
                if constexpr (DEGRID) {
                    // sum over my points of conj(Gv_j * Gu_i) * value: rows first (conj(Gu_i) * value), then conj(Gv_j)
                    const float2 meta = *vp;                   // {weight, where the result goes}
                    vp += P;
                    float2 part[PT];
#pragma unroll
                    for (int q = 0; q < PT; ++q) part[q] = make_float2(0.f, 0.f);
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb) {
#pragma unroll
                        for (int q = 0; q < PT; ++q) {
                            float rx = 0.f, ry_ = 0.f;
#pragma unroll
                            for (int a = 0; a < CU; ++a) {
                                rx = fmaf(gu[a].x, acc[bb][a][q].x, rx);
                                rx = fmaf(gu[a].y, acc[bb][a][q].y, rx);
                                ry_ = fmaf(gu[a].x, acc[bb][a][q].y, ry_);
                                ry_ = fmaf(-gu[a].y, acc[bb][a][q].x, ry_);
                            }
                            part[q].x = fmaf(gv[bb].x, rx, part[q].x);
                            part[q].x = fmaf(gv[bb].y, ry_, part[q].x);
                            part[q].y = fmaf(gv[bb].x, ry_, part[q].y);
                            part[q].y = fmaf(-gv[bb].y, rx, part[q].y);
                        }
                    }
                    // Team sum by recursive halving (the team's lanes are adjacent and aligned): at each step a
                    // lane keeps one half of its values and hands the other half to its partner, so the 2*PT
                    // floats end up spread over the lanes -- 2*PT-1 shuffles and adds instead of 2*PT*log2(TEAM).
                    float val[2 * PT];
#pragma unroll
                    for (int q = 0; q < PT; ++q) { val[2 * q] = part[q].x; val[2 * q + 1] = part[q].y; }
                    int first = 0;                             // my values are floats [first, first + width) of the result
                    constexpr int W0 = 2 * PT;
                    uint32_t dup = 0;                          // lane bits over which the result is replicated
#pragma unroll
                    constexpr int WT = TEAM < 32 ? TEAM : 32;  // lanes of the team inside this warp
                    for (int o = WT / 2, width = W0; o >= 1; o >>= 1) {
                        if (width > 1) {
                            const int h = width / 2;
                            const bool hi = (lt & o) != 0;
#pragma unroll
                            for (int i = 0; i < W0 / 2; ++i) {
                                if (i < h) {
                                    const float keep = hi ? val[i + h] : val[i];
                                    const float give = hi ? val[i] : val[i + h];
                                    val[i] = keep + __shfl_xor_sync(0xffffffffu, give, o);
                                }
                            }
                            if (hi) first += h;
                            width = h;
                        } else {
                            val[0] += __shfl_xor_sync(0xffffffffu, val[0], o);
                            dup |= (uint32_t)o;
                        }
                    }
                    constexpr int LOGT = WT >= 32 ? 5 : WT >= 16 ? 4 : WT >= 8 ? 3 : WT >= 4 ? 2 : WT >= 2 ? 1 : 0;
                    constexpr int WLAST = (W0 >> LOGT) > 1 ? (W0 >> LOGT) : 1;      // floats left per lane
                    const uint32_t code = __float_as_uint(meta.y);
                    if ((lt & dup & 31) == 0 && code != 0xffffffffu) {
                        float* o = reinterpret_cast<float*>(gp.vis_out + (out_base(my_cg) + (long long)(code & 0x7fffffffu)) * P) + first;
                        const float w = meta.x;
                        if constexpr (GW > 1 || NT > 1) {
                            // the team spans several warps (and, at S = 128, four tiles in other groups): every
                            // warp adds its share atomically; vis_out was zeroed by grid_degrid
#pragma unroll
                            for (int i = 0; i < WLAST; ++i)
                                if (!(code >> 31)) atomicAdd(o + i, w * val[i]);
                        } else {
#pragma unroll
                            for (int i = 0; i < WLAST; ++i) o[i] = (code >> 31) ? 0.f : w * val[i];
                        }
                    }
                    continue;
                }
                if constexpr (PT == 4) {
                    const float4 v01 = *reinterpret_cast<const float4*>(vp);
                    const float4 v23 = *reinterpret_cast<const float4*>(vp + 2);
                    v[0] = make_float2(v01.x, v01.y); v[1] = make_float2(v01.z, v01.w);
                    v[2] = make_float2(v23.x, v23.y); v[3] = make_float2(v23.z, v23.w);
                } else if constexpr (PT == 2) {
                    const float4 v01 = *reinterpret_cast<const float4*>(vp);
                    v[0] = make_float2(v01.x, v01.y); v[1] = make_float2(v01.z, v01.w);
                } else {
                    v[0] = *vp;
                }
                vp += P;
                if constexpr (PT < CU) {
                    // a6 reordered: T = Gv_j * V_p first, then Gu_i * T
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb) {
#pragma unroll
                        for (int q = 0; q < PT; ++q) {
                            const float tr = gv[bb].x * v[q].x - gv[bb].y * v[q].y;
                            const float ti = gv[bb].x * v[q].y + gv[bb].y * v[q].x;
#pragma unroll
                            for (int a = 0; a < CU; ++a) {                               // a7
                                acc[bb][a][q].x = fmaf(gu[a].x, tr, acc[bb][a][q].x);
                                acc[bb][a][q].x = fmaf(-gu[a].y, ti, acc[bb][a][q].x);
                                acc[bb][a][q].y = fmaf(gu[a].x, ti, acc[bb][a][q].y);
                                acc[bb][a][q].y = fmaf(gu[a].y, tr, acc[bb][a][q].y);
                            }
                        }
                    }
                } else {
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb) {
#pragma unroll
                        for (int a = 0; a < CU; ++a) {
                            const float gr = gv[bb].x * gu[a].x - gv[bb].y * gu[a].y;       // a6
                            const float gi = gv[bb].x * gu[a].y + gv[bb].y * gu[a].x;
#pragma unroll
                            for (int q = 0; q < PT; ++q) {                                   // a7
                                acc[bb][a][q].x = fmaf(gr, v[q].x, acc[bb][a][q].x);
                                acc[bb][a][q].x = fmaf(-gi, v[q].y, acc[bb][a][q].x);
                                acc[bb][a][q].y = fmaf(gr, v[q].y, acc[bb][a][q].y);
                                acc[bb][a][q].y = fmaf(gi, v[q].x, acc[bb][a][q].y);
                            }
                        }
                    }
                }
            }
        }
        if (live && !DEGRID) {                         // end of chunk: everything goes to the grid
#pragma unroll
            for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                for (int a = 0; a < CU; ++a) flush_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
        }
        cur = next;
        par = next_par;
    }
    cp_async_wait_all();
}

}  // namespace gridb200
