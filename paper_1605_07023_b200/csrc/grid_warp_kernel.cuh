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

// Tap t (< Sk) of row `row` of the table the kernel works with.  Supports that are not powers of two are
// zero-padded to Sk = S + pad: every row of the caller's table appears twice, copy 0 with the zeros behind the S
// taps, copy 1 with the zeros in front (gridder.cu, padded_support).
__device__ __forceinline__ float2 padded_tap(const float2* __restrict__ kern, long long row, int t, int S_real, int pad) {
    if (pad == 0) return __ldg(kern + row * S_real + t);
    const int src = (row & 1) ? t - pad : t;
    return (src >= 0 && src < S_real) ? __ldg(kern + (row >> 1) * S_real + src) : make_float2(0.f, 0.f);
}

// Row-doubled copy of the tap table in global memory (TG kernels): t[r][k] = kern[r][k mod S], k < 2S.
__global__ void __launch_bounds__(256) tap_table_kernel(const float2* __restrict__ kern, float2* __restrict__ out,
                                                        long long n_elems, int S, int pad) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_elems) return;
    const long long r = k / (2 * S);
    const int t = (int)(k - r * 2 * S) & (S - 1);
    out[k] = padded_tap(kern, r, t, S - pad, pad);
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

// Traversal geometry of one chunk (one team): 16 bytes in shared memory, 32-bit sample indices (the callers
// of this kernel require n_vis < 2^31).
struct WarpChunk {
    uint32_t base;            // mode 0: first position; mode 1: first sample of (baseline, time block)
    uint32_t total;           // positions in the chunk (mode 1: channels x time steps)
    uint32_t h_col;           // mode 1: time steps of this block | first channel << 16; mode 0 with layout: column of `base`
    uint32_t flags;           // bit 0: mode 0, parity of the time row of `base`; bits 4-5: tile of a 128 bin (x + 2 y)
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
// (An L2 evict-first hint on these copies -- cp.async ... .L2::cache_hint with a createpolicy value or with the fixed
//  encoding -- gained 1.5-3.5 % on every config and was taken out again: with it some kernels raised "illegal
//  instruction" on some boxes / driver versions and not on others, with the same binary; profiles/r2_experiments.md.)
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// PS ("polarisation split"): the P polarisations of a grid point are divided over PS adjacent lanes,
// each holding PT = P/PS of them.  With P = 4, PS = 2 the two 16-byte atomics that make up one
// 32-byte grid point come from neighbouring lanes of ONE instruction and reach the L2 as one sector
// operation instead of two -- the L2's atomic sector rate is the second bound of this kernel.
// Checked build (-DGRIDB200_CHECK; compute-sanitizer is closed on the measurement pool): every global address the
// kernel forms and every shared-memory slot it indexes is tested against its bounds; violations are counted in
// gp.counters[kCheckBase + code] (read back with grid_plan_debug_counters) and the access is suppressed.  The
// shipped library compiles these tests away.
static constexpr int kCheckBase = 40;            // counters[40..47]
enum { kChkGridCell = 0, kChkSampleIndex = 1, kChkRawSlot = 2, kChkCookedSlot = 3, kChkTapOffset = 4, kChkOutIndex = 5 };
#ifdef GRIDB200_CHECK
#define GRIDB200_CHK(cond, code) ((cond) ? true : (atomicAdd(gp.counters + kCheckBase + (code), 1u), false))
#else
#define GRIDB200_CHK(cond, code) true
#endif

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
    __host__ __device__ static constexpr size_t raw_bytes(int B) { return (size_t)TPG * B * (16 + 8 * P); }
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
// global memory (L1/L2) instead of Cu+Cv taps, and no GCF product is formed.  S <= 32.  DENSE = 2: one such table
// per polarisation, gp.dense_pol_stride elements apart (A-projection kernels depend on the polarisation).
// RS ("row skip"): the row pass of the flush skips the points its column pass has just flushed (see the flush).
template <int CU, int CV, int P, int LOGS, int PS = 1, bool DEGRID = false, bool TG = false, int DENSE = 0, bool RS = false>
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
    // raw stage layout: vis [slots][P] float2, then records [slots] {pos, rows, weight, -} of 16 bytes
    WarpChunk* geom = reinterpret_cast<WarpChunk*>(rbase + 2 * rstage);                  // [2][TPG]
    uint32_t* last_pos = reinterpret_cast<uint32_t*>(geom + 2 * TPG);                    // [2][TPG]
    uint32_t* ctrl = last_pos + 2 * TPG;

    if constexpr (!TG && !DENSE) {
        for (int k = tid; k < gp.n_rows * ROW; k += blockDim.x) {      // a4
            const int r = k / ROW, t = (k - r * ROW) & (S - 1);
            staps[k] = padded_tap(gp.kern, r, t, S - gp.tap_pad, gp.tap_pad);
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
        if (!GRIDB200_CHK(cell < (uint32_t)gp.N * (uint32_t)gp.N, kChkGridCell)) { clear_point(v); return; }
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
        if (!GRIDB200_CHK(skip || cell < (uint32_t)gp.N * (uint32_t)gp.N, kChkGridCell)) { clear_point(v); return; }
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

    const uint32_t n_vis32 = (uint32_t)gp.n_vis, n_chan = (uint32_t)gp.n_chan;
    const uint32_t tc = (uint32_t)gp.tc;               // a power of two (grid_plan_set_traversal)
    const int tshift = 31 - __clz((int)(tc > 0 ? tc : 1));

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
            uint32_t chunk_id = (uint32_t)(g / NT) * TPG + lg;      // tiled bins: NT consecutive queue entries share a chunk
            bool have = true;
            if (gp.order) {                            // locality-sorted queue (chunk_order.cuh)
                have = chunk_id < (uint32_t)chunk_count(gp, mode);
                if (have) chunk_id = __ldg(gp.order + chunk_id);
            }
            WarpChunk cg;
            cg.base = 0; cg.total = 0; cg.h_col = 1; cg.flags = (uint32_t)(g % NT) << 4;
            if (!have) {
            } else if (mode == 0) {
                const unsigned long long base = (unsigned long long)chunk_id * (uint32_t)gp.chunk;
                if (base < n_vis32) {
                    cg.base = (uint32_t)base;
                    const uint32_t left = n_vis32 - cg.base;
                    cg.total = left < (uint32_t)gp.chunk ? left : (uint32_t)gp.chunk;
                    if (n_chan > 0) {
                        const uint32_t row = cg.base / n_chan;
                        cg.h_col = cg.base - row * n_chan;
                        cg.flags |= row & 1u;
                    }
                }
            } else if (chunk_id < (uint32_t)gp.n_chunks_b) {
                // chunk = (baseline, block of tc time steps, block of chunk_cols channels)
                const uint32_t per_bl = (uint32_t)(gp.n_tblocks * gp.n_cblocks);
                const uint32_t bl = chunk_id / per_bl, rem = chunk_id - bl * per_bl;
                const uint32_t tb = rem / (uint32_t)gp.n_cblocks, cc = rem - tb * (uint32_t)gp.n_cblocks;
                const uint32_t tleft = (uint32_t)gp.n_times - tb * tc;
                const uint32_t h = tleft < tc ? tleft : tc;
                const uint32_t col0 = cc * (uint32_t)gp.chunk_cols;
                const uint32_t cleft = n_chan - col0;
                cg.base = (bl * (uint32_t)gp.n_times + tb * tc) * n_chan;
                cg.total = (cleft < (uint32_t)gp.chunk_cols ? cleft : (uint32_t)gp.chunk_cols) * h;
                cg.h_col = h | (col0 << 16);
            }
            *reinterpret_cast<uint4*>(&geom[par * TPG + lg]) = make_uint4(cg.base, cg.total, cg.h_col, cg.flags);
        }
        group_sync();
        return g;
    };

    auto count_of = [&](const WarpChunk& cg, int b) -> int {
        const int left = (int)cg.total - (b << bshift);
        return left < 0 ? 0 : (left < B ? left : B);
    };

    // sample (input index) at position q of the chunk's walk
    auto sample_of = [&](const WarpChunk& cg, int q) -> uint32_t {
        if (mode == 0) {
            uint32_t a = cg.base + (uint32_t)q;
            if (n_chan > 0) {                          // serpentine over time rows: odd rows are walked backwards
                uint32_t col = cg.h_col + (uint32_t)q, radd = 0;
                if (col >= n_chan) {                   // a chunk spans few rows: subtract instead of dividing
                    col -= n_chan; radd = 1;
                    if (col >= n_chan) { const uint32_t r2 = col / n_chan; col -= r2 * n_chan; radd += r2; }
                }
                if ((cg.flags + radd) & 1u) a += n_chan - 1u - 2u * col;
            }
            return a;
        }
        // columns of h time steps, walked one after another, odd columns backwards
        const uint32_t h = cg.h_col & 0xffffu, col0 = cg.h_col >> 16;
        uint32_t ci, tt;
        if (h == tc) { ci = (uint32_t)q >> tshift; tt = (uint32_t)q & (tc - 1u); }
        else { ci = (uint32_t)q / h; tt = (uint32_t)q - ci * h; }
        const uint32_t col = col0 + ci;
        const uint32_t ti = (col & 1u) ? h - 1u - tt : tt;
        return cg.base + ti * n_chan + col;
    };

    // a3: start the copies of batch b of the chunk group `par` into raw stage `st`: per sample one 16-byte
    // record {origin, tap rows, weight} (8 bytes + a separate weight for pre-quantised, compressed input)
    // and its visibilities
    auto issue = [&](int par, int b, int st) {
        unsigned char* rs = rbase + (size_t)st * rstage;
        float2* rvis = reinterpret_cast<float2*>(rs);
        uint4* rrec = reinterpret_cast<uint4*>(rs + (size_t)slots * 8 * P);
        for (int kk = lg; kk < slots; kk += GT) {
            const int t = kk >> bshift, k = kk & (B - 1);
            const uint4 g4 = *reinterpret_cast<const uint4*>(&geom[par * TPG + t]);
            const WarpChunk cg = {g4.x, g4.y, g4.z, g4.w};
            if (k >= count_of(cg, b)) continue;
            const uint32_t g = sample_of(cg, (b << bshift) + k);
            if (!GRIDB200_CHK(g < n_vis32, kChkSampleIndex) || !GRIDB200_CHK(kk < slots && st < 2, kChkRawSlot)) continue;
            if (gp.sorted) {
                // cell order: the record carries the index of its visibilities (P > 1) or the pre-weighted
                // visibility itself (P = 1)
                const uint4* src = reinterpret_cast<const uint4*>(gp.recs) + (size_t)g * gp.sorted_stride;
                cp_async_16(rrec + kk, src);
                if constexpr (!DEGRID) {
                    if (P > 1 || gp.sorted == 2) {
                        const uint32_t vi = __ldg(reinterpret_cast<const uint32_t*>(src) + 3);
                        if (!GRIDB200_CHK(vi < n_vis32, kChkSampleIndex)) continue;
                        if constexpr (P == 1) cp_async_8(rvis + kk, gp.vis + vi);
                        else {
#pragma unroll
                            for (int q = 0; q < P; q += 2) cp_async_16(rvis + (size_t)kk * P + q, gp.vis + (size_t)vi * P + q);
                        }
                    }
                }
                continue;
            }
            if (gp.rec16) {
                cp_async_16(rrec + kk, reinterpret_cast<const uint4*>(gp.recs) + g);
            } else {
                cp_async_8(rrec + kk, reinterpret_cast<const CycRec*>(gp.recs) + g);
                if (gp.weights) cp_async_4(&rrec[kk].z, gp.weights + g);   // null: pre-weighted (compressed) input
            }
            if constexpr (DEGRID) {
            } else if constexpr (P == 1) cp_async_8(rvis + kk, gp.vis + g);
            else {
#pragma unroll
                for (int q = 0; q < P; q += 2) cp_async_16(rvis + (size_t)kk * P + q, gp.vis + (size_t)g * P + q);
            }
        }
        cp_async_commit();
    };

    // a2: raw stage -> cooked records (tap offsets, moved masks) and pre-weighted visibilities
    auto cook = [&](int par, int b, int st) {
        const unsigned char* rs = rbase + (size_t)st * rstage;
        const float2* rvis = reinterpret_cast<const float2*>(rs);
        const uint4* rrec = reinterpret_cast<const uint4*>(rs + (size_t)slots * 8 * P);
        const bool unit_w = !gp.rec16 && !gp.weights;
        for (int kk = lg; kk < slots; kk += GT) {
            const int t = kk >> bshift, k = kk & (B - 1);
            const uint4 g4 = *reinterpret_cast<const uint4*>(&geom[par * TPG + t]);
            const WarpChunk cg = {g4.x, g4.y, g4.z, g4.w};
            const int cnt = count_of(cg, b);
            const int ck = t * BP + k;                 // slot in the cooked arrays
            if (!GRIDB200_CHK(ck < cslots && t < TPG, kChkCookedSlot)) continue;
            uint4 c = make_uint4(0u, 0u, 0u, 0u);
            if constexpr (W64) cmask[ck] = make_uint4(0u, 0u, 0u, 0u);
            uint32_t code = 0xffffffffu;               // DEGRID: where the result goes; all ones = no sample
            float w = 0.f;
            bool valid = false;
            if (k < cnt) {
                const uint4 rec = rrec[kk];
                mask_t mx = 0, my = 0;
                if (k > 0 || b > 0) {
                    const uint32_t pp = k > 0 ? rrec[kk - 1].x : last_pos[((b - 1) & 1) * TPG + t];
                    const int tile = (int)((cg.flags >> 4) & 3u);
                    if constexpr (NT > 1) {
                        mx = moved_mask_window128((int)(pp & 0x7fffu), (int)(rec.x & 0x7fffu), (tile & 1) * TS);
                        my = moved_mask_window128((int)(pp >> 16), (int)(rec.x >> 16), (tile >> 1) * TS);
                    } else if constexpr (W64) {
                        mx = moved_mask64((int)(pp & 0x7fffu), (int)(rec.x & 0x7fffu));
                        my = moved_mask64((int)(pp >> 16), (int)(rec.x >> 16));
                    } else {
                        mx = moved_mask<LOGS>((int)(pp & 0x7fffu), (int)(rec.x & 0x7fffu));
                        my = moved_mask<LOGS>((int)(pp >> 16), (int)(rec.x >> 16));
                    }
                }
                if (k == cnt - 1) last_pos[(b & 1) * TPG + t] = rec.x;
                const int i0 = (int)(rec.x & 0x7fffu), j0 = (int)(rec.x >> 16);
                const uint32_t xo = (rec.y & 0xffffu) * ROW + S - (i0 & (S - 1));
                const uint32_t yo = (rec.y >> 16) * ROW + S - (j0 & (S - 1));
                c.x = rec.x & 0xffff7fffu;
                if constexpr (DENSE) {
                    // table row ((wp*O + sv)*O + su), in elements of S*S
                    const uint32_t ru = rec.y & 0xffffu, rv = rec.y >> 16;
                    const uint32_t su = ru - (ru / (uint32_t)gp.oversample) * (uint32_t)gp.oversample;
                    c.y = (rv * (uint32_t)gp.oversample + su) * (uint32_t)(S * S);
                    c.z = mx; c.w = my;
                } else if constexpr (W64) {
                    c.y = rec.y;
                    cmask[ck] = make_uint4((uint32_t)mx, (uint32_t)((uint64_t)mx >> 32), (uint32_t)my, (uint32_t)((uint64_t)my >> 32));
                }
                else if constexpr (WIDE && TG) { c.y = rec.y; c.z = mx; c.w = my; }     // offsets exceed 16 bits
                else if constexpr (WIDE) { c.y = xo | (yo << 16); c.z = mx; c.w = my; }
                else { c.y = xo * 8u; c.z = yo * 8u; c.w = mx | (my << 16); }
                valid = (rec.x & 0x8000u) == 0;
                if (valid) w = unit_w ? 1.f : __uint_as_float(rec.z);
                if constexpr (DEGRID) code = (gp.sorted ? rec.w : sample_of(cg, (b << bshift) + k)) | (valid ? 0u : 0x80000000u);
            }
            crec[ck] = c;
            if constexpr (DEGRID) {
                cvis[(size_t)ck * P] = make_float2(w, __uint_as_float(code));
            } else if constexpr (P == 1) {
                float2 v = make_float2(0.f, 0.f);
                if (valid) {                                            // skipped: exact zeros, whatever the input holds
                    if (gp.sorted == 1) { const uint4 rec = rrec[kk]; v = make_float2(__uint_as_float(rec.z), __uint_as_float(rec.w)); }
                    else { v = rvis[kk]; v.x *= w; v.y *= w; }
                }
                cvis[ck] = v;
            } else {
                // pre-weighting, 16 bytes at a time
                const float4* src = reinterpret_cast<const float4*>(rvis + (size_t)kk * P);
                float4* dst = reinterpret_cast<float4*>(cvis + (size_t)ck * P);
#pragma unroll
                for (int q = 0; q < P / 2; ++q) {
                    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (valid) { v = src[q]; v.x *= w; v.y *= w; v.z *= w; v.w *= w; }
                    dst[q] = v;
                }
            }
        }
    };

    int par = 0;
    long long cur = fetch(par);
    if (cur < n_groups) issue(par, 0, 0);
    int st = 0;                                        // raw stage holding the next batch to cook
    while (cur < n_groups) {
        const uint4 my_g4 = *reinterpret_cast<const uint4*>(&geom[par * TPG + tg]);
        const WarpChunk my_cg = {my_g4.x, my_g4.y, my_g4.z, my_g4.w};
        const int my_tile = (int)((my_cg.flags >> 4) & 3u);
        // first owned column / row position (inside my tile of the bin when the bin is tiled)
        const int px0 = r0 + (NT > 1 ? (my_tile & 1) * TS : 0), py0 = s0 + (NT > 1 ? (my_tile >> 1) * TS : 0);
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
                            for (int a = 0; a < CU; ++a) {
                                // A point whose column has just been flushed holds zeros.  Adding them (at its old
                                // row and new column: inside the grid) is harmless and saves a branch per point:
                                // 5-12 % on the BASELINE configs whose grid is at most a few times the L2.  On much
                                // larger grids, where the atomics' DRAM sectors are the limit, the extra 6-10 % of
                                // atomics cost more (cfg3: -7 %): those use the RS instantiation, which skips them.
                                if constexpr (RS) flush_point_if(acc[bb][a], ry[bb] + (uint32_t)cx[a], (mxs & (mask_t(1) << (a * DU))) ? 1u : 0u);
                                else flush_point(acc[bb][a], ry[bb] + (uint32_t)cx[a]);
                            }
                            ry[bb] = (uint32_t)(j0 + ((py0 + bb * DV - j0) & (S - 1))) * (uint32_t)gp.N;
                        }
                    }
                    }
                }
                if constexpr (DENSE) {
                    const int mi = (px0 - (int)(c.x & 0x7fffu)) & (S - 1), mj = (py0 - (int)(c.x >> 16)) & (S - 1);
                    const float2* kb = gp.kern + c.y;
                    c = *++rp;                         // next sample's record
                    float2 v[PT];
#pragma unroll
                    for (int q = 0; q < PT; ++q) v[q] = vp[q];
                    vp += P;
                    if constexpr (DENSE == 2) {
                        // one table per polarisation: the values of polarisation q are fetched and used, then the next
#pragma unroll
                        for (int q = 0; q < PT; ++q) {
                            const float2* kq = kb + (size_t)(half * PT + q) * (size_t)gp.dense_pol_stride;
                            float2 g2[CV][CU];
#pragma unroll
                            for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                                for (int a = 0; a < CU; ++a)
                                    g2[bb][a] = __ldg(kq + ((mj + bb * DV) & (S - 1)) * S + ((mi + a * DU) & (S - 1)));
#pragma unroll
                            for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                                for (int a = 0; a < CU; ++a) {                               // a7
                                    acc[bb][a][q].x = fmaf(g2[bb][a].x, v[q].x, acc[bb][a][q].x);
                                    acc[bb][a][q].x = fmaf(-g2[bb][a].y, v[q].y, acc[bb][a][q].x);
                                    acc[bb][a][q].y = fmaf(g2[bb][a].x, v[q].y, acc[bb][a][q].y);
                                    acc[bb][a][q].y = fmaf(g2[bb][a].y, v[q].x, acc[bb][a][q].y);
                                }
                        }
                        continue;
                    }
                    float2 g2[CV][CU];
#pragma unroll
                    for (int bb = 0; bb < CV; ++bb)
#pragma unroll
                        for (int a = 0; a < CU; ++a)
                            g2[bb][a] = __ldg(kb + ((mj + bb * DV) & (S - 1)) * S + ((mi + a * DU) & (S - 1)));
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
                if constexpr (!TG) {                   // the taps this thread is about to read lie inside the table
                    (void)GRIDB200_CHK(tu >= staps && tu + (CU - 1) * DU < staps + (size_t)gp.n_rows * ROW &&
                                       tv >= staps && tv + (CV - 1) * DV < staps + (size_t)gp.n_rows * ROW, kChkTapOffset);
                }
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
                    if ((lt & dup & 31) == 0 && code != 0xffffffffu && GRIDB200_CHK((code & 0x7fffffffu) < n_vis32, kChkOutIndex)) {
                        float* o = reinterpret_cast<float*>(gp.vis_out + (size_t)(code & 0x7fffffffu) * P) + first;
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
