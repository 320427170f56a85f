// Shared declarations of the B200 gridder (product path; never includes anything from oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gridb200 {

// Quantised sample record written by the a1 pass ("the integer grid
// coordinates, the sub-grid coordinates for indexing the GCF, the w plane index"), already in the
// form the hot loop consumes for the plan's coarsening block (Cu x Cv) and bin (Bu x Bv):
//   x: X0 | Y0 << 16   origin of the block-aligned bounding box, X0 = floor(i0/Cu)*Cu
//                      0xFFFFFFFF marks a skipped sample (footprint outside the grid / non-finite)
//   y: (X0 mod Bu) | (Y0 mod Bv) << 16
//   z: element offset into the zero-padded u tap table: row(wp,su)*Lu + (Cu-1) - (i0-X0)
//   w: element offset into the zero-padded v tap table: row(wp,sv)*Lv + (Cv-1) - (j0-Y0)
typedef uint4 SampleRec;
static constexpr uint32_t kInvalidRec = 0xFFFFFFFFu;

// Record of the power-of-two-support kernel (grid_warp_kernel.cuh), 8 bytes:
//   pos : i0 | skipped << 15 | j0 << 16   (a skipped sample carries clamped in-grid coordinates)
//   rows: (wp*O + su) | (wp*O + sv) << 16
struct CycRec { uint32_t pos, rows; };

struct QuantParams {
    int format;           // 0: SampleRec (16 B), 1: CycRec (8 B), 2: CycRec + weight (16 B: pos, rows, weight, 0)
    double c_centre;      // O*floor(N/2) + 0.5
    int oversample;       // O
    int o_shift;          // log2(O) if O is a power of two, else -1
    int shift;            // O - ceil(O*S/2)
    int q_limit;          // (N-S+1)*O : valid iff 0 <= q < q_limit
    int n_wplanes;
    int cu, cv, bin_u, bin_v, row_u, row_v;   // coarsening block, bin, padded row lengths Lu, Lv
    int pad, sk, grid_size;                   // warp kernel on a support padded to sk = S + pad (a power of two); N
};

struct GridParams {
    const SampleRec* recs;
    const float2* vis;        // [n_vis][P]
    const float* weights;     // [n_vis]
    const float2* kern;       // [W][O][S]
    const float2* gtaps;      // variant 3, tap table too large for shared memory: rows doubled, in global memory
    float* grid;              // [N][N][P] complex64
    float2* vis_out;          // degridding only: [n_vis][P] complex64 result
    unsigned int* counters;   // [0]: next chunk group
    const float* hop_stats;   // [0] mean-hop sum along channels, [1] along time (quantise pass)
    long long n_vis;
    long long n_groups_a, n_groups_b, n_chunks_b;   // mode 0 / mode 1 work decomposition
    int N, S, n_rows;         // n_rows = W*O
    int oversample;           // O (dense tables: row = (wp*O + sv)*O + su)
    int bin_u, bin_v, row_u, row_v, nbx, nby;
    int team_threads, teams_per_cta, batch, chunk, batch_shift;
    int groups_per_cta;       // variant 3: warp groups per CTA (each its own queue consumer)
    // layout hint (0 = unknown) and time-innermost traversal: a mode-1 chunk is tc time steps x all
    // channels of one baseline; a batch is tc x (1 << cb_shift) samples
    int n_chan, n_times, tc, cb_shift, n_tblocks;
    const uint32_t* order;    // variant 3: queue position -> chunk id (chunk_order.cuh); null = identity
    int tile_shift;           // log2 of the tile side used for that order
    int n_cblocks, chunk_cols;   // variant 3, time-innermost: a chunk spans chunk_cols channels
    int force_mode;           // -1: pick from hop_stats, 0: channel-innermost, 1: time-innermost
    float fzero;              // 0.0f the compiler cannot see: accumulators are cleared by moves from the constant bank
    long long dense_pol_stride;   // dense GCF per polarisation: elements between the tables of two polarisations
    int tap_pad;              // warp kernel: zero taps added to each row (support padded to a power of two)
    int rec16;                // warp kernel: records are 16 bytes {pos, rows, weight, -} (quantise format 2), else CycRec
    int sorted_stride;        // cell order: records are this many 16-byte units apart
    int sorted;               // warp kernel: recs are in cell order (cell_sort.cuh), chunks are contiguous runs of them:
                              // 2 = {pos, rows, weight, sample index}, 1 = one polarisation, {pos, rows, weight * vis}
};

}  // namespace gridb200
