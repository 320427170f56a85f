// NEXT-2, first path: degridding -- the adjoint of the gridding operator ("the same
// approach applies to degridding", not measured by the paper).  For every valid sample
//     vis[n][p] = weight_n * sum_{tj,ti} conj(k[wp][sv][tj] * k[wp][su][ti]) * grid[j0+tj][i0+ti][p]
// (exactly oracle.degrid, the operator of pin P7); skipped samples (R7) get zeros.  A gather: no atomics.
//
// This first version keeps nothing in registers across samples: L lanes share one sample, lane r sums
// the footprint rows r, r+L, ... (contiguous S*P complex values each), then a shuffle tree adds the L
// partial sums.  Every grid value is read from L1/L2 once per sample that touches it: S*S*8P bytes per
// sample, so the kernel is bound by L2 bandwidth, not by FMAs.  The coarsened,
// register-resident variant (the paper's ownership scheme run backwards) is the next step.
#pragma once
#include "gridder_common.cuh"

namespace gridb200 {

template <int P, int L>
__global__ void __launch_bounds__(256)
degrid_gather_kernel(const CycRec* __restrict__ recs, const float* __restrict__ weights,
                     const float2* __restrict__ kern, const float2* __restrict__ grid, float2* __restrict__ vis_out,
                     long long n_vis, int N, int S) {
    const long long g = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / L;      // sample
    const int r = threadIdx.x % L;                                                     // my first footprint row
    const bool live = g < n_vis;                               // no early return: the shuffles need every lane
    CycRec rec;
    rec.pos = 0x8000u; rec.rows = 0u;
    if (live) rec = recs[g];
    const bool valid = (rec.pos & 0x8000u) == 0;
    const int i0 = (int)(rec.pos & 0x7fffu), j0 = (int)(rec.pos >> 16);
    const float2* ku = kern + (size_t)(rec.rows & 0xffffu) * S;
    const float2* kv = kern + (size_t)(rec.rows >> 16) * S;
    float2 acc[P];
#pragma unroll
    for (int q = 0; q < P; ++q) acc[q] = make_float2(0.f, 0.f);
    if (valid) {
        for (int tj = r; tj < S; tj += L) {
            const float2* row = grid + ((size_t)(j0 + tj) * N + i0) * P;
            float2 racc[P];
#pragma unroll
            for (int q = 0; q < P; ++q) racc[q] = make_float2(0.f, 0.f);
            for (int ti = 0; ti < S; ++ti) {
                const float2 a = __ldg(ku + ti);                       // conj(a) * cell
#pragma unroll
                for (int q = 0; q < P; ++q) {
                    const float2 c = row[(size_t)ti * P + q];
                    racc[q].x = fmaf(a.x, c.x, racc[q].x);
                    racc[q].x = fmaf(a.y, c.y, racc[q].x);
                    racc[q].y = fmaf(a.x, c.y, racc[q].y);
                    racc[q].y = fmaf(-a.y, c.x, racc[q].y);
                }
            }
            const float2 b = __ldg(kv + tj);                           // conj(b) * row sum
#pragma unroll
            for (int q = 0; q < P; ++q) {
                acc[q].x = fmaf(b.x, racc[q].x, acc[q].x);
                acc[q].x = fmaf(b.y, racc[q].y, acc[q].x);
                acc[q].y = fmaf(b.x, racc[q].y, acc[q].y);
                acc[q].y = fmaf(-b.y, racc[q].x, acc[q].y);
            }
        }
    }
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < P; ++q) {
            acc[q].x += __shfl_xor_sync(0xffffffffu, acc[q].x, o);
            acc[q].y += __shfl_xor_sync(0xffffffffu, acc[q].y, o);
        }
    }
    if (r == 0 && live) {
        const float w = valid ? weights[g] : 0.f;
#pragma unroll
        for (int q = 0; q < P; ++q)
            vis_out[g * P + q] = valid ? make_float2(w * acc[q].x, w * acc[q].y) : make_float2(0.f, 0.f);
    }
}

}  // namespace gridb200
