// Step a1: coordinate quantisation (device pass).  DESIGN.md R4, R5, R7.
// The paper does this offline and hands the kernel "the integer grid coordinates, the sub-grid
// coordinates for indexing the GCF, the w plane index" (section 4).
#pragma once
#include "gridder_common.cuh"

namespace gridb200 {

struct QuantOut { int i0, j0, su, sv, wp; bool valid; };

// One axis: nearest 1/O cell (half up) in IEEE binary64 -- the product x*O is exact in binary64 and
// the single rounding of the add cannot cross an integer (R4) -- then integer arithmetic.
__device__ __forceinline__ bool quantise_axis(float x, const QuantParams& qp, int* cell, int* sub) {
    const double pos = floor(fma((double)x, (double)qp.oversample, qp.c_centre));
    const double q = pos + (double)qp.shift;
    const bool ok = (q >= 0.0 && q < (double)qp.q_limit);        // false for NaN, Inf, outside the grid
    // skipped samples still get in-grid coordinates (fmax/fmin drop NaN): the bin == support kernel walks them
    const int qi = (int)fmin(fmax(q, 0.0), (double)(qp.q_limit - 1));
    // oversampling factors are powers of two in practice: a shift instead of a ~20-instruction division sequence
    const int c = qp.o_shift >= 0 ? (qi >> qp.o_shift) : qi / qp.oversample;
    *cell = c;
    *sub = qi - c * qp.oversample;
    return ok;
}

__device__ __forceinline__ QuantOut quantise_sample(float u, float v, float w, const QuantParams& qp) {
    QuantOut r;
    r.i0 = r.j0 = r.su = r.sv = r.wp = -1;
    bool ok = quantise_axis(u, qp, &r.i0, &r.su);
    ok = quantise_axis(v, qp, &r.j0, &r.sv) && ok;
    const float aw = fabsf(w);
    ok = ok && (aw <= 3.402823466e38f);                          // finite w (false for NaN)
    // floor(|w|) clamped to the last plane (R5); comparison in float is exact for these integers
    const int wp = (aw >= (float)(qp.n_wplanes - 1)) ? (qp.n_wplanes - 1) : (int)aw;
    r.wp = wp;
    r.valid = ok;
    return r;
}

__device__ __forceinline__ CycRec make_cyc_record(const QuantOut& q, const QuantParams& qp) {
    CycRec rec;
    int i0 = q.i0, j0 = q.j0;
    uint32_t ru = (uint32_t)(q.wp * qp.oversample + q.su), rv = (uint32_t)(q.wp * qp.oversample + q.sv);
    if (qp.pad) {
        // support padded to a power of two with zero taps: row copy 0 has the zeros behind the taps (origin
        // unchanged), copy 1 in front (origin moved down), used where the padded footprint would leave the grid
        const uint32_t bu = i0 + qp.sk > qp.grid_size ? 1u : 0u, bv = j0 + qp.sk > qp.grid_size ? 1u : 0u;
        i0 -= bu ? qp.pad : 0;
        j0 -= bv ? qp.pad : 0;
        ru = 2u * ru + bu;
        rv = 2u * rv + bv;
    }
    rec.pos = (uint32_t)i0 | ((uint32_t)j0 << 16) | (q.valid ? 0u : 0x8000u);
    rec.rows = ru | (rv << 16);
    return rec;
}

__device__ __forceinline__ SampleRec make_record(const QuantOut& q, const QuantParams& qp) {
    SampleRec rec;
    if (!q.valid) {
        rec.x = kInvalidRec; rec.y = 0; rec.z = 0; rec.w = 0;
        return rec;
    }
    const int X0 = (q.i0 / qp.cu) * qp.cu, Y0 = (q.j0 / qp.cv) * qp.cv;
    rec.x = (uint32_t)X0 | ((uint32_t)Y0 << 16);
    rec.y = (uint32_t)(X0 % qp.bin_u) | ((uint32_t)(Y0 % qp.bin_v) << 16);
    rec.z = (uint32_t)((q.wp * qp.oversample + q.su) * qp.row_u + (qp.cu - 1) - (q.i0 - X0));
    rec.w = (uint32_t)((q.wp * qp.oversample + q.sv) * qp.row_v + (qp.cv - 1) - (q.j0 - Y0));
    return rec;
}

// uvw is [n][3] float32.  Each thread handles 4 consecutive samples = three aligned float4 loads.
// It also measures, on every 64th block, how far consecutive samples move along the channel axis and
// along the time axis (layout hint: sample = (baseline*n_times + t)*n_chan + c), so that the gridding
// kernel can walk each chunk along the slower axis (hop_stats[0] channel, [1] time; capped per hop).
__global__ void __launch_bounds__(256)
quantise_kernel(const float* __restrict__ uvw, SampleRec* __restrict__ recs, long long n,
                QuantParams qp, float* __restrict__ hop_stats, int n_chan, int n_times, float hop_cap,
                const float* __restrict__ weights = nullptr) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long first = g * 4;
    if (n_chan > 0 && (blockIdx.x & 63) == 0) {
        float hc = 0.f, ht = 0.f;
        if (first < n) {
            const long long row = first / n_chan;
            const int col = (int)(first - row * n_chan);
            const int t = (int)(row % n_times);
            const float u = __ldg(uvw + 3 * first), v = __ldg(uvw + 3 * first + 1);
            if (col + 1 < n_chan)
                hc = fminf(fabsf(__ldg(uvw + 3 * (first + 1)) - u) + fabsf(__ldg(uvw + 3 * (first + 1) + 1) - v), hop_cap);
            if (t + 1 < n_times)
                ht = fminf(fabsf(__ldg(uvw + 3 * (first + n_chan)) - u) + fabsf(__ldg(uvw + 3 * (first + n_chan) + 1) - v), hop_cap);
            if (!(hc == hc)) hc = 0.f;           // NaN coordinates carry no information
            if (!(ht == ht)) ht = 0.f;
        }
        for (int o = 16; o > 0; o >>= 1) {
            hc += __shfl_xor_sync(0xffffffffu, hc, o);
            ht += __shfl_xor_sync(0xffffffffu, ht, o);
        }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(hop_stats, hc);
            atomicAdd(hop_stats + 1, ht);
        }
    }
    if (first >= n) return;
    float c[12];
    if (first + 4 <= n) {
        const float4* p = reinterpret_cast<const float4*>(uvw + first * 3);
        const float4 a = __ldg(p), b = __ldg(p + 1), d = __ldg(p + 2);
        c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w; c[4] = b.x; c[5] = b.y; c[6] = b.z;
        c[7] = b.w; c[8] = d.x; c[9] = d.y; c[10] = d.z; c[11] = d.w;
    } else {
        for (int k = 0; k < 12; ++k) c[k] = (first * 3 + k < n * 3) ? __ldg(uvw + first * 3 + k) : 0.f;
    }
    if (qp.format == 2) {                            // the warp kernel's records: the weight travels with the sample
        float w[4] = {1.f, 1.f, 1.f, 1.f};
        if (weights) {
            if (first + 4 <= n) {
                const float4 w4 = __ldg(reinterpret_cast<const float4*>(weights + first));
                w[0] = w4.x; w[1] = w4.y; w[2] = w4.z; w[3] = w4.w;
            } else {
                for (int k = 0; k < 4; ++k) if (first + k < n) w[k] = __ldg(weights + first + k);
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (first + k < n) {
                const CycRec r = make_cyc_record(quantise_sample(c[3 * k], c[3 * k + 1], c[3 * k + 2], qp), qp);
                recs[first + k] = make_uint4(r.pos, r.rows, __float_as_uint(w[k]), 0u);
            }
        }
        return;
    }
    if (qp.format == 1 && first + 4 <= n) {          // four 8-byte records = two 16-byte stores
        CycRec r[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) r[k] = make_cyc_record(quantise_sample(c[3 * k], c[3 * k + 1], c[3 * k + 2], qp), qp);
        uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<CycRec*>(recs) + first);
        dst[0] = make_uint4(r[0].pos, r[0].rows, r[1].pos, r[1].rows);
        dst[1] = make_uint4(r[2].pos, r[2].rows, r[3].pos, r[3].rows);
        return;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (first + k < n) {
            const QuantOut q = quantise_sample(c[3 * k], c[3 * k + 1], c[3 * k + 2], qp);
            if (qp.format == 0) recs[first + k] = make_record(q, qp);
            else reinterpret_cast<CycRec*>(recs)[first + k] = make_cyc_record(q, qp);
        }
    }
}

// Unpacked form for inspection / parity tests (grid_quantise): out[n][6].
__global__ void __launch_bounds__(256)
quantise_debug_kernel(const float* __restrict__ uvw, int* __restrict__ out, long long n, QuantParams qp) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
    const QuantOut q = quantise_sample(uvw[3 * g], uvw[3 * g + 1], uvw[3 * g + 2], qp);
    int* o = out + 6 * g;
    const int m = q.valid ? 0 : -1;               // skipped samples report -1 (their clamped walk
    o[0] = q.i0 | m; o[1] = q.j0 | m; o[2] = q.su | m; o[3] = q.sv | m; o[4] = q.wp | m;   // coordinates are internal)
    o[5] = q.valid ? 1 : 0;
}

}  // namespace gridb200
