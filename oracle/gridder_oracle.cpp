// TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT PATH.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code with paper_1605_07023_b200/csrc/.
//
// Plain float64 CPU convolutional gridder written from the paper's definition:
//   "each visibility sample is treated as a Dirac delta, convolved with some function, and then
//    sampled onto the grid"                                   (section 2.2)
//   GCF read from a precomputed, oversampled table            (section 2.2)
//   selected per sample by "the integer grid coordinates, the sub-grid coordinates for indexing
//   the GCF, the w plane index", values "pre-weighted"        (section 4)
//   separable GCF  G_ij = G^u_i G^v_j, polarisation-independent
// The readings of everything the paper leaves open (quantiser Q, plane selection W, layouts,
// edge handling) are DESIGN.md "Readings" R1-R24 == SURVEY.md 8(c) A1-A24.
//
// Pins (tests/test_oracle_pins.py): P1-P16 of DESIGN.md.  "Parity unpinned": the physical tap
// positions inside the table (which distance each k[.][su][t] represents) -- the paper gives no
// formula or worked example; only the synthetic table generator depends on it.
//
// Parallelism: OpenMP over interleaved grid rows.  Thread r of R applies only the taps whose grid
// row j has (j - row_lo) mod R == r, scanning the samples in input order, so every cell receives its contributions in input
// order for any thread count: the result is bit-identical for 1 or many threads (pin P15), no atomics.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;

namespace {

struct Quant { int64_t i0, j0; int su, sv, wp; bool valid; };

// Q(x): R4 (refines SURVEY A4; identical to it whenever O*S is even, i.e. for every config).
//   pos = floor(double(x)*O + (O*floor(N/2) + 0.5))   position in 1/O cells, nearest, half up;
//                                                      binary64: product exact, one rounding in the
//                                                      add, which never crosses an integer
//   q   = pos + O - ceil(O*S/2)                        integer
//   (cell, row) = (q div O, q mod O)                   floor division
// so the S cells are those at distance d in (-S/2, S/2] of the rounded position and tap t of row
// `row` lies at d = t - S/2 + 1 - row/O (R8, R24).
inline bool quant_axis(float x, int N, int S, int O, int64_t* cell, int* sub) {
    const double cN = (double)O * (double)(N / 2) + 0.5;
    const double pos = std::floor((double)x * (double)O + cN);
    const double q = pos + (double)(O - (O * S + 1) / 2);
    // valid footprints have 0 <= cell and cell + S <= N  <=>  0 <= q < (N-S+1)*O   (R7/A7)
    if (!(q >= 0.0) || !(q < (double)(N - S + 1) * (double)O)) return false;   // also rejects NaN
    const int64_t qi = (int64_t)q;
    *cell = qi / O;               // qi >= 0: truncation == floor
    *sub = (int)(qi % O);
    return true;
}

// W(w): R5/A5.  min(int(floor(|w|)), n_wplanes-1)
inline bool quant_w(float w, int n_wplanes, int* wp) {
    if (!std::isfinite(w)) return false;
    const double a = std::floor(std::fabs((double)w));
    *wp = (a >= (double)(n_wplanes - 1)) ? (n_wplanes - 1) : (int)a;
    return true;
}

inline Quant quantise(const float* uvw, int N, int S, int O, int n_wplanes) {
    Quant r{};
    r.valid = std::isfinite(uvw[0]) && std::isfinite(uvw[1]) && std::isfinite(uvw[2]);
    if (r.valid) r.valid = quant_axis(uvw[0], N, S, O, &r.i0, &r.su);
    if (r.valid) r.valid = quant_axis(uvw[1], N, S, O, &r.j0, &r.sv);
    if (r.valid) r.valid = quant_w(uvw[2], n_wplanes, &r.wp);
    return r;
}

inline bool bad_args(int N, int S, int O, int W, int P) {
    return N < 1 || S < 1 || S > N || O < 1 || W < 1 || P < 1;
}

}  // namespace

extern "C" {

// Per-sample integer outputs of Q and W (all int32; invalid samples get valid=0, others -1).
int oracle_quantise(int N, int S, int O, int n_wplanes, long long n_vis, const float* uvw,
                    int32_t* i0, int32_t* j0, int32_t* su, int32_t* sv, int32_t* wp, uint8_t* valid) {
    if (bad_args(N, S, O, n_wplanes, 1)) return -1;
    for (long long n = 0; n < n_vis; ++n) {
        Quant q = quantise(uvw + 3 * n, N, S, O, n_wplanes);
        valid[n] = q.valid ? 1 : 0;
        i0[n] = q.valid ? (int32_t)q.i0 : -1;
        j0[n] = q.valid ? (int32_t)q.j0 : -1;
        su[n] = q.valid ? q.su : -1;
        sv[n] = q.valid ? q.sv : -1;
        wp[n] = q.valid ? q.wp : -1;
    }
    return 0;
}

// grid[(j-row_lo)][i][p] (complex128, interleaved re/im) += contributions of all samples, for the
// rows row_lo <= j < row_hi only.  row_lo=0,row_hi=N gives the whole grid.  Returns #valid samples
// through *n_valid (may be null).
//   for n in input order:  (i0,su)=Q(u) (j0,sv)=Q(v) wp=W(w); skip unless the footprint is inside
//     for tj, ti, p:  grid[j0+tj][i0+ti][p] += weight_n * vis[n][p] * k[wp][sv][tj] * k[wp][su][ti]
int oracle_grid(int N, int S, int O, int n_wplanes, int P, long long n_vis,
                const float* uvw, const float* vis, const float* weights, const float* kernel,
                double* grid, int row_lo, int row_hi, int n_threads, long long* n_valid) {
    if (bad_args(N, S, O, n_wplanes, P) || row_lo < 0 || row_hi > N || row_lo > row_hi) return -1;
    const int rows = row_hi - row_lo;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = omp_get_max_threads();
#else
    n_threads = 1;
#endif
    if (n_threads > rows) n_threads = rows > 0 ? rows : 1;
    long long valid_count = 0;
    for (long long n = 0; n < n_vis; ++n)
        valid_count += quantise(uvw + 3 * n, N, S, O, n_wplanes).valid ? 1 : 0;
    if (n_valid) *n_valid = valid_count;
    if (rows == 0) return 0;
    cd* g = reinterpret_cast<cd*>(grid);
#pragma omp parallel num_threads(n_threads)
    {
#ifdef _OPENMP
        const int r = omp_get_thread_num(), R = omp_get_num_threads();
#else
        const int r = 0, R = 1;
#endif
        std::vector<cd> wv(P);
        for (long long n = 0; n < n_vis; ++n) {
            const Quant q = quantise(uvw + 3 * n, N, S, O, n_wplanes);
            if (!q.valid) continue;
            if (q.j0 + S <= row_lo || q.j0 >= row_hi) continue;
            const double wt = (double)weights[n];
            for (int p = 0; p < P; ++p)
                wv[p] = wt * cd((double)vis[2 * (n * P + p)], (double)vis[2 * (n * P + p) + 1]);
            const float* ku = kernel + 2 * (((size_t)q.wp * O + q.su) * S);
            const float* kv = kernel + 2 * (((size_t)q.wp * O + q.sv) * S);
            for (int tj = 0; tj < S; ++tj) {
                const int64_t j = q.j0 + tj;
                if (j < row_lo || j >= row_hi || (int)((j - row_lo) % R) != r) continue;   // not my row
                const cd gv((double)kv[2 * tj], (double)kv[2 * tj + 1]);
                for (int ti = 0; ti < S; ++ti) {
                    const cd gu((double)ku[2 * ti], (double)ku[2 * ti + 1]);
                    const cd gij = gv * gu;
                    cd* cell = g + ((size_t)(j - row_lo) * N + (size_t)(q.i0 + ti)) * P;
                    for (int p = 0; p < P; ++p) cell[p] += wv[p] * gij;
                }
            }
        }
    }
    return 0;
}

// Dense (non-separable) GCF, SURVEY NEXT-4 ("non-separable GCFs", 186): the same scatter with a
// full S x S table per (w-plane, v sub-offset, u sub-offset):
//   kernel2d[wp][sv][su][tj][ti] complex64;  grid[j0+tj][i0+ti][p] += weight_n * vis[n][p] * kernel2d[wp][sv][su][tj][ti]
// Serial, whole grid (complex128 [N][N][P]); small cases only.
int oracle_grid_dense(int N, int S, int O, int n_wplanes, int P, long long n_vis,
                      const float* uvw, const float* vis, const float* weights, const float* kernel2d, double* grid) {
    if (bad_args(N, S, O, n_wplanes, P)) return -1;
    cd* g = reinterpret_cast<cd*>(grid);
    for (long long n = 0; n < n_vis; ++n) {
        const Quant q = quantise(uvw + 3 * n, N, S, O, n_wplanes);
        if (!q.valid) continue;
        const double wt = (double)weights[n];
        const float* k = kernel2d + 2 * ((((size_t)q.wp * O + q.sv) * O + q.su) * S * S);
        for (int tj = 0; tj < S; ++tj)
            for (int ti = 0; ti < S; ++ti) {
                const cd gij((double)k[2 * (tj * S + ti)], (double)k[2 * (tj * S + ti) + 1]);
                cd* cell = g + ((size_t)(q.j0 + tj) * N + (size_t)(q.i0 + ti)) * P;
                for (int p = 0; p < P; ++p)
                    cell[p] += wt * cd((double)vis[2 * (n * P + p)], (double)vis[2 * (n * P + p) + 1]) * gij;
            }
    }
    return 0;
}

// Dense GCF per polarisation, SURVEY NEXT-4 remainder (the coarsened kernel "assumed that the GCF is
// polarization-independent ... cannot be directly applied to A-projection"; GCFs "dependent on time,
// frequency, polarization"): the same scatter with one full table per polarisation,
//   kernel2d[p][wp][sv][su][tj][ti] complex64;  grid[j0+tj][i0+ti][p] += weight_n * vis[n][p] * kernel2d[p][wp][sv][su][tj][ti]
// Serial, whole grid (complex128 [N][N][P]); small cases only.
int oracle_grid_dense_pol(int N, int S, int O, int n_wplanes, int P, long long n_vis,
                          const float* uvw, const float* vis, const float* weights, const float* kernel2d, double* grid) {
    if (bad_args(N, S, O, n_wplanes, P)) return -1;
    cd* g = reinterpret_cast<cd*>(grid);
    const size_t per_pol = (size_t)n_wplanes * O * O * S * S;
    for (long long n = 0; n < n_vis; ++n) {
        const Quant q = quantise(uvw + 3 * n, N, S, O, n_wplanes);
        if (!q.valid) continue;
        const double wt = (double)weights[n];
        const size_t entry = (((size_t)q.wp * O + q.sv) * O + q.su) * S * S;
        for (int p = 0; p < P; ++p) {
            const float* k = kernel2d + 2 * ((size_t)p * per_pol + entry);
            const cd v((double)vis[2 * (n * P + p)], (double)vis[2 * (n * P + p) + 1]);
            for (int tj = 0; tj < S; ++tj)
                for (int ti = 0; ti < S; ++ti) {
                    const cd gij((double)k[2 * (tj * S + ti)], (double)k[2 * (tj * S + ti) + 1]);
                    g[((size_t)(q.j0 + tj) * N + (size_t)(q.i0 + ti)) * P + p] += wt * v * gij;
                }
        }
    }
    return 0;
}

// Adjoint (degridding), written solely for pin P7 (north_star property 5):
//   out[n][p] = weight_n * sum_{tj,ti} conj(k[wp][sv][tj] * k[wp][su][ti]) * G[j0+tj][i0+ti][p]
// Invalid samples give 0.  grid is a full [N][N][P] complex128 array; out is complex128 [n_vis][P].
int oracle_degrid(int N, int S, int O, int n_wplanes, int P, long long n_vis,
                  const float* uvw, const float* weights, const float* kernel,
                  const double* grid, double* out) {
    if (bad_args(N, S, O, n_wplanes, P)) return -1;
    const cd* g = reinterpret_cast<const cd*>(grid);
    cd* o = reinterpret_cast<cd*>(out);
    for (long long n = 0; n < n_vis; ++n) {
        for (int p = 0; p < P; ++p) o[n * P + p] = cd(0.0, 0.0);
        const Quant q = quantise(uvw + 3 * n, N, S, O, n_wplanes);
        if (!q.valid) continue;
        const float* ku = kernel + 2 * (((size_t)q.wp * O + q.su) * S);
        const float* kv = kernel + 2 * (((size_t)q.wp * O + q.sv) * S);
        for (int tj = 0; tj < S; ++tj) {
            const cd gv((double)kv[2 * tj], (double)kv[2 * tj + 1]);
            for (int ti = 0; ti < S; ++ti) {
                const cd gu((double)ku[2 * ti], (double)ku[2 * ti + 1]);
                const cd c = std::conj(gv * gu);
                const cd* cell = g + ((size_t)(q.j0 + tj) * N + (size_t)(q.i0 + ti)) * P;
                for (int p = 0; p < P; ++p) o[n * P + p] += c * cell[p];
            }
        }
        for (int p = 0; p < P; ++p) o[n * P + p] *= (double)weights[n];
    }
    return 0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
