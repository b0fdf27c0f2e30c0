// rick_oracle.cpp -- CPU ORACLE for the w-stacking hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, fp64 restatement of what librick_b200 computes, written from the paper
// (/root/reference/PAPER.md, cited as P:<line>) and from the readings D1-D9 of SURVEY.md section 8(c)
// (restated in DESIGN.md "Readings").  It shares no code, header, table or constant with the CUDA
// path under paper_2411_07321_b200/csrc/ and neither includes the other.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// The method is an approximation (nearest-plane w-stacking; truncated-kernel convolutional
// gridding, Eq. 3; FFT per plane; phase screen and plane sum, Eq. 2), so the oracle
// follows the algorithm step by step in that order.  There is no blocking, fusion or reordering: the
// only parallelism is an OpenMP loop over independent output rows, which leaves every sum in the
// same order as the serial loop (results do not depend on the thread count).
//
// Pins (tests/test_oracle_*.py, all CPU): hand-computed keys; grid-sum and centre-pixel invariants;
// own radix-2 FFT against the literal double sum of D7; closed forms for a phase-centre and an
// on-pixel source; brute-force direct DFT of the visibilities (rick_oracle_direct_dft) on tiny
// inputs; linearity; Hermitian symmetry; input-order invariance.
// Parity unpinned: anything about real LOFAR images (no data in the container).
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC rick_oracle.cpp -o librick_oracle.so

#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cplx;
const double kPi = 3.14159265358979323846264338327950288;

// Gridding kernel family, selected process-wide by rick_oracle_set_kernel (the Python front end sets it
// from the Plan before every call):  0 = truncated Gaussian (BASELINE.json north_star; D6),
// 1 = Kaiser-Bessel (the kernel of the paper's own tests; D6-KB of DESIGN.md).
int g_kernel_kind = 0;
double g_kernel_beta = 0.0;

// Modified Bessel function of the first kind, order 0, by its power series
//   I0(x) = sum_k (x^2 / 4)^k / (k!)^2      (all terms positive: no cancellation)
double bessel_i0(double x) {
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

struct Geometry {
    int N, Nw, S, h;
    int kernel;      // 0 Gaussian, 1 Kaiser-Bessel
    double beta, i0_beta;   // KB shape parameter and I0(beta)
    double sigma, w_min, w_max, dl;
    double s;        // D2: (double)N * dl, one rounded multiply
    double inv_dw;   // D3: (double)Nw / (w_max - w_min)
    int T;           // D4: tiles per axis, N / 32
};

Geometry make_geometry(int N, int Nw, int S, double sigma, double w_min, double w_max, double dl) {
    Geometry g;
    g.N = N; g.Nw = Nw; g.S = S; g.h = (S - 1) / 2;
    g.sigma = sigma; g.w_min = w_min; g.w_max = w_max; g.dl = dl;
    g.kernel = g_kernel_kind; g.beta = g_kernel_beta;
    g.i0_beta = g.kernel == 1 ? bessel_i0(g.beta) : 1.0;
    g.s = (double)N * dl;
    g.inv_dw = (double)Nw / (w_max - w_min);
    g.T = N / 32;
    return g;
}

// D2 + D3 + D5: nearest cell, nearest plane, keep/drop.  Returns false when the visibility is dropped.
// P:53 "visibilities are mapped to the closest w-plane"; planes are centred in Nw equal sub-intervals
// of [w_min, w_max] (D3).  Whole-drop at the mesh edge and outside the w range (D5).
bool locate(const Geometry& g, float u, float v, float w, float vre, float vim, float wt,
            double* x_out, double* y_out, long* i0_out, long* j0_out, long* k_out) {
    if (!std::isfinite(u) || !std::isfinite(v) || !std::isfinite(w) || !std::isfinite(vre) ||
        !std::isfinite(vim) || !std::isfinite(wt))
        return false;
    const double half = (double)(g.N / 2);
    const double x = std::fma((double)u, g.s, half);
    const double y = std::fma((double)v, g.s, half);
    const double xr = std::floor(x + 0.5);
    const double yr = std::floor(y + 0.5);
    // the comparisons are done on the (exact, integer-valued) doubles so that no out-of-range cast occurs
    if (xr < (double)g.h || xr > (double)(g.N - 1 - g.h)) return false;
    if (yr < (double)g.h || yr > (double)(g.N - 1 - g.h)) return false;
    const double t = ((double)w - g.w_min) * g.inv_dw;
    double kf = std::floor(t);
    if (kf >= (double)g.Nw && (double)w <= g.w_max) kf = (double)(g.Nw - 1);
    if (kf < 0.0 || kf >= (double)g.Nw) return false;
    *x_out = x; *y_out = y;
    *i0_out = (long)xr; *j0_out = (long)yr; *k_out = (long)kf;
    return true;
}

// D6 tap.  Gaussian: g(d) = exp(-d^2 / 2 sigma^2), un-normalised, sigma in cells.
// D6-KB: g(d) = I0(beta sqrt(1 - (d / a_t)^2)) / I0(beta) for |d| <= a_t = h + 1/2 (the footprint offsets
// satisfy -a_t < d <= a_t), the Kaiser-Bessel window of full width 2 a_t = S cells.
inline double tap(double d, const Geometry& g) {
    if (g.kernel == 1) {
        const double a_t = (double)g.h + 0.5;
        const double r = d / a_t;
        const double arg = 1.0 - r * r;
        return bessel_i0(g.beta * std::sqrt(arg > 0.0 ? arg : 0.0)) / g.i0_beta;
    }
    return std::exp(-(d * d) / (2.0 * g.sigma * g.sigma));
}

// ---- own radix-2 FFT (sign +, unnormalised), used for D7 -------------------------------------
void fft1d_inverse(cplx* a, int n) {
    // bit reversal
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        const int half = len >> 1;
        for (int i = 0; i < n; i += len) {
            for (int j = 0; j < half; ++j) {
                const double ang = 2.0 * kPi * (double)j / (double)len;   // sign + (Eq. 2)
                const cplx wv(std::cos(ang), std::sin(ang));
                const cplx x = a[i + j];
                const cplx y = a[i + j + half] * wv;
                a[i + j] = x + y;
                a[i + j + half] = x - y;
            }
        }
    }
}

// D7: P[q][p] = sum_{j,i} G[j][i] exp(+2 pi i ((i-N/2)(p-N/2) + (j-N/2)(q-N/2)) / N), in place.
// Centred indices are handled with the checkerboard identity (N even):
//   P[q][p] = (-1)^(p+q) * IFFT2[(-1)^(i+j) G][q][p].
void plane_transform(cplx* plane, int N) {
#pragma omp parallel for schedule(static)
    for (int j = 0; j < N; ++j) {
        cplx* row = plane + (size_t)j * N;
        for (int i = 0; i < N; ++i)
            if ((i + j) & 1) row[i] = -row[i];
        fft1d_inverse(row, N);
    }
#pragma omp parallel
    {
        std::vector<cplx> col(N);
#pragma omp for schedule(static)
        for (int p = 0; p < N; ++p) {
            for (int j = 0; j < N; ++j) col[j] = plane[(size_t)j * N + p];
            fft1d_inverse(col.data(), N);
            for (int q = 0; q < N; ++q) plane[(size_t)q * N + p] = ((p + q) & 1) ? -col[q] : col[q];
        }
    }
}

// D8: n - 1 = -(l^2 + m^2) / (1 + sqrt(1 - l^2 - m^2))
inline double nm1_of(double l, double m) {
    const double r2 = l * l + m * m;
    return -r2 / (1.0 + std::sqrt(1.0 - r2));
}

// D8 1-D taper table: t[p] = c0 exp(-2 pi^2 sigma^2 nu_p^2), nu_p = (p - N/2)/N,
// c0 = sigma sqrt(2 pi) erf(a_t / (sigma sqrt 2)), a_t = h + 1/2 (integral of the truncated kernel).
// D8-KB: the exact transform of the compactly supported Kaiser-Bessel window,
//   t(nu) = int_{-a_t}^{a_t} g(d) e^{-2 pi i nu d} dd = (2 a_t / I0(beta)) sinh(z) / z,  z = sqrt(beta^2 - (2 pi a_t nu)^2)
// (sin(z') / z' with z' = sqrt((2 pi a_t nu)^2 - beta^2) beyond the main lobe; 1 at z = 0).
void taper_table(const Geometry& g, double* t) {
    const double a_t = (double)g.h + 0.5;
    if (g.kernel == 1) {
        for (int p = 0; p < g.N; ++p) {
            const double nu = (double)(p - g.N / 2) / (double)g.N;
            const double y = 2.0 * kPi * a_t * nu;
            const double z2 = g.beta * g.beta - y * y;
            double sc;
            if (z2 > 1e-24) { const double z = std::sqrt(z2); sc = std::sinh(z) / z; }
            else if (z2 < -1e-24) { const double z = std::sqrt(-z2); sc = std::sin(z) / z; }
            else sc = 1.0;
            t[p] = 2.0 * a_t * sc / g.i0_beta;
        }
        return;
    }
    const double c0 = g.sigma * std::sqrt(2.0 * kPi) * std::erf(a_t / (g.sigma * std::sqrt(2.0)));
    for (int p = 0; p < g.N; ++p) {
        const double nu = (double)(p - g.N / 2) / (double)g.N;
        t[p] = c0 * std::exp(-2.0 * kPi * kPi * g.sigma * g.sigma * nu * nu);
    }
}

// D6 for one plane: grid[j][i] += (wt V) g(i - x) g(j - y) over the S x S footprint of every kept
// visibility of plane k (Eq. 3).  `list` holds that plane's visibilities in input order.
// Rows are distributed over threads; each cell still receives its terms in input order.
void grid_plane(const Geometry& g, const std::vector<uint32_t>& list, const float* u, const float* v,
                const float* vis, const float* wt, cplx* plane) {
    const int N = g.N, h = g.h;
    const int RB = 8;   // rows per work item
#pragma omp parallel for schedule(dynamic, 1)
    for (int jb = 0; jb < N; jb += RB) {
        const int j_lo = jb, j_hi = std::min(N, jb + RB);   // [j_lo, j_hi)
        for (size_t n = 0; n < list.size(); ++n) {
            const uint32_t m = list[n];
            const double half = (double)(N / 2);
            const double y = std::fma((double)v[m], g.s, half);
            const long j0 = (long)std::floor(y + 0.5);
            if (j0 + h < j_lo || j0 - h >= j_hi) continue;
            const double x = std::fma((double)u[m], g.s, half);
            const long i0 = (long)std::floor(x + 0.5);
            const cplx val((double)wt[m] * (double)vis[2 * m], (double)wt[m] * (double)vis[2 * m + 1]);
            for (int b = -h; b <= h; ++b) {
                const long j = j0 + b;
                if (j < j_lo || j >= j_hi) continue;
                const double gy = tap((double)j - y, g);
                for (int a = -h; a <= h; ++a) {
                    const long i = i0 + a;
                    const double gx = tap((double)i - x, g);
                    plane[(size_t)j * N + i] += val * (gx * gy);
                }
            }
        }
    }
}

// D8 for one plane: acc[q][p] += Re{ exp(+2 pi i frac(w_k nm1)) P_k[q][p] }   (Eq. 2)
void wcorrect_plane(const Geometry& g, int k, const cplx* plane, double* acc) {
    const int N = g.N;
    const double wk = g.w_min + ((double)k + 0.5) * (g.w_max - g.w_min) / (double)g.Nw;
#pragma omp parallel for schedule(static)
    for (int q = 0; q < N; ++q) {
        const double m = (double)(q - N / 2) * g.dl;
        for (int p = 0; p < N; ++p) {
            const double l = (double)(p - N / 2) * g.dl;
            const double t = wk * nm1_of(l, m);
            const double phi = 2.0 * kPi * (t - std::floor(t));
            const cplx scr(std::cos(phi), std::sin(phi));
            acc[(size_t)q * N + p] += (scr * plane[(size_t)q * N + p]).real();
        }
    }
}

double seconds_since(std::chrono::steady_clock::time_point t0) {
    return std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
}

}  // namespace

extern "C" {

int rick_oracle_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Select the gridding kernel used by every later call: kind 0 Gaussian (sigma of each call), kind 1
// Kaiser-Bessel with shape parameter beta (sigma is then ignored).
void rick_oracle_set_kernel(int kind, double beta) {
    g_kernel_kind = kind == 1 ? 1 : 0;
    g_kernel_beta = beta;
}

double rick_oracle_bessel_i0(double x) { return bessel_i0(x); }

void rick_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// D2-D5.  key[m] = (k T + (j0 >> 5)) T + (i0 >> 5), sentinel Nw T^2 for dropped visibilities.
// i0/j0/k (nullable) receive the nearest cell and plane, -1 for dropped.  Returns n_kept.
long long rick_oracle_keys(int N, int Nw, int S, double w_min, double w_max, double dl, long long M,
                           const float* u, const float* v, const float* w, const float* vis,
                           const float* wt, uint32_t* key, int32_t* i0_out, int32_t* j0_out,
                           int32_t* k_out) {
    const Geometry g = make_geometry(N, Nw, S, 1.0, w_min, w_max, dl);
    const uint32_t sentinel = (uint32_t)Nw * (uint32_t)g.T * (uint32_t)g.T;
    long long kept = 0;
#pragma omp parallel for schedule(static) reduction(+ : kept)
    for (long long m = 0; m < M; ++m) {
        double x, y;
        long i0, j0, k;
        if (locate(g, u[m], v[m], w[m], vis[2 * m], vis[2 * m + 1], wt[m], &x, &y, &i0, &j0, &k)) {
            key[m] = (uint32_t)((k * g.T + (j0 >> 5)) * g.T + (i0 >> 5));
            if (i0_out) i0_out[m] = (int32_t)i0;
            if (j0_out) j0_out[m] = (int32_t)j0;
            if (k_out) k_out[m] = (int32_t)k;
            ++kept;
        } else {
            key[m] = sentinel;
            if (i0_out) i0_out[m] = -1;
            if (j0_out) j0_out[m] = -1;
            if (k_out) k_out[m] = -1;
        }
    }
    return kept;
}

// D4': the order rick_bin leaves the visibilities in.  BASELINE.json north_star (2) asks
// for a sort by (w-plane, 32x32 uv tile); D4' refines it so that visibilities sharing a nearest cell are
// adjacent: kept visibilities first, ordered by
//     w-plane k,  tile row j0 / 32,  tile column i0 / 32,  row inside the tile j0 % 32,
//     column inside the tile (i0 % 32) / 2^col_drop,  input index (the sort is stable);
// dropped visibilities (k < 0) follow, in input order.  col_drop = 0 (the exact cell) for every plan with
// Nw (N/32)^2 <= 2^22, which covers the five configurations; larger plans report their col_drop.
// i0 / j0 / k are the outputs of rick_oracle_keys.  perm[r] = input index of the visibility at rank r.
void rick_oracle_sort_cells(long long M, const int32_t* i0, const int32_t* j0, const int32_t* k, int col_drop,
                            uint32_t* perm) {
    std::iota(perm, perm + M, (uint32_t)0);
    std::stable_sort(perm, perm + M, [=](uint32_t a, uint32_t b) {
        const bool da = k[a] < 0, db = k[b] < 0;
        if (da || db) return !da && db;                      // kept before dropped; dropped stay in input order
        if (k[a] != k[b]) return k[a] < k[b];
        if (j0[a] / 32 != j0[b] / 32) return j0[a] / 32 < j0[b] / 32;
        if (i0[a] / 32 != i0[b] / 32) return i0[a] / 32 < i0[b] / 32;
        if (j0[a] % 32 != j0[b] % 32) return j0[a] % 32 < j0[b] % 32;
        const int ca = (i0[a] % 32) >> col_drop, cb = (i0[b] % 32) >> col_drop;
        return ca < cb;
    });
}

// D4: the stable order (tile key, input index).  perm[r] = input index of the visibility at sorted rank r.
void rick_oracle_sort(long long M, const uint32_t* key, uint32_t* perm) {
    std::iota(perm, perm + M, (uint32_t)0);
    std::stable_sort(perm, perm + M, [key](uint32_t a, uint32_t b) { return key[a] < key[b]; });
}

// The same order by a counting sort written out (pins rick_oracle_sort in the tests), plus the bin
// offsets: bin_start[b] = number of visibilities with key < b, for b = 0 .. n_bins + 1
// (bin_start[n_bins] = n_kept, bin_start[n_bins + 1] = M); n_bins = Nw T^2 (the sentinel is bin n_bins).
void rick_oracle_counting_sort(long long M, const uint32_t* key, uint32_t n_bins, uint32_t* perm,
                               uint64_t* bin_start) {
    std::vector<uint64_t> count((size_t)n_bins + 2, 0);
    for (long long m = 0; m < M; ++m) count[(size_t)key[m] + 1]++;
    for (size_t b = 1; b < count.size(); ++b) count[b] += count[b - 1];
    if (bin_start) std::memcpy(bin_start, count.data(), count.size() * sizeof(uint64_t));
    if (perm) {
        std::vector<uint64_t> next(count.begin(), count.end() - 1);
        for (long long m = 0; m < M; ++m) perm[next[key[m]]++] = (uint32_t)m;
    }
}

// D6, whole mesh: grid[k][j][i] complex128 (interleaved re, im), zeroed here.
void rick_oracle_grid(int N, int Nw, int S, double sigma, double w_min, double w_max, double dl,
                      long long M, const float* u, const float* v, const float* w, const float* vis,
                      const float* wt, double* grid) {
    const Geometry g = make_geometry(N, Nw, S, sigma, w_min, w_max, dl);
    std::vector<std::vector<uint32_t>> lists(Nw);
    for (long long m = 0; m < M; ++m) {
        double x, y;
        long i0, j0, k;
        if (locate(g, u[m], v[m], w[m], vis[2 * m], vis[2 * m + 1], wt[m], &x, &y, &i0, &j0, &k))
            lists[k].push_back((uint32_t)m);
    }
    cplx* mesh = reinterpret_cast<cplx*>(grid);
    const size_t plane_cells = (size_t)N * N;
    std::fill(mesh, mesh + plane_cells * Nw, cplx(0.0, 0.0));
    for (int k = 0; k < Nw; ++k) grid_plane(g, lists[k], u, v, vis, wt, mesh + plane_cells * k);
}

// D7 on one N x N plane, in place (own radix-2 FFT; N a power of two).
void rick_oracle_plane_transform(int N, double* plane) {
    plane_transform(reinterpret_cast<cplx*>(plane), N);
}

// D7 written out literally (O(N^4)): the pin for rick_oracle_plane_transform at N = 16, 32.
void rick_oracle_plane_transform_literal(int N, const double* in, double* out) {
    const cplx* G = reinterpret_cast<const cplx*>(in);
    cplx* P = reinterpret_cast<cplx*>(out);
    const int c = N / 2;
    for (int q = 0; q < N; ++q)
        for (int p = 0; p < N; ++p) {
            cplx acc(0.0, 0.0);
            for (int j = 0; j < N; ++j)
                for (int i = 0; i < N; ++i) {
                    const long e = (long)(i - c) * (p - c) + (long)(j - c) * (q - c);
                    const double ang = 2.0 * kPi * (double)e / (double)N;
                    acc += G[(size_t)j * N + i] * cplx(std::cos(ang), std::sin(ang));
                }
            P[(size_t)q * N + p] = acc;
        }
}

void rick_oracle_taper(int N, int S, double sigma, double* t) {
    const Geometry g = make_geometry(N, 1, S, sigma, 0.0, 1.0, 1.0);
    taper_table(g, t);
}

double rick_oracle_nm1(double l, double m) { return nm1_of(l, m); }

double rick_oracle_plane_centre(int Nw, double w_min, double w_max, int k) {
    return w_min + ((double)k + 0.5) * (w_max - w_min) / (double)Nw;
}

// D8 on transformed planes P[k][q][p] (complex128): image[q][p] = acc / (t[p] t[q]).
void rick_oracle_wcorrect(int N, int Nw, int S, double sigma, double w_min, double w_max, double dl,
                          const double* planes, double* image) {
    const Geometry g = make_geometry(N, Nw, S, sigma, w_min, w_max, dl);
    const size_t plane_cells = (size_t)N * N;
    std::fill(image, image + plane_cells, 0.0);
    const cplx* P = reinterpret_cast<const cplx*>(planes);
    for (int k = 0; k < Nw; ++k) wcorrect_plane(g, k, P + plane_cells * k, image);
    std::vector<double> t(N);
    taper_table(g, t.data());
    for (int q = 0; q < N; ++q)
        for (int p = 0; p < N; ++p) image[(size_t)q * N + p] /= (t[p] * t[q]);
}

// The whole path, D2-D8, one plane at a time (memory O(N^2) + inputs):
//   keys -> per-plane lists (the "array per slab" of P:76) -> for each plane: grid (Eq. 3),
//   transform, phase screen + sum (Eq. 2) -> taper division.
// stage_seconds[4] (nullable): keys+bucketing, gridding, FFT, w-correction+taper.  Returns n_kept.
long long rick_oracle_image(int N, int Nw, int S, double sigma, double w_min, double w_max, double dl,
                            long long M, const float* u, const float* v, const float* w,
                            const float* vis, const float* wt, double* image, double* stage_seconds) {
    const Geometry g = make_geometry(N, Nw, S, sigma, w_min, w_max, dl);
    double t_key = 0, t_grid = 0, t_fft = 0, t_wc = 0;
    auto t0 = std::chrono::steady_clock::now();
    std::vector<std::vector<uint32_t>> lists(Nw);
    long long kept = 0;
    for (long long m = 0; m < M; ++m) {
        double x, y;
        long i0, j0, k;
        if (locate(g, u[m], v[m], w[m], vis[2 * m], vis[2 * m + 1], wt[m], &x, &y, &i0, &j0, &k)) {
            lists[k].push_back((uint32_t)m);
            ++kept;
        }
    }
    t_key = seconds_since(t0);
    const size_t plane_cells = (size_t)N * N;
    std::vector<cplx> plane(plane_cells);
    std::fill(image, image + plane_cells, 0.0);
    for (int k = 0; k < Nw; ++k) {
        t0 = std::chrono::steady_clock::now();
        std::fill(plane.begin(), plane.end(), cplx(0.0, 0.0));
        grid_plane(g, lists[k], u, v, vis, wt, plane.data());
        t_grid += seconds_since(t0);
        t0 = std::chrono::steady_clock::now();
        plane_transform(plane.data(), N);
        t_fft += seconds_since(t0);
        t0 = std::chrono::steady_clock::now();
        wcorrect_plane(g, k, plane.data(), image);
        t_wc += seconds_since(t0);
    }
    t0 = std::chrono::steady_clock::now();
    std::vector<double> t(N);
    taper_table(g, t.data());
    for (int q = 0; q < N; ++q)
        for (int p = 0; p < N; ++p) image[(size_t)q * N + p] /= (t[p] * t[q]);
    t_wc += seconds_since(t0);
    if (stage_seconds) {
        stage_seconds[0] = t_key; stage_seconds[1] = t_grid; stage_seconds[2] = t_fft; stage_seconds[3] = t_wc;
    }
    return kept;
}

// Ground truth for the oracle itself (tiny inputs only, O(N^2 M)): the exact dirty image
//   D*(l, m) = Re sum_kept wt V exp(+2 pi i (u l + v m + w (n - 1))),  n = sqrt(1 - l^2 - m^2)
// (adjoint of Eq. 1; D9: no 1/n factor, no normalisation), summed over the visibilities the
// drop rule D5 keeps, on the pixel grid of D1.
void rick_oracle_direct_dft(int N, int Nw, int S, double w_min, double w_max, double dl, long long M,
                            const float* u, const float* v, const float* w, const float* vis,
                            const float* wt, double* image) {
    const Geometry g = make_geometry(N, Nw, S, 1.0, w_min, w_max, dl);
    std::vector<uint32_t> kept;
    for (long long m = 0; m < M; ++m) {
        double x, y;
        long i0, j0, k;
        if (locate(g, u[m], v[m], w[m], vis[2 * m], vis[2 * m + 1], wt[m], &x, &y, &i0, &j0, &k))
            kept.push_back((uint32_t)m);
    }
#pragma omp parallel for schedule(static)
    for (int q = 0; q < N; ++q) {
        const double mm = (double)(q - N / 2) * dl;
        for (int p = 0; p < N; ++p) {
            const double l = (double)(p - N / 2) * dl;
            const double r2 = l * l + mm * mm;
            const double nm1 = std::sqrt(1.0 - r2) - 1.0;
            double acc = 0.0;
            for (uint32_t m : kept) {
                const double ph = 2.0 * kPi * ((double)u[m] * l + (double)v[m] * mm + (double)w[m] * nm1);
                const cplx val((double)wt[m] * (double)vis[2 * m], (double)wt[m] * (double)vis[2 * m + 1]);
                acc += (val * cplx(std::cos(ph), std::sin(ph))).real();
            }
            image[(size_t)q * N + p] = acc;
        }
    }
}

}  // extern "C"
