// Internal definitions shared by the translation units of librick_b200 (sm_100a only).
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include "rick_b200.h"

#define RICK_TILE 32          // uv tile edge of the sort key (BASELINE.json north_star (2))
#define RICK_MAX_PASSES 4
#define RICK_KB_POLY_TERMS 10
#define RICK_IMAGE_PARTS 4            // rick_image_from_host_chunked: image parts copied out while the next is computed
#define RICK_GREC_PAD 4096    // gridder records are allocated in whole chunks of this many (one CTA's share)
#define RICK_RADIX_BITS_MAX 9

// Geometry constants handed to kernels by value.
struct RickGeom {
    int N, Nw, S, h, T;
    double s;        // (double)N * dl                      [D2]
    double half;     // (double)(N/2)
    double w_min, w_max;
    double inv_dw;   // (double)Nw / (w_max - w_min)         [D3]
    double dl;
    double dw;       // (w_max - w_min) / Nw
    double sigma;
    uint32_t n_bins; // Nw * T * T, also the sentinel tile key [D4]
    int cell_bits;   // cb: in-tile cell bits appended to the tile key in the sort key [D4']
    uint32_t sort_sentinel;  // sort key of a dropped visibility: (n_bins << cb) - 1, a key D5 never keeps
    double tap_c;    // 1 / (2 sigma^2)
    // Kaiser-Bessel taps (rick_plan_set_kernel): tables over |d| in [0, a_t], kb_n intervals of a_t / kb_n
    int kernel;                 // RICK_KERNEL_GAUSS / RICK_KERNEL_KB
    int kb_n;
    double kb_inv_h;            // kb_n / a_t
    const float2* kb_lut_f;     // [kb_n + 1] (g_i, g_{i+1} - g_i): linear interpolation, fp32 mesh
    const double2* kb_lut_d;    // [kb_n + 1] (g_i, (a_t / kb_n) g'_i): cubic Hermite, fp64 mesh
};

struct rick_plan {
    RickGeom g;
    int dtype;
    bool dtype_set;
    // sort layout
    int key_bits, n_pass;
    int digit_bits[RICK_MAX_PASSES], digit_shift[RICK_MAX_PASSES];
    double kb_beta;
    void *kb_lut_f_dev, *kb_lut_d_dev;
    // per-tap polynomials of the Kaiser-Bessel window for the fp32 gridder: tap a of a visibility with
    // fractional offset delta in [-1/2, 1/2] is sum_k kb_poly[a][k] (2 delta)^k (fitted in fp64 at
    // rick_plan_set_kernel, used when the fit is good to 5e-8 of the peak: kb_poly_ok)
    float kb_poly[15][RICK_KB_POLY_TERMS];
    bool kb_poly_ok;
    // taper: inv_t[p] = 1 / t[p], device double[N]
    double* inv_taper_dev;
    // fused column transform + w-correction (colfft.cu), opt-in
    int fused;               // rick_plan_set_fusion: 0 off; 1: rick_fft_planes does rows only, K6 finishes;
                             // 2: in addition only the mesh rows some footprint touches are cleared / read
    // row occupancy (mode 2), plan-owned: bit (k N + j) of occ_cur = row j of plane k is touched by a
    // footprint of the visibilities of the last rick_bin; occ_mesh = rows of the mesh that hold defined data
    uint32_t *occ_cur_dev, *occ_mesh_dev;
    uint32_t* row_list_dev;  // [Nw N] rows to clear, built by rick_grid
    uint32_t* n_rows_dev;
    // segment occupancy (mode 2 with the library's own long-row kernel, rowbig.cu): a mesh row is 64 segments of
    // N / 64 cells; bit s of seg_cur[k N + j] = segment s of that row is touched by a footprint of the bound
    // visibilities, seg_mesh = it holds defined data, seg_fresh = it is cleared by the rick_grid in progress.
    // Only defined segments are cleared and read by the row transform (which writes whole rows).
    bool segs;
    unsigned long long *seg_cur_dev, *seg_mesh_dev, *seg_fresh_dev;
    cufftHandle fft_rows;    // batched 1-D row transforms
    bool fft_rows_ready;
    size_t fft_rows_work_bytes;
    void* colfft_tw;         // device float2[N]: exp(+2 pi i j / N)
    // split column transform (colsplit.cu): N = split_N1 * split_N2, engine selected by rick_plan_set_fusion
    bool split;              // fused != 0: true = sweeps A + B of colsplit.cu, false = the one-sweep kernel of colfft.cu
    int split_N1, split_N2;
    void* split_tw;          // device float2[N] / double2[N] (mesh precision): exp(+2 pi i j / N)
    // cuFFT
    cufftHandle fft;
    bool fft_ready;
    int fft_batch;           // planes per exec call
    size_t fft_work_bytes;
    // binding made by rick_bin
    bool bound;
    long long M;
    const float *u_s, *v_s, *w_s, *weight_s;
    const void* vis_s;
    const long long* n_kept_dev;
    // gridder records of the sorted kept visibilities, written by rick_bin's gather into its workspace:
    //   a = (i0 | j0 << 16, k), b = (i0 - x, j0 - y) in fp32, c = +-weight * (re, im)
    const uint2* grec_a;
    const float2 *grec_b, *grec_c;
    // indirect mode (rick_bin without sorted SoA outputs, fp32 mesh): sorted input indices and sort keys (kept
    // visibilities first) and the staging records in INPUT order, each holding the gridder record
    // ((i0 | j0 << 16, k, i0 - x, j0 - y), (+-weight re, +-weight im, -, -)); the gridder fetches them by index
    bool indirect;
    const uint32_t *gidx, *gkey;
    const float4* grec;
    // stage timing
    cudaEvent_t ev_start[RICK_T_COUNT], ev_stop[RICK_T_COUNT];
    // rick_image_from_host_chunked: copy stream and the events that hand the two staging halves back and forth
    cudaStream_t copy_stream;
    cudaEvent_t ev_copied[2], ev_consumed[2], ev_entry, ev_part[RICK_IMAGE_PARTS];
    bool pipe_ready;
    bool ev_valid[RICK_T_COUNT];
    long long launches;
    int sm_count;
    int device;              // CUDA device the plan was created on (kernel attributes are set per device)
};

#define RICK_MAX_DEVICES 64

#define RICK_CUDA(call)                                  \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return RICK_ECUDA;        \
    } while (0)

#define RICK_LAUNCH_CHECK()                              \
    do {                                                 \
        if (cudaGetLastError() != cudaSuccess) {         \
            return RICK_ECUDA;                           \
        }                                                \
    } while (0)

static inline size_t rick_align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---- device helpers --------------------------------------------------------------------------

// D2/D3/D5 with explicitly rounded fp64 operations (never contracted), so that the indices are
// bit-identical to any other correctly rounded evaluation of the same rules.
struct RickLoc {
    double x, y;
    int i0, j0, k;
    bool keep;
};

__device__ __forceinline__ bool rick_finite(float a) { return fabsf(a) <= 3.402823466e+38f; }

__device__ __forceinline__ RickLoc rick_locate(const RickGeom& g, float u, float v, float w) {
    RickLoc r;
    r.x = __fma_rn((double)u, g.s, g.half);
    r.y = __fma_rn((double)v, g.s, g.half);
    const double xr = floor(__dadd_rn(r.x, 0.5));
    const double yr = floor(__dadd_rn(r.y, 0.5));
    const double lo = (double)g.h, hi = (double)(g.N - 1 - g.h);
    const double t = __dmul_rn(__dsub_rn((double)w, g.w_min), g.inv_dw);
    double kf = floor(t);
    if (kf >= (double)g.Nw && (double)w <= g.w_max) kf = (double)(g.Nw - 1);
    r.keep = (xr >= lo) && (xr <= hi) && (yr >= lo) && (yr <= hi) && (kf >= 0.0) && (kf < (double)g.Nw);
    r.i0 = r.keep ? (int)xr : 0;
    r.j0 = r.keep ? (int)yr : 0;
    r.k = r.keep ? (int)kf : 0;
    return r;
}

// D4: tile key.  D4': sort key = tile key refined by the top cell_bits of the in-tile cell index
// (j0 & 31) << 5 | (i0 & 31), so that equal nearest cells become runs in the sorted order.
__device__ __forceinline__ uint32_t rick_tile_key(const RickGeom& g, const RickLoc& r) {
    return (uint32_t)((r.k * g.T + (r.j0 >> 5)) * g.T + (r.i0 >> 5));
}
__device__ __forceinline__ uint32_t rick_sort_key(const RickGeom& g, const RickLoc& r) {
    const uint32_t cell = (uint32_t)(((r.j0 & 31) << 5) | (r.i0 & 31));
    return (rick_tile_key(g, r) << g.cell_bits) | (cell >> (10 - g.cell_bits));
}
__device__ __forceinline__ uint32_t rick_tile_of_sort_key(const RickGeom& g, uint32_t sk) {
    return sk == g.sort_sentinel ? g.n_bins : (sk >> g.cell_bits);
}

// n - 1 = -(l^2 + m^2) / (1 + sqrt(1 - l^2 - m^2)) without the library's IEEE square root and division (two
// subroutine calls per output): fp32 seeds refined by two Newton steps each in fp64 (error < 2 ulp).  Used by the
// fp32-mesh column kernels, whose threads need 16 of these before their first plane.
__device__ __forceinline__ double rick_nm1_fast(double r2) {
    const double y = 1.0 - r2;
    double x = (double)rsqrtf((float)y);
    x = x * fma(-0.5 * y, x * x, 1.5);
    x = x * fma(-0.5 * y, x * x, 1.5);
    const double d = fma(y, x, 1.0);                     // 1 + sqrt(y)
    double r = (double)__frcp_rn((float)d);
    r = r * fma(-d, r, 2.0);
    r = r * fma(-d, r, 2.0);
    return -r2 * r;
}

// translation-unit entry points (host side)
void rick_stage_begin(rick_plan* p, int stage, cudaStream_t st);
void rick_stage_end(rick_plan* p, int stage, cudaStream_t st);
int rick_bin_impl(rick_plan* p, long long M, const float* u, const float* v, const float* w,
                  const float2* vis, const float* weight, float* u_s, float* v_s, float* w_s,
                  float2* vis_s, float* weight_s, unsigned* key_out, unsigned* perm_out,
                  unsigned long long* bin_start_out, void* workspace, long long* n_kept_dev, cudaStream_t st);
size_t rick_bin_workspace_bytes(const rick_plan* p, long long M);
int rick_bin_init();   // one-time kernel attributes (dynamic shared memory opt-in)
int rick_grid_impl(rick_plan* p, void* grid, cudaStream_t st);
int rick_wcorrect_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st);
bool rick_colfft_supported(const rick_plan* p);
int rick_colfft_init(rick_plan* p);
int rick_colfft_wcorrect_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st,
                              int col_lo = 0, int col_hi = -1, bool clear_image = true);
int rick_colfft_split(const rick_plan* p);                              // 1 or 2 plane halves per column block
int rick_colfft_columns_per_cta();
bool rick_colsplit_supported(const rick_plan* p);
int rick_colsplit_init(rick_plan* p);
int rick_colsplit_a_impl(rick_plan* p, void* grid, cudaStream_t st);
int rick_colsplit_b_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st,
                         int col_lo = 0, int col_hi = -1);
bool rick_rowbig_supported(const rick_plan* p);
int rick_rowbig_impl(rick_plan* p, void* grid, cudaStream_t st);         // row transforms of the listed rows, N >= 4096
int rick_rows_mark(rick_plan* p, long long M, cudaStream_t st);          // rick_bin: occ_cur from the records
int rick_rows_clear(rick_plan* p, void* grid, int zero_first, cudaStream_t st);   // rick_grid: clear new rows
int rick_rows_list_all(rick_plan* p, cudaStream_t st);                   // row_list = all defined rows
int rick_rowfft_impl(rick_plan* p, void* grid, cudaStream_t st);         // row transforms of the listed rows
