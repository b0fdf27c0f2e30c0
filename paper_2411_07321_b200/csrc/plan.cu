// plan.cu -- plan lifetime, cuFFT stage, stage timers, host<->device entry points of librick_b200.
#include <cmath>
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "rick_internal.cuh"

void rick_stage_begin(rick_plan* p, int stage, cudaStream_t st) { cudaEventRecord(p->ev_start[stage], st); }
void rick_stage_end(rick_plan* p, int stage, cudaStream_t st) {
    cudaEventRecord(p->ev_stop[stage], st);
    p->ev_valid[stage] = true;
}

namespace {

int ceil_log2_u64(unsigned long long v) {   // smallest b with 2^b > v  (bits needed to store v)
    int b = 0;
    while (b < 63 && (1ull << b) <= v) ++b;
    return b;
}

struct StageTimer {
    rick_plan* p;
    int stage;
    cudaStream_t st;
    StageTimer(rick_plan* p_, int s_, cudaStream_t st_) : p(p_), stage(s_), st(st_) {
        cudaEventRecord(p->ev_start[stage], st);
    }
    ~StageTimer() {
        cudaEventRecord(p->ev_stop[stage], st);
        p->ev_valid[stage] = true;
    }
};

void destroy_fft(rick_plan* p) {
    if (p->fft_ready) {
        cufftDestroy(p->fft);
        p->fft_ready = false;
    }
    if (p->fft_rows_ready) {
        cufftDestroy(p->fft_rows);
        p->fft_rows_ready = false;
    }
    p->fft_rows_work_bytes = 0;
    p->fused = 0;
    p->split = false;
}

// batched 1-D inverse transforms of all Nw * N rows, in place (the row half of D7)
int build_fft_rows(rick_plan* p) {
    const long long N = p->g.N;
    cufftHandle h;
    if (cufftCreate(&h) != CUFFT_SUCCESS) return RICK_ECUFFT;
    if (cufftSetAutoAllocation(h, 0) != CUFFT_SUCCESS) { cufftDestroy(h); return RICK_ECUFFT; }
    long long n[1] = {N};
    size_t work = 0;
    const cufftType type = (p->dtype == RICK_C128) ? CUFFT_Z2Z : CUFFT_C2C;
    if (cufftMakePlanMany64(h, 1, n, NULL, 1, N, NULL, 1, N, type, N * p->g.Nw, &work) != CUFFT_SUCCESS) {
        cufftDestroy(h);
        return RICK_ECUFFT;
    }
    p->fft_rows = h;
    p->fft_rows_ready = true;
    p->fft_rows_work_bytes = work;
    return RICK_OK;
}

// Largest batch (a divisor of Nw) whose cuFFT work area stays within `limit` bytes.
int build_fft(rick_plan* p) {
    destroy_fft(p);
    const long long N = p->g.N;
    const cufftType type = (p->dtype == RICK_C128) ? CUFFT_Z2Z : CUFFT_C2C;
    const size_t limit = (size_t)8 << 30;
    for (int batch = p->g.Nw; batch >= 1; --batch) {
        if (p->g.Nw % batch) continue;
        cufftHandle h;
        if (cufftCreate(&h) != CUFFT_SUCCESS) return RICK_ECUFFT;
        if (cufftSetAutoAllocation(h, 0) != CUFFT_SUCCESS) { cufftDestroy(h); return RICK_ECUFFT; }
        long long n[2] = {N, N};
        size_t work = 0;
        cufftResult r = cufftMakePlanMany64(h, 2, n, NULL, 1, N * N, NULL, 1, N * N, type, batch, &work);
        if (r != CUFFT_SUCCESS) {
            cufftDestroy(h);
            if (batch == 1) return RICK_ECUFFT;
            continue;
        }
        if (work > limit && batch > 1) {
            cufftDestroy(h);
            continue;
        }
        p->fft = h;
        p->fft_ready = true;
        p->fft_batch = batch;
        p->fft_work_bytes = work;
        return RICK_OK;
    }
    return RICK_ECUFFT;
}


// Modified Bessel functions of the first kind through the C++17 special-function library (libstdc++'s
// std::cyl_bessel_i: series for small arguments, asymptotic / uniform expansions beyond).
double bessel_i0_lib(double x) { return std::cyl_bessel_i(0.0, fabs(x)); }
double bessel_i1_over_x_lib(double x) {        // I1(x) / x -> 1/2 at 0
    const double ax = fabs(x);
    if (ax < 1e-8) return 0.5;
    return std::cyl_bessel_i(1.0, ax) / ax;
}

// sinh(sqrt t) / sqrt t as one entire function of t (it continues to sin(sqrt -t) / sqrt -t for t < 0):
// the transform of the Kaiser-Bessel window is 2 a_t sinhc(beta^2 - (2 pi a_t nu)^2) / I0(beta) on both
// sides of the edge of the main lobe [D8-KB]
double sinhc_of_square(double t) {
    if (fabs(t) < 1e-3) return 1.0 + (t / 6.0) * (1.0 + (t / 20.0) * (1.0 + t / 42.0));
    const double r = sqrt(fabs(t));
    return t > 0.0 ? sinh(r) / r : sin(r) / r;
}

// D8 / D8-KB: 1 / t[p] on the device.  Gaussian: t[p] = c0 exp(-2 pi^2 sigma^2 nu_p^2),
// c0 = sigma sqrt(2 pi) erf(a_t / (sigma sqrt 2)).  Kaiser-Bessel: t = 2 a_t sinh(z) / (z I0(beta)),
// z = sqrt(beta^2 - (2 pi a_t nu)^2) (sin(z') / z' beyond the main lobe).
int upload_taper(rick_plan* p) {
    const RickGeom& g = p->g;
    const int N = g.N;
    double* inv_t = (double*)malloc(sizeof(double) * (size_t)N);
    if (!inv_t) return RICK_ENOMEM;
    const double pi = 3.14159265358979323846;
    const double a_t = (double)g.h + 0.5;
    if (g.kernel == RICK_KERNEL_KB) {
        const double scale = bessel_i0_lib(p->kb_beta) / (2.0 * a_t), b2 = p->kb_beta * p->kb_beta;
        for (int i = 0; i < N; ++i) {
            const double y = 2.0 * pi * a_t * ((double)(i - N / 2) / (double)N);
            inv_t[i] = scale / sinhc_of_square(b2 - y * y);
        }
    } else {
        const double sigma = g.sigma;
        const double c0 = sigma * sqrt(2.0 * pi) * erf(a_t / (sigma * sqrt(2.0)));
        for (int i = 0; i < N; ++i) {
            const double nu = (double)(i - N / 2) / (double)N;
            inv_t[i] = 1.0 / (c0 * exp(-2.0 * pi * pi * sigma * sigma * nu * nu));
        }
    }
    cudaError_t e = cudaSuccess;
    if (!p->inv_taper_dev) e = cudaMalloc((void**)&p->inv_taper_dev, sizeof(double) * (size_t)N);
    if (e == cudaSuccess) e = cudaMemcpy(p->inv_taper_dev, inv_t, sizeof(double) * (size_t)N, cudaMemcpyHostToDevice);
    free(inv_t);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RICK_ENOMEM : RICK_ECUDA;
    return RICK_OK;
}


// Degree-(T-1) interpolation polynomials (in t = 2 delta) of the Kaiser-Bessel taps g(delta + a - h) at the T
// Chebyshev nodes of [-1, 1]; returns the largest error of the fp32-rounded polynomials over a fine sample.
double fit_kb_polynomials(rick_plan* p) {
    const int T = RICK_KB_POLY_TERMS, S = p->g.S, h = p->g.h;
    const double a_t = (double)h + 0.5, beta = p->kb_beta, i0b = bessel_i0_lib(beta), pi = 3.14159265358979323846;
    auto win = [&](double d) {
        const double r = d / a_t, arg = 1.0 - r * r;
        return bessel_i0_lib(beta * sqrt(arg > 0.0 ? arg : 0.0)) / i0b;
    };
    double worst = 0.0;
    for (int a = 0; a < S; ++a) {
        long double A[RICK_KB_POLY_TERMS][RICK_KB_POLY_TERMS + 1];
        for (int r = 0; r < T; ++r) {
            const double t = cos(pi * (2.0 * r + 1.0) / (2.0 * T));
            long double pw = 1.0L;
            for (int c = 0; c < T; ++c) { A[r][c] = pw; pw *= (long double)t; }
            A[r][T] = (long double)win(0.5 * t + (double)(a - h));
        }
        for (int c = 0; c < T; ++c) {                      // Gauss-Jordan with partial pivoting
            int piv = c;
            for (int r = c + 1; r < T; ++r) if (fabsl(A[r][c]) > fabsl(A[piv][c])) piv = r;
            for (int k = 0; k <= T; ++k) { const long double tmp = A[c][k]; A[c][k] = A[piv][k]; A[piv][k] = tmp; }
            for (int r = 0; r < T; ++r) {
                if (r == c) continue;
                const long double f = A[r][c] / A[c][c];
                for (int k = c; k <= T; ++k) A[r][k] -= f * A[c][k];
            }
        }
        for (int c = 0; c < T; ++c) p->kb_poly[a][c] = (float)(A[c][T] / A[c][c]);
        for (int i = 0; i <= 400; ++i) {
            const double t = -1.0 + i / 200.0;
            double v = 0.0;
            for (int c = T - 1; c >= 0; --c) v = v * t + (double)p->kb_poly[a][c];
            const double e = fabs(v - win(0.5 * t + (double)(a - h)));
            if (e > worst) worst = e;
        }
    }
    return worst;
}

// copy stream and hand-over events of rick_image_from_host_chunked, created with the plan
int pipe_init(rick_plan* p) {
    if (p->pipe_ready) return RICK_OK;
    RICK_CUDA(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    for (int b = 0; b < 2; ++b) {
        RICK_CUDA(cudaEventCreateWithFlags(&p->ev_copied[b], cudaEventDisableTiming));
        RICK_CUDA(cudaEventCreateWithFlags(&p->ev_consumed[b], cudaEventDisableTiming));
    }
    RICK_CUDA(cudaEventCreateWithFlags(&p->ev_entry, cudaEventDisableTiming));
    for (int i = 0; i < RICK_IMAGE_PARTS; ++i) RICK_CUDA(cudaEventCreateWithFlags(&p->ev_part[i], cudaEventDisableTiming));
    p->pipe_ready = true;
    return RICK_OK;
}

}  // namespace

extern "C" {

int rick_plan_create(int N, int Nw, int support, double sigma, double w_min, double w_max, double dl,
                     rick_plan** out) {
    if (!out) return RICK_EINVAL;
    *out = NULL;
    if (N < 32 || N > 32768 || (N % RICK_TILE) != 0) return RICK_EINVAL;
    if (Nw < 1 || Nw > 4096) return RICK_EINVAL;
    if (support < 3 || support > 15 || (support % 2) == 0) return RICK_EINVAL;
    // sigma >= 1/4 cell: below that the tap recurrence g(d0 + s) = g(d0) E^s g(s) overflows E^s while g(s)
    // underflows (inf * 0), and a Gaussian that narrow is not a usable gridding kernel anyway
    if (!(sigma >= 0.25) || !isfinite(sigma)) return RICK_EINVAL;
    if (!isfinite(w_min) || !isfinite(w_max) || !(w_max > w_min)) return RICK_EINVAL;
    if (!(dl > 0.0) || !isfinite(dl) || !((double)N * dl < 1.4142135623730951)) return RICK_EINVAL;
    const long long T = N / RICK_TILE;
    const long long n_bins = (long long)Nw * T * T;
    if (n_bins > (1ll << 27)) return RICK_EINVAL;   // keeps >= 5 cell bits in the 32-bit sort key [D4']

    rick_plan* p = new (std::nothrow) rick_plan();
    if (!p) return RICK_ENOMEM;
    memset(p, 0, sizeof(*p));
    RickGeom& g = p->g;
    g.N = N; g.Nw = Nw; g.S = support; g.h = (support - 1) / 2; g.T = (int)T;
    g.s = (double)N * dl;
    g.half = (double)(N / 2);
    g.w_min = w_min; g.w_max = w_max;
    g.inv_dw = (double)Nw / (w_max - w_min);
    g.dl = dl;
    g.dw = (w_max - w_min) / (double)Nw;
    g.sigma = sigma;
    g.n_bins = (uint32_t)n_bins;
    g.tap_c = 1.0 / (2.0 * sigma * sigma);
    // D4': as many in-tile cell bits as fit a 32-bit sort key (10 = the exact cell)
    g.cell_bits = 10;
    while (g.cell_bits > 0 && ((unsigned long long)n_bins << g.cell_bits) > (1ull << 32)) --g.cell_bits;
    // the largest sort key belongs to row j0 = N-1 of the last tile (cb >= 5 keeps all of j0 & 31),
    // which D5 never keeps (h >= 1): it is free to mark dropped visibilities and costs no extra key bit
    g.sort_sentinel = (uint32_t)(((unsigned long long)n_bins << g.cell_bits) - 1ull);
    p->dtype = RICK_C64;

    if (rick_bin_init() != RICK_OK) { delete p; return RICK_ECUDA; }
    // radix-sort digit layout: sort keys take values 0 .. sort_sentinel, LSD passes of <= 9 bits
    p->key_bits = ceil_log2_u64((unsigned long long)g.sort_sentinel);
    if (p->key_bits < 1) p->key_bits = 1;
    // digits are 9 bits wide (up to 27 key bits: 1-3 passes) or 8 bits wide (28-32 key bits: 4 passes);
    // the top digit may extend past the key (those bits are zero)
    {
        const int width = p->key_bits <= 27 ? 9 : 8;
        p->n_pass = (p->key_bits + width - 1) / width;
        for (int i = 0; i < p->n_pass; ++i) {
            p->digit_bits[i] = width;
            p->digit_shift[i] = i * width;
        }
    }

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { delete p; return RICK_ECUDA; }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { delete p; return RICK_ECUDA; }
    p->sm_count = sms > 0 ? sms : 148;
    p->device = dev;

    {
        const int rc = upload_taper(p);
        if (rc != RICK_OK) { delete p; return rc; }
    }
    for (int i = 0; i < RICK_T_COUNT; ++i) {
        if (cudaEventCreate(&p->ev_start[i]) != cudaSuccess || cudaEventCreate(&p->ev_stop[i]) != cudaSuccess) {
            rick_plan_destroy(p);
            return RICK_ECUDA;
        }
    }
    if (pipe_init(p) != RICK_OK) {
        rick_plan_destroy(p);
        return RICK_ECUDA;
    }
    *out = p;
    return RICK_OK;
}

int rick_plan_set_dtype(rick_plan* p, int dtype) {
    if (!p || (dtype != RICK_C64 && dtype != RICK_C128)) return RICK_EINVAL;
    p->dtype = dtype;
    p->dtype_set = true;
    return build_fft(p);
}

int rick_plan_set_kernel(rick_plan* p, int kind, double param) {
    if (!p || (kind != RICK_KERNEL_GAUSS && kind != RICK_KERNEL_KB)) return RICK_EINVAL;
    if (kind == RICK_KERNEL_KB && !(param > 0.0 && param <= 64.0)) return RICK_EINVAL;
    RICK_CUDA(cudaDeviceSynchronize());       // the tables may be in use by queued work
    RickGeom& g = p->g;
    g.kernel = kind;
    if (kind == RICK_KERNEL_KB) {
        p->kb_beta = param;
        const int nL = 8192;
        const double a_t = (double)g.h + 0.5, hstep = a_t / nL, i0b = bessel_i0_lib(param);
        float2* lf = (float2*)malloc(sizeof(float2) * (nL + 1));
        double2* ld = (double2*)malloc(sizeof(double2) * (nL + 1));
        double* gv = (double*)malloc(sizeof(double) * (nL + 1));
        if (!lf || !ld || !gv) { free(lf); free(ld); free(gv); return RICK_ENOMEM; }
        for (int i = 0; i <= nL; ++i) {
            const double d = i * hstep, r = d / a_t;
            const double arg = 1.0 - r * r, z = param * sqrt(arg > 0.0 ? arg : 0.0);
            gv[i] = bessel_i0_lib(z) / i0b;
            // g'(d) = -(beta^2 d / a_t^2) (I1(z) / z) / I0(beta)
            ld[i] = make_double2(gv[i], hstep * (-(param * param) * d / (a_t * a_t) * bessel_i1_over_x_lib(z) / i0b));
        }
        for (int i = 0; i <= nL; ++i) lf[i] = make_float2((float)gv[i], i < nL ? (float)(gv[i + 1] - gv[i]) : 0.f);
        cudaError_t e = cudaSuccess;
        if (!p->kb_lut_f_dev) e = cudaMalloc(&p->kb_lut_f_dev, sizeof(float2) * (nL + 1));
        if (e == cudaSuccess && !p->kb_lut_d_dev) e = cudaMalloc(&p->kb_lut_d_dev, sizeof(double2) * (nL + 1));
        if (e == cudaSuccess) e = cudaMemcpy(p->kb_lut_f_dev, lf, sizeof(float2) * (nL + 1), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p->kb_lut_d_dev, ld, sizeof(double2) * (nL + 1), cudaMemcpyHostToDevice);
        free(lf); free(ld); free(gv);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RICK_ENOMEM : RICK_ECUDA;
        g.kb_n = nL;
        g.kb_inv_h = (double)nL / a_t;
        g.kb_lut_f = (const float2*)p->kb_lut_f_dev;
        g.kb_lut_d = (const double2*)p->kb_lut_d_dev;
        p->kb_poly_ok = fit_kb_polynomials(p) <= 5e-8;
    }
    return upload_taper(p);
}

int rick_plan_set_fusion(rick_plan* p, int on) {
    if (!p) return RICK_EINVAL;
    if (on < 0 || on > 2) return RICK_EINVAL;
    if (!on) { p->fused = 0; p->segs = false; return RICK_OK; }
    if (!p->dtype_set) return RICK_ESTATE;
    // engine: the one-sweep column kernel where a column block fits one SM (fp32 mesh, N <= 2048), else the
    // split column transform (two sweeps; N up to 16384, both mesh types)
    const bool one_sweep = rick_colfft_supported(p);
    if (!one_sweep && !rick_colsplit_supported(p)) return RICK_EINVAL;
    if (!p->fft_rows_ready) {
        int rc = build_fft_rows(p);
        if (rc != RICK_OK) return rc;
        if ((rc = one_sweep ? rick_colfft_init(p) : rick_colsplit_init(p)) != RICK_OK) return rc;
    }
    p->split = !one_sweep;
    if (on == 2 && !p->occ_cur_dev) {
        const size_t words = (size_t)p->g.Nw * p->g.N / 32, rows = (size_t)p->g.Nw * p->g.N;
        if (cudaMalloc((void**)&p->occ_cur_dev, 4 * words) != cudaSuccess ||
            cudaMalloc((void**)&p->occ_mesh_dev, 4 * words) != cudaSuccess ||
            cudaMalloc((void**)&p->row_list_dev, 4 * rows) != cudaSuccess ||
            cudaMalloc((void**)&p->n_rows_dev, 4) != cudaSuccess)
            return RICK_ENOMEM;
        RICK_CUDA(cudaMemset(p->occ_cur_dev, 0, 4 * words));
        RICK_CUDA(cudaMemset(p->occ_mesh_dev, 0, 4 * words));
    }
    // segment occupancy: where the library's own long-row kernel transforms the rows (it takes zeros for the
    // segments of a row no footprint touches)
    p->segs = (on == 2) && p->split && rick_rowbig_supported(p);
    if (p->segs && !p->seg_cur_dev) {
        const size_t rows = (size_t)p->g.Nw * p->g.N;
        if (cudaMalloc((void**)&p->seg_cur_dev, 8 * rows) != cudaSuccess ||
            cudaMalloc((void**)&p->seg_mesh_dev, 8 * rows) != cudaSuccess ||
            cudaMalloc((void**)&p->seg_fresh_dev, 8 * rows) != cudaSuccess)
            return RICK_ENOMEM;
        RICK_CUDA(cudaMemset(p->seg_cur_dev, 0, 8 * rows));
        RICK_CUDA(cudaMemset(p->seg_mesh_dev, 0, 8 * rows));
        RICK_CUDA(cudaMemset(p->seg_fresh_dev, 0, 8 * rows));
    }
    p->fused = on;
    return RICK_OK;
}

int rick_plan_cells_defined(rick_plan* p, long long* cells) {
    if (!p || !cells) return RICK_EINVAL;
    if (p->fused != 2 || !p->n_rows_dev) return RICK_ESTATE;
    RICK_CUDA(cudaDeviceSynchronize());
    if (!p->segs) {
        uint32_t n = 0;
        RICK_CUDA(cudaMemcpy(&n, p->n_rows_dev, sizeof(n), cudaMemcpyDeviceToHost));
        *cells = (long long)n * p->g.N;
        return RICK_OK;
    }
    const size_t rows = (size_t)p->g.Nw * p->g.N;
    unsigned long long* h = (unsigned long long*)malloc(8 * rows);
    if (!h) return RICK_ENOMEM;
    if (cudaMemcpy(h, p->seg_mesh_dev, 8 * rows, cudaMemcpyDeviceToHost) != cudaSuccess) { free(h); return RICK_ECUDA; }
    long long n = 0;
    for (size_t r = 0; r < rows; ++r) n += __builtin_popcountll(h[r]);
    free(h);
    *cells = n * (p->g.N / 64);
    return RICK_OK;
}

int rick_plan_rows_defined(rick_plan* p, long long* rows) {
    if (!p || !rows) return RICK_EINVAL;
    if (p->fused != 2 || !p->n_rows_dev) return RICK_ESTATE;
    uint32_t n = 0;
    RICK_CUDA(cudaDeviceSynchronize());
    RICK_CUDA(cudaMemcpy(&n, p->n_rows_dev, sizeof(n), cudaMemcpyDeviceToHost));
    *rows = (long long)n;
    return RICK_OK;
}

int rick_plan_workspace_bytes(const rick_plan* p, long long M, size_t* bin_bytes, size_t* fft_bytes) {
    if (!p || M < 0 || M >= 4294967295ll) return RICK_EINVAL;
    if (bin_bytes) *bin_bytes = rick_bin_workspace_bytes(p, M);
    if (fft_bytes) {
        if (!p->fft_ready) return RICK_ESTATE;
        // fused: only the batched row transforms go through cuFFT -- and in mode 2 not even those where the library
        // has a row kernel of its own (k_rowfft, k_row_big)
        const bool own_rows = p->fused == 2 && (!p->split || rick_rowbig_supported(p));
        *fft_bytes = p->fused ? (own_rows ? 0 : p->fft_rows_work_bytes) : p->fft_work_bytes;
    }
    return RICK_OK;
}

int rick_plan_sort_layout(const rick_plan* p, int* key_bits, int* n_pass, int* cell_bits) {
    if (!p) return RICK_EINVAL;
    if (key_bits) *key_bits = p->key_bits;
    if (n_pass) *n_pass = p->n_pass;
    if (cell_bits) *cell_bits = p->g.cell_bits;
    return RICK_OK;
}

int rick_plan_destroy(rick_plan* p) {
    if (!p) return RICK_EINVAL;
    destroy_fft(p);
    if (p->inv_taper_dev) cudaFree(p->inv_taper_dev);
    if (p->colfft_tw) cudaFree(p->colfft_tw);
    if (p->split_tw) cudaFree(p->split_tw);
    if (p->occ_cur_dev) cudaFree(p->occ_cur_dev);
    if (p->occ_mesh_dev) cudaFree(p->occ_mesh_dev);
    if (p->row_list_dev) cudaFree(p->row_list_dev);
    if (p->n_rows_dev) cudaFree(p->n_rows_dev);
    if (p->seg_cur_dev) cudaFree(p->seg_cur_dev);
    if (p->seg_mesh_dev) cudaFree(p->seg_mesh_dev);
    if (p->seg_fresh_dev) cudaFree(p->seg_fresh_dev);
    if (p->kb_lut_f_dev) cudaFree(p->kb_lut_f_dev);
    if (p->kb_lut_d_dev) cudaFree(p->kb_lut_d_dev);
    for (int i = 0; i < RICK_T_COUNT; ++i) {
        if (p->ev_start[i]) cudaEventDestroy(p->ev_start[i]);
        if (p->ev_stop[i]) cudaEventDestroy(p->ev_stop[i]);
    }
    if (p->pipe_ready) {
        cudaStreamDestroy(p->copy_stream);
        for (int b = 0; b < 2; ++b) { cudaEventDestroy(p->ev_copied[b]); cudaEventDestroy(p->ev_consumed[b]); }
        cudaEventDestroy(p->ev_entry);
        for (int i = 0; i < RICK_IMAGE_PARTS; ++i) cudaEventDestroy(p->ev_part[i]);
    }
    delete p;
    return RICK_OK;
}

int rick_bin(rick_plan* p, long long M, const float* u, const float* v, const float* w, const void* vis,
             const float* weight, float* u_s, float* v_s, float* w_s, void* vis_s, float* weight_s,
             unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out, void* workspace,
             size_t workspace_bytes, long long* n_kept_dev, void* stream) {
    if (!p || M < 0 || M >= 4294967295ll || !n_kept_dev) return RICK_EINVAL;
    if (M > 0 && (!u || !v || !w || !vis || !weight)) return RICK_EINVAL;
    // sorted SoA outputs: all five, or none (indirect mode: fp32 mesh only -- the fp64 gridder reads them)
    const int n_sorted = (u_s != NULL) + (v_s != NULL) + (w_s != NULL) + (vis_s != NULL) + (weight_s != NULL);
    if (n_sorted != 0 && n_sorted != 5) return RICK_EINVAL;
    if (n_sorted == 0 && p->dtype == RICK_C128) return RICK_EINVAL;
    if (!workspace || ((uintptr_t)workspace & 255)) return RICK_EINVAL;
    if (workspace_bytes < rick_bin_workspace_bytes(p, M)) return RICK_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    StageTimer tm(p, RICK_T_BIN, st);
    return rick_bin_impl(p, M, u, v, w, (const float2*)vis, weight, u_s, v_s, w_s, (float2*)vis_s, weight_s,
                         key_out, perm_out, bin_start_out, workspace, n_kept_dev, st);
}

int rick_grid(rick_plan* p, void* grid, int zero_first, void* stream) {
    if (!p || !grid || ((uintptr_t)grid & 15)) return RICK_EINVAL;     // 16-byte reductions, bulk copies
    if (!p->bound) return RICK_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->fused == 2) {          // clear only the rows the bound visibilities touch and that are not defined yet
        StageTimer tz(p, RICK_T_ZERO, st);
        const int rc = rick_rows_clear(p, grid, zero_first, st);
        if (rc != RICK_OK) return rc;
    } else if (zero_first) {
        StageTimer tz(p, RICK_T_ZERO, st);
        const size_t cell = (p->dtype == RICK_C128) ? 16 : 8;
        RICK_CUDA(cudaMemsetAsync(grid, 0, cell * (size_t)p->g.Nw * (size_t)p->g.N * (size_t)p->g.N, st));
    }
    StageTimer tm(p, RICK_T_GRID, st);
    return rick_grid_impl(p, grid, st);
}

int rick_fft_planes(rick_plan* p, void* grid, void* fft_work, size_t fft_work_bytes, void* stream) {
    if (!p || !grid || ((uintptr_t)grid & 15)) return RICK_EINVAL;
    if (!p->fft_ready) return RICK_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->fused == 2 && !p->split) {   // row transforms of the defined rows only, by the library's own kernel (colfft.cu)
        StageTimer tm(p, RICK_T_FFT, st);
        int rc = rick_rows_list_all(p, st);
        StageTimer tr(p, RICK_T_FFT_ROWS, st);
        if (rc == RICK_OK) rc = rick_rowfft_impl(p, grid, st);
        return rc;
    }
    if (p->fused == 2 && p->split && rick_rowbig_supported(p)) {
        // own row kernel on the defined rows only (rowbig.cu), then sweep A, which reads only those rows
        StageTimer tm(p, RICK_T_FFT, st);
        int rc = rick_rows_list_all(p, st);
        {
            StageTimer tr(p, RICK_T_FFT_ROWS, st);
            if (rc == RICK_OK) rc = rick_rowbig_impl(p, grid, st);
        }
        StageTimer ta(p, RICK_T_FFT_COL_A, st);
        if (rc == RICK_OK) rc = rick_colsplit_a_impl(p, grid, st);
        return rc;
    }
    if (p->fused) {   // rows only (+ sweep A of the split engine); rick_wcorrect_accumulate finishes the transform
        if (p->fft_rows_work_bytes > 0 && (!fft_work || fft_work_bytes < p->fft_rows_work_bytes)) return RICK_ENOMEM;
        if (cufftSetStream(p->fft_rows, st) != CUFFT_SUCCESS) return RICK_ECUFFT;
        if (p->fft_rows_work_bytes > 0 && cufftSetWorkArea(p->fft_rows, fft_work) != CUFFT_SUCCESS) return RICK_ECUFFT;
        StageTimer tm(p, RICK_T_FFT, st);
        {
            StageTimer tr(p, RICK_T_FFT_ROWS, st);
            const cufftResult r = p->dtype == RICK_C128
                ? cufftExecZ2Z(p->fft_rows, (cufftDoubleComplex*)grid, (cufftDoubleComplex*)grid, CUFFT_INVERSE)
                : cufftExecC2C(p->fft_rows, (cufftComplex*)grid, (cufftComplex*)grid, CUFFT_INVERSE);
            if (r != CUFFT_SUCCESS) return RICK_ECUFFT;
        }
        if (p->split) {
            // mode 2: rows no footprint touched hold undefined data; the library transforms them in place (each
            // row on its own) and sweep A reads only the touched ones
            int rc = p->fused == 2 ? rick_rows_list_all(p, st) : RICK_OK;
            StageTimer ta(p, RICK_T_FFT_COL_A, st);
            if (rc == RICK_OK) rc = rick_colsplit_a_impl(p, grid, st);
            return rc;
        }
        return RICK_OK;
    }
    if (p->fft_work_bytes > 0 && (!fft_work || fft_work_bytes < p->fft_work_bytes)) return RICK_ENOMEM;
    if (cufftSetStream(p->fft, st) != CUFFT_SUCCESS) return RICK_ECUFFT;
    if (p->fft_work_bytes > 0 && cufftSetWorkArea(p->fft, fft_work) != CUFFT_SUCCESS) return RICK_ECUFFT;
    StageTimer tm(p, RICK_T_FFT, st);
    const size_t plane = (size_t)p->g.N * (size_t)p->g.N;
    for (int k = 0; k < p->g.Nw; k += p->fft_batch) {
        cufftResult r;
        if (p->dtype == RICK_C128) {
            cufftDoubleComplex* d = (cufftDoubleComplex*)grid + plane * (size_t)k;
            r = cufftExecZ2Z(p->fft, d, d, CUFFT_INVERSE);
        } else {
            cufftComplex* d = (cufftComplex*)grid + plane * (size_t)k;
            r = cufftExecC2C(p->fft, d, d, CUFFT_INVERSE);
        }
        if (r != CUFFT_SUCCESS) return RICK_ECUFFT;
    }
    return RICK_OK;
}

int rick_wcorrect_accumulate(rick_plan* p, const void* grid, double* image, int zero_first, void* stream) {
    if (!p || !grid || !image || ((uintptr_t)grid & 15) || ((uintptr_t)image & 7)) return RICK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    StageTimer tm(p, RICK_T_WCORRECT, st);
    if (p->fused && p->split) return rick_colsplit_b_impl(p, grid, image, zero_first, st);
    if (p->fused) return rick_colfft_wcorrect_impl(p, grid, image, zero_first, st);
    return rick_wcorrect_impl(p, grid, image, zero_first, st);
}

int rick_image(rick_plan* p, const double* image_dev, double* out, int out_is_host, void* stream) {
    if (!p || !image_dev || !out) return RICK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    StageTimer tm(p, RICK_T_IMAGE, st);
    const size_t bytes = sizeof(double) * (size_t)p->g.N * (size_t)p->g.N;
    if (out == image_dev) return RICK_OK;
    RICK_CUDA(cudaMemcpyAsync(out, image_dev, bytes, out_is_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, st));
    return RICK_OK;
}

int rick_image_from_host(rick_plan* p, long long M, const float* u_h, const float* v_h, const float* w_h,
                         const void* vis_h, const float* weight_h, const rick_device_buffers* d,
                         double* image_host, void* stream) {
    if (!p || !d || !image_host || M < 0) return RICK_EINVAL;
    if (M > 0 && (!u_h || !v_h || !w_h || !vis_h || !weight_h)) return RICK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t m = (size_t)M;
    if (M > 0) {
        RICK_CUDA(cudaMemcpyAsync(d->u, u_h, 4 * m, cudaMemcpyHostToDevice, st));
        RICK_CUDA(cudaMemcpyAsync(d->v, v_h, 4 * m, cudaMemcpyHostToDevice, st));
        RICK_CUDA(cudaMemcpyAsync(d->w, w_h, 4 * m, cudaMemcpyHostToDevice, st));
        RICK_CUDA(cudaMemcpyAsync(d->vis, vis_h, 8 * m, cudaMemcpyHostToDevice, st));
        RICK_CUDA(cudaMemcpyAsync(d->weight, weight_h, 4 * m, cudaMemcpyHostToDevice, st));
    }
    int rc = rick_bin(p, M, d->u, d->v, d->w, d->vis, d->weight, d->u_s, d->v_s, d->w_s, d->vis_s, d->weight_s,
                      NULL, NULL, NULL, d->workspace, d->workspace_bytes, d->n_kept, stream);
    if (rc != RICK_OK) return rc;
    if ((rc = rick_grid(p, d->grid, 1, stream)) != RICK_OK) return rc;
    if ((rc = rick_fft_planes(p, d->grid, d->fft_work, d->fft_work_bytes, stream)) != RICK_OK) return rc;
    if ((rc = rick_wcorrect_accumulate(p, d->grid, d->image, 1, stream)) != RICK_OK) return rc;
    if ((rc = rick_image(p, d->image, image_host, 1, stream)) != RICK_OK) return rc;
    RICK_CUDA(cudaStreamSynchronize(st));
    return RICK_OK;
}

int rick_image_from_host_chunked(rick_plan* p, long long M, const float* u_h, const float* v_h,
                                 const float* w_h, const void* vis_h, const float* weight_h,
                                 const rick_device_buffers* d, int n_chunks, double* image_host,
                                 void* stream) {
    if (!p || !d || !image_host || M < 0 || n_chunks < 1) return RICK_EINVAL;
    if (n_chunks < 2 || M < 2 * 1024)
        return rick_image_from_host(p, M, u_h, v_h, w_h, vis_h, weight_h, d, image_host, stream);
    if (!u_h || !v_h || !w_h || !vis_h || !weight_h) return RICK_EINVAL;
    int rc = RICK_OK;
    cudaStream_t st = (cudaStream_t)stream, cs = p->copy_stream;
    // chunk length: a multiple of 1024 visibilities, two of them within the staging capacity M
    long long c = (M + n_chunks - 1) / n_chunks;
    c = (c + 1023) / 1024 * 1024;
    if (2 * c > M) c = M / 2 / 1024 * 1024;
    const long long n = (M + c - 1) / c;
    // the copy stream starts behind whatever `stream` holds (earlier users of the staging buffers)
    RICK_CUDA(cudaEventRecord(p->ev_entry, st));
    RICK_CUDA(cudaStreamWaitEvent(cs, p->ev_entry, 0));
    auto copy_chunk = [&](long long i) -> int {
        const int b = (int)(i & 1);
        const size_t o = (size_t)(i * c), ob = (size_t)b * (size_t)c;
        const size_t m = (size_t)((i + 1) * c <= M ? c : M - i * c);
        if (i >= 2) RICK_CUDA(cudaStreamWaitEvent(cs, p->ev_consumed[b], 0));
        RICK_CUDA(cudaMemcpyAsync(d->u + ob, u_h + o, 4 * m, cudaMemcpyHostToDevice, cs));
        RICK_CUDA(cudaMemcpyAsync(d->v + ob, v_h + o, 4 * m, cudaMemcpyHostToDevice, cs));
        RICK_CUDA(cudaMemcpyAsync(d->w + ob, w_h + o, 4 * m, cudaMemcpyHostToDevice, cs));
        RICK_CUDA(cudaMemcpyAsync((char*)d->vis + 8 * ob, (const char*)vis_h + 8 * o, 8 * m,
                                  cudaMemcpyHostToDevice, cs));
        RICK_CUDA(cudaMemcpyAsync(d->weight + ob, weight_h + o, 4 * m, cudaMemcpyHostToDevice, cs));
        RICK_CUDA(cudaEventRecord(p->ev_copied[b], cs));
        return RICK_OK;
    };
    if ((rc = copy_chunk(0)) != RICK_OK) return rc;
    for (long long i = 0; i < n; ++i) {
        const int b = (int)(i & 1);
        const size_t ob = (size_t)b * (size_t)c;
        const long long m = (i + 1) * c <= M ? c : M - i * c;
        // the next chunk's copies are queued before this chunk's kernels so that they overlap them
        if (i + 1 < n && (rc = copy_chunk(i + 1)) != RICK_OK) return rc;
        RICK_CUDA(cudaStreamWaitEvent(st, p->ev_copied[b], 0));
        rc = rick_bin(p, m, d->u + ob, d->v + ob, d->w + ob, (char*)d->vis + 8 * ob, d->weight + ob, d->u_s,
                      d->v_s, d->w_s, d->vis_s, d->weight_s, NULL, NULL, NULL, d->workspace,
                      d->workspace_bytes, d->n_kept, stream);
        if (rc != RICK_OK) return rc;
        RICK_CUDA(cudaEventRecord(p->ev_consumed[b], st));   // rick_bin has read the staging half
        if ((rc = rick_grid(p, d->grid, i == 0, stream)) != RICK_OK) return rc;
    }
    if ((rc = rick_fft_planes(p, d->grid, d->fft_work, d->fft_work_bytes, stream)) != RICK_OK) return rc;
    if (p->fused && p->split && p->g.N >= 1024) {
        // split engine: sweep B over RICK_IMAGE_PARTS column stripes; the copy stream takes a stripe to the host while
        // the next one is computed
        const int N = p->g.N, stripe = N / RICK_IMAGE_PARTS;
        StageTimer tm(p, RICK_T_WCORRECT, st);
        for (int part = 0; part < RICK_IMAGE_PARTS; ++part) {
            const int c_lo = part * stripe, c_hi = c_lo + stripe;
            if ((rc = rick_colsplit_b_impl(p, d->grid, d->image, 1, st, c_lo, c_hi)) != RICK_OK) return rc;
            RICK_CUDA(cudaEventRecord(p->ev_part[part], st));
            RICK_CUDA(cudaStreamWaitEvent(cs, p->ev_part[part], 0));
            RICK_CUDA(cudaMemcpy2DAsync(image_host + c_lo, sizeof(double) * (size_t)N, d->image + c_lo,
                                        sizeof(double) * (size_t)N, sizeof(double) * (size_t)stripe, (size_t)N,
                                        cudaMemcpyDeviceToHost, cs));
        }
        RICK_CUDA(cudaStreamSynchronize(st));
        RICK_CUDA(cudaStreamSynchronize(cs));
        return RICK_OK;
    }
    if (!p->fused || p->split) {
        if ((rc = rick_wcorrect_accumulate(p, d->grid, d->image, 1, stream)) != RICK_OK) return rc;
        if ((rc = rick_image(p, d->image, image_host, 1, stream)) != RICK_OK) return rc;
        RICK_CUDA(cudaStreamSynchronize(st));
        return RICK_OK;
    }
    // fused column kernel: the image comes out in parts of whole waves of CTAs (two waves each, at most
    // RICK_IMAGE_PARTS parts); the copy stream takes a part to the host while the next one is computed
    const int N = p->g.N, kc = rick_colfft_columns_per_cta(), items = N / kc;
    const int per_wave = p->sm_count / rick_colfft_split(p);          // column blocks per wave of CTAs
    const int waves = (items + per_wave - 1) / per_wave;
    int n_parts = (waves + 1) / 2;
    n_parts = n_parts < 1 ? 1 : (n_parts > RICK_IMAGE_PARTS ? RICK_IMAGE_PARTS : n_parts);
    const int waves_per_part = (waves + n_parts - 1) / n_parts;
    {
        StageTimer tm(p, RICK_T_WCORRECT, st);
        int b_lo = 0;
        for (int part = 0; part < n_parts && b_lo < items; ++part) {
            int b_hi = b_lo + waves_per_part * per_wave;
            if (b_hi > items || part == n_parts - 1) b_hi = items;
            const int c_lo = b_lo * kc, c_hi = b_hi * kc;
            if ((rc = rick_colfft_wcorrect_impl(p, d->grid, d->image, 1, st, c_lo, c_hi, part == 0)) != RICK_OK) return rc;
            RICK_CUDA(cudaEventRecord(p->ev_part[part], st));
            RICK_CUDA(cudaStreamWaitEvent(cs, p->ev_part[part], 0));
            RICK_CUDA(cudaMemcpy2DAsync(image_host + c_lo, sizeof(double) * (size_t)N, d->image + c_lo,
                                        sizeof(double) * (size_t)N, sizeof(double) * (size_t)(c_hi - c_lo), (size_t)N,
                                        cudaMemcpyDeviceToHost, cs));
            b_lo = b_hi;
        }
    }
    RICK_CUDA(cudaStreamSynchronize(st));
    RICK_CUDA(cudaStreamSynchronize(cs));
    return RICK_OK;
}

int rick_get_timings(rick_plan* p, double* ms, int n) {
    if (!p || !ms || n < 0 || n > RICK_T_COUNT) return RICK_EINVAL;
    for (int i = 0; i < n; ++i) {
        ms[i] = 0.0;
        if (!p->ev_valid[i]) continue;
        RICK_CUDA(cudaEventSynchronize(p->ev_stop[i]));
        float t = 0.f;
        RICK_CUDA(cudaEventElapsedTime(&t, p->ev_start[i], p->ev_stop[i]));
        ms[i] = (double)t;
    }
    return RICK_OK;
}

long long rick_launch_count(const rick_plan* p) { return p ? p->launches : 0; }

const char* rick_strerror(int status) {
    switch (status) {
        case RICK_OK: return "ok";
        case RICK_EINVAL: return "invalid argument";
        case RICK_ENOMEM: return "workspace too small or allocation failed";
        case RICK_ECUDA: return "CUDA runtime error";
        case RICK_ECUFFT: return "cuFFT error";
        case RICK_ESTATE: return "call order violated (bind/dtype missing)";
        case RICK_ELIMIT: return "M exceeds RICK_BIN_STATIC_MAX_M, the capacity of the static scratch (use rick_bin with a workspace)";
        default: return "unknown status";
    }
}

}  // extern "C"
