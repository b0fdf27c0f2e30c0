// grid.cu -- rick_grid: convolutional gridding, Eq. 3, with the separable truncated Gaussian [D6]
// or the separable Kaiser-Bessel window of the paper's own tests [D6-KB] (rick_plan_set_kernel).
//
// Run-accumulating gridders.  rick_bin leaves the kept visibilities sorted by (plane, tile, cell) [D4'],
// so visibilities that share a nearest cell (i0, j0, k) -- and therefore the same S x S footprint --
// are adjacent: 87 % of the "10M" workload sits in runs of >= 8.
// Each thread walks a range of consecutive sorted visibilities (16 .. 128) and keeps the whole footprint
// (or a block of RB rows of it per pass) in registers:
//
//     acc[b][a] += gx[a] * (gy[b] * weight * V)          2 FMAs per cell and visibility
//
// and only when the footprint window changes (or its range ends) adds it to the mesh with reductions in
// L2.  No shared-memory accumulation: fp32 atomicAdd on shared memory is a CAS loop on sm_100a.
// At the end of the ranges the lanes of a warp, which hold consecutive ranges, merge the windows they share
// (segmented sum over the lanes by shuffles) and one lane per window flushes: a hot cell spans many ranges
// (hotspot: 7 600 visibilities per core cell), and its per-range flushes would all land on the same few L2 lines.
//
//   k_grid_rec  (fp32 mesh)  reads the 24-byte gridder records the gather wrote (cell, plane, fractional
//               offsets, signed weight * V), staged through shared memory with coalesced cp.async copies;
//               the footprint columns live in an even-aligned window of S + 1 cells, so every flush is a
//               16-byte red.global.add.v4.f32 (two cells) and two neighbouring cells share one window.
//   k_grid_runs (fp64 mesh)  reads the sorted SoA, recomputes the coordinates in fp64 (bit-identical
//               indices to the key generation), red.global.add.f64 (no vector fp64 reduction exists).
//
// The checkerboard (-1)^(i+j) of the modulated mesh (rick_b200.h) costs nothing: the column and row
// signs are compile-time negations of the taps, the run-constant remainder is the sign of the weight.
#include <string.h>

#include "fft_radix.cuh"
#include "rick_internal.cuh"

namespace {

constexpr int kRunThreads = 128;

struct TapConst {
    double K[8];   // K[t] = exp(-t^2 / (2 sigma^2)), t = 0 .. h
    float Kf[8];   // the same, rounded to fp32
};
struct KbPoly {    // Kaiser-Bessel taps as polynomials in 2 delta (plan: kb_poly), fp32 gridder only
    float c[15][RICK_KB_POLY_TERMS];
    int ok;        // 0: use the table
};

__device__ __forceinline__ void red_add_cell(float2* addr, float re, float im) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(re), "f"(im) : "memory");
}
__device__ __forceinline__ void red_add_cell(double2* addr, double re, double im) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(re) : "memory");
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"((double*)addr + 1), "d"(im) : "memory");
}

__device__ __forceinline__ void red_add_pair(float2* addr, float re0, float im0, float re1, float im1) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(re0), "f"(im0), "f"(re1), "f"(im1)
                 : "memory");
}

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Taps of one axis with the alternating sign of the modulated mesh folded in:
//     t[a] = (-1)^a g(d0 + a - h),  a = 0 .. S-1,  d0 = i0 - x (formed in fp64, narrowed once),
// through the exact identity g(d0 + s) = g(d0) E^s g(s), E = exp(-d0 / sigma^2): three exponentials per
// axis instead of S (fp32: MUFU.EX2; fp64: two exp and one reciprocal).  The (-1)^a are compile-time
// negations (operand modifiers); the remaining run-constant factor (-1)^(i0+j0) multiplies weight * V.
template <int S, bool kSigned>
__device__ __forceinline__ void taps_f32(float* t, float d, float c2, const TapConst& tc) {
    constexpr int h = (S - 1) / 2;
    const float g0 = ex2_approx(d * d * c2);
    const float e = 2.0f * d * c2;
    const float E = ex2_approx(e), Ei = ex2_approx(-e);
    float pp = g0, pm = g0;
    t[h] = (kSigned && (h & 1)) ? -g0 : g0;
#pragma unroll
    for (int s = 1; s <= h; ++s) {
        pp *= E;
        pm *= Ei;
        const float a = pp * tc.Kf[s], b = pm * tc.Kf[s];
        t[h + s] = (kSigned && ((h + s) & 1)) ? -a : a;
        t[h - s] = (kSigned && ((h - s) & 1)) ? -b : b;
    }
}
template <int S, bool kSigned>
__device__ __forceinline__ void taps(float* t, double d0, const RickGeom& g, const TapConst& tc) {
    taps_f32<S, kSigned>(t, (float)d0, (float)(-g.tap_c * 1.4426950408889634), tc);   // c2 = -log2(e) / (2 sigma^2)
}
template <int S, bool kSigned>
__device__ __forceinline__ void taps(double* t, double d0, const RickGeom& g, const TapConst& tc) {
    constexpr int h = (S - 1) / 2;
    const double g0 = exp(-d0 * d0 * g.tap_c);
    const double E = exp(-2.0 * d0 * g.tap_c);
    const double Ei = 1.0 / E;
    t[h] = (kSigned && (h & 1)) ? -g0 : g0;
    double pp = g0, pm = g0;
#pragma unroll
    for (int s = 1; s <= h; ++s) {
        pp *= E;
        pm *= Ei;
        const double a = pp * tc.K[s], b = pm * tc.K[s];
        t[h + s] = (kSigned && ((h + s) & 1)) ? -a : a;
        t[h - s] = (kSigned && ((h - s) & 1)) ? -b : b;
    }
}

// Kaiser-Bessel taps [D6-KB]: g(|d|) from the plan's tables over [0, a_t] (built in fp64 on the host).
// fp32 mesh: linear interpolation between 8192 nodes (error < 4e-8 of the peak); fp64 mesh: cubic Hermite
// on values and derivatives (error < 1e-14).  d = d0 + a - h lies in (-a_t, a_t].
template <int S, bool kSigned>
__device__ __forceinline__ void taps_kb(float* t, float d0, const RickGeom& g) {
    constexpr int h = (S - 1) / 2;
    const float inv_h = (float)g.kb_inv_h;
#pragma unroll
    for (int a = 0; a < S; ++a) {
        const float x = fabsf(d0 + (float)(a - h)) * inv_h;
        int i = (int)x;
        i = i < g.kb_n ? i : g.kb_n - 1;
        const float2 e = __ldg(g.kb_lut_f + i);
        const float v = fmaf(e.y, x - (float)i, e.x);
        t[a] = (kSigned && (a & 1)) ? -v : v;
    }
}
// the same taps from the per-tap polynomials in 2 d0 (no memory access: coefficients are kernel parameters)
template <int S, bool kSigned>
__device__ __forceinline__ void taps_kb_poly(float* t, float d0, const KbPoly& kp) {
    const float x = 2.0f * d0;
#pragma unroll
    for (int a = 0; a < S; ++a) {
        float v = kp.c[a][RICK_KB_POLY_TERMS - 1];
#pragma unroll
        for (int k = RICK_KB_POLY_TERMS - 2; k >= 0; --k) v = fmaf(v, x, kp.c[a][k]);
        t[a] = (kSigned && (a & 1)) ? -v : v;
    }
}
template <int S, bool kSigned>
__device__ __forceinline__ void taps_kb(double* t, double d0, const RickGeom& g) {
    constexpr int h = (S - 1) / 2;
#pragma unroll
    for (int a = 0; a < S; ++a) {
        const double x = fabs(d0 + (double)(a - h)) * g.kb_inv_h;
        int i = (int)x;
        i = i < g.kb_n ? i : g.kb_n - 1;
        const double f = x - (double)i;
        const double2 e0 = __ldg(g.kb_lut_d + i), e1 = __ldg(g.kb_lut_d + i + 1);
        // cubic Hermite on [0, 1]: values e0.x, e1.x, scaled slopes e0.y, e1.y
        const double f2 = f * f, f3 = f2 * f;
        const double v = (2.0 * f3 - 3.0 * f2 + 1.0) * e0.x + (f3 - 2.0 * f2 + f) * e0.y +
                         (-2.0 * f3 + 3.0 * f2) * e1.x + (f3 - f2) * e1.y;
        t[a] = (kSigned && (a & 1)) ? -v : v;
    }
}

template <typename real> struct CellOf;
template <> struct CellOf<float> { typedef float2 type; };
template <> struct CellOf<double> { typedef double2 type; };

// four consecutive floats starting at p (p is a multiple of 4); entries at or beyond n are not read
__device__ __forceinline__ float4 load4(const float* __restrict__ a, long long p, long long n) {
    if (p + 4 <= n) return __ldg((const float4*)(a + p));
    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
    if (p < n) r.x = __ldg(a + p);
    if (p + 1 < n) r.y = __ldg(a + p + 1);
    if (p + 2 < n) r.z = __ldg(a + p + 2);
    return r;
}

template <typename real, int S, int RB, int KIND>
__global__ void __launch_bounds__(kRunThreads) k_grid_runs(RickGeom g, TapConst tc, const long long* __restrict__ n_kept,
                                                          const float* __restrict__ u_s, const float* __restrict__ v_s,
                                                          const float* __restrict__ w_s, const float2* __restrict__ vis_s,
                                                          const float* __restrict__ wt_s,
                                                          typename CellOf<real>::type* __restrict__ grid, int L) {
    typedef typename CellOf<real>::type cell;
    constexpr int h = (S - 1) / 2;
    constexpr int kPasses = (S + RB - 1) / RB;
    // fp32: the footprint columns live in an even-aligned window of W = S + 1 cells, so that every pair of
    // cells is one 16-byte red.global.add.v4.f32 (the extra column carries a zero tap); fp64: W = S.
    constexpr bool kWin = (sizeof(real) == 4);
    constexpr int W = kWin ? S + 1 : S;
    const long long n = *n_kept;
    const long long first = ((long long)blockIdx.x * kRunThreads + threadIdx.x) * L;   // L: a multiple of 4
    if ((long long)blockIdx.x * kRunThreads * L >= n) return;      // whole block past the end (lanes past it stay for the merge)
    const size_t N = (size_t)g.N;

#pragma unroll
    for (int pass = 0; pass < kPasses; ++pass) {
        const int b0 = pass * RB;
        real ar[RB][W], ai[RB][W];
#pragma unroll
        for (int r = 0; r < RB; ++r)
#pragma unroll
            for (int a = 0; a < W; ++a) ar[r][a] = ai[r][a] = (real)0;
        int ci = -1, cj = 0, ck = 0;

        auto flush = [&]() {
            const int iw = kWin ? ((ci - h) & ~1) : (ci - h);   // first column of the window
            cell* base = grid + ((size_t)ck * N + (size_t)(cj - h + b0)) * N + (size_t)iw;
            cell* rowp[RB];                      // one address register pair per row (see k_grid_rec)
#pragma unroll
            for (int r = 0; r < RB; ++r) rowp[r] = base + (size_t)r * N;
#pragma unroll
            for (int r = 0; r < RB; ++r) asm volatile("" : "+l"(rowp[r]));
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                if (b0 + r < S) {
                    if constexpr (kWin) {
#pragma unroll
                        for (int a = 0; a < W; a += 2) {
                            float2* dst = (float2*)(rowp[r] + a);
                            // the zero column may fall past the end of the row (only when i0 = N-1-h)
                            if (a + 2 == W && iw + W > (int)N)
                                red_add_cell(dst, (float)ar[r][a], (float)ai[r][a]);
                            else
                                red_add_pair(dst, (float)ar[r][a], (float)ai[r][a], (float)ar[r][a + 1], (float)ai[r][a + 1]);
                            ar[r][a] = ai[r][a] = ar[r][a + 1] = ai[r][a + 1] = (real)0;
                        }
                    } else {
#pragma unroll
                        for (int a = 0; a < W; ++a) {
                            red_add_cell(rowp[r] + a, ar[r][a], ai[r][a]);
                            ar[r][a] = ai[r][a] = (real)0;
                        }
                    }
                }
            }
        };

        auto one = [&](float uu, float vv, float ww, float re, float im, float wgt) {
            const RickLoc loc = rick_locate(g, uu, vv, ww);
            if (loc.i0 != ci || loc.j0 != cj || loc.k != ck) {
                if (ci >= 0) flush();
                ci = loc.i0; cj = loc.j0; ck = loc.k;
            }
            real gx[W], gy[S];
            if (KIND == RICK_KERNEL_KB) taps_kb<S, true>(gy, (real)((double)loc.j0 - loc.y), g);
            else taps<S, true>(gy, (double)loc.j0 - loc.y, g, tc);
            bool neg;
            if constexpr (kWin) {
                // window column c <-> cell iw + c, iw even: sign (-1)^c at compile time; tap index c - o
                real t[S];
                if (KIND == RICK_KERNEL_KB) taps_kb<S, false>(t, (real)((double)loc.i0 - loc.x), g);
                else taps<S, false>(t, (double)loc.i0 - loc.x, g, tc);
                const bool o = ((loc.i0 - h) & 1) != 0;
#pragma unroll
                for (int c = 0; c < W; ++c) {
                    const real lo = (c >= 1) ? t[c - 1] : (real)0, hi = (c < S) ? t[c] : (real)0;
                    const real v = o ? lo : hi;
                    gx[c] = (c & 1) ? -v : v;
                }
                neg = ((loc.j0 - h) & 1) != 0;            // (-1)^(j0-h): the rest of (-1)^(i+j)
            } else {
                if (KIND == RICK_KERNEL_KB) taps_kb<S, true>(gx, (real)((double)loc.i0 - loc.x), g);
                else taps<S, true>(gx, (double)loc.i0 - loc.x, g, tc);
                neg = ((loc.i0 + loc.j0) & 1) != 0;       // (-1)^(i0+j0)
            }
            const real ws = neg ? -(real)wgt : (real)wgt;
            const real vr = ws * (real)re, vi = ws * (real)im;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                if (b0 + r < S) {
                    const real yr = gy[b0 + r] * vr, yi = gy[b0 + r] * vi;
#pragma unroll
                    for (int a = 0; a < W; ++a) {
                        ar[r][a] = fma(gx[a], yr, ar[r][a]);
                        ai[r][a] = fma(gx[a], yi, ai[r][a]);
                    }
                }
            }
        };

#pragma unroll 1
        for (int i = 0; i < L; i += 4) {
            const long long p = first + i;
            if (p >= n) break;
            const float4 u4 = load4(u_s, p, n), v4 = load4(v_s, p, n), w4 = load4(w_s, p, n), t4 = load4(wt_s, p, n);
            const float4 va = load4((const float*)vis_s, 2 * p, 2 * n);
            const float4 vb = load4((const float*)vis_s, 2 * p + 4, 2 * n);
            one(u4.x, v4.x, w4.x, va.x, va.y, t4.x);
            if (p + 1 < n) one(u4.y, v4.y, w4.y, va.z, va.w, t4.y);
            if (p + 2 < n) one(u4.z, v4.z, w4.z, vb.x, vb.y, t4.z);
            if (p + 3 < n) one(u4.w, v4.w, w4.w, vb.z, vb.w, t4.w);
        }
        // end of the ranges: lanes that end on the same cell merge their accumulators, one lane flushes (see k_grid_rec)
        {
            const unsigned kFull = 0xffffffffu;
            const int lane = (int)(threadIdx.x & 31);
            const int up_i = __shfl_up_sync(kFull, ci, 1), up_j = __shfl_up_sync(kFull, cj, 1), up_k = __shfl_up_sync(kFull, ck, 1);
            const bool joins = lane > 0 && ci >= 0 && up_i == ci && up_j == cj && up_k == ck;
            const unsigned heads = ~__ballot_sync(kFull, joins);
            if (heads != kFull) {
                const int start = 31 - __clz((int)(heads & (kFull >> (31 - lane))));
#pragma unroll 1
                for (int d = 1; d < 32; d <<= 1) {
                    const bool take = lane - d >= start;
#pragma unroll
                    for (int r = 0; r < RB; ++r)
#pragma unroll
                        for (int a = 0; a < W; ++a) {
                            const real orr = __shfl_up_sync(kFull, ar[r][a], d), oi = __shfl_up_sync(kFull, ai[r][a], d);
                            if (take) {
                                ar[r][a] += orr;
                                ai[r][a] += oi;
                            }
                        }
                }
                const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
                if (!tail) ci = -1;
            }
        }
        if (ci >= 0) flush();
    }
}

// ---------------------------------------------------------------------------------------------
// fp32 mesh: the record-fed gridder.  A CTA stages its 128 x L gridder records (rick_bin's gather wrote
// them: cell, plane, fractional offsets, signed weight * V; 24 B per visibility in three 8-byte streams)
// into shared memory with coalesced 16-byte cp.async copies, every byte of HBM read exactly once and all
// copies of a CTA in flight together; the second CTA of the SM computes meanwhile.  The 16-byte pieces
// are XOR-swizzled so that the per-thread reads (thread t owns records t*L .. t*L+L-1: that is what
// makes runs) are bank-conflict free.  No fp64 and no global loads inside the accumulation loop.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}

// pieces of a record fetched at random (indirect mode): ask L2 for 64 bytes, not the whole 128-byte line
// (hotspot gridder 40.2 -> 37.7 ms: the random reads share the DRAM with the reductions' read-modify-writes)
__device__ __forceinline__ void cp_async16_rand(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global.L2::64B [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async8_rand(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global.L2::64B [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}

// kIdx = false: the three sorted record streams ga / gb / gc (written by rick_bin's gather).
// kIdx = true (indirect mode, rick_bin without sorted SoA outputs): the record of the sorted visibility at
// position i is the 32-byte staging record grec[gidx[i]] in INPUT order.  A stage's indices are copied to shared
// memory one stage ahead (coalesced 16-byte cp.async), then every record is fetched with one 16-byte and one
// 8-byte cp.async -- 2 x 128 x L random sector reads in flight per SM while the stage before is accumulated.
// The gather of the sort (bound by the GPU's random-access rate) disappears into this kernel.
template <int S, int RB, int L, int NBUF, int KIND, bool kIdx>
__global__ void __launch_bounds__(kRunThreads) k_grid_rec(RickGeom g, TapConst tc, const long long* __restrict__ n_kept,
                                                         const uint2* __restrict__ ga, const float2* __restrict__ gb,
                                                         const float2* __restrict__ gc, const uint32_t* __restrict__ gidx,
                                                         const float4* __restrict__ grec, float2* __restrict__ grid,
                                                         int n_stage, KbPoly kp) {
    constexpr int h = (S - 1) / 2;
    constexpr int kPasses = (S + RB - 1) / RB;
    constexpr int W = S + 1;                    // even-aligned window, see k_grid_runs
    constexpr int PPT = L / 2;                  // 16-byte pieces (two records) per thread, stream and stage
    constexpr int NP = kRunThreads * PPT;       // pieces per stream and stage
    static_assert((L & (L - 1)) == 0 && L >= (kIdx ? 8 : 16), "L: a power of two, >= 16 (>= 8 in indirect mode)");
    extern __shared__ uint4 stage[];            // direct: [2 buffers][3 streams][NP]; indirect: see below
    // indirect layout: A[2][128 L] uint4 (cell, plane, offsets), B[2][128 L] uint2 (weight * V), idx[2][128 L] u32
    constexpr int NR = kRunThreads * L;         // records per stage
    uint4* recA = stage;
    uint2* recB = reinterpret_cast<uint2*>(stage + 2 * NR);
    uint32_t* idxb = reinterpret_cast<uint32_t*>(recB + 2 * NR);
    const long long n = *n_kept;
    const long long per_thread = (long long)L * n_stage;
    const long long cta_first = (long long)blockIdx.x * (kRunThreads * per_thread);
    if (cta_first >= n) return;
    const int tid = threadIdx.x;
    const long long first = cta_first + (long long)tid * per_thread;   // the thread's run of records
    const size_t N = (size_t)g.N;
    const float c2 = (float)(-g.tap_c * 1.4426950408889634);
    const int sw = tid & 7;

    // stage st of every thread's range -> buffer st & 1 (16 lanes copy one thread's 16 * PPT bytes per stream)
    auto issue = [&](int st) {
        uint4* buf = stage + (st % NBUF) * (3 * NP);
#pragma unroll 4
        for (int q = tid; q < NP; q += kRunThreads) {
            const int t = q / PPT, piece = q % PPT;
            const long long rec = cta_first + (long long)t * per_thread + (long long)st * L + 2 * piece;
            if (rec < n) {
                const int phys = q ^ (t & 7);
                cp_async16(buf + phys, (const uint4*)(ga + rec));
                cp_async16(buf + NP + phys, (const uint4*)(gb + rec));
                cp_async16(buf + 2 * NP + phys, (const uint4*)(gc + rec));
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    // indirect mode: the thread's own L indices of stage st (contiguous), and the records of stage st
    auto issue_idx = [&](int st) {
        const long long pos = first + (long long)st * L;
        if (pos < n) {
            uint32_t* dst = idxb + (st & 1) * NR + tid * L;
#pragma unroll
            for (int x = 0; x < L; x += 4) cp_async16(dst + x, gidx + pos + x);
        }
    };
    auto issue_rec = [&](int st) {
        const uint32_t* ib = idxb + (st & 1) * NR;
#pragma unroll 4
        for (int q = tid; q < NR; q += kRunThreads) {
            const int t = q / L, r = q % L;
            const long long pos = cta_first + (long long)t * per_thread + (long long)st * L + r;
            if (pos < n) {
                const float4* src = grec + 2 * (size_t)ib[q];
                // swizzles: a quarter warp's 16-byte reads (a half warp's 8-byte reads) of one r hit distinct banks
                cp_async16_rand(recA + (st & 1) * NR + t * L + (r ^ (t & 7)), src);
                cp_async8_rand(recB + (st & 1) * NR + t * L + (r ^ (t & (L - 1) & 15)), src + 1);
            }
        }
    };

#pragma unroll
    for (int pass = 0; pass < kPasses; ++pass) {
        const int b0 = pass * RB;
        // (re, im) of a cell in one register pair: the accumulation is one packed fma.rn.f32x2 (FFMA2) per cell
        float2 acc[RB][W];
#pragma unroll
        for (int r = 0; r < RB; ++r)
#pragma unroll
            for (int a = 0; a < W; ++a) acc[r][a] = make_float2(0.f, 0.f);
        uint32_t cij = 0xFFFFFFFFu, ck = 0;

        auto flush = [&]() {
            const int iw = (int)(cij & 0xFFFFu), cj = (int)(cij >> 16);   // cij: window column | j0 << 16
            float2* base = grid + ((size_t)ck * N + (size_t)(cj - h + b0)) * N + (size_t)iw;
            const bool edge = iw + W > (int)N;      // the zero column would fall past the row (i0 = N-1-h)
            // every row's address in a register pair of its own: a reduction holds its address register
            // until the memory pipe has taken it, and reusing one pair for all rows stalled each row's
            // address arithmetic behind the last row's reductions (27 % of the kernel's stall samples)
            float2* rowp[RB];
#pragma unroll
            for (int r = 0; r < RB; ++r) rowp[r] = base + (size_t)r * N;
#pragma unroll
            for (int r = 0; r < RB; ++r) asm volatile("" : "+l"(rowp[r]));
            if (!edge) {
#pragma unroll
                for (int r = 0; r < RB; ++r)
                    if (b0 + r < S) {
#pragma unroll
                        for (int a = 0; a < W; a += 2)
                            red_add_pair(rowp[r] + a, acc[r][a].x, acc[r][a].y, acc[r][a + 1].x, acc[r][a + 1].y);
                    }
            } else {
#pragma unroll
                for (int r = 0; r < RB; ++r)
                    if (b0 + r < S) {
#pragma unroll
                        for (int a = 0; a < W; a += 2) {
                            if (a + 2 == W) red_add_cell(rowp[r] + a, acc[r][a].x, acc[r][a].y);
                            else red_add_pair(rowp[r] + a, acc[r][a].x, acc[r][a].y, acc[r][a + 1].x, acc[r][a + 1].y);
                        }
                    }
            }
#pragma unroll
            for (int r = 0; r < RB; ++r)
#pragma unroll
                for (int a = 0; a < W; ++a) acc[r][a] = make_float2(0.f, 0.f);
        };

        auto one = [&](uint32_t ij, uint32_t k, float dx, float dy, float vr, float vi) {
            // the even-aligned window of a cell: cells i0, i0 + 1 with i0 - h even share it, so a run of
            // visibilities on two neighbouring cells accumulates into the same registers
            const uint32_t wij = (ij - (uint32_t)h) & ~1u;          // i0 >= h: no borrow into j0
            if (wij != cij || k != ck) {
                if (cij != 0xFFFFFFFFu) flush();
                cij = wij; ck = k;
            }
            float t[S], gx[W], gy[S];
            if (KIND == RICK_KERNEL_KB) {
                if (kp.ok) {
                    taps_kb_poly<S, true>(gy, dy, kp);
                    taps_kb_poly<S, false>(t, dx, kp);
                } else {
                    taps_kb<S, true>(gy, dy, g);
                    taps_kb<S, false>(t, dx, g);
                }
            } else {
                taps_f32<S, true>(gy, dy, c2, tc);
                taps_f32<S, false>(t, dx, c2, tc);
            }
            const bool o = (((int)(ij & 0xFFFFu) - h) & 1) != 0;     // footprint starts on an odd column
#pragma unroll
            for (int c = 0; c < W; ++c) {
                const float lo = (c >= 1) ? t[c - 1] : 0.f, hi = (c < S) ? t[c] : 0.f;
                const float v = o ? lo : hi;
                gx[c] = (c & 1) ? -v : v;
            }
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                if (b0 + r < S) {
                    const float2 y = cx_scale(gy[b0 + r], make_float2(vr, vi));
#pragma unroll
                    for (int a = 0; a < W; ++a) acc[r][a] = cx_fma_real(gx[a], y, acc[r][a]);
                }
            }
        };

        if (pass > 0) __syncthreads();          // every thread is done with both buffers
        if constexpr (kIdx) {
            issue_idx(0);
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
            issue_rec(0);
            if (1 < n_stage) issue_idx(1);
            asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll 1
            for (int st = 0; st < n_stage; ++st) {
                asm volatile("cp.async.wait_group 0;" ::: "memory");      // records of stage st, indices of stage st + 1
                __syncthreads();
                if (st + 1 < n_stage) {
                    issue_rec(st + 1);
                    if (st + 2 < n_stage) issue_idx(st + 2);
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
                const long long left = n - (first + (long long)st * L);
                const int cnt = left >= L ? L : (left > 0 ? (int)left : 0);
                const uint4* myA = recA + (st & 1) * NR + tid * L;
                const uint2* myB = recB + (st & 1) * NR + tid * L;
                const int swB = tid & (L - 1) & 15;
#pragma unroll 1
                for (int i = 0; i < cnt; ++i) {
                    const uint4 a = myA[i ^ sw];
                    const uint2 c = myB[i ^ swB];
                    one(a.x, a.y, __uint_as_float(a.z), __uint_as_float(a.w), __uint_as_float(c.x), __uint_as_float(c.y));
                }
                __syncthreads();                    // buffer st & 1 is free for stage st + 2
            }
        } else {
        issue(0);
#pragma unroll 1
        for (int st = 0; st < n_stage; ++st) {
            if (NBUF == 2) {
                if (st + 1 < n_stage) issue(st + 1);
                else asm volatile("cp.async.commit_group;" ::: "memory");
                asm volatile("cp.async.wait_group 1;" ::: "memory");
            } else {
                if (st > 0) issue(st);
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            __syncthreads();
            const long long left = n - (first + (long long)st * L);
            const int cnt = left >= L ? L : (left > 0 ? (int)left : 0);
            const uint4* my = stage + (st % NBUF) * (3 * NP) + tid * PPT;
#pragma unroll 1
            for (int i = 0; i < cnt; i += 2) {
                const int piece = (i >> 1) ^ sw;
                const uint4 a = my[piece];
                const uint4 b = my[NP + piece];
                const uint4 c = my[2 * NP + piece];
                one(a.x, a.y, __uint_as_float(b.x), __uint_as_float(b.y), __uint_as_float(c.x), __uint_as_float(c.y));
                if (i + 1 < cnt)
                    one(a.z, a.w, __uint_as_float(b.z), __uint_as_float(b.w), __uint_as_float(c.z), __uint_as_float(c.w));
            }
            __syncthreads();                    // buffer st & 1 is free for stage st + 2
        }
        }
        // End of the ranges.  The lanes of a warp hold consecutive ranges of the sorted records, so where a hot cell
        // spans many ranges (hotspot: 7 600 visibilities per core cell against 256 per range) neighbouring lanes end on
        // the same window: those lanes merge their accumulators (segmented sum over the lanes) and only the last lane
        // of a segment flushes -- one footprint of reductions per warp and hot cell instead of one per lane, all of
        // them aimed at the same few L2 lines.  Warps whose lanes all end on different windows skip this.
        {
            const unsigned kFull = 0xffffffffu;
            const int lane = tid & 31;
            const uint32_t up_ij = __shfl_up_sync(kFull, cij, 1), up_k = __shfl_up_sync(kFull, ck, 1);
            const bool joins = lane > 0 && cij != 0xFFFFFFFFu && up_ij == cij && up_k == ck;
            const unsigned heads = ~__ballot_sync(kFull, joins);            // bit l: lane l starts a segment (bit 0 is set)
            if (heads != kFull) {                                            // warp-uniform
                const int start = 31 - __clz((int)(heads & (kFull >> (31 - lane))));   // first lane of this lane's segment
#pragma unroll 1
                for (int d = 1; d < 32; d <<= 1) {
                    const bool take = lane - d >= start;
#pragma unroll
                    for (int r = 0; r < RB; ++r)
#pragma unroll
                        for (int a = 0; a < W; ++a) {
                            const float ox = __shfl_up_sync(kFull, acc[r][a].x, d), oy = __shfl_up_sync(kFull, acc[r][a].y, d);
                            if (take) {
                                acc[r][a].x += ox;
                                acc[r][a].y += oy;
                            }
                        }
                }
                const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
                if (!tail) cij = 0xFFFFFFFFu;                                // its sum lives on in a later lane
            }
        }
        if (cij != 0xFFFFFFFFu) flush();
    }
}

template <int S, int RB, int KIND, bool kIdx>
int launch_rec_k(rick_plan* p, void* grid, cudaStream_t st) {
    // records per thread and stage; 8 in indirect mode: 57 KB of staging, so that two CTAs stay resident (16: 114 KB,
    // one CTA per SM, measured 48.5 against 40.2 ms on hotspot; a third record buffer -- two stages in flight --
    // 39.0 against 37.7 ms on hotspot, 12.6 against 13.9 ms on 500M: not kept)
    constexpr int L = kIdx ? 8 : 16;
    constexpr int NBUF = 2;                                 // double-buffered stages (1 was measured: no gain)
    // direct: NBUF buffers of three 8-byte streams; indirect: two buffers of 16 + 8 record bytes and 4 index bytes
    constexpr int smem = kIdx ? 2 * kRunThreads * L * (16 + 8 + 4) : NBUF * 3 * kRunThreads * (L / 2) * 16;
    static bool attr_done[RICK_MAX_DEVICES] = {};      // the opt-in is per device
    const int dv = p->device & (RICK_MAX_DEVICES - 1);
    if (!attr_done[dv]) {
        if (cudaFuncSetAttribute(k_grid_rec<S, RB, L, NBUF, KIND, kIdx>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
            return RICK_ECUDA;
        attr_done[dv] = true;
    }
    TapConst tc;
    for (int t = 0; t < 8; ++t) {
        tc.K[t] = exp(-(double)(t * t) * p->g.tap_c);
        tc.Kf[t] = (float)tc.K[t];
    }
    // records per thread: short ranges keep a CTA's threads on neighbouring cells (L2 locality of the reductions)
    // and balance the CTAs; the flushes at their ends cost little since the lanes of a warp merge the windows
    // they share.  Measured with that merge, indirect / direct mode: hotspot 32: 26.1 / --, 64: 25.7 / 17.9,
    // 128: 26.8 / 18.2, 256: 28.1 / 18.8 ms; 500M 32: 10.9 / 8.1, 64: 10.9 / 7.4, 128: 11.6 / 7.0, 256: 12.8 / 7.0 ms.
    constexpr int kMaxRange = kIdx ? 64 : 128;
    const long long want = p->M / ((long long)kRunThreads * p->sm_count * 2 * 12);
    int n_stage = (int)(want / L);
    n_stage = n_stage < 2 ? 2 : (n_stage > kMaxRange / L ? kMaxRange / L : n_stage);
    const long long per_block = (long long)kRunThreads * L * n_stage;
    const unsigned blocks = (unsigned)((p->M + per_block - 1) / per_block);
    KbPoly kp;
    memset(&kp, 0, sizeof(kp));
    if (KIND == RICK_KERNEL_KB && p->kb_poly_ok) {
        memcpy(kp.c, p->kb_poly, sizeof(kp.c));
        kp.ok = 1;
    }
    k_grid_rec<S, RB, L, NBUF, KIND, kIdx><<<blocks, kRunThreads, smem, st>>>(p->g, tc, p->n_kept_dev, p->grec_a, p->grec_b, p->grec_c,
                                                                 p->gidx, p->grec, (float2*)grid, n_stage, kp);
    return RICK_OK;
}

template <typename real, int S, int RB, int KIND>
void launch_runs_k(rick_plan* p, void* grid, cudaStream_t st) {
    typedef typename CellOf<real>::type cell;
    TapConst tc;
    for (int t = 0; t < 8; ++t) {
        tc.K[t] = exp(-(double)(t * t) * p->g.tap_c);
        tc.Kf[t] = (float)tc.K[t];
    }
    // consecutive sorted visibilities per thread: as for the record gridder (100M: 64: 5.72, 128: 5.57, 256: 5.85 ms)
    long long L = p->M / ((long long)kRunThreads * p->sm_count * 2 * 12) / 4 * 4;
    L = L < 32 ? 32 : (L > 128 ? 128 : L);
    const long long per_block = (long long)kRunThreads * L;
    const unsigned blocks = (unsigned)((p->M + per_block - 1) / per_block);
    k_grid_runs<real, S, RB, KIND><<<blocks, kRunThreads, 0, st>>>(p->g, tc, p->n_kept_dev, p->u_s, p->v_s, p->w_s,
                                                              (const float2*)p->vis_s, p->weight_s, (cell*)grid, (int)L);
}

template <int S, int RB>
int launch_rec(rick_plan* p, void* grid, cudaStream_t st) {
    if (p->indirect)
        return p->g.kernel == RICK_KERNEL_KB ? launch_rec_k<S, RB, RICK_KERNEL_KB, true>(p, grid, st)
                                             : launch_rec_k<S, RB, RICK_KERNEL_GAUSS, true>(p, grid, st);
    return p->g.kernel == RICK_KERNEL_KB ? launch_rec_k<S, RB, RICK_KERNEL_KB, false>(p, grid, st)
                                         : launch_rec_k<S, RB, RICK_KERNEL_GAUSS, false>(p, grid, st);
}
template <typename real, int S, int RB>
void launch_runs(rick_plan* p, void* grid, cudaStream_t st) {
    if (p->g.kernel == RICK_KERNEL_KB) launch_runs_k<real, S, RB, RICK_KERNEL_KB>(p, grid, st);
    else launch_runs_k<real, S, RB, RICK_KERNEL_GAUSS>(p, grid, st);
}

}  // namespace

int rick_grid_impl(rick_plan* p, void* grid, cudaStream_t st) {
    if (p->M == 0) return RICK_OK;
    const bool f64 = (p->dtype == RICK_C128);
    // <real, S, RB>: RB rows of the footprint are held in registers per pass
    int rc = RICK_OK;
    switch (p->g.S) {
        case 3:  if (f64) launch_runs<double, 3, 3>(p, grid, st);  else rc = launch_rec<3, 3>(p, grid, st); break;
        case 5:  if (f64) launch_runs<double, 5, 5>(p, grid, st);  else rc = launch_rec<5, 5>(p, grid, st); break;
        case 7:  if (f64) launch_runs<double, 7, 7>(p, grid, st);  else rc = launch_rec<7, 7>(p, grid, st); break;
        case 9:  if (f64) launch_runs<double, 9, 3>(p, grid, st);  else rc = launch_rec<9, 9>(p, grid, st); break;
        case 11: if (f64) launch_runs<double, 11, 2>(p, grid, st); else rc = launch_rec<11, 4>(p, grid, st); break;
        case 13: if (f64) launch_runs<double, 13, 2>(p, grid, st); else rc = launch_rec<13, 3>(p, grid, st); break;
        case 15: if (f64) launch_runs<double, 15, 2>(p, grid, st); else rc = launch_rec<15, 3>(p, grid, st); break;
        default: return RICK_EINVAL;
    }
    if (rc != RICK_OK) return rc;
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
