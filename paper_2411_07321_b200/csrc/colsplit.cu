// colsplit.cu -- split column transform: the column half of D7 in two sweeps, the second fused with D8
// (phase screen, plane sum, taper), for the meshes whose columns do not fit one SM: N = 4096 .. 16384, and
// every N = 256 .. 16384 of the fp64 mesh.  (N <= 2048 on the fp32 mesh keeps the one-sweep kernel of colfft.cu.)
//
// A column of N = N1 N2 mesh rows, j = N2 j1 + j2, transforms to frequencies q = q1 + N1 q2 as
//
//     X[q1 + N1 q2] = sum_j2  W_N2^(j2 q2)  .  W_N^(j2 q1)  sum_j1 x[N2 j1 + j2] W_N1^(j1 q1)        W_n = exp(+2 pi i / n)
//                     `------ sweep B -----'   `------------------- sweep A ----------------------'
//
// Sweep A (k_col_a, part of rick_fft_planes, after the row transforms): for every plane, every j2 and every
// block of C adjacent columns, the N1 rows j2, j2 + N2, j2 + 2 N2 ... are loaded straight into registers
// (a warp reads 256 contiguous bytes of one row per instruction), transformed (two radix passes, one trip
// through shared memory), multiplied by W_N^(j2 q1) and written back in place.  In fusion mode 2 only rows
// some footprint touched are read (the others count as zero); every row is written, so the mesh is dense
// afterwards.
// Sweep B (k_col_b, rick_wcorrect_accumulate): a CTA owns N2 CONSECUTIVE rows (one q1) of C adjacent columns.
// Plane after plane it pulls that N2 x C tile into shared memory with one 256-byte bulk copy per row
// (cp.async.bulk, completion on an mbarrier; double-buffered against the next plane), runs the N2-point
// transforms, multiplies every output by the phase screen exp(+2 pi i w_k nm1(q, p)) (Eq. 2) and adds the
// real part to fp64 accumulators that stay in registers for all planes; then (-1)^(p+q), taper, one write.
// The transformed planes are never stored: sweeps over the mesh are rows (r+w), A (r+w), B (r) instead of
// the library's rows + two column sweeps (3 x r+w) followed by the w-correction's read.
//
// Outputs of both sub-transforms are left in digit-reversed order in place (slot u R2 + q' holds frequency
// u + R1 q'); sweep B only needs to know which q1 its row block holds and which image row each output is.
#include "fft_radix.cuh"
#include "rick_internal.cuh"

namespace {

// L-point transform = radix R1 pass, then radix R2 pass (R2 = 1: single pass)
template <int L> struct Split;
template <> struct Split<16> { static constexpr int R1 = 16, R2 = 1; };
template <> struct Split<32> { static constexpr int R1 = 8, R2 = 4; };
template <> struct Split<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct Split<128> { static constexpr int R1 = 16, R2 = 8; };

template <typename C2> struct ColsOf { static constexpr int C = 256 / (int)sizeof(C2); };   // 256-byte row pieces

// slot (position in the transformed order) -> frequency, for an L-point split transform
template <int L> __host__ __device__ constexpr int slot_freq(int slot) {
    return Split<L>::R2 == 1 ? slot : (slot / Split<L>::R2) + Split<L>::R1 * (slot % Split<L>::R2);
}

// streaming load of one complex value when `live`, else zero -- predicated, no branch
template <typename C2> RICK_DI C2 ldg_cx_if(const C2* p, bool live);
template <> RICK_DI float2 ldg_cx_if<float2>(const float2* p, bool live) {
    float2 r;
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
                 "mov.f32 %0, 0f00000000;\n\tmov.f32 %1, 0f00000000;\n\t"
                 "@q ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];\n\t}"
                 : "=&f"(r.x), "=&f"(r.y) : "l"(p), "r"((unsigned)live));
    return r;
}
template <> RICK_DI double2 ldg_cx_if<double2>(const double2* p, bool live) {
    double2 r;
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
                 "mov.f64 %0, 0d0000000000000000;\n\tmov.f64 %1, 0d0000000000000000;\n\t"
                 "@q ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];\n\t}"
                 : "=&d"(r.x), "=&d"(r.y) : "l"(p), "r"((unsigned)live));
    return r;
}

// First pass of the L-point transforms of a tile: thread (g, c) owns butterfly m = g of column c, elements
// m + t R2.  Leaves y_u W_L^(m u) in v[u] (slot m + u R2).
template <int L, typename C2> RICK_DI void first_pass(C2* v, const C2* twL, int g) {
    constexpr int R1 = Split<L>::R1, R2 = Split<L>::R2;
    cx_dft<R1>(v);
    if constexpr (R2 > 1) {
#pragma unroll
        for (int u = 1; u < R1; ++u) v[u] = cx_mul(v[u], twL[g * u]);
    }
}

// ---------------------------------------------------------------------------------------------
// Sweep A.  N = N1 N2 is a compile-time constant: every row stride below is an immediate.
// ---------------------------------------------------------------------------------------------
template <typename C2, int N1, int N2>
__global__ void __launch_bounds__(N1 * ColsOf<C2>::C / Split<N1>::R1)
k_col_a(C2* __restrict__ planes, const C2* __restrict__ tw_g, const uint32_t* __restrict__ occ) {
    constexpr int L = N1, N = N1 * N2;
    constexpr int R1 = Split<L>::R1, R2 = Split<L>::R2, C = ColsOf<C2>::C;
    constexpr int T = L * C / R1;
    constexpr size_t rstride = (size_t)N2 * N;                          // mesh rows j2 + N2 j1 are N2 rows apart
    __shared__ C2 tile[R2 > 1 ? L * C : 1];
    __shared__ C2 twL[L];
    __shared__ C2 twq[L];                                               // W_N^(j2 q1), q1 < N1
    const int tid = threadIdx.x, c = tid % C, g = tid / C;
    const int j2 = blockIdx.y, k = blockIdx.z;
    C2* base = planes + ((size_t)k * N + j2) * N + (size_t)blockIdx.x * C + c;
    C2 v[R1];
    {
        bool live[R1];
#pragma unroll
        for (int t = 0; t < R1; ++t) {
            live[t] = true;
            if (occ) {
                const uint32_t r = (uint32_t)k * (uint32_t)N + (uint32_t)(N2 * (g + t * R2) + j2);
                live[t] = (__ldg(occ + (r >> 5)) >> (r & 31)) & 1u;
            }
        }
#pragma unroll
        for (int t = 0; t < R1; ++t) v[t] = ldg_cx_if(base + (size_t)(g + t * R2) * rstride, live[t]);
    }
    for (int i = tid; i < L; i += T) {
        twL[i] = tw_g[i * N2];                                          // W_L^i = W_N^(i N / L)
        twq[i] = tw_g[(j2 * i) & (N - 1)];
    }
    __syncthreads();
    first_pass<L>(v, twL, g);
    if constexpr (R2 == 1) {
#pragma unroll
        for (int u = 0; u < R1; ++u) base[(size_t)u * rstride] = cx_mul(v[u], twq[u]);      // slot u = frequency u
    } else {
#pragma unroll
        for (int u = 0; u < R1; ++u) tile[(g + u * R2) * C + c] = v[u];
        __syncthreads();
        // second pass: blocks u = g + R2 i of R2 consecutive slots
#pragma unroll
        for (int i = 0; i < R1 / R2; ++i) {
            const int u = g + R2 * i;
            C2 w[R2];
#pragma unroll
            for (int s = 0; s < R2; ++s) w[s] = tile[(u * R2 + s) * C + c];
            cx_dft<R2>(w);
#pragma unroll
            for (int s = 0; s < R2; ++s)                                // slot u R2 + s holds q1 = u + R1 s
                base[(size_t)(u * R2 + s) * rstride] = cx_mul(w[s], twq[u + R1 * s]);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Sweep B: bulk-copy pipeline (TMA unit, SASS UBLKCP) + N2-point transforms + phase screen + plane sum
// ---------------------------------------------------------------------------------------------
RICK_DI unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

RICK_DI void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
RICK_DI void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
RICK_DI bool mbar_try_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// global -> shared bulk copy of `bytes` (a multiple of 16, both addresses 16-byte aligned), completion on `bar`
RICK_DI void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// per-output state of the phase screen
template <typename real, int E> struct Screen;
// fp32 mesh: nm1 kept in fp64, the fraction of w_k nm1 rounded to 2^-23 turn without the conversion pipe,
// hardware sine / cosine on the reduced argument (same arithmetic as k_colfft_wcorrect, colfft.cu)
template <int E> struct Screen<float, E> {
    double nm1[E];
    RICK_DI void init(int e, double nm1v, const RickGeom&) { nm1[e] = nm1v; }
    RICK_DI double term(int e, float2 v, double wk) {
        const double z = fma(wk, nm1[e], 805306368.0);                     // 1.5 * 2^29: fraction in the low 23 bits
        uint32_t gbits;                                                     // 1 + fraction: (lo & mantissa) | one, one LOP3
        asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(gbits) : "r"((uint32_t)__double2loint(z)), "r"(0x007FFFFFu), "r"(0x3F800000u));
        const float gq = __uint_as_float(gbits);
        // 2 pi (fraction - 1/2), in [-pi, pi): one FFMA (rounding: 2^-24 pi rad, below the 2^-23-turn phase step)
        const float t = fmaf(gq, 6.283185307179586f, -9.42477796076938f);
        float sn, cs;
        __sincosf(t, &sn, &cs);
        return (double)(sn * v.y - cs * v.x);                              // the half turn negates sine and cosine
    }
    RICK_DI void next(int) {}
};
// fp64 mesh: exp(2 pi i (w_0 + k dw) nm1) advanced by one complex rotation per plane (as k_wcorrect_c128)
template <int E> struct Screen<double, E> {
    double c[E], s[E], cs[E], ss[E];
    RICK_DI void init(int e, double nm1v, const RickGeom& g) {
        double t0 = (g.w_min + 0.5 * g.dw) * nm1v;
        t0 -= floor(t0);
        double t1 = g.dw * nm1v;
        t1 -= floor(t1);
        sincospi(2.0 * t0, &s[e], &c[e]);
        sincospi(2.0 * t1, &ss[e], &cs[e]);
    }
    RICK_DI double term(int e, double2 v, double) { return c[e] * v.x - s[e] * v.y; }
    RICK_DI void next(int e) {
        const double n = c[e] * cs[e] - s[e] * ss[e];
        s[e] = c[e] * ss[e] + s[e] * cs[e];
        c[e] = n;
    }
};

template <typename real> RICK_DI double nm1_of(double r2);
template <> RICK_DI double nm1_of<float>(double r2) { return rick_nm1_fast(r2); }
template <> RICK_DI double nm1_of<double>(double r2) { return -r2 / (1.0 + sqrt(1.0 - r2)); }

template <typename C2, int L> struct ColB {
    static constexpr int R1 = Split<L>::R1, R2 = Split<L>::R2, C = ColsOf<C2>::C;
    static constexpr int T = L * C / R1;
    static constexpr int kIssuers = L < T ? L : T;                // threads that issue row copies
    static constexpr int kRowsPerIssuer = L / kIssuers;
    static constexpr size_t smem = 2 * sizeof(C2) * L * C + sizeof(C2) * L + 2 * sizeof(unsigned long long);
    // resident CTAs the register allocation must leave room for: three (of 256 threads: 80 registers, the fp64 sums
    // and n - 1 values partly in local memory, but 24 instead of 16 warps per SM: hotspot 9.45 -> 9.15 ms, 500M 4.39 ->
    // 4.36 ms; shared memory, 66 KB per CTA at N2 = 128, allows no more); the 128-row fp64 tile fits once
    static constexpr int kMinBlocks = (sizeof(C2) == 16 && L == 128) ? 1 : 3;
};

template <typename C2, int N1, int N2>
__global__ void __launch_bounds__(ColB<C2, N2>::T, ColB<C2, N2>::kMinBlocks)
k_col_b(RickGeom g, const C2* __restrict__ planes, const C2* __restrict__ tw_g, const double* __restrict__ inv_t,
        double* __restrict__ image, int accumulate, int col_first) {
    typedef typename RickRealOf<C2>::type real;
    constexpr int L = N2, N = N1 * N2;
    typedef ColB<C2, L> P;
    constexpr int R1 = P::R1, R2 = P::R2, C = P::C, T = P::T, E = R1;
    constexpr size_t plane_cells = (size_t)N * N;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C2* buf0 = reinterpret_cast<C2*>(smem_raw);
    C2* buf1 = buf0 + L * C;
    C2* twL = buf1 + L * C;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(twL + L);
    const int tid = threadIdx.x, c = tid % C, gq = tid / C;
    const int b = blockIdx.y;                                       // block of L consecutive mesh rows
    const int q1 = slot_freq<N1>(b);                                // the frequency sweep A left there
    const int col0 = col_first + blockIdx.x * C, p = col0 + c;     // col_first: first column of this launch's part of the image
    const C2* src0 = planes + (size_t)b * L * N + col0;             // row 0 of the tile in plane 0

    if (tid == 0) {
        mbar_init(bar + 0, P::kIssuers);
        mbar_init(bar + 1, P::kIssuers);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < L; i += T) twL[i] = tw_g[i * N1];         // W_L^i = W_N^(i N / L)
    __syncthreads();

    auto issue = [&](int k) {
        if (tid < P::kIssuers) {
            C2* dst = (k & 1) ? buf1 : buf0;
            mbar_arrive_expect_tx(bar + (k & 1), 256u * P::kRowsPerIssuer);
#pragma unroll
            for (int r = 0; r < P::kRowsPerIssuer; ++r) {
                const int row = tid + r * P::kIssuers;
                bulk_g2s(dst + row * C, src0 + (size_t)k * plane_cells + (size_t)row * N, 256u, bar + (k & 1));
            }
        }
    };
    issue(0);
    if (g.Nw > 1) issue(1);

    Screen<real, E> scr;
    double acc[E];
    // output e of this thread: R2 > 1: e = i R2 + s: block u = gq + R2 i, slot u R2 + s, q2 = u + R1 s; R2 = 1: q2 = e
    auto out_q = [&](int e) {
        const int q2 = R2 == 1 ? e : (gq + R2 * (e / R2)) + R1 * (e % R2);
        return q1 + N1 * q2;
    };
    {
        const double l = (double)(p - N / 2) * g.dl, l2 = l * l;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double m = (double)(out_q(e) - N / 2) * g.dl;
            scr.init(e, nm1_of<real>(fma(m, m, l2)), g);
            acc[e] = 0.0;
        }
    }

    for (int k = 0; k < g.Nw; ++k) {
        C2* buf = (k & 1) ? buf1 : buf0;
        const unsigned parity = (unsigned)(k >> 1) & 1u;
        while (!mbar_try_wait(bar + (k & 1), parity)) {}
        const double wk = g.w_min + ((double)k + 0.5) * g.dw;
        C2 v[R1];
#pragma unroll
        for (int t = 0; t < R1; ++t) v[t] = buf[(gq + t * R2) * C + c];
        first_pass<L>(v, twL, gq);
        if constexpr (R2 == 1) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                acc[e] += scr.term(e, v[e], wk);
                scr.next(e);
            }
        } else {
#pragma unroll
            for (int u = 0; u < R1; ++u) buf[(gq + u * R2) * C + c] = v[u];
            __syncthreads();
#pragma unroll
            for (int i = 0; i < R1 / R2; ++i) {
                const int u = gq + R2 * i;
                C2 w[R2];
#pragma unroll
                for (int s = 0; s < R2; ++s) w[s] = buf[(u * R2 + s) * C + c];
                cx_dft<R2>(w);
#pragma unroll
                for (int s = 0; s < R2; ++s) {
                    acc[i * R2 + s] += scr.term(i * R2 + s, w[s], wk);
                    scr.next(i * R2 + s);
                }
            }
        }
        // every thread is done with this buffer (its own generic-proxy writes included) before the bulk copy
        // of plane k + 2 overwrites it through the async proxy
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (k + 2 < g.Nw) issue(k + 2);
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int q = out_q(e);
        const double sg = ((p + q) & 1) ? -1.0 : 1.0;
        double out = acc[e] * (sg * inv_t[q] * inv_t[p]);
        const size_t o = (size_t)q * N + p;
        if (accumulate) out += image[o];
        image[o] = out;
    }
}

template <typename C2, int N1, int N2>
int launch_a(rick_plan* p, void* grid, cudaStream_t st) {
    constexpr int C = ColsOf<C2>::C, T = N1 * C / Split<N1>::R1, N = N1 * N2;
    const dim3 blocks((unsigned)(N / C), (unsigned)N2, (unsigned)p->g.Nw);
    const uint32_t* occ = p->fused == 2 ? p->occ_mesh_dev : nullptr;
    k_col_a<C2, N1, N2><<<blocks, T, 0, st>>>((C2*)grid, (const C2*)p->split_tw, occ);
    return RICK_OK;
}

template <typename C2, int N1, int N2>
int launch_b(rick_plan* p, const void* grid, double* image, int accumulate, cudaStream_t st, int col_lo, int col_hi) {
    typedef ColB<C2, N2> P;
    constexpr int N = N1 * N2;
    static bool attr_done[RICK_MAX_DEVICES] = {};
    bool& done = attr_done[p->device & (RICK_MAX_DEVICES - 1)];
    if (!done) {
        if (cudaFuncSetAttribute(k_col_b<C2, N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem) != cudaSuccess)
            return RICK_ECUDA;
        done = true;
    }
    if (col_hi < 0) col_hi = N;
    if (col_lo < 0 || col_hi > N || col_lo >= col_hi || (col_lo % P::C) || (col_hi % P::C)) return RICK_EINVAL;
    const dim3 blocks((unsigned)((col_hi - col_lo) / P::C), (unsigned)N1);
    k_col_b<C2, N1, N2><<<blocks, P::T, P::smem, st>>>(p->g, (const C2*)grid, (const C2*)p->split_tw, p->inv_taper_dev,
                                                        image, accumulate, col_lo);
    return RICK_OK;
}

// the (N1, N2) pairs of N = 256 .. 16384
#define RICK_SPLIT_DISPATCH(CALL)                                            \
    switch (p->g.N) {                                                        \
        case 256: return CALL(16, 16);                                       \
        case 512: return CALL(16, 32);                                       \
        case 1024: return CALL(32, 32);                                      \
        case 2048: return CALL(32, 64);                                      \
        case 4096: return CALL(64, 64);                                      \
        case 8192: return CALL(64, 128);                                     \
        case 16384: return CALL(128, 128);                                   \
        default: return RICK_EINVAL;                                         \
    }

template <typename C2>
int sweep_a(rick_plan* p, void* grid, cudaStream_t st) {
#define RICK_CALL_A(n1, n2) launch_a<C2, n1, n2>(p, grid, st)
    RICK_SPLIT_DISPATCH(RICK_CALL_A)
#undef RICK_CALL_A
}
template <typename C2>
int sweep_b(rick_plan* p, const void* grid, double* image, int accumulate, cudaStream_t st, int col_lo, int col_hi) {
#define RICK_CALL_B(n1, n2) launch_b<C2, n1, n2>(p, grid, image, accumulate, st, col_lo, col_hi)
    RICK_SPLIT_DISPATCH(RICK_CALL_B)
#undef RICK_CALL_B
}

}  // namespace

// N = N1 N2 with N2 = 2^ceil(log2(N)/2) consecutive rows per sweep-B tile; both factors in 16 .. 128
bool rick_colsplit_supported(const rick_plan* p) {
    const int N = p->g.N;
    if (N < 256 || N > 16384 || (N & (N - 1))) return false;
    if (p->dtype == RICK_C64) {
        // the fp32 screen takes the fraction of w_k nm1 from the low mantissa bits of w_k nm1 + 1.5 * 2^29
        const double w_abs = fmax(fabs(p->g.w_min), fabs(p->g.w_max));
        if (!(w_abs < 268435456.0)) return false;
    }
    return true;
}

int rick_colsplit_init(rick_plan* p) {
    const int N = p->g.N;
    int n = 0;
    while ((1 << n) < N) ++n;
    p->split_N2 = 1 << ((n + 1) / 2);
    p->split_N1 = N / p->split_N2;
    // twiddles exp(+2 pi i j / N) in the mesh's precision, fp64 values rounded once
    const bool f64 = p->dtype == RICK_C128;
    const size_t bytes = (f64 ? sizeof(double2) : sizeof(float2)) * (size_t)N;
    void* h = malloc(bytes);
    if (!h) return RICK_ENOMEM;
    const double two_pi = 6.283185307179586476925286766559;
    for (int j = 0; j < N; ++j) {
        const double cs = cos(two_pi * j / N), sn = sin(two_pi * j / N);
        if (f64) ((double2*)h)[j] = make_double2(cs, sn);
        else ((float2*)h)[j] = make_float2((float)cs, (float)sn);
    }
    if (p->split_tw) { cudaFree(p->split_tw); p->split_tw = nullptr; }
    cudaError_t e = cudaMalloc(&p->split_tw, bytes);
    if (e == cudaSuccess) e = cudaMemcpy(p->split_tw, h, bytes, cudaMemcpyHostToDevice);
    free(h);
    return e == cudaSuccess ? RICK_OK : (e == cudaErrorMemoryAllocation ? RICK_ENOMEM : RICK_ECUDA);
}

// sweep A, in place on the row-transformed mesh (rick_fft_planes)
int rick_colsplit_a_impl(rick_plan* p, void* grid, cudaStream_t st) {
    const int rc = p->dtype == RICK_C128 ? sweep_a<double2>(p, grid, st) : sweep_a<float2>(p, grid, st);
    if (rc != RICK_OK) return rc;
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}

// sweep B + phase screen + plane sum + taper (rick_wcorrect_accumulate) for the image columns [col_lo, col_hi)
// (multiples of 64; col_hi < 0: all): the chunked host entry copies one part out while the next is computed
int rick_colsplit_b_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st, int col_lo,
                         int col_hi) {
    const int acc = zero_first ? 0 : 1;
    const int rc = p->dtype == RICK_C128 ? sweep_b<double2>(p, grid, image, acc, st, col_lo, col_hi)
                                         : sweep_b<float2>(p, grid, image, acc, st, col_lo, col_hi);
    if (rc != RICK_OK) return rc;
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
