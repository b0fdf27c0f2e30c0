// rowbig.cu -- row transforms of the listed mesh rows for N = 4096 .. 16384 (fusion mode 2): the row half of D7
// on the rows some footprint touched only (51 .. 59 % of the rows of configs 3 - 5), one whole row per CTA
// in shared memory, natural order in and out, one read and one write of the row.
//
// The row of N = N1 N2 elements is the matrix [j1][j2] (j2 contiguous), and
//     X[q1 + N1 q2] = sum_j2 W_N2^(j2 q2) . W_N^(j2 q1) sum_j1 x[N2 j1 + j2] W_N1^(j1 q1)
// Step 1 (over j1, lanes over j2): global -> registers (coalesced), two radix passes with one exchange through
// shared memory in the natural layout; its results, times W_N^(j2 q1), are written TRANSPOSED with pitch N1 + 1
// (layout [j2][q1]: bank-conflict free for lanes over j2 on the write and for lanes over q1 afterwards).
// Step 2 (over j2, lanes over q1): two radix passes in place, the last straight to global memory, where a warp
// writes 32 consecutive frequencies q1 + N1 q2.
// A thread holds 32 elements; the twiddles W_N^(j2 q1) of its elements do not depend on the row: W_N^(j2 u) per
// butterfly and the powers of W_N^(j2 R1) stay in registers for all rows of the CTA.
// Segment occupancy (rows.cu): of a listed row only the segments (N / 64 cells each) some footprint touched hold
// defined data; the others are not read (nor prefetched) and count as zeros.  A segment is N1 / 64 whole lines j1 of
// the matrix, so the test is uniform over a warp.  The row is written whole.
#include "fft_radix.cuh"
#include "rick_internal.cuh"

namespace {

template <int L> struct Split;      // same factorisations as colsplit.cu
template <> struct Split<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct Split<128> { static constexpr int R1 = 16, R2 = 8; };

template <typename C2, int N1, int N2> struct RowBig {
    static constexpr int N = N1 * N2, T = N / 32;
    static constexpr int PB = N1 + 1;                                  // pitch of the transposed layout
    static constexpr size_t elems = (size_t)N2 * PB;                   // >= N
    static constexpr size_t smem = sizeof(C2) * (elems + N1 + N2);
    // resident CTAs per SM the register allocation leaves room for: by shared memory, at 128 (fp32) / 255 (fp64) registers per thread
    static constexpr int kBySmem = (int)((227 * 1024) / (smem + 1024));
    static constexpr int kByRegs = 65536 / (T * (sizeof(C2) == 16 ? 255 : 128));      // 32 complex values per thread: 64 / 128 registers
    static constexpr int kMinBlocks = kBySmem < kByRegs ? (kBySmem < 1 ? 1 : kBySmem) : (kByRegs < 1 ? 1 : kByRegs);
};

// streaming load of one complex value when `live`, else zero -- predicated, no branch
template <typename C2> RICK_DI C2 ldg_stream_if(const C2* p, bool live);
template <> RICK_DI float2 ldg_stream_if<float2>(const float2* p, bool live) {
    float2 r;
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
                 "mov.f32 %0, 0f00000000;\n\tmov.f32 %1, 0f00000000;\n\t"
                 "@q ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];\n\t}"
                 : "=&f"(r.x), "=&f"(r.y) : "l"(p), "r"((unsigned)live));
    return r;
}
template <> RICK_DI double2 ldg_stream_if<double2>(const double2* p, bool live) {
    double2 r;
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
                 "mov.f64 %0, 0d0000000000000000;\n\tmov.f64 %1, 0d0000000000000000;\n\t"
                 "@q ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];\n\t}"
                 : "=&d"(r.x), "=&d"(r.y) : "l"(p), "r"((unsigned)live));
    return r;
}

// asks the L2 for `bytes` (a multiple of 16) at p: no register, no completion to wait for
RICK_DI void prefetch_l2(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

template <typename C2, int N1, int N2>
__global__ void __launch_bounds__(RowBig<C2, N1, N2>::T, RowBig<C2, N1, N2>::kMinBlocks)
k_row_big(C2* __restrict__ planes, const C2* __restrict__ tw_g, const uint32_t* __restrict__ list,
          const uint32_t* __restrict__ n_rows, const unsigned long long* __restrict__ seg) {
    typedef RowBig<C2, N1, N2> P;
    constexpr int N = P::N, T = P::T, PB = P::PB;
    constexpr int Ra1 = Split<N1>::R1, Ra2 = Split<N1>::R2, Rb1 = Split<N2>::R1, Rb2 = Split<N2>::R2;
    static_assert(T % N2 == 0 && T % N1 == 0, "a thread keeps its j2 (step 1) and its q1 (step 2) for all butterflies");
    static_assert(N1 % 64 == 0 && N2 % 32 == 0, "a segment (N / 64 cells) is N1 / 64 whole lines j1, and a warp stays within one line");
    constexpr int kSegLines = N1 / 64;                                // lines j1 per segment
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C2* buf = reinterpret_cast<C2*>(smem_raw);
    C2* twA = buf + P::elems;           // W_N1^i
    C2* twB = twA + N1;                 // W_N2^i
    const int tid = threadIdx.x;
    const int n = (int)*n_rows;
    if ((int)blockIdx.x >= n) return;
    for (int i = tid; i < N1; i += T) twA[i] = tw_g[i * N2];
    for (int i = tid; i < N2; i += T) twB[i] = tw_g[i * N1];
    // step 1: j2 = tid % N2; pass 1 butterflies m = tid / N2 + i T / N2 (m < Ra2); pass 2 blocks u likewise (u < Ra1)
    const int j2 = tid % N2, a0 = tid / N2;
    constexpr int aStep = T / N2;
    // step 2: q1 = tid % N1; pass 1 butterflies m = tid / N1 + i T / N1 (m < Rb2); pass 2 blocks u likewise (u < Rb1)
    const int q1 = tid % N1, b0 = tid / N1;
    constexpr int bStep = T / N1;
    // row-independent twiddles of this thread's step-1 outputs: W_N^(j2 (u + Ra1 s)) = base[i] * pw[s]
    C2 base[32 / Ra2], pw[Ra2];
#pragma unroll
    for (int i = 0; i < 32 / Ra2; ++i) base[i] = tw_g[(j2 * (a0 + i * aStep)) & (N - 1)];
#pragma unroll
    for (int s = 0; s < Ra2; ++s) pw[s] = tw_g[(j2 * Ra1 * s) & (N - 1)];
    __syncthreads();

    // the inputs of the first pass (radix Ra1 over j1 = m + t Ra2) come straight from global memory; the next row's
    // are requested as soon as this row's last butterflies have left the registers, before the closing barrier
    C2 v[32];
    auto fetch = [&](uint32_t row, unsigned long long segs) {
        const C2* x = planes + (size_t)row * N;
#pragma unroll
        for (int i = 0; i < 32 / Ra1; ++i) {
            const int m = a0 + i * aStep;
#pragma unroll
            for (int t = 0; t < Ra1; ++t) {
                const int j1 = m + t * Ra2;
                v[i * Ra1 + t] = ldg_stream_if(x + j1 * N2 + j2, (segs >> (j1 / kSegLines)) & 1ull);
            }
        }
    };
    // row numbers and segment masks run one row ahead of the loads, which run one row ahead of the arithmetic
    const int G = (int)gridDim.x;
    uint32_t row_cur = __ldg(list + blockIdx.x), row_nxt = 0;
    unsigned long long m_nxt = 0;
    if ((int)blockIdx.x + G < n) {
        row_nxt = __ldg(list + blockIdx.x + G);
        m_nxt = seg ? __ldg(seg + row_nxt) : ~0ull;
    }
    fetch(row_cur, seg ? __ldg(seg + row_cur) : ~0ull);
    for (int r = blockIdx.x; r < n; r += G) {
        C2* x = planes + (size_t)row_cur * N;
        // the defined segments of the row after this one travel from DRAM to the L2 while this one is transformed: the
        // loads at the end of the loop body then wait for the L2 only (one warp asks, two segments per lane)
        if (tid < 32 && r + G < n) {
            const C2* xn = planes + (size_t)row_nxt * N + (size_t)tid * (N / 32);
            if ((m_nxt >> (2 * tid)) & 1ull) prefetch_l2(xn, (unsigned)(sizeof(C2) * (N / 64)));
            if ((m_nxt >> (2 * tid + 1)) & 1ull) prefetch_l2(xn + N / 64, (unsigned)(sizeof(C2) * (N / 64)));
        }
        uint32_t row_n2 = 0;
        unsigned long long m_n2 = 0;
        if (r + 2 * G < n) {
            row_n2 = __ldg(list + r + 2 * G);
            m_n2 = seg ? __ldg(seg + row_n2) : ~0ull;
        }
        // ---- step 1, pass 1
#pragma unroll
        for (int i = 0; i < 32 / Ra1; ++i) {
            const int m = a0 + i * aStep;
            cx_dft<Ra1>(v + i * Ra1);
#pragma unroll
            for (int u = 1; u < Ra1; ++u) v[i * Ra1 + u] = cx_mul(v[i * Ra1 + u], twA[m * u]);
#pragma unroll
            for (int u = 0; u < Ra1; ++u) buf[(m + u * Ra2) * N2 + j2] = v[i * Ra1 + u];
        }
        __syncthreads();
        // ---- step 1, pass 2: radix Ra2 over the slots u Ra2 + s; result q1 = u + Ra1 s, times W_N^(j2 q1), transposed
#pragma unroll
        for (int i = 0; i < 32 / Ra2; ++i) {
            const int u = a0 + i * aStep;
#pragma unroll
            for (int s = 0; s < Ra2; ++s) v[i * Ra2 + s] = buf[(u * Ra2 + s) * N2 + j2];
        }
        __syncthreads();                         // the natural layout is dead: the transposed one takes its place
#pragma unroll
        for (int i = 0; i < 32 / Ra2; ++i) {
            const int u = a0 + i * aStep;
            cx_dft<Ra2>(v + i * Ra2);
#pragma unroll
            for (int s = 0; s < Ra2; ++s)
                buf[j2 * PB + (u + Ra1 * s)] = cx_mul(v[i * Ra2 + s], cx_mul(base[i], pw[s]));
        }
        __syncthreads();
        // ---- step 2, pass 1: radix Rb1 over j2 = m + t Rb2, in place
#pragma unroll
        for (int i = 0; i < 32 / Rb1; ++i) {
            const int m = b0 + i * bStep;
#pragma unroll
            for (int t = 0; t < Rb1; ++t) v[i * Rb1 + t] = buf[(m + t * Rb2) * PB + q1];
            cx_dft<Rb1>(v + i * Rb1);
#pragma unroll
            for (int u = 1; u < Rb1; ++u) v[i * Rb1 + u] = cx_mul(v[i * Rb1 + u], twB[m * u]);
#pragma unroll
            for (int u = 0; u < Rb1; ++u) buf[(m + u * Rb2) * PB + q1] = v[i * Rb1 + u];
        }
        __syncthreads();
        // ---- step 2, pass 2: radix Rb2 over the slots u Rb2 + s; frequency q1 + N1 (u + Rb1 s), to global memory
#pragma unroll
        for (int i = 0; i < 32 / Rb2; ++i) {
            const int u = b0 + i * bStep;
#pragma unroll
            for (int s = 0; s < Rb2; ++s) v[i * Rb2 + s] = buf[(u * Rb2 + s) * PB + q1];
            cx_dft<Rb2>(v + i * Rb2);
#pragma unroll
            for (int s = 0; s < Rb2; ++s) x[q1 + N1 * (u + Rb1 * s)] = v[i * Rb2 + s];
        }
        if (r + G < n) fetch(row_nxt, m_nxt);
        __syncthreads();                         // the buffer is free for the next row
        row_cur = row_nxt;
        row_nxt = row_n2;
        m_nxt = m_n2;
    }
}

template <typename C2, int N1, int N2>
int launch_row_big(rick_plan* p, void* grid, cudaStream_t st) {
    typedef RowBig<C2, N1, N2> P;
    static bool attr_done[RICK_MAX_DEVICES] = {};
    bool& done = attr_done[p->device & (RICK_MAX_DEVICES - 1)];
    if (!done) {
        if (cudaFuncSetAttribute(k_row_big<C2, N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem) != cudaSuccess)
            return RICK_ECUDA;
        done = true;
    }
    const int ctas = p->sm_count * P::kMinBlocks;       // persistent: every CTA walks its share of the row list
    k_row_big<C2, N1, N2><<<ctas, P::T, P::smem, st>>>((C2*)grid, (const C2*)p->split_tw, p->row_list_dev, p->n_rows_dev,
                                                       p->segs ? p->seg_mesh_dev : nullptr);
    return RICK_OK;
}

}  // namespace

// N = 4096, 8192, 16384 on the fp32 mesh; 4096, 8192 on the fp64 mesh (a 16384-point fp64 row does not fit one SM)
bool rick_rowbig_supported(const rick_plan* p) {
    const int N = p->g.N;
    if (p->dtype == RICK_C128) return N == 4096 || N == 8192;
    return N == 4096 || N == 8192 || N == 16384;
}

// row transforms of the rows of p->row_list_dev (rick_rows_list_all), in place
int rick_rowbig_impl(rick_plan* p, void* grid, cudaStream_t st) {
    int rc = RICK_EINVAL;
    if (p->dtype == RICK_C128) {
        switch (p->g.N) {
            case 4096: rc = launch_row_big<double2, 64, 64>(p, grid, st); break;
            case 8192: rc = launch_row_big<double2, 64, 128>(p, grid, st); break;
            default: break;
        }
    } else {
        switch (p->g.N) {
            case 4096: rc = launch_row_big<float2, 64, 64>(p, grid, st); break;
            case 8192: rc = launch_row_big<float2, 64, 128>(p, grid, st); break;
            case 16384: rc = launch_row_big<float2, 128, 128>(p, grid, st); break;
            default: break;
        }
    }
    if (rc != RICK_OK) return rc;
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
