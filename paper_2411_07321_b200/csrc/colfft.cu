// colfft.cu -- fused column transform + w-correction (RICK_C64, N = 256 .. 2048, opt-in through
// rick_plan_set_fusion): the second half of D7 and all of D8 in ONE read of the mesh.
//
// With fusion on, rick_fft_planes only runs the contiguous row transforms (batched 1-D cuFFT, which
// streams at the copy rate); the strided column pass -- the slow half of a 2-D cuFFT (profiles/) -- is
// done here.  A CTA owns kC = 4 adjacent image columns.  For every plane it pulls the N x 4 column block
// (32-byte rows, full sectors) into shared memory with cp.async (double-buffered against the next
// plane), runs four in-place length-N inverse DFTs (decimation in frequency, radix 16 x 16 x {1,2,4,8},
// butterflies in registers, digit-reversed output left in place), multiplies each output by the phase
// screen exp(+2 pi i w_k nm1(q,p)) (Eq. 2) and adds the real part to fp64 accumulators that stay
// in registers for all planes.  At the end: (-1)^(p+q), the taper division, one write of the image.
// The transformed planes are never written back: the column pass of a 2-D FFT (read + write of the
// mesh) and the K5 sweep (another read) collapse into one read.
//
// Phase: w_k * nm1 in fp64 (nm1 of a thread's pixels kept in registers), its fraction rounded to 2^-23 turns
// (3.7e-7 rad at worst) and reduced to [-1/2, 1/2), then the hardware sine / cosine in fp32 on the reduced
// argument (abs error < 5e-7, the precision of the fp32 planes themselves); the product in fp32, the plane
// sum in fp64.
#include "fft_radix.cuh"
#include "rick_internal.cuh"

namespace {

constexpr int kC = 4;            // columns per CTA
constexpr int kT = 512;          // threads per CTA
constexpr int kPadShift = 5;     // 4 float2 of padding after every 32 float2 (bank-conflict-free passes)

// X = 0: the column kernel's layout.  X = 2 (row kernel): two more slots after every 512, so that the last
// pass can take its butterflies in frequency order (lanes 4 KB apart in the plain layout) at a 2-way conflict.
template <int X = 0>
__device__ __forceinline__ constexpr int padded(int idx) { return idx + ((idx >> kPadShift) << 2) + (idx >> 9) * X; }

// complex product and the small inverse DFTs (natural order in and out) in the packed fp32 arithmetic of
// fft_radix.cuh (add / mul / fma .f32x2: one issue slot per (re, im) pair)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return cx_mul<float2>(a, b); }
template <int R> __device__ __forceinline__ void dft(float2* v) { cx_dft<R, float2>(v); }

// One in-place decimation-in-frequency pass of radix R over sub-transforms of length n = 2^LOG2n of the
// N = 2^LOG2N point columns:  for every sub-block B, offset m < n/R, column c:
//   x[B n + m + t n/R], t < R  ->  R-point DFT  ->  y_u * W_n^(m u) stored at the same slots (u for t).
// tw[j] = exp(+2 pi i j / N).  Everything but m is a compile-time constant: the R slots of a butterfly
// are the padded base plus constant offsets.
// In the second pass (n = N/16) a warp holds only N/256 <= 8 distinct m, and their table entries lie
// 128 u bytes apart -- all in one bank (4 wavefronts per load, 12 % of the kernel's shared-memory wavefronts).
// That pass reads a compact copy instead: tw2[ui q + m] = W_n^(m 2^ui), q = N/256 consecutive entries per power.
template <int LOG2N, int R, int LOG2n, int X = 0>
__device__ __forceinline__ void dif_pass(float2* buf, const float2* tw, int tid, const float2* tw2 = nullptr) {
    constexpr int N = 1 << LOG2N, n = 1 << LOG2n;
    constexpr int q = n / R;                     // stride between the R inputs (rows)
    constexpr int stride = q * kC;               // ... in float2 slots
    constexpr int per_block = stride;            // butterflies per sub-block = q * kC
    constexpr int total = N * kC / R;            // butterflies per pass
    constexpr int tw_step = N / n;
    // the padding is affine over the butterfly when its slots step by whole padding groups, or stay inside one
    constexpr bool kConstOff = (X == 0 ? (stride % 32) == 0 : ((stride % 512) == 0 || ((stride % 32) == 0 && R * stride <= 512))) ||
                               (R * stride <= 32);
#pragma unroll
    for (int w0 = 0; w0 < total; w0 += kT) {
        const int w = w0 + tid;
        if (total % kT != 0 && w >= total) break;
        const int B = w / per_block, rem = w % per_block;     // powers of two: shifts
        const int base = B * (n * kC) + rem;                  // ((B n + m) kC + c), rem = m kC + c
        const int pb = padded<X>(base);
        float2 v[R];
#pragma unroll
        for (int t = 0; t < R; ++t)
            v[t] = kConstOff ? buf[pb + t * padded<X>(stride)] : buf[padded<X>(base + t * stride)];
        dft<R>(v);
        if (q > 1) {
            // W_n^(m u), u < R: the powers of two come from the table, the rest are products of at
            // most three of them (shared-memory bandwidth, not arithmetic, bounds this kernel)
            const int ts = (rem / kC) * tw_step;              // m * N / n
            float2 wp[R];
            if (LOG2n == LOG2N - 4 && R == 16) {
#pragma unroll
                for (int ui = 0; ui < 4; ++ui) wp[1 << ui] = tw2[ui * q + rem / kC];
            } else {
#pragma unroll
                for (int u = 1; u < R; u <<= 1) wp[u] = tw[(ts * u) & (N - 1)];
            }
#pragma unroll
            for (int u = 3; u < R; ++u)
                if (u & (u - 1)) {                            // not a power of two: lowest set bit times the rest
                    const int lo = u & -u;
                    wp[u] = cmul(wp[u - lo], wp[lo]);
                }
#pragma unroll
            for (int u = 1; u < R; ++u) v[u] = cmul(v[u], wp[u]);
        }
#pragma unroll
        for (int u = 0; u < R; ++u) {
            if (kConstOff) buf[pb + u * padded<X>(stride)] = v[u];
            else buf[padded<X>(base + u * stride)] = v[u];
        }
    }
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}


// digit-reversed slot -> frequency: slot = u1 N/16 + u2 N/256 + u3  ->  q = u1 + 16 u2 + 256 u3
__device__ __forceinline__ int slot_to_freq(int slot, int N) {
    const int u1 = slot / (N >> 4), r1 = slot - u1 * (N >> 4);
    const int u2 = r1 / (N >> 8), u3 = r1 - u2 * (N >> 8);
    return u1 + (u2 << 4) + (u3 << 8);
}

template <int LOG2N>
__global__ void __launch_bounds__(kT, 1) k_colfft_wcorrect(RickGeom g, const float2* __restrict__ planes,
                                                           const float2* __restrict__ tw_g,
                                                           const double* __restrict__ inv_t,
                                                           double* __restrict__ image, int accumulate,
                                                           const uint32_t* __restrict__ occ, int col0) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int N = 1 << LOG2N;
    constexpr int R3 = N >> 8;                        // radices 16 x 16 x R3
    constexpr int n_slots = N * kC;                   // complex values of one column block
    constexpr int buf_elems = n_slots + ((n_slots >> kPadShift) << 2);   // float2 per buffer
    float2* buf0 = reinterpret_cast<float2*>(smem_raw);
    float2* buf1 = buf0 + buf_elems;
    float2* tw = buf1 + buf_elems;                    // [N]
    float2* tw2 = tw + N;                             // [4 R3] second-pass twiddles, compact
    const int tid = threadIdx.x;
    const int p0 = col0 + blockIdx.x * kC;           // col0: first column of this launch's part of the image
    constexpr int per_thread = n_slots / kT;          // outputs owned by a thread: 2 .. 16
    // Ownership: with a third pass (R3 > 1) a thread keeps the R3 outputs of each of its last-pass
    // butterflies (entry e = bi R3 + u: butterfly w = bi kT + tid, sub-block B = w / kC, column c = w % kC,
    // slot (B R3 + u) kC + c) -- they go from registers straight into the screen, never back to shared
    // memory; without one (N = 256) entry e is slot e kT + tid, read back from shared memory.
    auto owned_slot = [&](int e) {
        if (R3 > 1) {
            const int bi = e / R3, u = e % R3, w = bi * kT + tid;
            return ((w / kC) * R3 + u) * kC + (w % kC);
        }
        return e * kT + tid;
    };

    auto issue = [&](int k, float2* buf) {
        const float2* src = planes + (size_t)k * N * N + p0;
        // row j: kC float2 = 32 B = two 16-byte pieces.  Fusion mode 2 (occ != NULL): rows no footprint
        // touched hold undefined data and are not read -- their slots are zero-filled instead.
        // A warp's 32 pieces of one iteration are 16 consecutive rows, all in one word of the bitmap: lane
        // `it` fetches the word of iteration `it` (one load per lane, all in flight together) and the
        // iterations take theirs by shuffle.  (One dependent load per iteration cost 8 % of the kernel.)
        constexpr int kIt = N * 2 / kT;
        static_assert(kIt <= 32 && (kT / 2) % 32 == 0, "one bitmap word per warp and iteration");
        uint32_t live = 0xFFFFFFFFu;
        if (occ) {
            const int lane = tid & 31, row0 = (tid & ~31) >> 1;          // first row of the warp, iteration 0
            const uint32_t wv = lane < kIt ? __ldg(occ + ((k * N + row0 + lane * (kT / 2)) >> 5)) : 0u;
            live = 0;
#pragma unroll
            for (int it = 0; it < kIt; ++it)
                live |= ((__shfl_sync(0xffffffffu, wv, it) >> ((row0 + (lane >> 1)) & 31)) & 1u) << it;
        }
#pragma unroll 1
        for (int it = 0; it < kIt; ++it) {
            const int q = tid + it * kT, j = q >> 1, half = q & 1;
            float2* dst = buf + padded(j * kC + half * 2);
            if ((live >> it) & 1u) cp_async16(dst, src + (size_t)j * N + half * 2);
            else *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // planes of this CTA: gridDim.y splits the plane range (two halves fill the last wave of CTAs)
    const int k_per = (g.Nw + (int)gridDim.y - 1) / (int)gridDim.y;
    const int k_lo = (int)blockIdx.y * k_per;
    const int k_hi = (k_lo + k_per < g.Nw) ? k_lo + k_per : g.Nw;
    if (k_lo >= k_hi) return;
    issue(k_lo, buf0);
    for (int i = tid; i < N; i += kT) tw[i] = tw_g[i];
    for (int i = tid; i < 4 * R3; i += kT) tw2[i] = tw_g[(((i % R3) * 16) << (i / R3)) & (N - 1)];
    double acc[per_thread], nm1r[per_thread];         // plane sum and n - 1 of the owned pixels
#pragma unroll
    for (int e = 0; e < per_thread; ++e) {
        const int idx = owned_slot(e);
        const int q = slot_to_freq(idx / kC, N), p = p0 + (idx % kC);
        const double l = (double)(p - N / 2) * g.dl, m = (double)(q - N / 2) * g.dl;
        nm1r[e] = rick_nm1_fast(l * l + m * m);
        acc[e] = 0.0;
    }
    auto screen_add = [&](int e, float2 v, double wk) {
        // fraction of w_k nm1 in fixed point, without the conversion pipe (rint and the fp64 -> fp32 narrowing
        // are XU instructions, 4 lanes per clock and scheduler: with the two MUFUs and the widening below they
        // made the screen XU-bound): adding 1.5 * 2^29 rounds the product (one DFMA) to 2^-23 turns and leaves
        // the fraction, two's complement, in the low 23 mantissa bits (|w_k nm1| < 2^28 turns).
        const double z = fma(wk, nm1r[e], 805306368.0);
        uint32_t gbits;                                                     // 1 + fraction: (lo & mantissa) | one, one LOP3
        asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(gbits) : "r"((uint32_t)__double2loint(z)), "r"(0x007FFFFFu), "r"(0x3F800000u));
        const float gq = __uint_as_float(gbits);   // 1 + fraction
        // 2 pi (fraction - 1/2), in [-pi, pi): one FFMA (rounding: 2^-24 pi rad, below the 2^-23-turn phase step)
        const float t = fmaf(gq, 6.283185307179586f, -9.42477796076938f);
        float sn, cs;
        __sincosf(t, &sn, &cs);                                // MUFU on [-pi, pi]: abs error < 5e-7
        acc[e] += (double)(sn * v.y - cs * v.x);               // the half turn negates sine and cosine
    };

    for (int k = k_lo; k < k_hi; ++k) {
        const int par = (k - k_lo) & 1;
        float2* buf = par ? buf1 : buf0;
        if (k + 1 < k_hi) issue(k + 1, par ? buf0 : buf1);
        else asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        dif_pass<LOG2N, 16, LOG2N>(buf, tw, tid);
        __syncthreads();
        dif_pass<LOG2N, 16, LOG2N - 4>(buf, tw, tid, tw2);
        __syncthreads();
        const double wk = g.w_min + ((double)k + 0.5) * g.dw;
        if (R3 > 1) {
            // last pass (sub-length R3, no twiddles) fused with the screen: outputs stay in registers
#pragma unroll
            for (int bi = 0; bi < per_thread / R3; ++bi) {
                const int w = bi * kT + tid;
                const int pb = padded((w / kC) * (R3 * kC) + (w % kC));   // R3 * kC <= 32: one padding group
                float2 v[R3];
#pragma unroll
                for (int t = 0; t < R3; ++t) v[t] = buf[pb + t * kC];
                dft<R3>(v);
#pragma unroll
                for (int u = 0; u < R3; ++u) screen_add(bi * R3 + u, v[u], wk);
            }
        } else {
#pragma unroll
            for (int e = 0; e < per_thread; ++e) screen_add(e, buf[padded(e * kT + tid)], wk);
        }
        __syncthreads();                              // buf is free for plane k + 2
    }
#pragma unroll
    for (int e = 0; e < per_thread; ++e) {
        const int idx = owned_slot(e);
        const int q = slot_to_freq(idx / kC, N), p = p0 + (idx % kC);
        const double sg = ((p + q) & 1) ? -1.0 : 1.0;
        double out = acc[e] * (sg * inv_t[q] * inv_t[p]);
        const size_t o = (size_t)q * N + p;
        if (gridDim.y > 1) {
            atomicAdd(image + o, out);       // two addends onto a zeroed or given image: order-independent
        } else {
            if (accumulate) out += image[o];
            image[o] = out;
        }
    }
}

// Row transforms of the listed mesh rows only (fusion mode 2), in place: four rows per step go through the
// same shared-memory layout and DIF passes as four columns do in k_colfft_wcorrect; the last pass takes its
// butterflies in frequency order and writes the rows back in natural order.
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}

constexpr int kRowPad = 2;   // extra padding of the row kernel's layout (see padded<X>)

template <int LOG2N>
__global__ void __launch_bounds__(kT, 1) k_rowfft(float2* __restrict__ planes, const float2* __restrict__ tw_g,
                                                  const uint32_t* __restrict__ list, const uint32_t* __restrict__ n_rows) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int N = 1 << LOG2N;
    constexpr int R3 = N >> 8;
    constexpr int n_slots = N * kC;
    constexpr int buf_elems = padded<kRowPad>(n_slots);
    float2* buf0 = reinterpret_cast<float2*>(smem_raw);
    float2* buf1 = buf0 + buf_elems;
    float2* tw = buf1 + buf_elems;
    float2* tw2 = tw + N;
    const int tid = threadIdx.x;
    const int n = (int)*n_rows;
    const int n_groups = (n + kC - 1) / kC;

    auto issue = [&](int grp, float2* buf) {
        // slot (i, c) <- element i of row list[4 grp + c]; consecutive threads take consecutive i (coalesced)
        // (the group's row numbers are fetched before the copies: the copies clobber memory as far as the
        // compiler knows, and one dependent load per copy iteration is what cost K6 8 %)
        uint32_t row[kC];
#pragma unroll
        for (int c = 0; c < kC; ++c) row[c] = (grp * kC + c < n) ? __ldg(list + grp * kC + c) : 0xFFFFFFFFu;
#pragma unroll
        for (int it = 0; it < N * kC / kT; ++it) {
            const int q = tid + it * kT;
            const int c = q >> LOG2N, i = q & (N - 1);
            uint32_t rw = row[0];
#pragma unroll
            for (int x = 1; x < kC; ++x) rw = (c == x) ? row[x] : rw;
            if (rw != 0xFFFFFFFFu) cp_async8(buf + padded<kRowPad>(i * kC + c), planes + (size_t)rw * N + i);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    int grp = blockIdx.x;
    if (grp >= n_groups) return;
    issue(grp, buf0);
    for (int i = tid; i < N; i += kT) tw[i] = tw_g[i];
    for (int i = tid; i < 4 * R3; i += kT) tw2[i] = tw_g[(((i % R3) * 16) << (i / R3)) & (N - 1)];
    int par = 0;
    for (; grp < n_groups; grp += gridDim.x, par ^= 1) {
        float2* buf = par ? buf1 : buf0;
        const int next = grp + gridDim.x;
        if (next < n_groups) issue(next, par ? buf0 : buf1);
        else asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        dif_pass<LOG2N, 16, LOG2N, kRowPad>(buf, tw, tid);
        __syncthreads();
        dif_pass<LOG2N, 16, LOG2N - 4, kRowPad>(buf, tw, tid, tw2);
        __syncthreads();
        // Last pass straight to global memory, in NATURAL frequency order: the butterfly (u1, u2, c) holds
        // frequencies u1 + 16 u2 + 256 u3, u3 < R3 (slots (u1 16 + u2) R3 + u3).  Lanes run over u1, so that
        // every store instruction writes 16 consecutive frequencies of a row (full sectors).
#pragma unroll
        for (int bi = 0; bi < n_slots / kT / R3; ++bi) {
            const int w = bi * kT + tid;
            const int u1 = w & 15, c = (w >> 4) % kC, u2 = w / (16 * kC);
            const int r = grp * kC + c;
            float2 v[R3];
#pragma unroll
            for (int t = 0; t < R3; ++t) v[t] = buf[padded<kRowPad>(((u1 * 16 + u2) * R3 + t) * kC + c)];
            dft<R3>(v);
            if (r < n) {
                float2* dst = planes + (size_t)list[r] * N + (u1 + 16 * u2);
#pragma unroll
                for (int u = 0; u < R3; ++u) dst[256 * u] = v[u];
            }
        }
        __syncthreads();                              // buf is free for the group after next
    }
}

size_t colfft_smem_bytes(int N) {
    const int n_slots = N * kC;
    const size_t buf = (size_t)(n_slots + ((n_slots >> kPadShift) << 2)) * sizeof(float2);
    return 2 * buf + (size_t)(N + 32) * sizeof(float2);      // + twiddles + compact second-pass twiddles
}

}  // namespace

bool rick_colfft_supported(const rick_plan* p) {
    const int N = p->g.N;
    // the screen takes the fraction of w_k nm1 (|nm1| < 1) from the low mantissa bits of w_k nm1 + 1.5 * 2^29:
    // |w| must stay below 2^28 wavelengths (2.7e8; the longest baselines on Earth are ~1e7 at 1 GHz)
    const double w_abs = fmax(fabs(p->g.w_min), fabs(p->g.w_max));
    return p->dtype == RICK_C64 && (N == 256 || N == 512 || N == 1024 || N == 2048) && w_abs < 268435456.0;
}

int rick_colfft_init(rick_plan* p) {
    // twiddles exp(+2 pi i j / N), fp64 values rounded once, on the device
    const int N = p->g.N;
    float2* h = (float2*)malloc(sizeof(float2) * (size_t)N);
    if (!h) return RICK_ENOMEM;
    const double two_pi = 6.283185307179586476925286766559;
    for (int j = 0; j < N; ++j) h[j] = make_float2((float)cos(two_pi * j / N), (float)sin(two_pi * j / N));
    if (p->colfft_tw) { cudaFree(p->colfft_tw); p->colfft_tw = nullptr; }
    cudaError_t e = cudaMalloc((void**)&p->colfft_tw, sizeof(float2) * (size_t)N);
    if (e == cudaSuccess) e = cudaMemcpy(p->colfft_tw, h, sizeof(float2) * (size_t)N, cudaMemcpyHostToDevice);
    free(h);
    if (e != cudaSuccess) return RICK_ECUDA;
    const int smem = (int)colfft_smem_bytes(N);
    const cudaFuncAttribute a = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t ea = cudaSuccess;
    switch (N) {
        case 256: ea = cudaFuncSetAttribute(k_colfft_wcorrect<8>, a, smem); break;
        case 512: ea = cudaFuncSetAttribute(k_colfft_wcorrect<9>, a, smem); break;
        case 1024: ea = cudaFuncSetAttribute(k_colfft_wcorrect<10>, a, smem); break;
        case 2048: ea = cudaFuncSetAttribute(k_colfft_wcorrect<11>, a, smem); break;
        default: return RICK_EINVAL;
    }
    if (ea != cudaSuccess) return RICK_ECUDA;
    return RICK_OK;
}

int rick_colfft_columns_per_cta() { return kC; }

int rick_colfft_split(const rick_plan* p) {
    // split the planes in two when that fills the last wave of CTAs better (one CTA per SM)
    const int items = p->g.N / kC, sms = p->sm_count;
    const double r1 = (double)((items + sms - 1) / sms), r2 = 0.5 * (double)((2 * items + sms - 1) / sms);
    return (p->g.Nw >= 2 && r2 < 0.95 * r1) ? 2 : 1;
}

// Columns [col_lo, col_hi) of the image (multiples of kC = 4).  The whole image in one call, or part by part
// (rick_image_from_host_chunked copies one part to the host while the next is computed); clear_image:
// the plane halves of a split launch add onto a zeroed image -- zero it in the first part's call only.
int rick_colfft_wcorrect_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st,
                              int col_lo, int col_hi, bool clear_image) {
    const RickGeom& g = p->g;
    const int N = g.N;
    if (col_hi < 0) col_hi = N;
    if (col_lo < 0 || col_hi > N || col_lo >= col_hi || (col_lo % kC) || (col_hi % kC)) return RICK_EINVAL;
    const int ksplit = rick_colfft_split(p);
    if (ksplit > 1 && zero_first && clear_image)
        RICK_CUDA(cudaMemsetAsync(image, 0, sizeof(double) * (size_t)N * N, st));
    const dim3 blocks((unsigned)((col_hi - col_lo) / kC), (unsigned)ksplit);
    const size_t smem = colfft_smem_bytes(N);
    const float2* planes = (const float2*)grid;
    const float2* tw = (const float2*)p->colfft_tw;
    const int acc = zero_first ? 0 : 1;
    const uint32_t* occ = p->fused == 2 ? p->occ_mesh_dev : nullptr;
    switch (N) {
        case 256: k_colfft_wcorrect<8><<<blocks, kT, smem, st>>>(g, planes, tw, p->inv_taper_dev, image, acc, occ, col_lo); break;
        case 512: k_colfft_wcorrect<9><<<blocks, kT, smem, st>>>(g, planes, tw, p->inv_taper_dev, image, acc, occ, col_lo); break;
        case 1024: k_colfft_wcorrect<10><<<blocks, kT, smem, st>>>(g, planes, tw, p->inv_taper_dev, image, acc, occ, col_lo); break;
        case 2048: k_colfft_wcorrect<11><<<blocks, kT, smem, st>>>(g, planes, tw, p->inv_taper_dev, image, acc, occ, col_lo); break;
        default: return RICK_EINVAL;
    }
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}

int rick_rowfft_impl(rick_plan* p, void* grid, cudaStream_t st) {
    const int N = p->g.N;
    const size_t smem = colfft_smem_bytes(N) + 2 * (size_t)(N * kC / 512) * kRowPad * sizeof(float2);
    static bool attr_done_dev[RICK_MAX_DEVICES] = {};      // the opt-in is per device
    bool& attr_done = attr_done_dev[p->device & (RICK_MAX_DEVICES - 1)];
    if (!attr_done) {
        const cudaFuncAttribute a = cudaFuncAttributeMaxDynamicSharedMemorySize;
        if (cudaFuncSetAttribute(k_rowfft<8>, a, (int)(colfft_smem_bytes(256) + 2 * (256 * kC / 512) * kRowPad * sizeof(float2))) != cudaSuccess ||
            cudaFuncSetAttribute(k_rowfft<9>, a, (int)(colfft_smem_bytes(512) + 2 * (512 * kC / 512) * kRowPad * sizeof(float2))) != cudaSuccess ||
            cudaFuncSetAttribute(k_rowfft<10>, a, (int)(colfft_smem_bytes(1024) + 2 * (1024 * kC / 512) * kRowPad * sizeof(float2))) != cudaSuccess ||
            cudaFuncSetAttribute(k_rowfft<11>, a, (int)(colfft_smem_bytes(2048) + 2 * (2048 * kC / 512) * kRowPad * sizeof(float2))) != cudaSuccess)
            return RICK_ECUDA;
        attr_done = true;
    }
    float2* planes = (float2*)grid;
    const float2* tw = (const float2*)p->colfft_tw;
    const unsigned blocks = (unsigned)p->sm_count;      // one CTA per SM, each walks its share of row groups
    switch (N) {
        case 256: k_rowfft<8><<<blocks, kT, smem, st>>>(planes, tw, p->row_list_dev, p->n_rows_dev); break;
        case 512: k_rowfft<9><<<blocks, kT, smem, st>>>(planes, tw, p->row_list_dev, p->n_rows_dev); break;
        case 1024: k_rowfft<10><<<blocks, kT, smem, st>>>(planes, tw, p->row_list_dev, p->n_rows_dev); break;
        case 2048: k_rowfft<11><<<blocks, kT, smem, st>>>(planes, tw, p->row_list_dev, p->n_rows_dev); break;
        default: return RICK_EINVAL;
    }
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
