// peaks.cu -- measurement helper, not part of the imaging path: the fp32 issue rates of this GPU, measured.
// bench.py reports the instruction-issue view of the FFT / gridding kernels against these numbers instead of a
// spec-sheet product (SMs x lanes x clock).  Each thread runs a dependent chain of kChains independent
// accumulators through n_iter fused multiply-adds (or adds); the grid fills every SM with full occupancy.
#include "rick_internal.cuh"

namespace {

constexpr int kChains = 8;

template <bool kFma>
__global__ void __launch_bounds__(256) k_fp32_rate(float* out, int n_iter, float a, float b) {
    float x[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) x[i] = kFma ? fmaf(x[i], a, b) : (x[i] + b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;      // keeps the chains alive; practically never true
}

// the same chain with the packed instruction of sm_100 (fma.rn.f32x2 -> FFMA2: two fused multiply-adds per lane)
__global__ void __launch_bounds__(256) k_fp32x2_rate(float* out, int n_iter, float a, float b) {
    unsigned long long x[kChains], pa, pb;
    asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
#pragma unroll
    for (int i = 0; i < kChains; ++i) asm("mov.b64 %0, {%1, %2};" : "=l"(x[i]) : "f"((float)(threadIdx.x + i)), "f"((float)i));
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(pa), "l"(pb));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[i]));
        s += lo + hi;
    }
    if (s == 12345.678f) out[0] = s;
}

// random 32-byte record reads (two 16-byte loads of one sector, 64-byte L2 fetches): the access pattern of a gather
__global__ void __launch_bounds__(256) k_random_read_rate(const float4* __restrict__ rec, unsigned long long mask,
                                                          unsigned long long n, float* out) {
    float acc = 0.f;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        unsigned long long z = i * 0x9E3779B97F4A7C15ull;                 // splitmix64 of the counter
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        const float4* p = rec + 2 * ((z ^ (z >> 31)) & mask);
        float4 a, b;
        asm volatile("ld.global.nc.L2::64B.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w) : "l"(p));
        asm volatile("ld.global.nc.L2::64B.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p + 1));
        acc += a.x + b.w;
    }
    if (acc == 12345.678f) out[0] = acc;
}

}  // namespace

extern "C" int rick_measure_random_read_rate(double* grecords_per_s, void* stream) {
    if (!grecords_per_s) return RICK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    RICK_CUDA(cudaGetDevice(&dev));
    RICK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const unsigned long long n_rec = 1ull << 26;            // 2 GB of 32-byte records: 16 x the L2
    float4* rec = nullptr;
    float* out = nullptr;
    if (cudaMalloc((void**)&rec, n_rec * 32) != cudaSuccess) return RICK_ENOMEM;
    if (cudaMalloc((void**)&out, sizeof(float)) != cudaSuccess) { cudaFree(rec); return RICK_ENOMEM; }
    cudaMemsetAsync(rec, 0, n_rec * 32, st);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const unsigned long long n = 1ull << 27;
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {                     // first repetition warms up
        cudaEventRecord(e0, st);
        k_random_read_rate<<<sms * 8, 256, 0, st>>>(rec, n_rec - 1, n, out);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)n / ((double)ms * 1e-3) / 1e9;
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(rec);
    cudaFree(out);
    RICK_LAUNCH_CHECK();
    *grecords_per_s = best;
    return RICK_OK;
}

extern "C" int rick_measure_fp32_rate(double* fma_tflops, double* add_tinst, double* fma2_tflops, void* stream) {
    if (!fma_tflops || !add_tinst || !fma2_tflops) return RICK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    RICK_CUDA(cudaGetDevice(&dev));
    RICK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* out = nullptr;
    RICK_CUDA(cudaMalloc((void**)&out, sizeof(float)));
    cudaEvent_t e0, e1;
    RICK_CUDA(cudaEventCreate(&e0));
    RICK_CUDA(cudaEventCreate(&e1));
    const int blocks = sms * 8, n_iter = 8192;
    const double ops = (double)blocks * 256.0 * (double)n_iter * (double)kChains;
    double best[3] = {0.0, 0.0, 0.0};
    for (int kind = 0; kind < 3; ++kind) {
        for (int rep = 0; rep < 4; ++rep) {      // first repetition warms up
            RICK_CUDA(cudaEventRecord(e0, st));
            if (kind == 0) k_fp32_rate<true><<<blocks, 256, 0, st>>>(out, n_iter, 0.999f, 0.001f);
            else if (kind == 1) k_fp32_rate<false><<<blocks, 256, 0, st>>>(out, n_iter, 0.999f, 0.001f);
            else k_fp32x2_rate<<<blocks, 256, 0, st>>>(out, n_iter, 0.999f, 0.001f);
            RICK_CUDA(cudaEventRecord(e1, st));
            RICK_CUDA(cudaEventSynchronize(e1));
            float ms = 0.f;
            RICK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
            const double rate = ops / ((double)ms * 1e-3) / 1e12;
            if (rep > 0 && rate > best[kind]) best[kind] = rate;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    RICK_LAUNCH_CHECK();
    *fma_tflops = 2.0 * best[0];      // 2 flop per fused multiply-add
    *add_tinst = best[1];             // 1e12 fp32 add instructions (lane-ops) per second
    *fma2_tflops = 4.0 * best[2];     // packed: 2 fused multiply-adds = 4 flop per lane-op
    return RICK_OK;
}
