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

}  // namespace

extern "C" int rick_measure_fp32_rate(double* fma_tflops, double* add_tinst, void* stream) {
    if (!fma_tflops || !add_tinst) return RICK_EINVAL;
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
    double best[2] = {0.0, 0.0};
    for (int kind = 0; kind < 2; ++kind) {
        for (int rep = 0; rep < 4; ++rep) {      // first repetition warms up
            RICK_CUDA(cudaEventRecord(e0, st));
            if (kind == 0) k_fp32_rate<true><<<blocks, 256, 0, st>>>(out, n_iter, 0.999f, 0.001f);
            else k_fp32_rate<false><<<blocks, 256, 0, st>>>(out, n_iter, 0.999f, 0.001f);
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
    return RICK_OK;
}
