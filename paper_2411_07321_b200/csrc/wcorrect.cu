// wcorrect.cu -- rick_wcorrect_accumulate: w phase screen, plane sum and taper division in one
// bandwidth-bound sweep.  Eq. 2, step 4  [D8].
//
// Every transformed plane is read exactly once (Nw*N*N*cell bytes), the fp64 image is written once.
// Per pixel the screen of plane k is exp(2 pi i (w_0 + k dw) nm1): it is advanced by a complex rotation
// per plane (two sincospi per pixel instead of Nw), all in fp64, so the kernel stays HBM-bound.
// The (-1)^(p+q) factor undoes the un-shifted FFT of the modulated mesh (see rick_b200.h).
#include "rick_internal.cuh"

namespace {

constexpr int kUnroll = 8;

__device__ __forceinline__ void screen_init(const RickGeom& g, int p, int q, double& c, double& s, double& cs,
                                            double& ss) {
    const double l = (double)(p - g.N / 2) * g.dl;
    const double m = (double)(q - g.N / 2) * g.dl;
    const double r2 = l * l + m * m;
    const double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
    const double w0 = g.w_min + 0.5 * g.dw;
    double t0 = w0 * nm1;
    t0 -= floor(t0);
    double t1 = g.dw * nm1;
    t1 -= floor(t1);
    sincospi(2.0 * t0, &s, &c);
    sincospi(2.0 * t1, &ss, &cs);
}

__device__ __forceinline__ float4 ldg_stream(const float4* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(p));
    return r;
}

__device__ __forceinline__ double2 ldg_stream(const double2* p) {
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

// c64 mesh: one thread per two adjacent pixels (one 16-byte load per plane)
__global__ void __launch_bounds__(256) k_wcorrect_c64(RickGeom g, const float4* __restrict__ planes,
                                                       const double* __restrict__ inv_t, double2* __restrict__ image,
                                                       int accumulate) {
    const size_t pairs_per_plane = (size_t)g.N * g.N / 2;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= pairs_per_plane) return;
    const int q = (int)(t / (g.N / 2));
    const int p = (int)(t % (g.N / 2)) * 2;
    double c0, s0, cs0, ss0, c1, s1, cs1, ss1;
    screen_init(g, p, q, c0, s0, cs0, ss0);
    screen_init(g, p + 1, q, c1, s1, cs1, ss1);
    double a0 = 0.0, a1 = 0.0;
    const float4* src = planes + t;
    int k = 0;
    for (; k + kUnroll <= g.Nw; k += kUnroll) {
        float4 vbuf[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) vbuf[j] = ldg_stream(src + (size_t)(k + j) * pairs_per_plane);
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            a0 += c0 * (double)vbuf[j].x - s0 * (double)vbuf[j].y;
            a1 += c1 * (double)vbuf[j].z - s1 * (double)vbuf[j].w;
            const double n0 = c0 * cs0 - s0 * ss0;
            s0 = c0 * ss0 + s0 * cs0;
            c0 = n0;
            const double n1 = c1 * cs1 - s1 * ss1;
            s1 = c1 * ss1 + s1 * cs1;
            c1 = n1;
        }
    }
    for (; k < g.Nw; ++k) {
        const float4 vv = ldg_stream(src + (size_t)k * pairs_per_plane);
        a0 += c0 * (double)vv.x - s0 * (double)vv.y;
        a1 += c1 * (double)vv.z - s1 * (double)vv.w;
        const double n0 = c0 * cs0 - s0 * ss0;
        s0 = c0 * ss0 + s0 * cs0;
        c0 = n0;
        const double n1 = c1 * cs1 - s1 * ss1;
        s1 = c1 * ss1 + s1 * cs1;
        c1 = n1;
    }
    const double tq = inv_t[q];
    const double sg = ((p + q) & 1) ? -1.0 : 1.0;
    double2 out;
    out.x = a0 * (sg * tq * inv_t[p]);
    out.y = a1 * (-sg * tq * inv_t[p + 1]);
    if (accumulate) {
        const double2 old = image[t];
        out.x += old.x;
        out.y += old.y;
    }
    image[t] = out;
}

// c128 mesh: one thread per pixel (one 16-byte load per plane)
__global__ void __launch_bounds__(256) k_wcorrect_c128(RickGeom g, const double2* __restrict__ planes,
                                                        const double* __restrict__ inv_t, double* __restrict__ image,
                                                        int accumulate) {
    const size_t cells = (size_t)g.N * g.N;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= cells) return;
    const int q = (int)(t / g.N);
    const int p = (int)(t % g.N);
    double c, s, cs, ss;
    screen_init(g, p, q, c, s, cs, ss);
    double acc = 0.0;
    const double2* src = planes + t;
    int k = 0;
    for (; k + kUnroll <= g.Nw; k += kUnroll) {
        double2 vbuf[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) vbuf[j] = ldg_stream(src + (size_t)(k + j) * cells);
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            acc += c * vbuf[j].x - s * vbuf[j].y;
            const double n = c * cs - s * ss;
            s = c * ss + s * cs;
            c = n;
        }
    }
    for (; k < g.Nw; ++k) {
        const double2 vv = ldg_stream(src + (size_t)k * cells);
        acc += c * vv.x - s * vv.y;
        const double n = c * cs - s * ss;
        s = c * ss + s * cs;
        c = n;
    }
    const double sg = ((p + q) & 1) ? -1.0 : 1.0;
    double out = acc * (sg * inv_t[q] * inv_t[p]);
    if (accumulate) out += image[t];
    image[t] = out;
}

}  // namespace

int rick_wcorrect_impl(rick_plan* p, const void* grid, double* image, int zero_first, cudaStream_t st) {
    const RickGeom& g = p->g;
    const size_t cells = (size_t)g.N * g.N;
    if (p->dtype == RICK_C128) {
        const unsigned blocks = (unsigned)((cells + 255) / 256);
        k_wcorrect_c128<<<blocks, 256, 0, st>>>(g, (const double2*)grid, p->inv_taper_dev, image, zero_first ? 0 : 1);
    } else {
        const unsigned blocks = (unsigned)((cells / 2 + 255) / 256);
        k_wcorrect_c64<<<blocks, 256, 0, st>>>(g, (const float4*)grid, p->inv_taper_dev, (double2*)image, zero_first ? 0 : 1);
    }
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
