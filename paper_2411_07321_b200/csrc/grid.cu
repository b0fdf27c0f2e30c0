// grid.cu -- rick_grid: convolutional gridding, Eq. 3 with the separable truncated Gaussian [D6].
//
// v0 (first correct path): one thread per sorted visibility, S*S vector reductions straight into the
// mesh in L2 (red.global.add).  Sorted order keeps the reductions of a warp inside one 32x32 tile.
#include "rick_internal.cuh"

namespace {

constexpr int kMaxS = 15;

__device__ __forceinline__ void red_add_v2(float2* addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

// Taps of one axis: g(i0 + a - x) for a = -h..h, with the checkerboard sign (-1)^(i0+a) folded in
// (modulated mesh, see rick_b200.h).  d0 = i0 - x is formed in fp64 and narrowed once.
template <typename real>
__device__ __forceinline__ void taps(real* t, int S, int h, int i0, double x, real inv_2s2) {
    const real d0 = (real)((double)i0 - x);
    for (int a = 0; a < S; ++a) {
        const real d = d0 + (real)(a - h);
        real val = (sizeof(real) == 4) ? (real)expf(-(float)(d * d) * (float)inv_2s2) : (real)exp(-(double)(d * d) * (double)inv_2s2);
        t[a] = ((i0 + a - h) & 1) ? -val : val;
    }
}

template <typename real, typename cell>
__global__ void __launch_bounds__(128) k_grid_naive(RickGeom g, const long long* __restrict__ n_kept,
                                                     const float* __restrict__ u_s, const float* __restrict__ v_s,
                                                     const float* __restrict__ w_s, const float2* __restrict__ vis_s,
                                                     const float* __restrict__ wt_s, cell* __restrict__ grid) {
    const long long n = *n_kept;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const real inv_2s2 = (real)(1.0 / (2.0 * g.sigma * g.sigma));
    for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += stride) {
        const RickLoc r = rick_locate(g, u_s[m], v_s[m], w_s[m]);
        const float2 vi = vis_s[m];
        const float wgt = wt_s[m];
        const real vr = (real)wgt * (real)vi.x, vim = (real)wgt * (real)vi.y;
        real gx[kMaxS], gy[kMaxS];
        taps<real>(gx, g.S, g.h, r.i0, r.x, inv_2s2);
        taps<real>(gy, g.S, g.h, r.j0, r.y, inv_2s2);
        cell* base = grid + ((size_t)r.k * g.N + (size_t)(r.j0 - g.h)) * g.N + (size_t)(r.i0 - g.h);
        for (int b = 0; b < g.S; ++b) {
            const real yr = gy[b] * vr, yi = gy[b] * vim;
            cell* row = base + (size_t)b * g.N;
            for (int a = 0; a < g.S; ++a) {
                if (sizeof(real) == 4) {
                    red_add_v2((float2*)(row + a), (float)(gx[a] * yr), (float)(gx[a] * yi));
                } else {
                    double* c = (double*)(row + a);
                    atomicAdd(c, (double)(gx[a] * yr));
                    atomicAdd(c + 1, (double)(gx[a] * yi));
                }
            }
        }
    }
}

}  // namespace

int rick_grid_impl(rick_plan* p, void* grid, cudaStream_t st) {
    if (p->M == 0) return RICK_OK;
    const long long want = (p->M + 127) / 128;
    const long long cap = (long long)p->sm_count * 64;
    const int blocks = (int)(want > cap ? cap : want);
    if (p->dtype == RICK_C128)
        k_grid_naive<double, double2><<<blocks, 128, 0, st>>>(p->g, p->n_kept_dev, p->u_s, p->v_s, p->w_s,
                                                               (const float2*)p->vis_s, p->weight_s, (double2*)grid);
    else
        k_grid_naive<float, float2><<<blocks, 128, 0, st>>>(p->g, p->n_kept_dev, p->u_s, p->v_s, p->w_s,
                                                             (const float2*)p->vis_s, p->weight_s, (float2*)grid);
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
