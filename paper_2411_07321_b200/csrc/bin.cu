// bin.cu -- rick_bin: key generation, hand-written stable LSD radix sort (one-sweep style, decoupled
// look-back), gather of the SoA payload, optional bin offsets.   [D2-D5], BASELINE.json north_star (2).
//
// The key that is sorted is the (w-plane, 32x32 tile) key of D4 refined by the in-tile cell index
// [D4']: the order is still grouped by plane and tile, and visibilities with the same nearest cell
// are adjacent, which is what lets rick_grid accumulate whole runs in registers.
//
// Passes and traffic per visibility (algorithmic):
//   K1 keygen+histograms   read 24 B, write 4 B key
//   K2 one-sweep pass x n_pass (n_pass = ceil(key_bits / 8) <= 3 for the five configs)
//                          read 8 B (4 B in the first pass: the index is implicit), write 8 B
//   K3 gather              read 4 B index + 24 B payload (sector-amplified: random rows), write 24 B
#include "rick_internal.cuh"

namespace {

constexpr int kRadix = 1 << RICK_RADIX_BITS_MAX;   // 256 digit values at most
constexpr int kSortThreads = 512;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;   // 8192 keys per tile
constexpr int kSortWarps = kSortThreads / 32;

struct SortLayout {
    int n_pass;
    int shift[RICK_MAX_PASSES];
    int bits[RICK_MAX_PASSES];
};

struct Workspace {
    uint32_t *key_a, *key_b, *idx_a, *idx_b;
    uint32_t* hist;                  // [RICK_MAX_PASSES][kRadix] digit counts -> exclusive bases
    uint32_t* ticket;                // [RICK_MAX_PASSES] dynamic tile ids
    unsigned long long* status;      // [n_tiles][kRadix] look-back words
    size_t zero_offset, zero_bytes;  // the region cleared at the start of every rick_bin
    size_t total;
};

Workspace carve(void* base, long long M) {
    Workspace ws;
    const size_t m = (size_t)(M > 0 ? M : 1);
    const size_t n_tiles = (m + kSortTile - 1) / kSortTile;
    size_t off = 0;
    char* b = (char*)base;
    ws.key_a = (uint32_t*)(b + off); off += rick_align256(4 * m);
    ws.key_b = (uint32_t*)(b + off); off += rick_align256(4 * m);
    ws.idx_a = (uint32_t*)(b + off); off += rick_align256(4 * m);
    ws.idx_b = (uint32_t*)(b + off); off += rick_align256(4 * m);
    ws.zero_offset = off;
    ws.hist = (uint32_t*)(b + off); off += rick_align256(sizeof(uint32_t) * RICK_MAX_PASSES * kRadix);
    ws.ticket = (uint32_t*)(b + off); off += rick_align256(sizeof(uint32_t) * RICK_MAX_PASSES);
    ws.status = (unsigned long long*)(b + off); off += rick_align256(sizeof(unsigned long long) * n_tiles * kRadix);
    ws.zero_bytes = off - ws.zero_offset;
    ws.total = off;
    return ws;
}

// ---------------------------------------------------------------------------------------------
// K1: keys + global digit histograms of every pass + n_kept
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_keygen(RickGeom g, long long M, const float* __restrict__ u,
                                                const float* __restrict__ v, const float* __restrict__ w,
                                                const float2* __restrict__ vis, const float* __restrict__ wt,
                                                uint32_t* __restrict__ key, uint32_t* __restrict__ tile_key_out,
                                                uint32_t* __restrict__ hist,
                                                unsigned long long* __restrict__ n_kept, SortLayout lay) {
    __shared__ uint32_t sh[RICK_MAX_PASSES][kRadix];
    for (int i = threadIdx.x; i < RICK_MAX_PASSES * kRadix; i += blockDim.x) (&sh[0][0])[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    unsigned kept = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    // warp-uniform trip count so that every lane reaches the match instructions
    for (long long base = (long long)blockIdx.x * blockDim.x; base < M; base += stride) {
        const long long m = base + threadIdx.x;
        const bool valid = m < M;
        uint32_t kk = 0xFFFFFFFFu;
        if (valid) {
            const float uu = u[m], vv = v[m], ww = w[m], wgt = wt[m];
            const float2 vi = vis[m];
            RickLoc r = rick_locate(g, uu, vv, ww);
            const bool fin = rick_finite(uu) && rick_finite(vv) && rick_finite(ww) && rick_finite(wgt) &&
                             rick_finite(vi.x) && rick_finite(vi.y);
            const bool keep = r.keep && fin;
            kk = keep ? rick_sort_key(g, r) : g.sort_sentinel;
            kept += keep ? 1u : 0u;
            key[m] = kk;
            if (tile_key_out) tile_key_out[m] = keep ? rick_tile_key(g, r) : g.n_bins;
        }
#pragma unroll
        for (int p = 0; p < RICK_MAX_PASSES; ++p) {
            if (p < lay.n_pass) {
                const uint32_t d = valid ? ((kk >> lay.shift[p]) & ((1u << lay.bits[p]) - 1u)) : (0x10000u | lane);
                const unsigned peers = __match_any_sync(0xffffffffu, d);
                if (valid && lane == (__ffs(peers) - 1)) atomicAdd(&sh[p][d], (uint32_t)__popc(peers));
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < lay.n_pass * kRadix; i += blockDim.x) {
        const uint32_t c = (&sh[0][0])[i];
        if (c) atomicAdd(&hist[i], c);
    }
    for (int o = 16; o > 0; o >>= 1) kept += __shfl_xor_sync(0xffffffffu, kept, o);
    if (lane == 0 && kept) atomicAdd(n_kept, (unsigned long long)kept);
}

// exclusive scan of each pass's 256 digit counts, in place (one block per pass)
__global__ void __launch_bounds__(kRadix) k_scan_hist(uint32_t* __restrict__ hist) {
    __shared__ uint32_t s[kRadix];
    uint32_t* h = hist + blockIdx.x * kRadix;
    const int t = threadIdx.x;
    const uint32_t mine = h[t];
    s[t] = mine;
    __syncthreads();
    for (int o = 1; o < kRadix; o <<= 1) {
        const uint32_t add = (t >= o) ? s[t - o] : 0u;
        __syncthreads();
        s[t] += add;
        __syncthreads();
    }
    h[t] = s[t] - mine;
}

// ---------------------------------------------------------------------------------------------
// K2: one stable LSD pass.  Tiles take their id from a ticket (so that every predecessor is already
// running), rank their keys per warp with match.any (stable: items are warp-striped and visited in
// order), publish per-digit tile counts and resolve their global offsets by decoupled look-back.
// status word: [63:62] state (1 = tile aggregate, 2 = inclusive prefix) | [61:32] epoch | [31:0] count
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long pack_status(uint32_t state, uint32_t epoch, uint32_t value) {
    return ((unsigned long long)state << 62) | ((unsigned long long)epoch << 32) | (unsigned long long)value;
}

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

template <bool kFirst>
__global__ void __launch_bounds__(kSortThreads) k_onesweep(const uint32_t* __restrict__ key_in,
                                                            const uint32_t* __restrict__ idx_in,
                                                            uint32_t* __restrict__ key_out,
                                                            uint32_t* __restrict__ idx_out, long long M, int shift,
                                                            int bits, const uint32_t* __restrict__ digit_base,
                                                            unsigned long long* __restrict__ status,
                                                            uint32_t* __restrict__ ticket, uint32_t epoch) {
    __shared__ uint32_t warp_hist[kSortWarps][kRadix + 1];
    __shared__ uint32_t tile_base[kRadix];
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < kSortWarps * (kRadix + 1); i += kSortThreads) (&warp_hist[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long base = (long long)tile * kSortTile + (long long)warp * (kSortItems * 32) + lane;
    const uint32_t mask = (1u << bits) - 1u;

    uint32_t k[kSortItems], id[kSortItems], rank[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const long long gidx = base + j * 32;
        const bool valid = gidx < M;
        k[j] = valid ? key_in[gidx] : 0u;
        id[j] = kFirst ? (uint32_t)gidx : (valid ? idx_in[gidx] : 0u);
    }
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const bool valid = (base + j * 32) < M;
        const uint32_t d = valid ? ((k[j] >> shift) & mask) : (uint32_t)kRadix;
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        const int leader = __ffs(peers) - 1;
        uint32_t c = 0;
        if (lane == leader) {
            c = warp_hist[warp][d];
            warp_hist[warp][d] = c + (uint32_t)__popc(peers);
        }
        c = __shfl_sync(0xffffffffu, c, leader);
        rank[j] = c + (uint32_t)__popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    if (tid < kRadix) {
        uint32_t running = 0;
#pragma unroll
        for (int wv = 0; wv < kSortWarps; ++wv) {
            const uint32_t c = warp_hist[wv][tid];
            warp_hist[wv][tid] = running;
            running += c;
        }
        unsigned long long* mine = status + (size_t)tile * kRadix + tid;
        uint32_t excl = 0;
        if (tile == 0) {
            st_status(mine, pack_status(2u, epoch, running));
        } else {
            st_status(mine, pack_status(1u, epoch, running));
            long long t = (long long)tile - 1;
            while (true) {
                const unsigned long long* pred = status + (size_t)t * kRadix + tid;
                unsigned long long sv;
                do {
                    sv = ld_status(pred);
                } while ((uint32_t)((sv >> 32) & 0x3FFFFFFFu) != epoch || (sv >> 62) == 0ull);
                excl += (uint32_t)sv;
                if ((sv >> 62) == 2ull || t == 0) break;
                --t;
            }
            st_status(mine, pack_status(2u, epoch, excl + running));
        }
        tile_base[tid] = digit_base[tid] + excl;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const bool valid = (base + j * 32) < M;
        if (valid) {
            const uint32_t d = (k[j] >> shift) & mask;
            const uint32_t pos = tile_base[d] + warp_hist[warp][d] + rank[j];
            key_out[pos] = k[j];
            idx_out[pos] = id[j];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K3: gather the kept visibilities into sorted SoA arrays
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather(const long long* __restrict__ n_kept, const uint32_t* __restrict__ idx,
                                                const float* __restrict__ u, const float* __restrict__ v,
                                                const float* __restrict__ w, const float2* __restrict__ vis,
                                                const float* __restrict__ wt, float* __restrict__ u_s,
                                                float* __restrict__ v_s, float* __restrict__ w_s,
                                                float2* __restrict__ vis_s, float* __restrict__ wt_s) {
    const long long n = *n_kept;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint32_t src = idx[i];
        u_s[i] = u[src];
        v_s[i] = v[src];
        w_s[i] = w[src];
        vis_s[i] = vis[src];
        wt_s[i] = wt[src];
    }
}

// bin_start[b] = number of sorted tile keys < b, b = 0 .. n_bins + 1
__global__ void __launch_bounds__(256) k_bin_start(RickGeom g, long long M, const uint32_t* __restrict__ key_sorted,
                                                   unsigned long long* __restrict__ bin_start) {
    const uint32_t n_bins = g.n_bins;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i <= M; i += stride) {
        const long long prev = (i == 0) ? -1ll : (long long)rick_tile_of_sort_key(g, key_sorted[i - 1]);
        const long long cur = (i == M) ? (long long)n_bins + 1 : (long long)rick_tile_of_sort_key(g, key_sorted[i]);
        for (long long b = prev + 1; b <= cur; ++b) bin_start[b] = (unsigned long long)i;
    }
}

}  // namespace

size_t rick_bin_workspace_bytes(const rick_plan* p, long long M) {
    (void)p;
    return carve(nullptr, M).total;
}

int rick_bin_impl(rick_plan* p, long long M, const float* u, const float* v, const float* w, const float2* vis,
                  const float* weight, float* u_s, float* v_s, float* w_s, float2* vis_s, float* weight_s,
                  unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out, void* workspace,
                  size_t workspace_bytes, long long* n_kept_dev, cudaStream_t st) {
    (void)workspace_bytes;
    const RickGeom& g = p->g;
    Workspace ws = carve(workspace, M);
    p->bound = false;
    RICK_CUDA(cudaMemsetAsync(n_kept_dev, 0, sizeof(long long), st));
    if (M == 0) {
        if (bin_start_out) {
            RICK_CUDA(cudaMemsetAsync(bin_start_out, 0, sizeof(unsigned long long) * ((size_t)g.n_bins + 2), st));
        }
    } else {
        RICK_CUDA(cudaMemsetAsync((char*)workspace + ws.zero_offset, 0, ws.zero_bytes, st));
        SortLayout lay;
        lay.n_pass = p->n_pass;
        for (int i = 0; i < RICK_MAX_PASSES; ++i) {
            lay.shift[i] = p->digit_shift[i];
            lay.bits[i] = p->digit_bits[i];
        }
        rick_stage_begin(p, RICK_T_KEYGEN, st);
        {
            const long long want = (M + 256 * 8 - 1) / (256 * 8);
            const long long cap = (long long)p->sm_count * 16;
            const int blocks = (int)(want < 1 ? 1 : (want > cap ? cap : want));
            k_keygen<<<blocks, 256, 0, st>>>(g, M, u, v, w, vis, weight, ws.key_a, key_out, ws.hist,
                                             (unsigned long long*)n_kept_dev, lay);
            RICK_LAUNCH_CHECK();
            p->launches++;
        }
        rick_stage_end(p, RICK_T_KEYGEN, st);
        rick_stage_begin(p, RICK_T_SORT, st);
        k_scan_hist<<<p->n_pass, kRadix, 0, st>>>(ws.hist);
        RICK_LAUNCH_CHECK();
        p->launches++;

        const unsigned n_tiles = (unsigned)((M + kSortTile - 1) / kSortTile);
        uint32_t *kin = ws.key_a, *iin = ws.idx_a, *kout = ws.key_b, *iout = ws.idx_b;
        for (int pass = 0; pass < p->n_pass; ++pass) {
            if (pass == 0)
                k_onesweep<true><<<n_tiles, kSortThreads, 0, st>>>(kin, iin, kout, iout, M, lay.shift[pass], lay.bits[pass],
                                                                    ws.hist + pass * kRadix, ws.status, ws.ticket + pass,
                                                                    (uint32_t)(pass + 1));
            else
                k_onesweep<false><<<n_tiles, kSortThreads, 0, st>>>(kin, iin, kout, iout, M, lay.shift[pass], lay.bits[pass],
                                                                     ws.hist + pass * kRadix, ws.status, ws.ticket + pass,
                                                                     (uint32_t)(pass + 1));
            RICK_LAUNCH_CHECK();
            p->launches++;
            uint32_t* t;
            t = kin; kin = kout; kout = t;
            t = iin; iin = iout; iout = t;
        }
        rick_stage_end(p, RICK_T_SORT, st);
        // sorted (key, index) now live in kin / iin
        if (perm_out) {
            RICK_CUDA(cudaMemcpyAsync(perm_out, iin, 4 * (size_t)M, cudaMemcpyDeviceToDevice, st));
        }
        if (bin_start_out) {
            const long long want = (M + 1 + 255) / 256;
            const long long cap = (long long)p->sm_count * 16;
            k_bin_start<<<(int)(want > cap ? cap : want), 256, 0, st>>>(g, M, kin, bin_start_out);
            RICK_LAUNCH_CHECK();
            p->launches++;
        }
        rick_stage_begin(p, RICK_T_GATHER, st);
        {
            const long long want = (M + 255) / 256;
            const long long cap = (long long)p->sm_count * 32;
            k_gather<<<(int)(want > cap ? cap : want), 256, 0, st>>>(n_kept_dev, iin, u, v, w, vis, weight, u_s, v_s, w_s,
                                                                     vis_s, weight_s);
            RICK_LAUNCH_CHECK();
            p->launches++;
        }
        rick_stage_end(p, RICK_T_GATHER, st);
    }
    p->M = M;
    p->u_s = u_s; p->v_s = v_s; p->w_s = w_s; p->vis_s = vis_s; p->weight_s = weight_s;
    p->n_kept_dev = n_kept_dev;
    p->bound = true;
    return RICK_OK;
}
