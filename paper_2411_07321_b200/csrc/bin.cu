// bin.cu -- rick_bin: key generation, hand-written stable LSD radix sort (one-sweep style, decoupled
// look-back), gather of the SoA payload, optional bin offsets.   [D2-D5], BASELINE.json north_star (2).
//
// The key that is sorted is the (w-plane, 32x32 tile) key of D4 refined by the in-tile cell index
// [D4']: the order is still grouped by plane and tile, and visibilities with the same nearest cell
// are adjacent, which is what lets rick_grid accumulate whole runs in registers.
//
// Passes and traffic per visibility (algorithmic):
//   K1 keygen+histograms   read 24 B, write 4 B key + 32 B staging record (one sector per visibility)
//   K2 one-sweep pass x n_pass (n_pass = ceil(key_bits / 9): 3 for 27-bit keys, 4 for 28-32 bits)
//                          read 8 B (4 B in the first pass: the index is implicit), write 8 B
//   K3 gather              read 4 B index + one 32-B record (random rows), write 24 B
#include "rick_internal.cuh"
#include <type_traits>

namespace {

constexpr int kRadix = 1 << RICK_RADIX_BITS_MAX;   // 512 digit values at most
constexpr int kSortTile = 8192;                        // keys per tile
// shape of a one-sweep CTA: 256 threads x 32 keys, or, for the plain passes over 9-bit digits, 512 threads x 16 keys
// (one digit per thread, 64 registers, two CTAs = 32 warps per SM: 0.269 -> 0.228 ms for the three passes of config 10M;
// the same shape on 8-bit digits, where half the threads would own no digit, measured slower: 22.2 against 19.6 ms on
// hotspot, and 54 against 46 ms for the gather variant at one CTA per SM)
template <int kBits, bool kGather> struct SortShape {
    static constexpr int kThreads = (kBits == 9 && !kGather) ? 512 : 256;
    static constexpr int kItems = kSortTile / kThreads;
    static constexpr int kWarps = kThreads / 32;
    static constexpr int kMinBlocks = kThreads == 512 ? 2 : ((kBits == 8 && !kGather) ? 3 : 2);
};
constexpr int kSortAhead = 48;     // tickets between a tile and the one whose input it sends on its way to the L2

struct SortLayout {
    int n_pass;
    int shift[RICK_MAX_PASSES];
    int bits[RICK_MAX_PASSES];
};

struct Workspace {
    uint32_t *key_a, *key_b, *idx_a, *idx_b;
    float4* rec;                     // [M][2]: (u, v, w, re), (im, weight, -, -): one 32-B sector per visibility
    float2 *grec_b, *grec_c;         // gridder records b[], c[] of the sorted kept visibilities (rick_internal.cuh)
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
    const size_t mp = (m + RICK_GREC_PAD - 1) / RICK_GREC_PAD * RICK_GREC_PAD;   // whole gridder chunks
    // (key, index) ping and pong, each pair contiguous: the pair that is dead after the last pass is
    // reused for the 8-byte gridder records a[]
    ws.key_a = (uint32_t*)(b + off); off += 4 * mp;
    ws.idx_a = (uint32_t*)(b + off); off += 4 * mp;
    ws.key_b = (uint32_t*)(b + off); off += 4 * mp;
    ws.idx_b = (uint32_t*)(b + off); off += 4 * mp;
    ws.rec = (float4*)(b + off); off += rick_align256(32 * m);
    ws.grec_b = (float2*)(b + off); off += rick_align256(8 * mp);
    ws.grec_c = (float2*)(b + off); off += rick_align256(8 * mp);
    ws.zero_offset = off;
    ws.hist = (uint32_t*)(b + off); off += rick_align256(sizeof(uint32_t) * RICK_MAX_PASSES * kRadix);
    ws.ticket = (uint32_t*)(b + off); off += rick_align256(sizeof(uint32_t) * RICK_MAX_PASSES);
    ws.status = (unsigned long long*)(b + off); off += rick_align256(sizeof(unsigned long long) * n_tiles * kRadix);
    ws.zero_bytes = off - ws.zero_offset;
    ws.total = off;
    return ws;
}

// ---------------------------------------------------------------------------------------------
// K1: sort keys + AoS staging records + global digit histograms of every pass + n_kept
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_keygen(RickGeom g, long long M, const float* __restrict__ u,
                                                const float* __restrict__ v, const float* __restrict__ w,
                                                const float2* __restrict__ vis, const float* __restrict__ wt,
                                                uint32_t* __restrict__ key, float4* __restrict__ rec,
                                                uint32_t* __restrict__ tile_key_out, uint32_t* __restrict__ hist,
                                                unsigned long long* __restrict__ n_kept, SortLayout lay, int rec_form) {
    __shared__ uint32_t sh[RICK_MAX_PASSES][kRadix];
    for (int i = threadIdx.x; i < RICK_MAX_PASSES * kRadix; i += blockDim.x) (&sh[0][0])[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    unsigned kept = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    // warp-uniform trip count so that every lane reaches the votes
    // the loads of the next trip are issued before this trip's arithmetic and votes (twice the bytes in
    // flight per thread: the kernel waits on DRAM latency, not on bandwidth)
    float uu = 0.f, vv = 0.f, ww = 0.f, wgt = 0.f;
    float2 vi = make_float2(0.f, 0.f);
    {
        const long long m0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (m0 < M) { uu = __ldg(u + m0); vv = __ldg(v + m0); ww = __ldg(w + m0); wgt = __ldg(wt + m0); vi = __ldg(vis + m0); }
    }
    for (long long base = (long long)blockIdx.x * blockDim.x; base < M; base += stride) {
        const long long m = base + threadIdx.x;
        const bool valid = m < M;
        uint32_t kk = 0;
        const float uu_c = uu, vv_c = vv, ww_c = ww, wgt_c = wgt;
        const float2 vi_c = vi;
        if (m + stride < M) {
            const long long mn = m + stride;
            uu = __ldg(u + mn); vv = __ldg(v + mn); ww = __ldg(w + mn); wgt = __ldg(wt + mn); vi = __ldg(vis + mn);
        }
        if (valid) {
            const float uu = uu_c, vv = vv_c, ww = ww_c, wgt = wgt_c;
            const float2 vi = vi_c;
            RickLoc r = rick_locate(g, uu, vv, ww);
            const bool fin = rick_finite(uu) && rick_finite(vv) && rick_finite(ww) && rick_finite(wgt) &&
                             rick_finite(vi.x) && rick_finite(vi.y);
            const bool keep = r.keep && fin;
            kk = keep ? rick_sort_key(g, r) : g.sort_sentinel;
            kept += keep ? 1u : 0u;
            key[m] = kk;
            if (rec_form == 0) {     // raw visibility: the gather copies it to the sorted SoA and derives the gridder record
                rec[2 * m] = make_float4(uu, vv, ww, vi.x);
                rec[2 * m + 1] = make_float4(vi.y, wgt, 0.f, 0.f);
            } else {                 // the gridder record itself (rick_internal.cuh): the fp32 gridder fetches it by index
                const float ws = ((r.j0 - g.h) & 1) ? -wgt : wgt;
                rec[2 * m] = make_float4(__uint_as_float((uint32_t)r.i0 | ((uint32_t)r.j0 << 16)), __uint_as_float((uint32_t)r.k),
                                         (float)((double)r.i0 - r.x), (float)((double)r.j0 - r.y));
                rec[2 * m + 1] = make_float4(ws * vi.x, ws * vi.y, 0.f, 0.f);
            }
            if (tile_key_out) tile_key_out[m] = keep ? rick_tile_key(g, r) : g.n_bins;
        }
        // digit histograms: lanes that share lane 0's digit (the common case in the skewed high
        // digits) are counted with one vote, the rest with one shared-memory atomic each
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        const int first = __ffs(act) - 1;
#pragma unroll
        for (int p = 0; p < RICK_MAX_PASSES; ++p) {
            if (p < lay.n_pass) {
                const uint32_t d = (kk >> lay.shift[p]) & ((1u << lay.bits[p]) - 1u);
                const uint32_t d0 = __shfl_sync(0xffffffffu, d, first);
                const unsigned same = __ballot_sync(0xffffffffu, valid && d == d0);
                if (lane == first) atomicAdd(&sh[p][d0], (uint32_t)__popc(same));
                else if (valid && d != d0) atomicAdd(&sh[p][d], 1u);
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

// exclusive scan of each pass's kRadix digit counts, in place (one block per pass)
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
// K2: one stable LSD pass (one-sweep).  Tiles take their id from a ticket (so that every predecessor
// is already running), rank their keys per warp with ballots (stable: items are warp-striped and
// visited in order), publish per-digit tile counts and resolve their global offsets by decoupled
// look-back, exchange the tile through shared memory into digit order and write it out in runs.
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

// Outputs of the gather: sorted SoA copies and gridder records (rick_internal.cuh) of the kept visibilities.
struct GatherOut {
    RickGeom g;
    const float4* rec;
    float *u_s, *v_s, *w_s;
    float2* vis_s;
    float* wt_s;
    uint2* ga;
    float2 *gb, *gc;
};

// input visibility `src` goes to sorted position `pos`: one 32-byte record read, SoA + record writes; the
// fp64 coordinate arithmetic is repeated here because the kernel waits on memory anyway
__device__ __forceinline__ void gather_one(const GatherOut& o, size_t src, size_t pos) {
    const float4 a = __ldg(o.rec + 2 * src);
    const float4 b = __ldg(o.rec + 2 * src + 1);
    o.u_s[pos] = a.x;
    o.v_s[pos] = a.y;
    o.w_s[pos] = a.z;
    o.vis_s[pos] = make_float2(a.w, b.x);
    o.wt_s[pos] = b.y;
    const RickLoc r = rick_locate(o.g, a.x, a.y, a.z);
    const float ws = ((r.j0 - o.g.h) & 1) ? -b.y : b.y;       // (-1)^(j0-h): checkerboard factor of the fp32 gridder
    o.ga[pos] = make_uint2((uint32_t)r.i0 | ((uint32_t)r.j0 << 16), (uint32_t)r.k);
    o.gb[pos] = make_float2((float)((double)r.i0 - r.x), (float)((double)r.j0 - r.y));
    o.gc[pos] = make_float2(ws * a.w, ws * b.x);
}

// sized by the digit width and the CTA shape: 74 KB for 8-bit digits (256 threads, three CTAs per SM), 84 KB for the
// gather passes over 9-bit digits (256 threads, two CTAs), 100 KB for the plain ones (512 threads, two CTAs)
template <int kBits, int kSortWarps> struct SortSmem {
    uint32_t warp_cnt[kSortWarps][1 << kBits];   // per-warp digit counts -> exclusive offsets over warps
    uint32_t tile_excl[1 << kBits];              // first slot of each digit in the exchanged tile
    uint32_t glob[1 << kBits];                   // global position of slot i of digit d = glob[d] + i
    uint32_t xkey[kSortTile];
    uint32_t xidx[kSortTile];
    uint32_t warp_sum[kSortWarps];
    uint32_t tile;
};

template <int kBits, bool kGather> constexpr int sort_smem_bytes() {
    return (int)sizeof(SortSmem<kBits, SortShape<kBits, kGather>::kWarps>);
}

// kGather: this is the last pass and nobody asked for the sorted (key, index) arrays: instead of writing them,
// the tile gathers its visibilities straight to their final positions (the gather's random reads hide
// under the pass's arithmetic, and 12 bytes per visibility of key/index traffic disappear).
// Registers: only the keys and their ranks live through the ranking loop (the kernel is latency-bound: resident
// warps are what it needs -- three CTAs per SM for the plain 8-bit passes, 23.0 -> 21.6 ms for the four passes of
// hotspot; the gather variant keeps two CTAs of 128 registers, it needs them for the fp64 coordinates); the keys go to their exchange slots before the look-back, and the input indices are
// loaded only then, in flight during the look-back, and follow into the slots the ranks (now slot numbers) name.
template <bool kFirst, int kBits, bool kGather>
__global__ void __launch_bounds__((SortShape<kBits, kGather>::kThreads), (SortShape<kBits, kGather>::kMinBlocks)) k_onesweep(const uint32_t* __restrict__ key_in,
                                                               const uint32_t* __restrict__ idx_in,
                                                               uint32_t* __restrict__ key_out,
                                                               uint32_t* __restrict__ idx_out, long long M, int shift,
                                                               const uint32_t* __restrict__ digit_base,
                                                               unsigned long long* __restrict__ status,
                                                               uint32_t* __restrict__ ticket, uint32_t epoch,
                                                               GatherOut go, uint32_t ahead) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    typedef SortShape<kBits, kGather> Shape;
    constexpr int kSortThreads = Shape::kThreads, kSortItems = Shape::kItems, kSortWarps = Shape::kWarps;
    typedef SortSmem<kBits, kSortWarps> Smem;
    Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) sm.tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < kSortWarps * (1 << kBits); i += kSortThreads) (&sm.warp_cnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = sm.tile;
    const long long tile_base = (long long)tile * kSortTile;
    // the tile a CTA will take `ahead` tickets from now starts its way from DRAM to the L2: 8 lanes x 4 KB of keys
    // (and of indices).  Any distance from 8 to 110 tickets measures the same (hotspot: 21.9 -> 19.6 ms for the four
    // passes); a whole wave of resident CTAs (444) is too far: the lines are evicted before use (13.1 instead of
    // 8.2 GB of DRAM reads per pass).
    if (tid < 8) {
        const long long pf = ((long long)tile + ahead) * kSortTile;
        if (pf + kSortTile <= M) {
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(key_in + pf + tid * (kSortTile / 8)), "r"(kSortTile / 8 * 4) : "memory");
            if (!kFirst)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(idx_in + pf + tid * (kSortTile / 8)), "r"(kSortTile / 8 * 4) : "memory");
        }
    }
    const long long base = tile_base + (long long)warp * (kSortItems * 32) + lane;
    constexpr uint32_t mask = (1u << kBits) - 1u;
    constexpr int kDigitsPerThread = (1 << kBits) / kSortThreads;   // 2 (9-bit digits) or 1 (8-bit digits)
    static_assert(kDigitsPerThread >= 1, "digit width too small for the block size");

    uint32_t k[kSortItems];
    typedef typename std::conditional<(kSortItems <= 16), uint32_t, uint16_t>::type rank_t;
    rank_t rank[kSortItems];                // rank in the warp's digit bucket, later the exchange slot (< 8192)
    const unsigned lt = (1u << lane) - 1u;
    const bool full = tile_base + kSortTile <= M;     // every tile but the last: no validity tests
    // rank of an item among the items of its warp with the same digit (stable: lanes in order), by one
    // ballot per digit bit; the warp's running count of the digit is kept by the lowest peer lane
    auto rank_items = [&](auto full_c) {
        constexpr bool kFull = decltype(full_c)::value;
#pragma unroll
        for (int j = 0; j < kSortItems; ++j) {
            const long long gidx = base + j * 32;
            const bool valid = kFull || gidx < M;
            k[j] = valid ? __ldg(key_in + gidx) : 0u;
        }
#pragma unroll
        for (int j = 0; j < kSortItems; ++j) {
            const bool valid = kFull || (base + j * 32) < M;
            const uint32_t d = (k[j] >> shift) & mask;
            unsigned peers = kFull ? 0xffffffffu : __ballot_sync(0xffffffffu, valid);
#pragma unroll
            for (int b = 0; b < kBits; ++b) {
                unsigned m;      // lanes whose bit b equals this lane's
                asm("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\t"
                    "and.b32 t, %1, %2;\n\t"
                    "setp.ne.u32 p, t, 0;\n\t"
                    "vote.sync.ballot.b32 %0, p, 0xffffffff;\n\t"
                    "@!p not.b32 %0, %0;\n\t}"
                    : "=r"(m) : "r"(d), "r"(1u << b));
                peers &= m;
            }
            const int leader = __ffs(peers) - 1;   // valid lanes always contain themselves
            uint32_t c = 0;
            if (valid && lane == leader) {
                c = sm.warp_cnt[warp][d];
                sm.warp_cnt[warp][d] = c + (uint32_t)__popc(peers);
            }
            c = __shfl_sync(0xffffffffu, c, valid ? leader : lane);
            rank[j] = (rank_t)(c + (uint32_t)__popc(peers & lt));
            __syncwarp();
        }
    };
    if (full) rank_items(std::true_type{});
    else rank_items(std::false_type{});
    __syncthreads();

    // per-digit totals over the warps (thread t owns digits 2t, 2t+1), exclusive offsets in place
    uint32_t tot[kDigitsPerThread];
#pragma unroll
    for (int q = 0; q < kDigitsPerThread; ++q) {
        const int d = tid * kDigitsPerThread + q;
        uint32_t running = 0;
#pragma unroll
        for (int wv = 0; wv < kSortWarps; ++wv) {
            const uint32_t c = sm.warp_cnt[wv][d];
            sm.warp_cnt[wv][d] = running;
            running += c;
        }
        tot[q] = running;
    }
    // publish the tile aggregate as early as possible
    if (tile == 0) {
#pragma unroll
        for (int q = 0; q < kDigitsPerThread; ++q)
            st_status(status + (size_t)tile * kRadix + tid * kDigitsPerThread + q, pack_status(2u, epoch, tot[q]));
    } else {
#pragma unroll
        for (int q = 0; q < kDigitsPerThread; ++q)
            st_status(status + (size_t)tile * kRadix + tid * kDigitsPerThread + q, pack_status(1u, epoch, tot[q]));
    }
    // exclusive scan of the digit totals over the tile (slot of each digit in the exchanged order)
    uint32_t mine = 0;
#pragma unroll
    for (int q = 0; q < kDigitsPerThread; ++q) mine += tot[q];
    uint32_t incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) sm.warp_sum[warp] = incl;
    __syncthreads();
    uint32_t before = 0;
#pragma unroll
    for (int wv = 0; wv < kSortWarps; ++wv) before += (wv < warp) ? sm.warp_sum[wv] : 0u;
    uint32_t excl_tile = before + incl - mine;
    uint32_t texcl[kDigitsPerThread];
#pragma unroll
    for (int q = 0; q < kDigitsPerThread; ++q) {
        texcl[q] = excl_tile;
        sm.tile_excl[tid * kDigitsPerThread + q] = excl_tile;
        excl_tile += tot[q];
    }
    __syncthreads();                                  // tile_excl and the warp offsets are complete
    // the keys take their places in digit order now: the ranks become slot numbers and the key registers are free
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const bool valid = full || (base + j * 32) < M;
        if (valid) {
            const uint32_t d = (k[j] >> shift) & mask;
            const uint32_t lp = sm.tile_excl[d] + sm.warp_cnt[warp][d] + rank[j];
            sm.xkey[lp] = k[j];
            rank[j] = (rank_t)lp;
        }
    }
    // the input indices, in flight during the look-back
    uint32_t id[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const long long gidx = base + j * 32;
        id[j] = kFirst ? (uint32_t)gidx : ((full || gidx < M) ? __ldg(idx_in + gidx) : 0u);
    }
    // decoupled look-back: a window of kLookWin predecessors per digit is loaded at once (independent
    // loads in flight), then consumed from the nearest tile backwards up to the first inclusive prefix
    if (tile != 0) {
        // the digits of a thread walk back together, so that their polls are in flight at the same time
        constexpr int kLookWin = 4 / kDigitsPerThread;
        uint32_t excl[kDigitsPerThread];
        long long t[kDigitsPerThread];
        bool done[kDigitsPerThread];
#pragma unroll
        for (int q = 0; q < kDigitsPerThread; ++q) { excl[q] = 0; t[q] = (long long)tile - 1; done[q] = false; }
        bool all_done = false;
        while (!all_done) {
            unsigned long long sv[kDigitsPerThread][kLookWin];
#pragma unroll
            for (int q = 0; q < kDigitsPerThread; ++q)
#pragma unroll
                for (int x = 0; x < kLookWin; ++x) {
                    const long long tt = t[q] - x;
                    sv[q][x] = (!done[q] && tt >= 0)
                                   ? ld_status(status + (size_t)tt * kRadix + tid * kDigitsPerThread + q) : 0ull;
                }
            all_done = true;
#pragma unroll
            for (int q = 0; q < kDigitsPerThread; ++q) {
#pragma unroll
                for (int x = 0; x < kLookWin; ++x) {
                    if (done[q] || t[q] < 0) continue;
                    const unsigned long long v = sv[q][x];
                    const bool ready = (uint32_t)((v >> 32) & 0x3FFFFFFFu) == epoch && (v >> 62) != 0ull;
                    if (!ready) break;           // re-poll from this tile
                    excl[q] += (uint32_t)v;
                    if ((v >> 62) == 2ull || t[q] == 0) done[q] = true;
                    --t[q];
                }
                all_done = all_done && done[q];
            }
        }
#pragma unroll
        for (int q = 0; q < kDigitsPerThread; ++q) {
            const int d = tid * kDigitsPerThread + q;
            st_status(status + (size_t)tile * kRadix + d, pack_status(2u, epoch, excl[q] + tot[q]));
            sm.glob[d] = digit_base[d] + excl[q] - texcl[q];
        }
    } else {
#pragma unroll
        for (int q = 0; q < kDigitsPerThread; ++q) {
            const int d = tid * kDigitsPerThread + q;
            sm.glob[d] = digit_base[d] - texcl[q];
        }
    }
    // the indices follow the keys into digit order
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        if (full || (base + j * 32) < M) sm.xidx[rank[j]] = id[j];
    }
    __syncthreads();
    const long long left = M - tile_base;
    const int n_valid = left < (long long)kSortTile ? (int)left : kSortTile;
    for (int i = tid; i < n_valid; i += kSortThreads) {
        const uint32_t kk = sm.xkey[i];
        const uint32_t d = (kk >> shift) & mask;
        const uint32_t pos = sm.glob[d] + (uint32_t)i;
        if (kGather) {
            if (kk != go.g.sort_sentinel) gather_one(go, (size_t)sm.xidx[i], (size_t)pos);   // kept: pos < n_kept
        } else {
            key_out[pos] = kk;
            idx_out[pos] = sm.xidx[i];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K3: gather the kept visibilities into sorted SoA arrays (one 32-B record read per visibility) and
// write the gridder records: nearest cell, plane, fractional offsets (fp64 difference narrowed once)
// and weight * V with the run-constant checkerboard factor (-1)^(j0-h) of the fp32 gridder folded in.
// The kernel waits on memory, so the fp64 coordinate arithmetic is free here.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather(GatherOut o, const long long* __restrict__ n_kept,
                                                const uint32_t* __restrict__ idx) {
    const long long n = *n_kept;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        gather_one(o, (size_t)__ldg(idx + i), (size_t)i);
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

int rick_bin_init() {
    const cudaFuncAttribute a = cudaFuncAttributeMaxDynamicSharedMemorySize;
    if (cudaFuncSetAttribute(k_onesweep<true, 8, false>, a, sort_smem_bytes<8, false>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<true, 9, false>, a, sort_smem_bytes<9, false>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<false, 8, false>, a, sort_smem_bytes<8, false>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<false, 9, false>, a, sort_smem_bytes<9, false>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<true, 8, true>, a, sort_smem_bytes<8, true>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<true, 9, true>, a, sort_smem_bytes<9, true>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<false, 8, true>, a, sort_smem_bytes<8, true>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_onesweep<false, 9, true>, a, sort_smem_bytes<9, true>()) != cudaSuccess)
        return RICK_ECUDA;
    return RICK_OK;
}

int rick_bin_impl(rick_plan* p, long long M, const float* u, const float* v, const float* w, const float2* vis,
                  const float* weight, float* u_s, float* v_s, float* w_s, float2* vis_s, float* weight_s,
                  unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out, void* workspace,
                  long long* n_kept_dev, cudaStream_t st) {
    const RickGeom& g = p->g;
    Workspace ws = carve(workspace, M);
    p->bound = false;
    // No sorted SoA asked for (fp32 mesh only): nothing is gathered.  The staging records are the gridder records,
    // the sort ends with the sorted (key, index) pairs, and the gridder fetches its records through the index
    // -- the 1e9 random 32-byte reads of the gather (the GPU's random-access rate bounds them) then run under the
    // gridder's arithmetic instead of under a sort pass that has none.
    const bool indirect = (u_s == nullptr);
    p->indirect = indirect;
    p->gidx = nullptr;
    p->grec = nullptr;
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
            k_keygen<<<blocks, 256, 0, st>>>(g, M, u, v, w, vis, weight, ws.key_a, ws.rec, key_out, ws.hist,
                                             (unsigned long long*)n_kept_dev, lay, indirect ? 1 : 0);
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
        (void)iout;
        // the gather rides in the last pass unless the caller wants the sorted (key, index) arrays
        const bool fuse_gather = !indirect && !perm_out && !bin_start_out;
        GatherOut go;
        go.g = g; go.rec = ws.rec;
        go.u_s = u_s; go.v_s = v_s; go.w_s = w_s; go.vis_s = vis_s; go.wt_s = weight_s;
        go.ga = nullptr; go.gb = ws.grec_b; go.gc = ws.grec_c;
        for (int pass = 0; pass < p->n_pass; ++pass) {
            const bool first = (pass == 0);
            const bool nine = (lay.bits[pass] == 9);
            const bool gath = fuse_gather && pass == p->n_pass - 1;
            if (gath) go.ga = (uint2*)kout;       // this pass writes no (key, index): the pair holds records a[]
            auto kern = gath ? (first ? (nine ? k_onesweep<true, 9, true> : k_onesweep<true, 8, true>)
                                      : (nine ? k_onesweep<false, 9, true> : k_onesweep<false, 8, true>))
                             : (first ? (nine ? k_onesweep<true, 9, false> : k_onesweep<true, 8, false>)
                                      : (nine ? k_onesweep<false, 9, false> : k_onesweep<false, 8, false>));
            const int threads = gath ? (nine ? SortShape<9, true>::kThreads : SortShape<8, true>::kThreads)
                                     : (nine ? SortShape<9, false>::kThreads : SortShape<8, false>::kThreads);
            const int smem = gath ? (nine ? sort_smem_bytes<9, true>() : sort_smem_bytes<8, true>())
                                  : (nine ? sort_smem_bytes<9, false>() : sort_smem_bytes<8, false>());
            kern<<<n_tiles, threads, smem, st>>>(kin, iin, kout, iout, M, lay.shift[pass],
                                                                 ws.hist + pass * kRadix, ws.status, ws.ticket + pass,
                                                                 (uint32_t)(pass + 1), go,
                                                                 (uint32_t)kSortAhead);
            RICK_LAUNCH_CHECK();
            p->launches++;
            if (gath) break;
            uint32_t* t;
            t = kin; kin = kout; kout = t;
            t = iin; iin = iout; iout = t;
        }
        rick_stage_end(p, RICK_T_SORT, st);
        rick_stage_begin(p, RICK_T_GATHER, st);
        if (fuse_gather) {
            p->grec_a = (const uint2*)kout;
        } else if (indirect) {
            // sorted (key, index) live in kin / iin; kept visibilities come first
            if (perm_out) RICK_CUDA(cudaMemcpyAsync(perm_out, iin, 4 * (size_t)M, cudaMemcpyDeviceToDevice, st));
            if (bin_start_out) {
                const long long want = (M + 1 + 255) / 256;
                const long long cap = (long long)p->sm_count * 16;
                k_bin_start<<<(int)(want > cap ? cap : want), 256, 0, st>>>(g, M, kin, bin_start_out);
                RICK_LAUNCH_CHECK();
                p->launches++;
            }
            p->gidx = iin;
            p->gkey = kin;
            p->grec = ws.rec;
        } else {
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
            const long long want = (M + 255) / 256;
            const long long cap = (long long)p->sm_count * 32;
            go.ga = (uint2*)kout;
            k_gather<<<(int)(want > cap ? cap : want), 256, 0, st>>>(go, n_kept_dev, iin);
            RICK_LAUNCH_CHECK();
            p->launches++;
            p->grec_a = (const uint2*)kout;
        }
        rick_stage_end(p, RICK_T_GATHER, st);
    }
    if (M == 0) p->indirect = false;
    if (p->fused == 2) {
        p->n_kept_dev = n_kept_dev;
        const int rc = rick_rows_mark(p, M, st);
        if (rc != RICK_OK) return rc;
    }
    p->M = M;
    p->u_s = u_s; p->v_s = v_s; p->w_s = w_s; p->vis_s = vis_s; p->weight_s = weight_s;
    p->n_kept_dev = n_kept_dev;
    p->grec_b = ws.grec_b; p->grec_c = ws.grec_c;
    p->bound = true;
    return RICK_OK;
}

// ---------------------------------------------------------------------------------------------
// rick_bin_static (rick_b200.h): rick_bin for callers that cannot allocate.  The workspace rick_bin_impl carves
// (sort keys and indices, staging records, histograms, tickets, look-back words) is this file-scope device array.
// Every GPU that loads the library holds it until exit; every plan and call on a device shares it, and it keeps
// the last call's contents: rick_bin_impl clears the region that must start at zero on the caller's stream, as it
// does for a caller workspace.  Calls that overlap on the GPU race on it (rick_b200.h).
// In host code the array's name is a host-side stand-in, not a device address: the address handed to the kernels
// comes from cudaGetSymbolAddress, looked up once per device with that device current.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char rick_bin_static_scratch[RICK_BIN_STATIC_BYTES];

extern "C" int rick_bin_static(rick_plan* p, long long M, const float* u, const float* v, const float* w,
                               const void* vis, const float* weight, float* u_s, float* v_s, float* w_s, void* vis_s,
                               float* weight_s, unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out,
                               long long* n_kept_dev, void* stream) {
    if (!p || M < 0 || !n_kept_dev) return RICK_EINVAL;
    if (M > RICK_BIN_STATIC_MAX_M || carve(nullptr, M).total > (size_t)RICK_BIN_STATIC_BYTES) return RICK_ELIMIT;
    if (M > 0 && (!u || !v || !w || !vis || !weight)) return RICK_EINVAL;
    const int n_sorted = (u_s != nullptr) + (v_s != nullptr) + (w_s != nullptr) + (vis_s != nullptr) + (weight_s != nullptr);
    if (n_sorted != 0 && n_sorted != 5) return RICK_EINVAL;
    if (n_sorted == 0 && p->dtype == RICK_C128) return RICK_EINVAL;
    int dev = -1;
    RICK_CUDA(cudaGetDevice(&dev));
    if (dev != p->device || dev < 0 || dev >= RICK_MAX_DEVICES) return RICK_EINVAL;   // the look-up below needs the plan's device current
    static void* scratch_of_device[RICK_MAX_DEVICES] = {};
    void* scratch = scratch_of_device[dev];
    if (!scratch) {
        RICK_CUDA(cudaGetSymbolAddress(&scratch, rick_bin_static_scratch));
        if (!scratch || ((uintptr_t)scratch & 255)) return RICK_ECUDA;
        scratch_of_device[dev] = scratch;
    }
    cudaStream_t st = (cudaStream_t)stream;
    rick_stage_begin(p, RICK_T_BIN, st);
    const int rc = rick_bin_impl(p, M, u, v, w, (const float2*)vis, weight, u_s, v_s, w_s, (float2*)vis_s, weight_s,
                                 key_out, perm_out, bin_start_out, scratch, n_kept_dev, st);
    rick_stage_end(p, RICK_T_BIN, st);
    return rc;
}
