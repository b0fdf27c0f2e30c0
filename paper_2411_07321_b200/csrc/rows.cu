// rows.cu -- row occupancy of the mesh (rick_plan_set_fusion mode 2).
//
// The synthetic LOFAR-shaped workloads leave most (plane, row) pairs of the mesh untouched (60 % on config
// 10M: the outer w-planes hold a few tracks each).  In fusion mode 2 the library keeps a bitmap of the rows
// some footprint touches and spends memory traffic only on those: rick_grid clears only rows that are
// touched and not yet defined, the fused column transform reads only defined rows (and takes zeros for the
// others).  Untouched rows of the mesh hold undefined data in this mode.
//   occ_cur   rows touched by the visibilities bound by the last rick_bin (rows j0-h .. j0+h of plane k)
//   occ_mesh  rows that hold defined data (cleared or gridded) since the last rick_grid(zero_first != 0)
// Where the library's own long-row kernel runs (rowbig.cu: N >= 4096) the same is kept per SEGMENT of a row
// (64 segments of N / 64 cells, one 64-bit mask per row: seg_cur, seg_mesh): the tracks of the outer planes cross a
// row in a few places only (hotspot: 29 % of the segments of the touched rows, 5.8 of 20.3 GB), so rick_grid clears
// only touched segments and the row transform reads only defined ones and takes zeros for the rest of the row.
#include "rick_internal.cuh"

namespace {

// (j0 << 16 | i0, k) of the sorted kept visibility i: from the gridder records, or decoded from the sorted sort keys
// (then i0 = the first column of the visibility's tile: only i0 >> 5 is used)
// (indirect mode: sort key = tile key << cb | cell bits, rick_internal.cuh)
struct RowsFromRecords {
    const uint2* ga;
    __device__ __forceinline__ uint2 operator()(const RickGeom&, long long i) const { return __ldg(ga + i); }
};
struct RowsFromKeys {
    const uint32_t* key;
    int log2T;           // >= 0: T = N / 32 is a power of two (shifts instead of two integer divisions per key)
    __device__ __forceinline__ uint2 decode(const RickGeom& g, uint32_t sk) const {
        const uint32_t tile = sk >> g.cell_bits, cell = (sk & ((1u << g.cell_bits) - 1u)) << (10 - g.cell_bits);
        uint32_t tx, ty, k;
        if (log2T >= 0) {
            tx = tile & ((1u << log2T) - 1u);
            ty = (tile >> log2T) & ((1u << log2T) - 1u);
            k = tile >> (2 * log2T);
        } else {
            const uint32_t T = (uint32_t)g.T;
            tx = tile % T;
            ty = (tile / T) % T;
            k = tile / (T * T);
        }
        return make_uint2(((ty * 32u + (cell >> 5)) << 16) | (tx * 32u), k);       // (j0 << 16 | first column of the tile, k)
    }
};

// rows j0-h .. j0+h of plane k as one or two word masks; bits only ever get set, so a plain (L2) read that
// already shows them saves the atomic: the many tiles of a mesh row would otherwise all hit one word
__device__ __forceinline__ void mark_rows(const RickGeom& g, uint32_t j0, uint32_t k, uint32_t tx, uint32_t* __restrict__ occ,
                                          unsigned long long* __restrict__ seg, int seg_shift) {
    const uint32_t lo = k * (uint32_t)g.N + (j0 - (uint32_t)g.h), hi = lo + 2u * (uint32_t)g.h;
    if (seg) {
        // segment mode: the footprints of the visibilities of tile column tx lie in columns 32 tx - h .. 32 tx + 31 + h:
        // one or two segments (a segment is at least 64 cells wide), marked on the CENTRE row j0 only; k_segs_dilate
        // spreads them over j0 - h .. j0 + h afterwards, and the row bitmap follows from the masks (k_segs_new)
        const int c_lo = (int)(tx * 32u) - g.h, c_hi = (int)(tx * 32u) + 31 + g.h;
        const int s_lo = (c_lo < 0 ? 0 : c_lo) >> seg_shift, s_hi = (c_hi > g.N - 1 ? g.N - 1 : c_hi) >> seg_shift;
        const unsigned long long m = (1ull << s_lo) | (1ull << s_hi);
        unsigned long long* c = seg + (k * (uint32_t)g.N + j0);
        if ((__ldcg(c) & m) != m) atomicOr(c, m);
        return;
    }
    const uint32_t w0 = lo >> 5, w1 = hi >> 5;
    const uint32_t span = (2u * (uint32_t)g.h + 1u);
    const uint32_t m0 = (span >= 32u ? 0xffffffffu : ((1u << span) - 1u)) << (lo & 31);
    if ((__ldcg(occ + w0) & m0) != m0) atomicOr(occ + w0, m0);
    if (w1 != w0) {
        const uint32_t m1 = (1u << ((hi & 31) + 1u)) - 1u;
        if ((__ldcg(occ + w1) & m1) != m1) atomicOr(occ + w1, m1);
    }
}

// one thread per sorted kept visibility: the first of every (plane, row j0, tile column) group sets the 2h+1 bits
template <typename Src>
__global__ void __launch_bounds__(256) k_rows_mark(RickGeom g, const long long* __restrict__ n_kept,
                                                   Src ga, uint32_t* __restrict__ occ,
                                                   unsigned long long* __restrict__ seg, int seg_shift) {
    const long long n = *n_kept;
    const long long stride = (long long)gridDim.x * blockDim.x;
    // four records (and their predecessors) per trip, all loads first: one dependent DRAM wait per four
    // records instead of one per record (the kernel was 90 % long-scoreboard stalls at 1.8 TB/s)
    constexpr int kU = 4;
    for (long long i0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; i0 < n; i0 += kU * stride) {
        uint2 a[kU], b[kU];
#pragma unroll
        for (int x = 0; x < kU; ++x) {
            const long long i = i0 + x * stride;
            a[x] = b[x] = make_uint2(0xffffffffu, 0xffffffffu);          // no record: never a group start's equal
            if (i < n) {
                a[x] = ga(g, i);
                if (i > 0) b[x] = ga(g, i - 1);
            }
        }
#pragma unroll
        for (int x = 0; x < kU; ++x) {
            if (i0 + x * stride >= n) break;
            const uint32_t j0 = a[x].x >> 16, k = a[x].y, tx = (a[x].x & 0xffffu) >> 5;
            if ((b[x].x >> 16) == j0 && b[x].y == k && ((b[x].x & 0xffffu) >> 5) == tx) continue;   // same (plane, row, tile)
            mark_rows(g, j0, k, tx, occ, seg, seg_shift);
        }
    }
}

// The same from the sorted sort keys (indirect mode), eight consecutive keys per thread and trip with two 16-byte
// loads: a key with its column bits shifted out names its (plane, tile, row); only the first key of every such
// group decodes and marks.  (One key per thread through the generic kernel waited on its two dependent loads:
// 2.8 ms on hotspot.)
__global__ void __launch_bounds__(256) k_rows_mark_keys(RickGeom g, const long long* __restrict__ n_kept,
                                                        const uint32_t* __restrict__ key, int log2T,
                                                        uint32_t* __restrict__ occ,
                                                        unsigned long long* __restrict__ seg, int seg_shift) {
    const long long n = *n_kept;
    const int col_bits = g.cell_bits - 5;                 // cell_bits >= 5: the row-in-tile bits are always kept
    const RowsFromKeys dec{key, log2T};
    const long long stride = (long long)gridDim.x * blockDim.x * 8;
    for (long long base = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 8; base < n; base += stride) {
        // the key array is padded to whole multiples of 4096 entries: the two loads stay inside it
        const uint4 a = __ldg(reinterpret_cast<const uint4*>(key + base));
        const uint4 b = __ldg(reinterpret_cast<const uint4*>(key + base + 4));
        const uint32_t prev = base > 0 ? __ldg(key + base - 1) : 0u;
        const uint32_t k8[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            if (base + x >= n) break;
            const uint32_t before = x ? k8[x - 1] : prev;
            if ((base + x > 0) && (before >> col_bits) == (k8[x] >> col_bits)) continue;
            const uint2 r = dec.decode(g, k8[x]);
            mark_rows(g, r.x >> 16, r.y, (r.x & 0xffffu) >> 5, occ, seg, seg_shift);
        }
    }
}

// all == 0: rows to clear = occ_cur & ~occ_mesh, as a list, and occ_mesh |= occ_cur;
// all != 0: the list of all rows of occ_mesh (for the row transforms).  One warp per bitmap word; the
// words take their places in the list with one atomicAdd each on *n_rows (zeroed by the caller), so the
// order of the list is arbitrary -- its users (k_rows_zero, k_rowfft) take the rows in any order.
__global__ void __launch_bounds__(256) k_rows_new(int n_words, const uint32_t* __restrict__ occ_cur,
                                                  uint32_t* __restrict__ occ_mesh, uint32_t* __restrict__ list,
                                                  uint32_t* __restrict__ n_rows, int all) {
    const int w = (int)blockIdx.x * 8 + (int)(threadIdx.x >> 5), lane = (int)(threadIdx.x & 31);
    if (w >= n_words) return;
    uint32_t fresh = 0, pos = 0;
    if (lane == 0) {
        const uint32_t m = occ_mesh[w];
        if (all) {
            fresh = m;
        } else {
            const uint32_t c = occ_cur[w];
            fresh = c & ~m;
            if (fresh) occ_mesh[w] = m | c;
        }
        if (fresh) pos = atomicAdd(n_rows, (uint32_t)__popc(fresh));
    }
    fresh = __shfl_sync(0xffffffffu, fresh, 0);
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if ((fresh >> lane) & 1u) list[pos + (uint32_t)__popc(fresh & ((1u << lane) - 1u))] = (uint32_t)w * 32u + (uint32_t)lane;
}

// clear the listed rows (N cells of cell_bytes each)
__global__ void __launch_bounds__(256) k_rows_zero(const uint32_t* __restrict__ list, const uint32_t* __restrict__ n_rows,
                                                   uint4* __restrict__ grid, int row_vec /* 16-byte pieces per row */) {
    const uint32_t n = *n_rows;
    for (uint32_t r = blockIdx.x; r < n; r += gridDim.x) {
        uint4* row = grid + (size_t)list[r] * row_vec;
        for (int i = threadIdx.x; i < row_vec; i += 256) row[i] = make_uint4(0u, 0u, 0u, 0u);
    }
}

// Segment mode: cur[r] = OR of the centre-row masks c0[r - h .. r + h] (rows j0 < h and j0 > N - 1 - h are never
// centres, D5, so nothing leaks across a plane boundary)
__global__ void __launch_bounds__(256) k_segs_dilate(int n_rows, int h, const unsigned long long* __restrict__ c0,
                                                     unsigned long long* __restrict__ cur) {
    const int r = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (r >= n_rows) return;
    unsigned long long m = 0;
    for (int d = -h; d <= h; ++d) {
        const int q = r + d;
        if (q >= 0 && q < n_rows) m |= __ldg(c0 + q);
    }
    cur[r] = m;
}

// Segment mode.  One warp per 32 rows: rows with a touched segment that is not defined yet go on the list, with the
// mask of those segments in seg_fresh; seg_mesh |= seg_cur; the row bitmap occ_mesh |= "some segment touched".
__global__ void __launch_bounds__(256) k_segs_new(int n_words, const unsigned long long* __restrict__ seg_cur,
                                                  unsigned long long* __restrict__ seg_mesh,
                                                  unsigned long long* __restrict__ seg_fresh, uint32_t* __restrict__ occ_mesh,
                                                  uint32_t* __restrict__ list, uint32_t* __restrict__ n_rows) {
    const int w = (int)blockIdx.x * 8 + (int)(threadIdx.x >> 5), lane = (int)(threadIdx.x & 31);
    if (w >= n_words) return;
    const uint32_t row = (uint32_t)w * 32u + (uint32_t)lane;
    const unsigned long long c = seg_cur[row], m = seg_mesh[row], f = c & ~m;
    const uint32_t touched = __ballot_sync(0xffffffffu, c != 0ull), fresh = __ballot_sync(0xffffffffu, f != 0ull);
    if (f) {
        seg_mesh[row] = m | c;
        seg_fresh[row] = f;
    }
    uint32_t pos = 0;
    if (lane == 0) {
        if (touched) occ_mesh[w] |= touched;
        if (fresh) pos = atomicAdd(n_rows, (uint32_t)__popc(fresh));
    }
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if (f) list[pos + (uint32_t)__popc(fresh & ((1u << lane) - 1u))] = row;
}

// clear the fresh segments of the listed rows (seg_vec 16-byte pieces per segment); the warps of a block share a
// row's segments round robin
__global__ void __launch_bounds__(256) k_segs_zero(const uint32_t* __restrict__ list, const uint32_t* __restrict__ n_rows,
                                                   const unsigned long long* __restrict__ seg_fresh,
                                                   uint4* __restrict__ grid, int row_vec, int seg_vec) {
    const uint32_t n = *n_rows;
    const int warp = (int)(threadIdx.x >> 5), lane = (int)(threadIdx.x & 31);
    for (uint32_t r = blockIdx.x; r < n; r += gridDim.x) {
        const uint32_t row = list[r];
        unsigned long long f = seg_fresh[row];
        uint4* base = grid + (size_t)row * row_vec;
        for (int o = 0; f; ++o) {
            const int s = __ffsll((long long)f) - 1;
            f &= f - 1;
            if ((o & 7) != warp) continue;
            uint4* p = base + (size_t)s * seg_vec;
            for (int i = lane; i < seg_vec; i += 32) p[i] = make_uint4(0u, 0u, 0u, 0u);
        }
    }
}

}  // namespace

int rick_rows_mark(rick_plan* p, long long M, cudaStream_t st) {
    const size_t words = (size_t)p->g.Nw * p->g.N / 32;
    RICK_CUDA(cudaMemsetAsync(p->occ_cur_dev, 0, 4 * words, st));
    // segment mode: centre-row masks into seg_fresh (free between two rick_grid calls), dilated into seg_cur below
    unsigned long long* seg = p->segs ? p->seg_fresh_dev : nullptr;
    const int n_rows = p->g.Nw * p->g.N;
    int seg_shift = 0;
    while ((64 << seg_shift) < p->g.N) ++seg_shift;                     // a segment is N / 64 = 2^seg_shift cells
    if (seg) RICK_CUDA(cudaMemsetAsync(seg, 0, 8 * (size_t)n_rows, st));
    if (M == 0) {
        if (seg) RICK_CUDA(cudaMemsetAsync(p->seg_cur_dev, 0, 8 * (size_t)n_rows, st));
        return RICK_OK;
    }
    const long long want = (M + 255) / 256;
    const long long cap = (long long)p->sm_count * 16;
    if (p->indirect) {
        int log2T = -1;
        for (int b = 0; b < 16; ++b) if ((1 << b) == p->g.T) log2T = b;
        const long long want8 = (M / 8 + 255) / 256 + 1;
        k_rows_mark_keys<<<(int)(want8 > cap ? cap : want8), 256, 0, st>>>(p->g, p->n_kept_dev, p->gkey, log2T, p->occ_cur_dev, seg, seg_shift);
    }
    else
        k_rows_mark<<<(int)(want > cap ? cap : want), 256, 0, st>>>(p->g, p->n_kept_dev, RowsFromRecords{p->grec_a}, p->occ_cur_dev, seg, seg_shift);
    RICK_LAUNCH_CHECK();
    p->launches++;
    if (seg) {
        k_segs_dilate<<<(n_rows + 255) / 256, 256, 0, st>>>(n_rows, p->g.h, seg, p->seg_cur_dev);
        RICK_LAUNCH_CHECK();
        p->launches++;
    }
    return RICK_OK;
}

int rick_rows_clear(rick_plan* p, void* grid, int zero_first, cudaStream_t st) {
    const int words = (int)((size_t)p->g.Nw * p->g.N / 32);
    if (zero_first) RICK_CUDA(cudaMemsetAsync(p->occ_mesh_dev, 0, 4 * (size_t)words, st));
    RICK_CUDA(cudaMemsetAsync(p->n_rows_dev, 0, 4, st));
    if (p->segs) {      // clear the touched segments that are not defined yet
        const int cell = (p->dtype == RICK_C128) ? 16 : 8;
        if (zero_first) RICK_CUDA(cudaMemsetAsync(p->seg_mesh_dev, 0, 8 * (size_t)words * 32, st));
        k_segs_new<<<(words + 7) / 8, 256, 0, st>>>(words, p->seg_cur_dev, p->seg_mesh_dev, p->seg_fresh_dev, p->occ_mesh_dev,
                                                    p->row_list_dev, p->n_rows_dev);
        RICK_LAUNCH_CHECK();
        k_segs_zero<<<p->sm_count * 8, 256, 0, st>>>(p->row_list_dev, p->n_rows_dev, p->seg_fresh_dev, (uint4*)grid,
                                                     p->g.N * cell / 16, p->g.N / 64 * cell / 16);
        RICK_LAUNCH_CHECK();
        p->launches += 2;
        return RICK_OK;
    }
    k_rows_new<<<(words + 7) / 8, 256, 0, st>>>(words, p->occ_cur_dev, p->occ_mesh_dev, p->row_list_dev, p->n_rows_dev, 0);
    RICK_LAUNCH_CHECK();
    const int cell = (p->dtype == RICK_C128) ? 16 : 8;
    k_rows_zero<<<p->sm_count * 8, 256, 0, st>>>(p->row_list_dev, p->n_rows_dev, (uint4*)grid, p->g.N * cell / 16);
    RICK_LAUNCH_CHECK();
    p->launches += 2;
    return RICK_OK;
}

// list of all defined rows (for rick_fft_planes in fusion mode 2)
int rick_rows_list_all(rick_plan* p, cudaStream_t st) {
    const int words = (int)((size_t)p->g.Nw * p->g.N / 32);
    RICK_CUDA(cudaMemsetAsync(p->n_rows_dev, 0, 4, st));
    k_rows_new<<<(words + 7) / 8, 256, 0, st>>>(words, p->occ_cur_dev, p->occ_mesh_dev, p->row_list_dev, p->n_rows_dev, 1);
    RICK_LAUNCH_CHECK();
    p->launches++;
    return RICK_OK;
}
