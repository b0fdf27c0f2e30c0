/* rick_b200.h -- C ABI of librick_b200: the single-GPU w-stacking imaging hot path on NVIDIA B200 (sm_100a).
 *
 * What it computes (citations: P:n = PAPER.md line n of arXiv 2411.07321; D1-D9 = the readings listed
 * in DESIGN.md "Readings of the paper"):
 *
 *   rick_bin                   per-visibility nearest cell / nearest w-plane / keep-drop decision and a
 *                              stable device radix sort by (w-plane, 32x32 uv tile) key.  Replaces the
 *                              paper's per-slab bucket arrays; "visibilities are mapped to the
 *                              closest w-plane".                                     [D2-D5]
 *   rick_grid                  convolutional gridding, Eq. 3, with the separable truncated
 *                              Gaussian G = g(i-x) g(j-y), g(d) = exp(-d^2 / 2 sigma^2).         [D6]
 *   rick_fft_planes            un-normalised inverse 2-D DFT (sign +) of every w-plane,
 *                              batched cuFFT C2C / Z2Z, in place.                                [D7]
 *   rick_wcorrect_accumulate   phase screen exp(+2 pi i w_k (sqrt(1-l^2-m^2)-1)), sum over planes
 *                              (Eq. 2; step 4) and division by the kernel taper.     [D8]
 *   rick_image                 hands the fp64 N x N dirty image to the caller.
 *
 * Conventions
 *   - Every function returns RICK_OK (0) or a negative rick_status; nothing throws or exits.
 *   - "device" pointers are CUDA device pointers on the current device, "host" pointers are host memory.
 *     The caller owns every buffer it passes; the library owns only the plan (geometry constants, the
 *     1-D taper table, the cuFFT handle, stage-timing events, the copy stream and hand-over events of
 *     rick_image_from_host_chunked).  Allocation happens only in the rick_plan_* calls (create, set_dtype,
 *     set_kernel, set_fusion); the path calls (rick_bin ... rick_image_from_host_chunked) allocate nothing.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is
 *     enqueued asynchronously on it unless stated otherwise.
 *   - Geometry [D1]: du = 1/(N dl).  Mesh node i <-> u = (i - N/2) du; pixel p <-> l = (p - N/2) dl.
 *   - Layouts: mesh grid[k][j][i], i (u) fastest, interleaved (re, im), float2 (RICK_C64) or double2
 *     (RICK_C128), 16-byte aligned (RICK_EINVAL otherwise: 16-byte reductions and bulk copies);
 *     image[q][p], p (l) fastest, q <-> m, fp64.
 *   - Modulated mesh: rick_grid stores (-1)^(i+j) * V~(u_i, v_j, w_k) and rick_wcorrect_accumulate
 *     applies (-1)^(p+q); with the plain (un-shifted) cuFFT in between this equals the centred
 *     transform of D7 exactly (sign flips only, N even).  A caller comparing the mesh with Eq. 3 must
 *     multiply by the checkerboard.
 *   - Precision: RICK_C64 keeps visibility x weight x taps, the mesh and the FFT in fp32;
 *     coordinates, indices, the fractional offsets (before narrowing), the w phase, the plane sum and
 *     the image are fp64.  RICK_C128 is fp64 throughout.
 */
#ifndef RICK_B200_H
#define RICK_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rick_plan rick_plan; /* opaque */

typedef enum {
    RICK_OK = 0,
    RICK_EINVAL = -1,  /* bad argument (see each function) */
    RICK_ENOMEM = -2,  /* a caller-provided workspace is too small, or plan allocation failed */
    RICK_ECUDA = -3,   /* a CUDA runtime call or kernel launch failed */
    RICK_ECUFFT = -4,  /* a cuFFT call failed */
    RICK_ESTATE = -5,  /* call order: rick_grid before rick_bin, FFT before rick_plan_set_dtype, ... */
    RICK_ELIMIT = -6   /* rick_bin_static: M exceeds RICK_BIN_STATIC_MAX_M, the capacity of the library's static scratch */
} rick_status;

typedef enum { RICK_C64 = 0, RICK_C128 = 1 } rick_dtype;

/* gridding kernel families of rick_plan_set_kernel */
typedef enum { RICK_KERNEL_GAUSS = 0, RICK_KERNEL_KB = 1 } rick_kernel;

/* stage indices of rick_get_timings */
enum { RICK_T_BIN = 0, RICK_T_ZERO = 1, RICK_T_GRID = 2, RICK_T_FFT = 3, RICK_T_WCORRECT = 4,
       RICK_T_IMAGE = 5,
       /* parts of RICK_T_BIN */
       RICK_T_KEYGEN = 6, RICK_T_SORT = 7, RICK_T_GATHER = 8,
       /* parts of RICK_T_FFT when the column transform is fused (rick_plan_set_fusion): the row transforms and
          sweep A of the split column transform */
       RICK_T_FFT_ROWS = 9, RICK_T_FFT_COL_A = 10, RICK_T_COUNT = 11 };

/* Create a plan (BASELINE.json north_star (1)).  Host-synchronous.
 *   N        mesh and image size per axis; a multiple of 32 (tile size), 32 <= N <= 32768
 *   Nw       number of w-planes, 1 <= Nw <= 4096, Nw (N/32)^2 <= 2^27
 *   support  full footprint width S in cells, odd, 3 <= S <= 15  (h = (S-1)/2)
 *   sigma    Gaussian width in cells, >= 0.25 (narrower kernels are refused: RICK_EINVAL)
 *   w_min, w_max   w range covered by the Nw planes, w_max > w_min; plane k is centred at
 *            w_min + (k + 1/2)(w_max - w_min)/Nw  [D3]
 *   dl       pixel size (direction cosine per pixel), > 0, N dl < sqrt(2)
 * Errors: RICK_EINVAL, RICK_ENOMEM, RICK_ECUDA.  The mesh dtype defaults to RICK_C64. */
int rick_plan_create(int N, int Nw, int support, double sigma, double w_min, double w_max, double dl,
                     rick_plan** out);

/* Select the mesh dtype and (re)build the cuFFT plan for it.  Host-synchronous. */
int rick_plan_set_dtype(rick_plan* plan, int dtype);

/* Gridding kernel G of Eq. 3.  Default: the separable truncated Gaussian of rick_plan_create
 * (BASELINE.json north_star) [D6].  RICK_KERNEL_KB selects the separable Kaiser-Bessel window the paper's
 * own tests use: g(d) = I0(beta sqrt(1 - (d / a_t)^2)) / I0(beta), |d| <= a_t = support / 2, with
 * shape parameter `param` = beta > 0 (sigma is then unused), and the taper table becomes its exact
 * transform 2 a_t sinh(z) / (z I0(beta)), z = sqrt(beta^2 - (2 pi a_t nu)^2)  [D6-KB, D8-KB].
 * Host-synchronous (rebuilds the taper and tap tables); call before rick_grid / rick_wcorrect_accumulate.
 * Errors: RICK_EINVAL (unknown kind, beta <= 0 or > 64), RICK_ENOMEM, RICK_ECUDA. */
int rick_plan_set_kernel(rick_plan* plan, int kind, double param);

/* Fused column transform (optional; N a power of two, 256 <= N <= 16384, either mesh dtype, and on the fp32 mesh
 * |w| < 2^28 wavelengths; RICK_EINVAL otherwise; call after rick_plan_set_dtype, which switches it off, and before
 * rick_bin).  RICK_C64 with N <= 2048 uses the one-sweep kernel (whole column blocks in shared memory); larger N and
 * RICK_C128 use the split engine: rick_fft_planes also runs the first half of the column transform in place, and
 * rick_wcorrect_accumulate the second half.
 * on = 1: rick_fft_planes runs only the row transforms of D7 (the mesh then holds row-transformed planes),
 * and rick_wcorrect_accumulate performs the column transforms itself, fused with the phase screen, the plane
 * sum and the taper division, in one read of the mesh [D7, D8]; the image is the same within fp32 round-off.
 * on = 2: in addition the library tracks which mesh rows (plane, j) some footprint touches: rick_grid clears
 * only touched rows that are not defined yet (instead of the whole mesh) and the fused kernel reads only
 * defined rows; mesh rows no footprint touches then hold UNDEFINED data (only the image is an output).  Where the
 * library's own long-row kernel runs (N >= 4096; RICK_C128: N <= 8192) the same holds per segment of a row
 * (64 segments of N / 64 cells): only touched segments are cleared and read, the rest of a touched row is
 * undefined between rick_grid and rick_fft_planes as well.
 * on = 0: off. */
int rick_plan_set_fusion(rick_plan* plan, int on);

/* Fusion mode 2 only: number of mesh rows (plane, j) that held defined data at the last rick_fft_planes
 * (of Nw * N).  Host-synchronous.  RICK_ESTATE in other modes. */
int rick_plan_rows_defined(rick_plan* plan, long long* rows);

/* Fusion mode 2 only: number of mesh cells that hold defined data since the last rick_grid(zero_first != 0) -- the
 * cells of the defined segments, or of the defined rows where rows are the unit.  Host-synchronous (copies the
 * segment masks to the host).  RICK_ESTATE in other modes. */
int rick_plan_cells_defined(rick_plan* plan, long long* cells);

/* Sizes of the two caller-provided scratch buffers: `bin_bytes` for rick_bin with up to M
 * visibilities, `fft_bytes` for rick_fft_planes (0 if cuFFT needs none).  Either pointer may be NULL. */
int rick_plan_workspace_bytes(const rick_plan* plan, long long M, size_t* bin_bytes, size_t* fft_bytes);

int rick_plan_destroy(rick_plan* plan);

/* Layout of the key rick_bin sorts by [D4']: total key bits, number of radix passes (digits of <= 9
 * bits) and the number of in-tile cell bits appended to the tile key.  Any pointer may be NULL. */
int rick_plan_sort_layout(const rick_plan* plan, int* key_bits, int* n_pass, int* cell_bits);

/* Key generation + stable radix sort + gather.  [D2-D5], BASELINE.json north_star (2).
 *   M                     number of visibilities, 0 <= M < 2^32 - 1
 *   u, v, w               device float[M], baseline coordinates in wavelengths
 *   vis                   device float2[M] (complex64), weight: device float[M]
 *   u_s .. weight_s       device outputs of capacity M: the kept visibilities in the stable order [D4'];
 *                         only the first n_kept entries are written.  Either all five, or all five NULL
 *                         (RICK_C64 plans only): then nothing is gathered -- the library keeps the sorted
 *                         input indices in the workspace and rick_grid fetches its 32-byte records through
 *                         them ("indirect mode": the random reads of the gather run under the gridder's
 *                         arithmetic instead of under a sort pass).  RICK_C128 plans need the five outputs
 *                         (the fp64 gridder reads them): RICK_EINVAL otherwise
 *   key_out               nullable device unsigned[M]: key of every input visibility,
 *                         key = (k T + (j0 >> 5)) T + (i0 >> 5), T = N/32; dropped -> Nw T^2
 *   perm_out              nullable device unsigned[M]: sorted rank -> input index (all M, dropped ones last; in
 *                         indirect mode a copy of the index the gridder uses)
 *   bin_start_out         nullable device unsigned long long[Nw T^2 + 2]: number of visibilities with
 *                         key < b (entry Nw T^2 is n_kept, the last entry is M)
 *   workspace             device scratch of at least rick_plan_workspace_bytes(M) bytes, 256-byte aligned
 *   n_kept_dev            device long long: number of kept visibilities
 * A visibility is dropped whole (never clipped or wrapped) when any of its six numbers is non-finite,
 * its footprint would leave the mesh, or w lies outside [w_min, w_max]  [D5]; that is not an error.
 * The sorted arrays, n_kept_dev and the workspace are bound to the plan and must stay valid and
 * unmodified until the last rick_grid call that uses them.
 * Errors: RICK_EINVAL (null pointer, M out of range), RICK_ENOMEM (workspace too small), RICK_ECUDA. */
int rick_bin(rick_plan* plan, long long M, const float* u, const float* v, const float* w,
             const void* vis, const float* weight, float* u_s, float* v_s, float* w_s, void* vis_s,
             float* weight_s, unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out,
             void* workspace, size_t workspace_bytes, long long* n_kept_dev, void* stream);

/* rick_bin without a caller workspace, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * serving loops, harnesses that forbid allocation): the same kernels, the same arguments minus `workspace`, the same
 * outputs [D2-D5]; the scratch (sort keys and indices, staging records, digit histograms, look-back words: about
 * 64.5 bytes per visibility) lives in ONE file-scope device array of the library, RICK_BIN_STATIC_BYTES (17 MiB),
 * which every GPU that loads the library holds until the process exits.
 *   M    0 <= M <= RICK_BIN_STATIC_MAX_M (262144); a larger M is refused with RICK_ELIMIT before anything is enqueued
 *        (use rick_bin with a workspace of your own for larger inputs)
 * The call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating library routine): it looks up the
 * array's device address once per device (cudaGetSymbolAddress, with the plan's device current -- RICK_EINVAL if
 * another device is current) and hands it to rick_bin's kernels.  Everything else is rick_bin: the plan is bound
 * to the static scratch until the last rick_grid that uses it.
 * The array is shared by EVERY plan and every call on that device and keeps the last call's contents; the call
 * clears the part that must start at zero (histograms, tickets, look-back words) itself, on `stream`.  Two calls
 * (or one call and a rick_grid bound to an earlier one) that overlap on the GPU -- different streams, or two host
 * threads -- race on it: order them on one stream or with events.
 * Errors: those of rick_bin, plus RICK_ELIMIT. */
#define RICK_BIN_STATIC_MAX_M 262144
#define RICK_BIN_STATIC_BYTES (17u << 20)
int rick_bin_static(rick_plan* plan, long long M, const float* u, const float* v, const float* w,
                    const void* vis, const float* weight, float* u_s, float* v_s, float* w_s, void* vis_s,
                    float* weight_s, unsigned* key_out, unsigned* perm_out, unsigned long long* bin_start_out,
                    long long* n_kept_dev, void* stream);

/* Gridding, Eq. 3 [D6], of the visibilities bound by the last rick_bin into
 * grid[Nw][N][N] (device, dtype of the plan, caller-owned).  zero_first != 0 clears the mesh first;
 * zero_first == 0 accumulates onto its contents (chunked inputs).
 * Errors: RICK_ESTATE (no rick_bin yet), RICK_EINVAL, RICK_ECUDA. */
int rick_grid(rick_plan* plan, void* grid, int zero_first, void* stream);

/* In-place un-normalised inverse 2-D DFT of every plane [D7].  fft_work: device scratch of at least
 * the `fft_bytes` reported by rick_plan_workspace_bytes (may be NULL when that is 0).
 * Errors: RICK_ESTATE (dtype never set), RICK_ENOMEM, RICK_ECUFFT. */
int rick_fft_planes(rick_plan* plan, void* grid, void* fft_work, size_t fft_work_bytes, void* stream);

/* image[q][p] (+)= (1 / (t[p] t[q])) sum_k Re{ exp(+2 pi i w_k nm1(q,p)) P_k[q][p] },
 * nm1 = -(l^2+m^2)/(1+sqrt(1-l^2-m^2)), t = 1-D taper of the truncated Gaussian [D8].
 * Reads every transformed plane once.  image: device double[N*N]. */
int rick_wcorrect_accumulate(rick_plan* plan, const void* grid, double* image, int zero_first,
                             void* stream);

/* Copy the fp64 image to `out` (device if out_is_host == 0, host otherwise; asynchronous either way:
 * synchronise the stream before reading a host buffer). */
int rick_image(rick_plan* plan, const double* image_dev, double* out, int out_is_host, void* stream);

/* Device buffers for rick_image_from_host (all caller-owned, capacity M where per-visibility). */
typedef struct {
    float *u, *v, *w; void* vis; float* weight;          /* staging for the inputs */
    float *u_s, *v_s, *w_s; void* vis_s; float* weight_s;/* sorted copies */
    void* workspace; size_t workspace_bytes;             /* rick_bin scratch */
    void* grid;                                          /* Nw*N*N complex mesh */
    void* fft_work; size_t fft_work_bytes;
    double* image;                                       /* N*N */
    long long* n_kept;                                   /* device scalar */
} rick_device_buffers;

/* The whole path from HOST buffers to a HOST image: H2D copies of the five input arrays, rick_bin,
 * rick_grid (zero_first), rick_fft_planes, rick_wcorrect_accumulate (zero_first), D2H of the image.
 * Everything is enqueued on `stream`; the call returns after synchronising it.  Host buffers should
 * be pinned for the copies to run at full speed. */
int rick_image_from_host(rick_plan* plan, long long M, const float* u_host, const float* v_host,
                         const float* w_host, const void* vis_host, const float* weight_host,
                         const rick_device_buffers* dev, double* image_host, void* stream);

/* rick_image_from_host with the input split into n_chunks time slices ("the data are read and
 * gridded in chunks"): the host-to-device copies of slice i+1 run on a second stream while slice i is binned
 * and gridded onto the mesh (rick_grid with zero_first only for slice 0), then one rick_fft_planes,
 * rick_wcorrect_accumulate and the image copy.  The staging arrays of `dev` (capacity M) are used as two
 * halves, so a slice holds at most M/2 visibilities (rounded to a multiple of 1024); n_chunks < 2 or
 * M < 2048 falls back to rick_image_from_host.  The image equals the single-slice one up to the order of
 * the floating-point additions on the mesh.  With the fused column kernels (rick_plan_set_fusion) the image
 * is computed in up to four stripes of whole columns, each copied to image_host by the second stream while the
 * next stripe is computed.  Returns after synchronising `stream` and the copies. */
int rick_image_from_host_chunked(rick_plan* plan, long long M, const float* u_host, const float* v_host,
                                 const float* w_host, const void* vis_host, const float* weight_host,
                                 const rick_device_buffers* dev, int n_chunks, double* image_host,
                                 void* stream);

/* CUDA-event times (milliseconds) of the most recent call of each stage, indexed by RICK_T_*;
 * stages never run report 0.  Synchronises on the recorded events.  n <= RICK_T_COUNT. */
int rick_get_timings(rick_plan* plan, double* ms, int n);

/* Number of launches of the library's own kernels issued through this plan so far (memsets, copies and
 * cuFFT's internal kernels are not counted). */
long long rick_launch_count(const rick_plan* plan);

/* Measurement helper (not part of the imaging path; host-synchronous, allocates 4 bytes and frees them):
 * the fp32 rates of the current device from a register-resident microbenchmark on all SMs at full occupancy.
 *   fma_tflops   2 x 1e12 fused multiply-adds per second (the fp32 FMA peak, TFLOP/s)
 *   add_tinst    1e12 fp32 additions per second
 *   fma2_tflops  the same FMA chain with the packed fma.rn.f32x2 of sm_100 (4 flop per lane-op), TFLOP/s
 * bench.py reports issue-bound kernels against these measured numbers. */
int rick_measure_fp32_rate(double* fma_tflops, double* add_tinst, double* fma2_tflops, void* stream);

/* Measurement helper (host-synchronous; allocates 2 GB of device memory and frees it): how many random 32-byte
 * records per second (1e9 / s) this GPU reads from a 2 GB array at full occupancy -- the rate that bounds a
 * gather (the gridder's record fetch in indirect mode). */
int rick_measure_random_read_rate(double* grecords_per_s, void* stream);

const char* rick_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* RICK_B200_H */
