/*
 * rick.h -- C ABI of librick_b200: the w-stacking imaging hot path of RICK 2.0
 * (arxiv/paper_2601_19714) for one NVIDIA B200 (sm_100a).
 *
 * Path, every step a CUDA kernel:
 *   a0  w range + per-channel scale                       (reading R4)
 *   a1  cell / plane index + sort key                     ("closest w-plane", Eq. 5 :129)
 *   a2  stable device radix sort by (image, plane, uv tile)  (single-GPU analogue of the
 *                                                          paper's bucket sort, :82, :102)
 *   a3  convolutional gridding, Kaiser-Bessel             (Eq. 3 :64, :62)
 *   a4  2-D complex FFT of every w-plane                  (:53, :68)
 *   a5  w-term phase screen + sum over planes             (Eq. 2 :50, :69)
 *   a6  grid correction (division by the kernel transform)  (paper silent; reading R12)
 *
 * Notation: R rows (baseline x time), C channels, M = R*C visibilities (k = r*C + c),
 * N grid edge, N_w w-planes, S kernel support (odd), h = (S-1)/2, dl pixel scale [rad],
 * du = 1/(N dl) cell size [wavelengths].  Grid cell (j,i): row j = v, column i = u,
 * u fastest; cell i <-> u = (i - N/2) du.  Image pixel (q,p): row q = m, column p = l,
 * pixel p <-> l = (p - N/2) dl.
 *
 * Conventions
 *   Pointers: "device" = CUDA device memory of the current device, 16-byte aligned (checked:
 *     RICK_ERR_INVALID otherwise -- the kernels use vector loads); "host" = ordinary host memory
 *     (pinned memory makes the copies asynchronous).  Said per argument.
 *   Ownership: the caller owns every input and output buffer; the library borrows
 *     them until the work it enqueued on the plan's stream has completed and never
 *     frees them.  The plan owns sort items, plane stack, image, tables (for the fp32 grid with
 *     N >= 8192 also a transposed accumulation image of N*N doubles and the per-plane row maps) and
 *     frees them in rick_plan_destroy.
 *   Stream: every call enqueues on the plan's stream and returns without
 *     synchronising, except rick_get_stats, rick_image_host and rick_plan_destroy.
 *   Errors: int return, 0 = RICK_OK, negative = error.  Nothing throws, traps or aborts
 *     across the ABI.  Argument errors (RICK_ERR_INVALID, RICK_ERR_STATE) are detected before
 *     any work is enqueued and leave the plan usable; so does RICK_ERR_OOM (the scratch that
 *     could not grow is re-grown by the next call).  A CUDA failure (RICK_ERR_CUDA: a failed
 *     launch or copy, or the device-side failure flag of the radix sort, which the
 *     synchronising calls read) is STICKY: every later call on that plan returns
 *     RICK_ERR_CUDA until rick_plan_destroy; rick_last_error gives the text of the first failure.
 *   State machine: rick_grid -> rick_fft_wplanes -> rick_wcorrect_accumulate ->
 *     rick_gridcorrect; out of order returns RICK_ERR_STATE.  With
 *     plane_batch < n_wplanes or cube = 1 only rick_image / rick_image_host are
 *     valid (the staged calls need the whole stack of one image resident).
 *   Off-grid visibilities (footprint leaves the grid) are not an error: they are
 *     skipped and counted in n_dropped.  So are visibilities with a non-finite u, v or w
 *     (reading R23); a non-finite w takes no part in the w range.
 *   Threading: a plan is not thread-safe; distinct plans are independent.
 *   There is no CPU fallback: without a CUDA device rick_plan returns RICK_ERR_CUDA.
 */
#ifndef RICK_B200_H
#define RICK_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rick_plan_s rick_plan_t; /* opaque; owns all device scratch */

enum { RICK_OK = 0, RICK_ERR_INVALID = -1, RICK_ERR_STATE = -2, RICK_ERR_CUDA = -3, RICK_ERR_OOM = -4 };
enum { RICK_GRID_F64 = 0, RICK_GRID_F32 = 1 };
enum { RICK_VIS_C64 = 0, RICK_VIS_C128 = 1 };

typedef struct {
    int32_t n;           /* grid edge N: power of two, 64 <= N <= 16384; <= 8192 for F64: one row or
                          * column of the plane (N * 16 B) must fit one SM's shared memory, which is how
                          * every 1-D pass reads and writes the stack exactly once                     */
    int32_t n_wplanes;   /* N_w >= 1                                                            */
    int32_t support;     /* S, odd, 3..15 for F64, 3..9 for F32 (Eq. 5: full kernel width in cells; the
                          * unclamped taper, reading R12, amplifies fp32 rounding beyond the 1e-4 bar
                          * of the fp32 path from S = 11 on)                                    */
    double  pixel_rad;   /* dl, radians per pixel, > 0                                          */
    double  kb_beta;     /* Kaiser-Bessel beta; <= 0 -> 2.34*S (reading R5).  Accepted range: the taper
                          * c(nu) must stay above 1e-12 c(0) on the N pixels (beta >~ pi S / 2 - 1; a
                          * smaller beta puts a zero of c inside the image) and the per-tap polynomial
                          * fit of the kernel must hold to 1e-14 (beta <~ 4 S, and <= 60)        */
    int32_t grid_prec;   /* RICK_GRID_F64 (complex double mesh) | RICK_GRID_F32   */
    int32_t tile;        /* uv-tile edge B in cells (power of two, 8..32); 0 -> 16              */
    int32_t plane_batch; /* w-planes resident at once; 0 -> all N_w                             */
    int32_t cube;        /* 0: all channels into one image; 1: one image per channel (R16)      */
    int32_t flags;       /* RICK_FLAG_* bits, others must be 0                                  */
    double  w_min, w_max; /* wavelengths; NaN -> derived from the data in rick_grid (R4)        */
    int32_t z_begin;     /* w-plane SHARD: this plan owns  */
    int32_t z_count;     /* the planes z_begin .. z_begin + z_count - 1 of the n_wplanes; z_count = 0 ->
                          * all of them (z_begin must be 0).  The w range and the plane of every visibility
                          * are those of the whole problem; visibilities of other planes are skipped (not
                          * counted), off-grid ones are counted by the shard with z_begin = 0 only, so the
                          * statistics of the shards add up.  The image of a shard is its planes' share of
                          * the sum (a5), taper applied (a6 is linear): the shards' images ADD UP to the
                          * image of the whole problem (one reduction over the ranks).  The resident stack
                          * holds min(plane_batch, z_count) planes.  cube = 1 shards by channels instead
                          * (disjoint channel lists, nothing to reduce): z_count must be 0.        */
} rick_plan_desc;

/* flags */
enum { RICK_FLAG_FOLD_W = 1 };  /* reading R24: rows with w < 0 are imaged as (-u,-v,-w)
                                 * with conjugated visibilities (V(-u,-v,-w) = conj V, Eq. 1; the
                                 * image keeps the real part only, R13): every w >= 0, the planes cover half the
                                 * range.  Same direct sum; the w-stacked image differs from the unfolded one
                                 * within the w-quantisation error (it is the more accurate one).        */

typedef struct {
    int64_t n_vis;       /* M of the last rick_grid / rick_image                                */
    int64_t n_gridded;   /* on-grid visibilities                                                */
    int64_t n_dropped;   /* off-grid visibilities, incl. non-finite u, v or w (key = all ones of key_bits) */
    double  sum_w;       /* sum of weights over gridded visibilities                            */
    double  w_min, w_max; /* of image 0 (wavelengths)                                           */
    int64_t n_launches;  /* kernels launched by this plan since creation                        */
    int64_t occ_rows;    /* (plane, row) pairs some footprint reaches, of the last sort: the rows the
                          * row pass transforms and writes, out of n_planes * N                  */
    int64_t occ_tiles;   /* (plane, B x B tile) pairs some footprint reaches: what the zero-fill clears
                          * and the row pass reads, out of n_planes * (N/B)^2                    */
    int64_t n_planes;    /* planes of the last call: N_w, or C * N_w for a cube                 */
    int64_t occ_windows; /* (plane, window of N/32 consecutive rows) pairs with an occupied row, out of
                          * 32 * n_planes: what the fused N = 8192 fp64 column pass fetches     */
} rick_stats;

/* Create a plan: validates `d`, allocates the plane stack
 * (min(plane_batch, N_w) * N*N complex of grid_prec; with cube = 1 and every plane of an
 * image resident, the stacks of up to 8 channel images at once, 48 GB at most, so that one
 * zero-fill, gridder launch and row pass serve a group of channels), the image (N*N double,
 * or the caller's cube slice by slice), tables (FFT twiddles, taper, kernel coefficients)
 * -- the tables are computed by kernels on `cuda_stream` (a cudaStream_t, may be 0).
 * Returns RICK_ERR_INVALID (bad descriptor), RICK_ERR_CUDA (no device / CUDA
 * failure), RICK_ERR_OOM.  *out is NULL on failure.  A cube plan that cannot get the memory for a
 * group of images falls back to one resident image (same results, more launches). */
int rick_plan(rick_plan_t** out, const rick_plan_desc* d, void* cuda_stream);

/* Synchronises the plan's stream and frees everything the plan owns. NULL is OK. */
int rick_plan_destroy(rick_plan_t* p);

/* a0..a3: w range, index + key, stable sort, zero the stack, grid (Eq. 3).
 *   vis          device, [R][C] interleaved (re,im); float pairs if vis_dtype ==
 *                RICK_VIS_C64, double pairs if RICK_VIS_C128
 *   uvw_m        device, [R][3] double, metres
 *   weights      device, [R][C] float, or NULL (all 1: natural weighting)
 *   chan_freq_hz HOST, [C] double, > 0
 *   n_chan       C >= 1;  n_rows  R >= 0 (R = 0 gives an all-zero stack)
 * M = R*C must be < 2^32 - 1, and bits(n_img N_w N^2) + bits(M) <= 64 (one sort item per
 * visibility).  Scratch for the sort items grows as needed
 * (RICK_ERR_OOM if it cannot).  Requires plane_batch == N_w and cube == 0. */
int rick_grid(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
              const float* weights, const double* chan_freq_hz, int32_t n_chan, int64_t n_rows);

/* a4: centred, unnormalised, + sign 2-D transform of every resident plane, in place:
 * P_z[q][p] = sum_{j,i} G_z[j][i] exp(+2 pi i ((i-N/2)(p-N/2) + (j-N/2)(q-N/2))/N). */
int rick_fft_wplanes(rick_plan_t* p);

/* a5: I_raw[q][p] = sum_z Re(P_z[q][p] exp(+2 pi i w_z (n-1))), n = sqrt(1-l^2-m^2),
 * w_z = w_min + (z+0.5)(w_max-w_min)/N_w; pixels with l^2+m^2 >= 1 are 0.  Into the
 * plan's image (no taper). */
int rick_wcorrect_accumulate(rick_plan_t* p);

/* a6: I[q][p] = I_raw[q][p] / (c((p-N/2)/N) c((q-N/2)/N)), c = transform of the kernel. */
int rick_gridcorrect(rick_plan_t* p);

/* a0..a6 in one call, fused / streamed as the plan requires (plane batches, cube).
 * Arguments as rick_grid.  image_out: device, [N][N] double, or [C][N][N] when
 * cube = 1; may be NULL (the result stays in the plan, cube = 0 only). */
int rick_image(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
               const float* weights, const double* chan_freq_hz, int32_t n_chan,
               int64_t n_rows, double* image_out);

/* Same as rick_image with every buffer in HOST memory (pinned memory makes the copies
 * asynchronous): copies the inputs to plan-owned device staging, runs a0..a6, copies
 * the image back to image_out_host and SYNCHRONISES the stream before returning.  Sets of 2^22 or more
 * visibilities on a plan with N <= 4096, plane_batch == N_w and cube == 0 are processed as
 * rick_image_stream_host with two chunks (same image up to summation order, same statistics). */
int rick_image_host(rick_plan_t* p, const void* vis_host, int32_t vis_dtype, const double* uvw_m_host,
                    const float* weights_host, const double* chan_freq_hz, int32_t n_chan,
                    int64_t n_rows, double* image_out_host);

/* Out-of-core visibilities: rick_image_host for a visibility set that need not fit device memory.
 * The host arrays are as in rick_image_host; the visibilities (and weights) cross to the device in
 * chunks of rows_per_chunk rows (>= 1; the last chunk may be shorter) through a two-slot plan-owned
 * staging buffer, the copy of chunk c+1 overlapping index + sort + gridding of chunk c into the same
 * resident stack (gridding is linear in the visibilities, Eq. 3; the single-node analogue of
 * the I/O-compute overlap of PAPER.md:312).  uvw_m_host is copied whole first (24 B per row) and a0 runs
 * over ALL rows, so planes, cells and statistics equal those of one rick_image call; only the summation
 * order differs.  Per-chunk limits as rick_grid with R = rows_per_chunk.  Requires plane_batch == N_w
 * and cube == 0 (RICK_ERR_STATE otherwise).  SYNCHRONISES the stream before returning.  The debug item
 * accessor afterwards describes the last chunk only. */
int rick_image_stream_host(rick_plan_t* p, const void* vis_host, int32_t vis_dtype, const double* uvw_m_host,
                           const float* weights_host, const double* chan_freq_hz, int32_t n_chan,
                           int64_t n_rows, int64_t rows_per_chunk, double* image_out_host);

/* Histogram of the w-planes ("histogram-based balancing"): runs a0 and the
 * index step over all visibilities and counts the on-grid ones per plane of the WHOLE problem (the plan's
 * shard is ignored, RICK_FLAG_FOLD_W is honoured).  uvw_m device [R][3]; chan_freq_hz HOST [C];
 * hist_host HOST [n_wplanes] int64.  cube = 0 only (RICK_ERR_STATE).  SYNCHRONISES the stream. */
int rick_plane_histogram(rick_plan_t* p, const double* uvw_m, const double* chan_freq_hz, int32_t n_chan,
                         int64_t n_rows, int64_t* hist_host);

/* rick_plane_histogram for callers that must not allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, same kernels, same result, and NO cudaMalloc /
 * cudaFree / allocating library routine inside -- the per-call histogram accumulators, the channel scales, the
 * w range and the a0 counters live in one file-scope device array of RICK_NOALLOC_SCRATCH_BYTES bytes that every
 * GPU which loads the library holds until exit.  Limits: n_wplanes <= RICK_NOALLOC_MAX_PLANES and
 * n_chan <= RICK_NOALLOC_MAX_CHAN (RICK_ERR_INVALID with a message otherwise; rick_plane_histogram has no such
 * limit).  The array is shared by every call of every plan on the device and keeps the last call's contents;
 * each call clears what must start at zero.  Calls that overlap on the GPU (plans on different streams, or
 * several host threads) RACE on it: serialise them.  The plan's own state (w range, statistics, channel scales
 * of its last rick_grid / rick_image) is left alone.  SYNCHRONISES the stream. */
enum { RICK_NOALLOC_MAX_PLANES = 4096, RICK_NOALLOC_MAX_CHAN = 1024, RICK_NOALLOC_SCRATCH_BYTES = 41216 };
int rick_plane_histogram_noalloc(rick_plan_t* p, const double* uvw_m, const double* chan_freq_hz, int32_t n_chan,
                                 int64_t n_rows, int64_t* hist_host);

/* Host-only arithmetic (no device, no plan): cut n_wplanes planes into n_parts CONTIGUOUS ranges whose largest
 * cost is minimal, cost(range) = sum over its planes of (hist[z] + plane_cost) -- hist[z] visibilities to sort
 * and grid, plane_cost = what one plane's FFT + correction costs, in visibilities (>= 0).  bounds: [n_parts + 1],
 * range r = planes bounds[r] .. bounds[r+1] - 1; every range holds at least one plane when
 * n_parts <= n_wplanes, else the trailing ranges are empty.  Returns RICK_ERR_INVALID on bad arguments. */
int rick_partition_planes(const int64_t* hist, int32_t n_wplanes, int32_t n_parts, double plane_cost, int32_t* bounds);

/* Copy of the plan's image ([N][N] double) into dst_device (cube = 0 only). */
int rick_get_image(rick_plan_t* p, double* dst_device);

/* SYNCHRONISES the stream; fills *out. */
int rick_get_stats(rick_plan_t* p, rick_stats* out);

/* Text of the last error on this plan ("" if none); valid until the next call. */
const char* rick_last_error(const rick_plan_t* p);

/* Debug accessors for stage-wise parity: device pointers owned by the plan, valid
 * until the next rick_* call on it; NULL if that stage has not run. */
/* [M] sort items (key << *idx_bits) | k, key = ((((img N_w + i_p) T + i_v/B) T + i_u/B) B + i_v%B) B + i_u%B
 * (T = N/B; image, plane, uv tile, cell inside the tile: DESIGN.md step 4), the all-ones pattern
 * of *key_bits bits for a dropped visibility.  sorted = 0: in visibility order (item k describes
 * visibility k); sorted = 1: after the stable sort by key -- the low parts are then the permutation. */
const uint64_t* rick_debug_items(rick_plan_t* p, int32_t sorted, int32_t* idx_bits, int32_t* key_bits);
void*           rick_debug_planes(rick_plan_t* p); /* [N_w][N][N] complex of grid_prec; meaningful after the
                                                    * STAGED calls only: rick_image leaves the stack
                                                    * half-transformed (occupied rows transformed along u, the
                                                    * column pass fused with the correction never writes planes;
                                                    * on the two-pass fallback also the first column pass) */

/* Per-kernel timing with CUDA events on the plan's stream (for roofline reporting).
 * rick_profile(p, 1) clears the records and brackets every later kernel launch with a
 * pair of events; rick_profile(p, 0) stops.  Both SYNCHRONISE the stream.
 * rick_profile_read SYNCHRONISES and returns, for one kernel class, the summed duration in
 * milliseconds and the number of launches since profiling was enabled.
 * rick_kernel_name(id): "grid", "fft_rows", "fft_cols", "wcorrect", ...; NULL past the end. */
int rick_profile(rick_plan_t* p, int32_t enable);
int rick_profile_read(rick_plan_t* p, int32_t kernel_id, double* total_ms, int64_t* launches);
const char* rick_kernel_name(int32_t kernel_id);

/* Library identification, e.g. "librick_b200 0.1 sm_100a". */
const char* rick_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RICK_B200_H */
