// common.cuh -- internal declarations of librick_b200 (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>
#include <string>
#include <vector>

#include "../../include/rick.h"

#define RICK_C0 299792458.0
#define RICK_MAX_CHAN 4096
#define RICK_KB_DEG 18          // degree of the per-tap polynomial of the Kaiser-Bessel kernel

// Per-image w-plane geometry, computed on the device by k_wrange_finish (a0).
struct WRange {
    double w_min, w_max, dw, inv_dw;
};

// Small block of device-resident scalars (zeroed at the start of every rick_grid).
struct DevCounters {
    unsigned long long wmin_bits;   // ordered encoding of min over rows of w [m]
    unsigned long long wmax_bits;   // ordered encoding of max over rows of w [m]
    unsigned long long n_gridded;   // on-grid visibilities
    unsigned long long n_dropped;
    double sum_w;                   // sum of weights over gridded visibilities
    unsigned int grid_chunk;        // dynamic work counter of the gridder
    unsigned int error;             // sticky device-side failure flag (a radix tile lost its predecessor)
};

struct rick_plan_s {
    rick_plan_desc d;
    int N, Nw, S, h, B, T, log2N, log2B;
    int Nw_total, z0;        // the whole problem's planes and this plan's first one (Nw = planes of this shard)
    int fold;                // RICK_FLAG_FOLD_W
    int f32;                 // grid precision
    int batch;               // resident planes
    double beta, dl, inv_du;
    cudaStream_t stream;
    cudaStream_t stream2;    // low-priority side stream: the zero-fill runs beside index + sort
    cudaStream_t stream3;    // copy stream of rick_image_host (visibilities in, image parts out)
    cudaEvent_t ev_fork, ev_join, ev_vis, ev_part, ev_wgt;
    int n_sm;
    int state;               // 0 idle, 1 gridded, 2 transformed, 3 corrected, 4 tapered
    int failed;              // sticky: the first CUDA failure (RICK_ERR_CUDA); every later call returns it
    std::string err;
    int64_t n_launches;

    // tables
    void* twiddle;           // [N] complex of grid_prec: e^{+2 pi i k/N}
    void* twiddle2;          // [N/16] e^{+2 pi i k/(N/16)}: the long-column two-pass transform (N >= 8192), else null
    double* taper;           // [2N]: c((p-N/2)/N), then the reciprocals 1/c
    double kb_poly[15 * (RICK_KB_DEG + 1)];   // host: [S][DEG+1], tap a on d = (a-h) - s/2, s in [-1,1]

    // resident buffers
    void* stack;             // [batch][N][N] complex of grid_prec
    size_t plane_bytes;
    double* image;           // [N][N]

    // per-call visibility scratch (grows)
    int64_t cap_vis;
    // sort items (key << idx_bits) | k: unsorted, and the two ping-pong buffers of the radix sort
    unsigned long long *items, *items_a, *items_b;
    unsigned long long* sorted_items;      // points at items / items_a / items_b after the sort
    int idx_bits, key_bits;                // item layout of the last rick_grid / rick_image
    // onesweep radix passes: digit histograms + tickets, digit bases, look-back status words
    unsigned int* os_small;
    unsigned long long* os_gbase;
    unsigned long long* os_status; size_t os_status_cap;
    int64_t* plane_start;    // [n_planes_total + 1] offsets into the sorted order
    int64_t plane_start_cap;
    // row occupancy: row_occ[pg][row] = 1 when some visibility of global
    // plane pg has row in its footprint band (tile-row granularity), rebuilt by every sort;
    // row_dirty[slot][row] = 1 when that row of the resident slot may hold non-zero data.  Rows that
    // are neither are zero in HBM and stay untouched by zero-fill, gridder and the row pass.
    unsigned char* row_occ; size_t row_occ_cap;
    // win_mask[pg]: bit k = some row of the k-th 32nd of the plane (rows k N/32 ..) is occupied; written by the row
    // pass's launcher, read by the fused N = 8192 column pass (which fetches occupied windows only)
    uint32_t* win_mask; size_t win_mask_cap;
    uint32_t* cols_arrivals; size_t cols_arrivals_cap;   // pacing counters of the fused N = 8192 column pass (one per item of a CTA)
    unsigned char* row_dirty;
    // tile occupancy: tile_occ[pg][tv][tu] = 1 when the footprint of some
    // visibility of global plane pg reaches the B x B tile (tv, tu); rebuilt by every sort.  In rick_image
    // the zero-fill clears, and the row pass reads, only those tiles of an occupied row.
    unsigned char* tile_occ; size_t tile_occ_cap;
    unsigned int* row_list; size_t row_list_cap;   // work list of the row pass (+ its counter at [cap])
    double* chan_scale;      // [C] device, s_c = f_c / c0
    WRange* wrange;          // [n_img] device
    int chan_cap;
    double* h_scale;         // pinned host staging of s_c (RICK_MAX_CHAN)
    cudaEvent_t ev_scale;    // completion of the last upload from h_scale
    std::vector<double> last_freq;
    DevCounters* counters;   // device
    int64_t M; int32_t C; int64_t R; int n_img;

    // optional per-kernel CUDA-event timing (rick_profile)
    int prof_on;
    std::vector<cudaEvent_t> prof_ev;       // pool: 2 events per record
    std::vector<int> prof_id;               // kernel class of each record
    size_t prof_n;                          // records in use
    double prof_ms[32];                     // aggregated by rick_profile_read
    long long prof_cnt[32];

    // chunked gridding (rick_image_stream_host): visibility chunk c uses staging half c & 1
    cudaEvent_t ev_chunk_in[2], ev_chunk_free[2];

    // N = 4096 fp64 column kernels (fft_cols12.cu): TMA tensor map over the resident stack
    // cube plans with all planes of an image resident keep img_batch images' stacks resident (slots = batch *
    // img_batch) so that zero-fill, gridder and row pass run once per group of images, not once per channel
    int img_batch, slots;
    int cols12_ok;               // N = 4096 fp64: k_cols12_fft / k_cols12_wcorrect
    int cols13_ok;               // N = 8192 fp64: k_cols13_wcorrect (one column per SM, tensor map in cols12_tmap_sw)
    alignas(64) unsigned char cols12_tmap[128];
    alignas(64) unsigned char cols12_tmap_sw[128];   // same view, 32-byte swizzle (k_cols12_wcorrect)

    // fp32 grid with long columns (fft_cols_sparse.cu): per-plane row lists / bitmaps / prefix sums of the occupied
    // rows, the largest count (sp_count[Nw]) and the transposed accumulation image
    int sp_ok;
    unsigned int *sp_bits, *sp_prefix;
    unsigned short* sp_list;
    int* sp_count;
    double* sp_imageT;

    // host-buffer staging for rick_image_host
    void* st_vis; size_t st_vis_cap;
    double* st_uvw; size_t st_uvw_cap;
    float* st_wgt; size_t st_wgt_cap;
    double* st_img; size_t st_img_cap;
};

#define RICK_CUDA(p, call)                                                             \
    do {                                                                               \
        cudaError_t e__ = (call);                                                      \
        if (e__ != cudaSuccess) {                                                      \
            (p)->err = std::string(#call) + ": " + cudaGetErrorString(e__);            \
            if (e__ == cudaErrorMemoryAllocation) { cudaGetLastError(); return RICK_ERR_OOM; } \
            (p)->failed = RICK_ERR_CUDA;                                               \
            return RICK_ERR_CUDA;                                                      \
        }                                                                              \
    } while (0)

// kernel classes for rick_profile_read / rick_kernel_name
enum { RK_TABLES = 0, RK_RESET, RK_WRANGE, RK_INDEX_KEY, RK_RADIX_HIST, RK_SCAN, RK_RADIX_SCATTER,
       RK_PLANE_STARTS, RK_ZERO, RK_GRID, RK_FFT_ROWS, RK_FFT_COLS, RK_WCORRECT, RK_TAPER, RK_COLS_WCORRECT,
       RK_ROW_OCC, RK_NKERNELS };

void rick_prof_begin(rick_plan_t* p, int id, cudaStream_t st);   // plan.cu; no-ops unless profiling is on
void rick_prof_end(rick_plan_t* p, cudaStream_t st);

// launch one kernel: optional CUDA-event bracket, launch counter, launch-error check
#define RICK_KERNEL(p, id, ...) RICK_KERNEL_ON(p, (p)->stream, id, __VA_ARGS__)
#define RICK_KERNEL_ON(p, st, id, ...)                                                 \
    do {                                                                               \
        rick_prof_begin((p), (id), (st));                                              \
        __VA_ARGS__;                                                                   \
        rick_prof_end((p), (st));                                                      \
        RICK_LAUNCHED(p);                                                              \
    } while (0)

#define RICK_LAUNCHED(p)                                                               \
    do {                                                                               \
        (p)->n_launches++;                                                             \
        cudaError_t e__ = cudaGetLastError();                                          \
        if (e__ != cudaSuccess) {                                                      \
            (p)->err = std::string("kernel launch: ") + cudaGetErrorString(e__);       \
            (p)->failed = RICK_ERR_CUDA;                                               \
            return RICK_ERR_CUDA;                                                      \
        }                                                                              \
    } while (0)

// stage entry points (each enqueues on p->stream)
int rick_tables_build(rick_plan_t* p);                                   // tables.cu
// flags of rick_index_sort (chunked gridding, rick_image_stream_host): keep the w range and the statistics
// counters of the plan (set up once over ALL rows by rick_wrange_all), OR the occupancy maps into the
// existing ones instead of rebuilding them
#define RICK_SORT_KEEP_RANGE 1
#define RICK_SORT_OCC_ACCUM 2
int rick_index_sort(rick_plan_t* p, const double* uvw_m, const float* weights, int flags = 0);   // index_sort.cu
int rick_wrange_all(rick_plan_t* p, const double* uvw_m, int64_t n_rows);                         // index_sort.cu
int rick_plane_hist(rick_plan_t* p, const double* uvw_m, unsigned long long* hist_dev);          // index_sort.cu
int rick_zero_dirty(rick_plan_t* p, int n_slots, cudaStream_t st);        // grid.cu: zero the dirty rows of slots 0..n_slots-1
// grid.cu: occupied rows by tile; stale rows whole unless keep_stale (the two-pass column transform never reads
// a row that is not occupied, so rick_image leaves such rows dirty instead of clearing them)
int rick_zero_sparse(rick_plan_t* p, int plane_first, int n_slots, int keep_stale = 0);
int rick_mark_dirty(rick_plan_t* p, int plane_first, int n_planes);      // grid.cu: dirty |= occupancy of the batch
int rick_all_dirty(rick_plan_t* p, int n_slots);                         // grid.cu: after an in-place column pass
int rick_grid_planes(rick_plan_t* p, const void* vis, int vis_dtype, const double* uvw_m,
                     const float* weights, int plane_first, int n_planes);      // grid.cu
int rick_fft_planes(rick_plan_t* p, int plane_first, int n_planes);      // fft.cu: rows then columns (in place)
int rick_fft_rows(rick_plan_t* p, int plane_first, int n_planes);        // fft.cu: occupied rows only
int rick_fft_cols(rick_plan_t* p, int n_planes);                         // fft.cu (generic strided pass)
// fft.cu: column pass of rick_image for long columns (N >= 8192, rick_cols2_on) in two passes at full line
// width: rick_fft_cols2 = pass A (strided N/16-point transforms + twiddles, in place; reads occupied rows only,
// writes every row), rick_cols2_wcorrect = pass B (16-point transforms in registers) fused with a5 (+ a6):
// the transformed planes are never written
int rick_fft_cols2(rick_plan_t* p, int plane_first, int n_planes);
int rick_cols2_on(const rick_plan_t* p);     // 1 when the two-pass transform applies to this plan (N >= 8192)
int rick_cols2_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image, int accumulate,
                        int fuse_taper, int slot_first = 0, int col_begin = 0, int col_end = -1);   // columns [col_begin, col_end), multiples of 16; -1 = N
// fft_cols_sparse.cu: single fused column pass of the fp32 grid with long columns over the occupied rows only;
// every launch returns at once on the device when some plane has more than N/2 occupied rows (the two-pass
// kernels then run: they return at once in the other case -- rick_sparse_maxcount / rick_sparse_cap)
int rick_sparse_init(rick_plan_t* p);
void rick_sparse_free(rick_plan_t* p);
int rick_sparse_prepare(rick_plan_t* p);
int rick_sparse_wcorrect(rick_plan_t* p, int z_first, int n_planes, int accumulate, int col_begin = 0, int col_end = -1);
int rick_sparse_finish(rick_plan_t* p, double* image, int fuse_taper, int col_begin = 0, int col_end = -1);
const int* rick_sparse_maxcount(const rick_plan_t* p);
int rick_sparse_cap(const rick_plan_t* p);
int rick_cols12_init(rick_plan_t* p);                                    // fft_cols12.cu
int rick_cols12_fft(rick_plan_t* p, int n_planes);                       // fft_cols12.cu
int rick_cols12_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image,
                         int accumulate, int fuse_taper, int strip_begin, int strip_end, int slot_first = 0);   // fft_cols12.cu
int rick_cols12_strips(const rick_plan_t* p);                            // fft_cols12.cu: work units of the fused pass
int rick_cols12_unit_cols(const rick_plan_t* p);                         // columns per unit (2 at N = 4096, 1 at N = 8192)
int rick_cols_fused(const rick_plan_t* p);                               // 1 when the single fused column pass serves this plan
int rick_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image,
                  int accumulate, int fuse_taper, int slot_first = 0);   // wcorrect.cu
int rick_taper_divide(rick_plan_t* p, double* image);                    // wcorrect.cu

// ordered (monotone) encoding of doubles for atomicMin/atomicMax on u64
__host__ __device__ inline unsigned long long rick_ord_encode(double x)
{
#ifdef __CUDA_ARCH__
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
#else
    unsigned long long b;
    memcpy(&b, &x, sizeof(b));
#endif
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__host__ __device__ inline double rick_ord_decode(unsigned long long e)
{
    unsigned long long b = (e & 0x8000000000000000ull) ? (e & 0x7FFFFFFFFFFFFFFFull) : ~e;
#ifdef __CUDA_ARCH__
    return __longlong_as_double((long long)b);
#else
    double x;
    memcpy(&x, &b, sizeof(x));
    return x;
#endif
}
