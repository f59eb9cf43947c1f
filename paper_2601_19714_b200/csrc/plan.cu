// plan.cu -- the C ABI of librick_b200 (include/rick.h): plan lifetime, argument checks,
// the state machine and the host-side sequencing of a0..a6.  All arithmetic of the path runs
// in the kernels of index_sort.cu / grid.cu / fft.cu / wcorrect.cu.
#include "common.cuh"

#include <math.h>
#include <new>
#include <vector>

static bool is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }

// every entry point: a plan that has seen a CUDA failure stays failed (rick.h "Errors"); the text of the
// first failure stays readable through rick_last_error
#define RICK_ENTER(p)                                   \
    do {                                                \
        if (!(p)) return RICK_ERR_INVALID;              \
        if ((p)->failed) return (p)->failed;            \
        (p)->err.clear();                               \
    } while (0)

static bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

// closed form of the taper (tables.cu k_taper) on the host, for the plan-time check of kb_beta
static double taper_host(double nu, int S, double beta, double i0_beta)
{
    const double x = 3.14159265358979323846 * (double)S * nu, a = beta * beta - x * x;
    double f;
    if (fabs(a) < 1e-6) f = 1.0 + a / 6.0;
    else if (a > 0.0) { const double r = sqrt(a); f = sinh(r) / r; }
    else { const double r = sqrt(-a); f = sin(r) / r; }
    return (double)S / i0_beta * f;
}

static void free_dev(void* q)
{
    if (q) cudaFree(q);
}

// ---------------------------------------------------------------------------------------
// per-kernel CUDA-event timing
static const char* const k_names[RK_NKERNELS] = {
    "tables", "reset", "wrange", "index_key", "radix_hist", "scan", "radix_scatter", "plane_starts",
    "zero", "grid", "fft_rows", "fft_cols", "wcorrect", "taper", "fft_cols_wcorrect", "row_occupancy"};

void rick_prof_begin(rick_plan_t* p, int id, cudaStream_t st)
{
    if (!p->prof_on) return;
    if (p->prof_ev.size() < 2 * (p->prof_n + 1)) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { p->prof_on = 0; return; }
        p->prof_ev.push_back(a);
        p->prof_ev.push_back(b);
    }
    if (p->prof_id.size() <= p->prof_n) p->prof_id.push_back(id); else p->prof_id[p->prof_n] = id;
    cudaEventRecord(p->prof_ev[2 * p->prof_n], st);
}

void rick_prof_end(rick_plan_t* p, cudaStream_t st)
{
    if (!p->prof_on) return;
    cudaEventRecord(p->prof_ev[2 * p->prof_n + 1], st);
    p->prof_n++;
}

static void prof_collect(rick_plan_t* p)
{
    cudaStreamSynchronize(p->stream);
    if (p->stream2) cudaStreamSynchronize(p->stream2);
    for (size_t i = 0; i < p->prof_n; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p->prof_ev[2 * i], p->prof_ev[2 * i + 1]) == cudaSuccess) {
            p->prof_ms[p->prof_id[i]] += (double)ms;
            p->prof_cnt[p->prof_id[i]]++;
        }
    }
    p->prof_n = 0;
}

extern "C" int rick_profile(rick_plan_t* p, int32_t enable)
{
    if (!p) return RICK_ERR_INVALID;
    prof_collect(p);
    if (enable) {
        for (int i = 0; i < 32; ++i) { p->prof_ms[i] = 0.0; p->prof_cnt[i] = 0; }
    }
    p->prof_on = enable ? 1 : 0;
    return RICK_OK;
}

extern "C" int rick_profile_read(rick_plan_t* p, int32_t kernel_id, double* total_ms, int64_t* launches)
{
    if (!p || kernel_id < 0 || kernel_id >= RK_NKERNELS) return RICK_ERR_INVALID;
    prof_collect(p);
    if (total_ms) *total_ms = p->prof_ms[kernel_id];
    if (launches) *launches = (int64_t)p->prof_cnt[kernel_id];
    return RICK_OK;
}

extern "C" const char* rick_kernel_name(int32_t kernel_id)
{
    return (kernel_id >= 0 && kernel_id < RK_NKERNELS) ? k_names[kernel_id] : nullptr;
}

extern "C" const char* rick_version(void) { return "librick_b200 0.1 sm_100a"; }

extern "C" const char* rick_last_error(const rick_plan_t* p) { return p ? p->err.c_str() : "null plan"; }

extern "C" int rick_plan_destroy(rick_plan_t* p)
{
    if (!p) return RICK_OK;
    cudaStreamSynchronize(p->stream);
    free_dev(p->twiddle); free_dev(p->twiddle2); free_dev(p->taper); free_dev(p->stack); free_dev(p->image);
    free_dev(p->items); free_dev(p->items_a); free_dev(p->items_b);
    free_dev(p->os_small); free_dev(p->os_gbase); free_dev(p->os_status); free_dev(p->plane_start); free_dev(p->chan_scale);
    free_dev(p->row_occ); free_dev(p->win_mask); free_dev(p->cols_arrivals); free_dev(p->row_dirty); free_dev(p->tile_occ); free_dev(p->row_list);
    free_dev(p->wrange); free_dev(p->counters);
    rick_sparse_free(p);
    free_dev(p->st_vis); free_dev(p->st_uvw); free_dev(p->st_wgt); free_dev(p->st_img);
    for (cudaEvent_t e : p->prof_ev) cudaEventDestroy(e);
    if (p->h_scale) cudaFreeHost(p->h_scale);
    if (p->ev_scale) cudaEventDestroy(p->ev_scale);
    if (p->stream2) { cudaStreamSynchronize(p->stream2); cudaStreamDestroy(p->stream2); }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->stream3) { cudaStreamSynchronize(p->stream3); cudaStreamDestroy(p->stream3); }
    if (p->ev_vis) cudaEventDestroy(p->ev_vis);
    if (p->ev_part) cudaEventDestroy(p->ev_part);
    if (p->ev_wgt) cudaEventDestroy(p->ev_wgt);
    for (int i = 0; i < 2; ++i) {
        if (p->ev_chunk_in[i]) cudaEventDestroy(p->ev_chunk_in[i]);
        if (p->ev_chunk_free[i]) cudaEventDestroy(p->ev_chunk_free[i]);
    }
    delete p;
    return RICK_OK;
}

static int plan_init(rick_plan_t* p)
{
    int dev = 0;
    RICK_CUDA(p, cudaGetDevice(&dev));
    RICK_CUDA(p, cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev));
    const size_t cell = p->f32 ? 8 : 16;
    p->plane_bytes = (size_t)p->N * p->N * cell;
    if (p->img_batch > 1 && cudaMalloc(&p->stack, p->plane_bytes * (size_t)p->slots) != cudaSuccess) {
        // no room for a group of images: fall back to one image's stack at a time
        cudaGetLastError();
        p->stack = nullptr;
        p->img_batch = 1;
        p->slots = p->batch;
    }
    if (!p->stack) RICK_CUDA(p, cudaMalloc(&p->stack, p->plane_bytes * (size_t)p->slots));
    // the resident stack starts all-zero and no row is dirty: from here on only rows that were written
    // are ever cleared again (rick_zero_dirty)
    RICK_CUDA(p, cudaMemsetAsync(p->stack, 0, p->plane_bytes * (size_t)p->slots, p->stream));
    RICK_CUDA(p, cudaMalloc(&p->row_dirty, (size_t)p->slots * p->N));
    RICK_CUDA(p, cudaMemsetAsync(p->row_dirty, 0, (size_t)p->slots * p->N, p->stream));
    RICK_CUDA(p, cudaMalloc(&p->image, sizeof(double) * (size_t)p->N * p->N));
    RICK_CUDA(p, cudaMallocHost(&p->h_scale, sizeof(double) * RICK_MAX_CHAN));
    RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_scale, cudaEventDisableTiming));
    {
        int lo = 0, hi = 0;
        RICK_CUDA(p, cudaDeviceGetStreamPriorityRange(&lo, &hi));      // lo = least priority
        RICK_CUDA(p, cudaStreamCreateWithPriority(&p->stream2, cudaStreamNonBlocking, lo));
        RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
        RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming));
        RICK_CUDA(p, cudaStreamCreateWithFlags(&p->stream3, cudaStreamNonBlocking));
        RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_vis, cudaEventDisableTiming));
        RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_part, cudaEventDisableTiming));
        RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_wgt, cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) {
            RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_chunk_in[i], cudaEventDisableTiming));
            RICK_CUDA(p, cudaEventCreateWithFlags(&p->ev_chunk_free[i], cudaEventDisableTiming));
        }
    }
    RICK_CUDA(p, cudaMalloc(&p->counters, sizeof(DevCounters)));
    RICK_CUDA(p, cudaMemsetAsync(p->counters, 0, sizeof(DevCounters), p->stream));
    const int rc = rick_tables_build(p);
    if (rc) return rc;
    const int rc2 = rick_sparse_init(p);
    if (rc2) return rc2;
    return rick_cols12_init(p);
}

extern "C" int rick_plan(rick_plan_t** out, const rick_plan_desc* d, void* cuda_stream)
{
    if (!out) return RICK_ERR_INVALID;
    *out = nullptr;
    if (!d) return RICK_ERR_INVALID;
    if (!is_pow2(d->n) || d->n < 64 || d->n > 16384) return RICK_ERR_INVALID;
    if (d->n_wplanes < 1 || d->n_wplanes > 65536) return RICK_ERR_INVALID;
    if (d->support < 3 || d->support > 15 || (d->support & 1) == 0) return RICK_ERR_INVALID;
    if (!(d->pixel_rad > 0.0) || !isfinite(d->pixel_rad)) return RICK_ERR_INVALID;
    if (d->grid_prec != RICK_GRID_F64 && d->grid_prec != RICK_GRID_F32) return RICK_ERR_INVALID;
    if (d->grid_prec == RICK_GRID_F64 && d->n > 8192) return RICK_ERR_INVALID;
    const int B = d->tile ? d->tile : 16;
    if (!is_pow2(B) || B < 8 || B > 32 || B > d->n) return RICK_ERR_INVALID;
    if (d->plane_batch < 0 || d->plane_batch > (d->z_count > 0 ? d->z_count : d->n_wplanes)) return RICK_ERR_INVALID;
    if (d->cube != 0 && d->cube != 1) return RICK_ERR_INVALID;
    if (d->flags & ~RICK_FLAG_FOLD_W) return RICK_ERR_INVALID;
    if (d->z_count < 0 || d->z_begin < 0 || (d->z_count == 0 && d->z_begin != 0)) return RICK_ERR_INVALID;
    if (d->z_count > 0 && ((int64_t)d->z_begin + d->z_count > d->n_wplanes || d->cube)) return RICK_ERR_INVALID;
    if (isinf(d->w_min) || isinf(d->w_max)) return RICK_ERR_INVALID;
    if (d->w_min == d->w_min && d->w_max == d->w_max && d->w_max < d->w_min) return RICK_ERR_INVALID;
    if (d->kb_beta == d->kb_beta && d->kb_beta > 60.0) return RICK_ERR_INVALID;
    // fp32 grid: the taper is not clamped (reading R12) and its corner value falls with S (S = 7: 3.8e-4 of
    // the centre, S = 11: ~1e-8), so beyond S = 9 the fp32 rounding of the planes, amplified at the corners,
    // exceeds the 1e-4 bar of the fp32 path (measured 3e-4 at S = 11): such plans are refused
    if (d->grid_prec == RICK_GRID_F32 && d->support > 9) return RICK_ERR_INVALID;
    {
        // kb_beta too SMALL: for beta < pi S / 2 the taper c(nu) enters its sin(r)/r branch inside
        // |nu| <= 1/2 and can cross zero, and a6 would divide by ~0.  Refuse a plan whose taper falls below
        // 1e-12 of its centre value anywhere on the N pixels.
        const double beta = d->kb_beta > 0.0 ? d->kb_beta : 2.34 * (double)d->support;
        const double c0 = taper_host(0.0, d->support, beta, 1.0);
        double cmin = c0;
        for (int p = 0; p < d->n; ++p) {
            const double c = taper_host((double)(p - d->n / 2) / (double)d->n, d->support, beta, 1.0);
            if (!(c >= cmin)) cmin = c;
        }
        if (!(cmin > 1e-12 * c0)) return RICK_ERR_INVALID;
    }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return RICK_ERR_CUDA;   // no CPU fallback

    rick_plan_t* p = new (std::nothrow) rick_plan_s();
    if (!p) return RICK_ERR_OOM;
    p->d = *d;
    p->N = d->n;
    p->Nw_total = d->n_wplanes;
    p->z0 = d->z_begin;
    p->Nw = d->z_count > 0 ? d->z_count : d->n_wplanes;
    p->fold = (d->flags & RICK_FLAG_FOLD_W) ? 1 : 0;
    p->S = d->support;
    p->h = (d->support - 1) / 2;
    p->B = B;
    p->T = d->n / B;
    p->log2N = 0;
    while ((1 << p->log2N) < d->n) p->log2N++;
    p->log2B = 0;
    while ((1 << p->log2B) < B) p->log2B++;
    p->f32 = d->grid_prec == RICK_GRID_F32;
    p->batch = d->plane_batch ? d->plane_batch : p->Nw;
    // cube with every plane of an image resident: keep up to 8 images' stacks (at most 48 GB) resident
    p->img_batch = 1;
    if (d->cube && p->batch == p->Nw) {
        const double img_bytes = (double)d->n * d->n * (p->f32 ? 8.0 : 16.0) * (double)p->Nw;
        int k = (int)(48.0e9 / img_bytes);
        p->img_batch = k < 1 ? 1 : (k > 8 ? 8 : k);
    }
    p->slots = p->batch * p->img_batch;
    p->beta = d->kb_beta > 0.0 ? d->kb_beta : 2.34 * (double)d->support;
    p->dl = d->pixel_rad;
    p->inv_du = (double)d->n * d->pixel_rad;
    p->stream = (cudaStream_t)cuda_stream;
    const int rc = plan_init(p);
    if (rc != RICK_OK) {
        rick_plan_destroy(p);
        return rc;
    }
    *out = p;
    return RICK_OK;
}

// ---------------------------------------------------------------------------------------
// Sort item = (key << idx_bits) | k.  key < n_img * N_w * N^2 (image, plane, tile, cell in tile); the
// all-ones pattern of key_bits is reserved for dropped visibilities.
static void item_bits(const rick_plan_t* p, int32_t n_chan, unsigned long long M, int* key_bits, int* idx_bits)
{
    const unsigned long long n_img = p->d.cube ? (unsigned long long)n_chan : 1ull;
    const unsigned long long nkeys = n_img * (unsigned long long)p->Nw * (unsigned long long)p->N * (unsigned long long)p->N;
    int kb = 1;
    while (kb < 63 && ((1ull << kb) - 1ull) < nkeys) ++kb;
    int ib = 1;
    while (ib < 32 && (1ull << ib) < M) ++ib;
    *key_bits = kb;
    *idx_bits = ib;
}

// dev_ptrs: the buffers are device memory the kernels read directly (alignment matters); dev_w / dev_out: the
// optional weights and image_out of that call (may be null)
static int check_inputs(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
                        const double* chan_freq_hz, int32_t n_chan, int64_t n_rows, bool dev_ptrs = false,
                        const void* dev_w = nullptr, const void* dev_out = nullptr)
{
    if (vis_dtype != RICK_VIS_C64 && vis_dtype != RICK_VIS_C128) { p->err = "bad vis_dtype"; return RICK_ERR_INVALID; }
    if (n_chan < 1 || n_chan > RICK_MAX_CHAN || !chan_freq_hz) { p->err = "bad channels"; return RICK_ERR_INVALID; }
    if (n_rows < 0) { p->err = "negative n_rows"; return RICK_ERR_INVALID; }
    if (n_rows > 0 && (!vis || !uvw_m)) { p->err = "null input"; return RICK_ERR_INVALID; }
    for (int c = 0; c < n_chan; ++c)
        if (!(chan_freq_hz[c] > 0.0) || !isfinite(chan_freq_hz[c])) { p->err = "bad frequency"; return RICK_ERR_INVALID; }
    // the kernels read vis with 8- / 16-byte vector loads: a misaligned pointer would fault the context
    if (dev_ptrs && (!aligned16(vis) || !aligned16(uvw_m) || !aligned16(dev_w) || !aligned16(dev_out))) {
        p->err = "device pointer not 16-byte aligned (vis / uvw_m / weights / image_out)";
        return RICK_ERR_INVALID;
    }
    const unsigned long long M = (unsigned long long)n_rows * (unsigned long long)n_chan;
    if (M >= 0xFFFFFFFFull) { p->err = "too many visibilities for 32-bit indices"; return RICK_ERR_INVALID; }
    int kb, ib;
    item_bits(p, n_chan, M, &kb, &ib);
    if (kb + ib > 64) { p->err = "image x plane x cell key and visibility index do not fit one 64-bit sort item"; return RICK_ERR_INVALID; }
    return RICK_OK;
}

template <typename Tp> static int grow(rick_plan_t* p, Tp** buf, size_t n)
{
    free_dev(*buf);
    *buf = nullptr;
    RICK_CUDA(p, cudaMalloc(buf, sizeof(Tp) * (n ? n : 1)));
    return RICK_OK;
}

static int prepare_scales(rick_plan_t* p, const double* chan_freq_hz, int32_t n_chan);

static int prepare(rick_plan_t* p, const double* chan_freq_hz, int32_t n_chan, int64_t n_rows)
{
    p->C = n_chan;
    p->R = n_rows;
    p->M = n_rows * (int64_t)n_chan;
    p->n_img = p->d.cube ? n_chan : 1;
    int rc;
    item_bits(p, n_chan, (unsigned long long)p->M, &p->key_bits, &p->idx_bits);
    if (p->M > p->cap_vis) {
        p->cap_vis = 0;
        if ((rc = grow(p, &p->items, (size_t)p->M))) return rc;
        if ((rc = grow(p, &p->items_a, (size_t)p->M))) return rc;
        if ((rc = grow(p, &p->items_b, (size_t)p->M))) return rc;
        p->cap_vis = p->M;
    }
    if (!p->items) {   // M == 0 on a fresh plan: keep the pointers valid
        if ((rc = grow(p, &p->items, 1))) return rc;
        if ((rc = grow(p, &p->items_a, 1))) return rc;
        if ((rc = grow(p, &p->items_b, 1))) return rc;
    }
    const int64_t n_pl = (int64_t)p->n_img * p->Nw + 1;
    if (n_pl > p->plane_start_cap) {
        if ((rc = grow(p, &p->plane_start, (size_t)n_pl))) return rc;
        p->plane_start_cap = n_pl;
    }
    const size_t occ_bytes = (size_t)(n_pl - 1) * p->N;
    if (occ_bytes > p->row_occ_cap) {
        p->row_occ_cap = 0;
        if ((rc = grow(p, &p->row_occ, occ_bytes))) return rc;
        p->row_occ_cap = occ_bytes;
    }
    if ((size_t)(n_pl - 1) > p->win_mask_cap) {
        p->win_mask_cap = 0;
        if ((rc = grow(p, &p->win_mask, (size_t)(n_pl - 1)))) return rc;
        p->win_mask_cap = (size_t)(n_pl - 1);
    }
    const size_t tocc_bytes = (size_t)(n_pl - 1) * p->T * p->T;
    if (tocc_bytes > p->tile_occ_cap) {
        p->tile_occ_cap = 0;
        if ((rc = grow(p, &p->tile_occ, tocc_bytes))) return rc;
        p->tile_occ_cap = tocc_bytes;
    }
    return prepare_scales(p, chan_freq_hz, n_chan);
}

// per-channel scales s_c = f_c / c0 on the device (+ room for the w range of every image)
static int prepare_scales(rick_plan_t* p, const double* chan_freq_hz, int32_t n_chan)
{
    int rc;
    if (n_chan > p->chan_cap) {
        if ((rc = grow(p, &p->chan_scale, (size_t)n_chan))) return rc;
        if ((rc = grow(p, &p->wrange, (size_t)n_chan))) return rc;
        p->chan_cap = n_chan;
    }
    const bool same = (int)p->last_freq.size() == n_chan &&
                      memcmp(p->last_freq.data(), chan_freq_hz, sizeof(double) * (size_t)n_chan) == 0;
    if (!same) {
        // pinned staging; wait for the previous upload before overwriting it (normally done long ago)
        RICK_CUDA(p, cudaEventSynchronize(p->ev_scale));
        for (int c = 0; c < n_chan; ++c) p->h_scale[c] = chan_freq_hz[c] / RICK_C0;   // s_c = f_c / c0
        RICK_CUDA(p, cudaMemcpyAsync(p->chan_scale, p->h_scale, sizeof(double) * (size_t)n_chan,
                                     cudaMemcpyHostToDevice, p->stream));
        RICK_CUDA(p, cudaEventRecord(p->ev_scale, p->stream));
        p->last_freq.assign(chan_freq_hz, chan_freq_hz + n_chan);
    }
    return RICK_OK;
}

// a0..a2 on the plan's stream while the rows the previous call left dirty are cleared on the side
// stream (that needs nothing from the sort, only that earlier readers of the stack are done); joined
// before a3.  Afterwards the whole resident stack is zero.
static int sort_and_zero(rick_plan_t* p, const double* uvw_m, const float* weights, int n_planes_first)
{
    int rc;
    (void)n_planes_first;
    RICK_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
    RICK_CUDA(p, cudaStreamWaitEvent(p->stream2, p->ev_fork, 0));
    if ((rc = rick_zero_dirty(p, p->batch, p->stream2))) return rc;
    RICK_CUDA(p, cudaEventRecord(p->ev_join, p->stream2));
    if ((rc = rick_index_sort(p, uvw_m, weights))) return rc;
    RICK_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_join, 0));
    return RICK_OK;
}

extern "C" int rick_grid(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
                         const float* weights, const double* chan_freq_hz, int32_t n_chan, int64_t n_rows)
{
    RICK_ENTER(p);
    if (p->batch != p->Nw || p->d.cube) { p->err = "staged calls need the whole stack resident and cube = 0"; return RICK_ERR_STATE; }
    int rc = check_inputs(p, vis, vis_dtype, uvw_m, chan_freq_hz, n_chan, n_rows, true, weights);
    if (rc) return rc;
    p->state = 0;
    if ((rc = prepare(p, chan_freq_hz, n_chan, n_rows))) return rc;
    if ((rc = sort_and_zero(p, uvw_m, weights, p->Nw))) return rc;
    if ((rc = rick_mark_dirty(p, 0, p->Nw))) return rc;
    if ((rc = rick_grid_planes(p, vis, vis_dtype, uvw_m, weights, 0, p->Nw))) return rc;
    p->state = 1;
    return RICK_OK;
}

extern "C" int rick_fft_wplanes(rick_plan_t* p)
{
    RICK_ENTER(p);
    if (p->state != 1) { p->err = "rick_fft_wplanes needs a gridded stack"; return RICK_ERR_STATE; }
    const int rc = rick_fft_planes(p, 0, p->Nw);
    if (rc) return rc;
    p->state = 2;
    return RICK_OK;
}

extern "C" int rick_wcorrect_accumulate(rick_plan_t* p)
{
    RICK_ENTER(p);
    if (p->state != 2) { p->err = "rick_wcorrect_accumulate needs a transformed stack"; return RICK_ERR_STATE; }
    const int rc = rick_wcorrect(p, 0, 0, p->Nw, p->image, 0, 0);
    if (rc) return rc;
    p->state = 3;
    return RICK_OK;
}

extern "C" int rick_gridcorrect(rick_plan_t* p)
{
    RICK_ENTER(p);
    if (p->state != 3) { p->err = "rick_gridcorrect needs a w-corrected image"; return RICK_ERR_STATE; }
    const int rc = rick_taper_divide(p, p->image);
    if (rc) return rc;
    p->state = 4;
    return RICK_OK;
}

// a4..a6 of one resident batch (planes z0 .. z0 + nb - 1 of image img): row pass, then either the fused
// column pass + w-correction (N = 4096 fp64) or the generic column pass and correction.  host_out (cube = 0,
// last batch only): the image leaves for HOST memory part by part on the copy stream while the next part
// of the last pass is still running; *host_done says whether that happened.
static int transform_and_correct(rick_plan_t* p, int img, int z0, int nb, double* dst, int last, double* host_out,
                                 bool* host_done)
{
    int rc;
    if (rick_cols_fused(p)) {   // column pass fused with the w-correction: the transformed planes are never written
        if ((rc = rick_fft_rows(p, img * p->Nw + z0, nb))) return rc;
        const int strips = rick_cols12_strips(p), ucols = rick_cols12_unit_cols(p);
        if (host_out && last && !p->d.cube) {
            // whole rounds of the persistent grid per part.  N = 4096 (the pass is about as long as the copy of its image):
            // 4 + 4 + 3 + rest rounds of n_sm strips.  N = 8192 (26 ms of kernel against 10 ms of copy at configs[2]): seven
            // shrinking parts + the rest, so that the copy left over after the last kernel is 2 % of the image, not 26 %
            // (host entry 46.8 -> 44.5 ms; at N = 4096 the same split costs 0.1-0.7 ms)
            int rounds[8];
            const int total = (strips + p->n_sm - 1) / p->n_sm;
            if (p->cols13_ok) {
                static const int pct[7] = {28, 24, 18, 12, 8, 5, 3};
                for (int k = 0; k < 7; ++k) rounds[k] = (pct[k] * total + 50) / 100 > 0 ? (pct[k] * total + 50) / 100 : 1;
                rounds[7] = 1 << 20;
            } else {
                const int r4 = (strips / p->n_sm + 3) / 4;
                rounds[0] = rounds[1] = r4 > 0 ? r4 : 1;
                rounds[2] = r4 > 1 ? r4 - 1 : 1;
                for (int k = 3; k < 8; ++k) rounds[k] = 1 << 20;
            }
            int s0 = 0;
            for (int k = 0; k < 8 && s0 < strips; ++k) {
                long long s1 = (long long)s0 + (long long)rounds[k] * p->n_sm;
                if (s1 > strips) s1 = strips;
                if ((rc = rick_cols12_wcorrect(p, img, z0, nb, dst, z0 > 0, last, s0, (int)s1))) return rc;
                RICK_CUDA(p, cudaEventRecord(p->ev_part, p->stream));
                RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_part, 0));
                const size_t c0 = (size_t)ucols * (size_t)s0, nc = (size_t)ucols * (size_t)(s1 - s0);
                RICK_CUDA(p, cudaMemcpy2DAsync(host_out + c0, sizeof(double) * p->N, dst + c0, sizeof(double) * p->N,
                                               sizeof(double) * nc, (size_t)p->N, cudaMemcpyDeviceToHost, p->stream3));
                s0 = (int)s1;
            }
            *host_done = true;
        } else {
            if ((rc = rick_cols12_wcorrect(p, img, z0, nb, dst, z0 > 0, last, 0, strips))) return rc;
        }
    } else {
        const int two_pass = rick_cols2_on(p);
        if (two_pass) {       // long columns: pass A at full line width, pass B fused with the correction
            if ((rc = rick_fft_rows(p, img * p->Nw + z0, nb))) return rc;
            // fp32 grid: one fused pass over the occupied rows only, when every plane of the image has few
            // enough of them (decided on the device: either these launches or the two-pass ones return at
            // once).  It accumulates a transposed image, turned (and tapered) after the last batch.
            if (p->sp_ok && z0 == 0 && (rc = rick_sparse_prepare(p))) return rc;
            if (p->sp_ok && host_out && last && !p->d.cube) {
                // last batch through the host entry: the two-pass kernels first (the whole image, or nothing), then the
                // sparse pass, its transposition and the copy to the host by column ranges -- a short first range so
                // that the copy engine starts early (the 2.1 GB image of configs[3] takes longer to cross PCIe than
                // the last batch takes to compute), each range's copy under the next range's kernels
                if ((rc = rick_fft_cols2(p, img * p->Nw + z0, nb))) return rc;
                if ((rc = rick_cols2_wcorrect(p, img, z0, nb, dst, z0 > 0, last))) return rc;
                const int first = p->N / 16, step = (p->N - first + 2) / 3 / 32 * 32 + 32;
                for (int c0 = 0; c0 < p->N;) {
                    int c1 = c0 + (c0 == 0 ? first : step);
                    if (c1 > p->N) c1 = p->N;
                    if ((rc = rick_sparse_wcorrect(p, z0, nb, z0 > 0, c0, c1))) return rc;
                    if ((rc = rick_sparse_finish(p, dst, 1, c0, c1))) return rc;
                    RICK_CUDA(p, cudaEventRecord(p->ev_part, p->stream));
                    RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_part, 0));
                    RICK_CUDA(p, cudaMemcpy2DAsync(host_out + c0, sizeof(double) * p->N, dst + c0, sizeof(double) * p->N,
                                                   sizeof(double) * (size_t)(c1 - c0), (size_t)p->N, cudaMemcpyDeviceToHost, p->stream3));
                    c0 = c1;
                }
                *host_done = true;
                return RICK_OK;
            }
            if (p->sp_ok && (rc = rick_sparse_wcorrect(p, z0, nb, z0 > 0))) return rc;
            if ((rc = rick_fft_cols2(p, img * p->Nw + z0, nb))) return rc;
            if (p->sp_ok) {
                if ((rc = rick_cols2_wcorrect(p, img, z0, nb, dst, z0 > 0, last))) return rc;
                if (last && (rc = rick_sparse_finish(p, dst, 1))) return rc;
            } else if (host_out && last && !p->d.cube) {
                // four column ranges: the image columns of one part cross to the host under the next part
                const int step = p->N / 4;
                for (int c0 = 0; c0 < p->N; c0 += step) {
                    if ((rc = rick_cols2_wcorrect(p, img, z0, nb, dst, z0 > 0, last, 0, c0, c0 + step))) return rc;
                    RICK_CUDA(p, cudaEventRecord(p->ev_part, p->stream));
                    RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_part, 0));
                    RICK_CUDA(p, cudaMemcpy2DAsync(host_out + c0, sizeof(double) * p->N, dst + c0, sizeof(double) * p->N,
                                                   sizeof(double) * (size_t)step, (size_t)p->N, cudaMemcpyDeviceToHost, p->stream3));
                }
                *host_done = true;
            } else {
                if ((rc = rick_cols2_wcorrect(p, img, z0, nb, dst, z0 > 0, last))) return rc;
            }
        } else {
            if ((rc = rick_fft_planes(p, img * p->Nw + z0, nb))) return rc;
            if ((rc = rick_wcorrect(p, img, z0, nb, dst, z0 > 0, last))) return rc;
        }
    }
    return RICK_OK;
}

// a0..a6.  vis_ready (may be null): event the gridder must wait for (visibilities still being copied
// by rick_image_host).  host_out (may be null; cube = 0 only): the image goes to HOST memory, part by
// part on the copy stream while the next part of the last pass is still running.
static int image_impl(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
                      const float* weights, const double* chan_freq_hz, int32_t n_chan,
                      int64_t n_rows, double* image_out, cudaEvent_t vis_ready, double* host_out,
                      cudaEvent_t wgt_ready = nullptr)
{
    int rc = check_inputs(p, vis, vis_dtype, uvw_m, chan_freq_hz, n_chan, n_rows, true, weights, image_out);
    if (rc) return rc;
    if (p->d.cube && !image_out) { p->err = "cube mode needs image_out"; return RICK_ERR_INVALID; }
    p->state = 0;
    if ((rc = prepare(p, chan_freq_hz, n_chan, n_rows))) return rc;
    // a0..a2, then the zero-fill that needs this sort's occupancy (stale rows whole, occupied rows by tile)
    // (the index step sums the WEIGHTS of the gridded visibilities: with weights it must not start before the
    // copy stream has delivered them -- ADVICE r1, sum_w could come from stale staging)
    if (wgt_ready && weights) RICK_CUDA(p, cudaStreamWaitEvent(p->stream, wgt_ready, 0));
    if ((rc = rick_index_sort(p, uvw_m, weights))) return rc;
    if (vis_ready) RICK_CUDA(p, cudaStreamWaitEvent(p->stream, vis_ready, 0));
    const size_t NN = (size_t)p->N * p->N;
    bool host_done = false;
    if (p->d.cube && p->img_batch > 1) {
        // groups of img_batch images: one zero-fill, one gridder launch and one row pass per group (a
        // channel's 5e5 visibilities are too few to fill the machine), the column pass + correction per image
        const int two_pass = rick_cols2_on(p);
        for (int img0 = 0; img0 < p->n_img; img0 += p->img_batch) {
            const int kk = p->n_img - img0 < p->img_batch ? p->n_img - img0 : p->img_batch;
            const int pf = img0 * p->Nw, ns = kk * p->Nw;
            if ((rc = rick_zero_sparse(p, pf, ns, two_pass))) return rc;
            if ((rc = rick_mark_dirty(p, pf, ns))) return rc;
            if ((rc = rick_grid_planes(p, vis, vis_dtype, uvw_m, weights, pf, ns))) return rc;
            if ((rc = rick_fft_rows(p, pf, ns))) return rc;
            if (!rick_cols_fused(p)) {
                if (two_pass) rc = rick_fft_cols2(p, pf, ns);
                else rc = rick_fft_cols(p, ns);
                if (rc) return rc;
            }
            for (int j = 0; j < kk; ++j) {
                double* dst = image_out + (size_t)(img0 + j) * NN;
                if (rick_cols_fused(p)) rc = rick_cols12_wcorrect(p, img0 + j, 0, p->Nw, dst, 0, 1, 0, rick_cols12_strips(p), j * p->Nw);
                else if (two_pass) rc = rick_cols2_wcorrect(p, img0 + j, 0, p->Nw, dst, 0, 1, j * p->Nw);
                else rc = rick_wcorrect(p, img0 + j, 0, p->Nw, dst, 0, 1, j * p->Nw);
                if (rc) return rc;
            }
            if (host_out) {      // this group's images leave for the host while the next group is imaged
                RICK_CUDA(p, cudaEventRecord(p->ev_part, p->stream));
                RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_part, 0));
                RICK_CUDA(p, cudaMemcpyAsync(host_out + (size_t)img0 * NN, image_out + (size_t)img0 * NN,
                                             sizeof(double) * NN * (size_t)kk, cudaMemcpyDeviceToHost, p->stream3));
                host_done = true;
            }
        }
    } else
    for (int img = 0; img < p->n_img; ++img) {
        double* dst = p->d.cube ? image_out + (size_t)img * NN : p->image;
        for (int z0 = 0; z0 < p->Nw; z0 += p->batch) {
            const int nb = p->Nw - z0 < p->batch ? p->Nw - z0 : p->batch;
            const int last = z0 + nb >= p->Nw;
            // (the two-pass column transform reads occupied rows only: stale rows need no clearing)
            if ((rc = rick_zero_sparse(p, img * p->Nw + z0, nb, rick_cols2_on(p)))) return rc;
            if ((rc = rick_mark_dirty(p, img * p->Nw + z0, nb))) return rc;
            if ((rc = rick_grid_planes(p, vis, vis_dtype, uvw_m, weights, img * p->Nw + z0, nb))) return rc;
            if ((rc = transform_and_correct(p, img, z0, nb, dst, last, host_out, &host_done))) return rc;
        }
    }
    if (!p->d.cube) {
        if (image_out)
            RICK_CUDA(p, cudaMemcpyAsync(image_out, p->image, sizeof(double) * NN, cudaMemcpyDeviceToDevice, p->stream));
        // the staged state machine may continue only if the whole stack is what is resident
        p->state = 4;
    }
    if (host_out && !host_done) {
        const size_t n_img = p->d.cube ? (size_t)n_chan : 1;
        RICK_CUDA(p, cudaMemcpyAsync(host_out, p->d.cube ? image_out : p->image, sizeof(double) * NN * n_img,
                                     cudaMemcpyDeviceToHost, p->stream));
    }
    return RICK_OK;
}

extern "C" int rick_image(rick_plan_t* p, const void* vis, int32_t vis_dtype, const double* uvw_m,
                          const float* weights, const double* chan_freq_hz, int32_t n_chan,
                          int64_t n_rows, double* image_out)
{
    RICK_ENTER(p);
    return image_impl(p, vis, vis_dtype, uvw_m, weights, chan_freq_hz, n_chan, n_rows, image_out, nullptr, nullptr);
}

// the sticky device-side failure flag (DevCounters::error; a radix tile that lost its predecessor), read by
// the calls that synchronise anyway: turns into a sticky RICK_ERR_CUDA
static int check_device_error(rick_plan_t* p)
{
    unsigned int e = 0;
    RICK_CUDA(p, cudaMemcpy(&e, &p->counters->error, sizeof(e), cudaMemcpyDeviceToHost));
    if (e) {
        p->err = "device-side failure in the radix sort (a tile never saw its predecessor's status)";
        p->failed = RICK_ERR_CUDA;
        return RICK_ERR_CUDA;
    }
    return RICK_OK;
}

template <typename Tp> static int ensure_bytes(rick_plan_t* p, Tp** buf, size_t* cap, size_t bytes)
{
    if (*cap >= bytes) return RICK_OK;
    free_dev(*buf);
    *buf = nullptr;
    *cap = 0;
    RICK_CUDA(p, cudaMalloc(buf, bytes ? bytes : 16));
    *cap = bytes;
    return RICK_OK;
}

extern "C" int rick_image_stream_host(rick_plan_t* p, const void* vis_host, int32_t vis_dtype, const double* uvw_m_host,
                                      const float* weights_host, const double* chan_freq_hz, int32_t n_chan,
                                      int64_t n_rows, int64_t rows_per_chunk, double* image_out_host);

extern "C" int rick_image_host(rick_plan_t* p, const void* vis_host, int32_t vis_dtype, const double* uvw_m_host,
                               const float* weights_host, const double* chan_freq_hz, int32_t n_chan,
                               int64_t n_rows, double* image_out_host)
{
    RICK_ENTER(p);
    if (!image_out_host) { p->err = "null image_out_host"; return RICK_ERR_INVALID; }
    int rc = check_inputs(p, vis_host, vis_dtype, uvw_m_host, chan_freq_hz, n_chan, n_rows);
    if (rc) return rc;
    const size_t M = (size_t)n_rows * (size_t)n_chan;
    // large sets with the whole stack resident go through the chunked path in two halves: the second half
    // of the visibilities is still crossing PCIe while the first is sorted and gridded (measured on
    // configs[1]: 8.06 ms against 8.64 ms for copy-everything-then-sort; more chunks cost more in sorts)
    // (N <= 4096 only: the chunked path clears every dirty row of the stack before the first chunk, the one-shot
    // path only the tiles it grids into -- at configs[2], N = 8192, that is 5.3 ms against 0.5 ms, more than the
    // overlapped half of the copy saves: 53.0 ms chunked against 49.1 ms one-shot)
    if (!p->d.cube && p->batch == p->Nw && M >= ((size_t)1 << 22) && n_rows >= 2 && p->log2N <= 12)
        return rick_image_stream_host(p, vis_host, vis_dtype, uvw_m_host, weights_host, chan_freq_hz, n_chan, n_rows,
                                      (n_rows + 1) / 2, image_out_host);
    const size_t vis_bytes = M * (vis_dtype == RICK_VIS_C128 ? 16 : 8);
    const size_t NN = (size_t)p->N * p->N;
    const size_t n_img = p->d.cube ? (size_t)n_chan : 1;
    if ((rc = ensure_bytes(p, &p->st_vis, &p->st_vis_cap, vis_bytes))) return rc;
    if ((rc = ensure_bytes(p, &p->st_uvw, &p->st_uvw_cap, sizeof(double) * 3 * (size_t)n_rows))) return rc;
    if (weights_host && (rc = ensure_bytes(p, &p->st_wgt, &p->st_wgt_cap, sizeof(float) * M))) return rc;
    if (p->d.cube && (rc = ensure_bytes(p, &p->st_img, &p->st_img_cap, sizeof(double) * NN * n_img))) return rc;
    // uvw first on the plan's stream (a0..a2 need nothing else); the visibilities follow on the copy
    // stream and land while index + sort + zero-fill run; the gridder waits for ev_vis.
    if (M) {
        RICK_CUDA(p, cudaMemcpyAsync(p->st_uvw, uvw_m_host, sizeof(double) * 3 * (size_t)n_rows, cudaMemcpyHostToDevice, p->stream));
        RICK_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
        RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_fork, 0));
        // weights first: the index step (which sums them) waits for ev_wgt only, the gridder for ev_vis
        if (weights_host) {
            RICK_CUDA(p, cudaMemcpyAsync(p->st_wgt, weights_host, sizeof(float) * M, cudaMemcpyHostToDevice, p->stream3));
            RICK_CUDA(p, cudaEventRecord(p->ev_wgt, p->stream3));
        }
        RICK_CUDA(p, cudaMemcpyAsync(p->st_vis, vis_host, vis_bytes, cudaMemcpyHostToDevice, p->stream3));
        RICK_CUDA(p, cudaEventRecord(p->ev_vis, p->stream3));
    }
    rc = image_impl(p, p->st_vis, vis_dtype, p->st_uvw, weights_host ? p->st_wgt : nullptr, chan_freq_hz,
                    n_chan, n_rows, p->d.cube ? p->st_img : nullptr, M ? p->ev_vis : nullptr, image_out_host,
                    (M && weights_host) ? p->ev_wgt : nullptr);
    if (rc) return rc;
    RICK_CUDA(p, cudaStreamSynchronize(p->stream));
    RICK_CUDA(p, cudaStreamSynchronize(p->stream3));
    return check_device_error(p);
}


// Out-of-core visibilities (the single-node analogue of the I/O-compute overlap the
// paper plans).  The visibilities stay in HOST memory and cross to the device in chunks of
// rows_per_chunk rows through a two-slot staging buffer: chunk c + 1 is copied on the copy stream while
// chunk c is indexed, sorted and gridded INTO the same resident stack (gridding is linear in the
// visibilities, Eq. 3).  a0 runs once over all rows first (uvw is 24 B per row and is copied whole), so
// every chunk sees the same w range and lands on the same planes as in one rick_image call; the occupancy
// maps are the union over the chunks.  a4..a6 run once at the end.
extern "C" int rick_image_stream_host(rick_plan_t* p, const void* vis_host, int32_t vis_dtype, const double* uvw_m_host,
                                      const float* weights_host, const double* chan_freq_hz, int32_t n_chan,
                                      int64_t n_rows, int64_t rows_per_chunk, double* image_out_host)
{
    RICK_ENTER(p);
    if (!image_out_host) { p->err = "null image_out_host"; return RICK_ERR_INVALID; }
    if (p->batch != p->Nw || p->d.cube) { p->err = "chunked gridding needs the whole stack resident and cube = 0"; return RICK_ERR_STATE; }
    if (rows_per_chunk < 1) { p->err = "rows_per_chunk < 1"; return RICK_ERR_INVALID; }
    if (n_rows < 0) { p->err = "negative n_rows"; return RICK_ERR_INVALID; }
    if (rows_per_chunk > n_rows) rows_per_chunk = n_rows > 0 ? n_rows : 1;
    // the 32-bit index / 64-bit item limits apply to ONE chunk, not to the whole set
    int rc = check_inputs(p, vis_host, vis_dtype, uvw_m_host, chan_freq_hz, n_chan, n_rows > 0 ? rows_per_chunk : 0);
    if (rc) return rc;
    const size_t C = (size_t)n_chan, vsz = vis_dtype == RICK_VIS_C128 ? 16 : 8;
    const size_t chunk_vis = (size_t)rows_per_chunk * C * vsz, chunk_wgt = (size_t)rows_per_chunk * C * sizeof(float);
    const size_t NN = (size_t)p->N * p->N;
    if ((rc = ensure_bytes(p, &p->st_vis, &p->st_vis_cap, 2 * chunk_vis))) return rc;
    if ((rc = ensure_bytes(p, &p->st_uvw, &p->st_uvw_cap, sizeof(double) * 3 * (size_t)n_rows))) return rc;
    if (weights_host && (rc = ensure_bytes(p, &p->st_wgt, &p->st_wgt_cap, 2 * chunk_wgt))) return rc;
    p->state = 0;
    if ((rc = prepare(p, chan_freq_hz, n_chan, rows_per_chunk))) return rc;      // sort scratch for ONE chunk
    const int n_planes_total = p->Nw;
    if (n_rows > 0)
        RICK_CUDA(p, cudaMemcpyAsync(p->st_uvw, uvw_m_host, sizeof(double) * 3 * (size_t)n_rows, cudaMemcpyHostToDevice, p->stream));
    // the copy stream may touch the staging only after everything enqueued so far (earlier calls) is done
    RICK_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
    RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_fork, 0));
    if ((rc = rick_wrange_all(p, p->st_uvw, n_rows))) return rc;                 // a0 over ALL rows
    if ((rc = rick_zero_dirty(p, p->batch, p->stream))) return rc;               // the whole stack is zero again
    RICK_CUDA(p, cudaMemsetAsync(p->row_occ, 0, (size_t)n_planes_total * p->N, p->stream));
    RICK_CUDA(p, cudaMemsetAsync(p->tile_occ, 0, (size_t)n_planes_total * p->T * p->T, p->stream));
    int c = 0;
    for (int64_t r0 = 0; r0 < n_rows; r0 += rows_per_chunk, ++c) {
        const int64_t nr = n_rows - r0 < rows_per_chunk ? n_rows - r0 : rows_per_chunk;
        const int b = c & 1;
        const size_t off = (size_t)r0 * C;
        unsigned char* dv = reinterpret_cast<unsigned char*>(p->st_vis) + (size_t)b * chunk_vis;
        float* dw = weights_host ? reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(p->st_wgt) + (size_t)b * chunk_wgt) : nullptr;
        if (c >= 2) RICK_CUDA(p, cudaStreamWaitEvent(p->stream3, p->ev_chunk_free[b], 0));
        RICK_CUDA(p, cudaMemcpyAsync(dv, reinterpret_cast<const unsigned char*>(vis_host) + off * vsz, (size_t)nr * C * vsz,
                                     cudaMemcpyHostToDevice, p->stream3));
        if (dw)
            RICK_CUDA(p, cudaMemcpyAsync(dw, weights_host + off, (size_t)nr * C * sizeof(float), cudaMemcpyHostToDevice, p->stream3));
        RICK_CUDA(p, cudaEventRecord(p->ev_chunk_in[b], p->stream3));
        p->R = nr;
        p->M = nr * (int64_t)n_chan;
        const double* du = p->st_uvw + 3 * (size_t)r0;
        if (dw) RICK_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_chunk_in[b], 0));   // the index step sums the weights
        if ((rc = rick_index_sort(p, du, dw, RICK_SORT_KEEP_RANGE | RICK_SORT_OCC_ACCUM))) return rc;
        if (!dw) RICK_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_chunk_in[b], 0));
        if ((rc = rick_mark_dirty(p, 0, p->Nw))) return rc;
        if ((rc = rick_grid_planes(p, dv, vis_dtype, du, dw, 0, p->Nw))) return rc;
        RICK_CUDA(p, cudaEventRecord(p->ev_chunk_free[b], p->stream));
    }
    p->R = n_rows;
    p->M = n_rows * (int64_t)n_chan;
    bool host_done = false;
    if ((rc = transform_and_correct(p, 0, 0, p->Nw, p->image, 1, image_out_host, &host_done))) return rc;
    p->state = 4;
    if (!host_done)
        RICK_CUDA(p, cudaMemcpyAsync(image_out_host, p->image, sizeof(double) * NN, cudaMemcpyDeviceToHost, p->stream));
    RICK_CUDA(p, cudaStreamSynchronize(p->stream));
    RICK_CUDA(p, cudaStreamSynchronize(p->stream3));
    return check_device_error(p);
}

extern "C" int rick_plane_histogram(rick_plan_t* p, const double* uvw_m, const double* chan_freq_hz, int32_t n_chan,
                                    int64_t n_rows, int64_t* hist_host)
{
    RICK_ENTER(p);
    if (!hist_host) { p->err = "null hist_host"; return RICK_ERR_INVALID; }
    if (p->d.cube) { p->err = "rick_plane_histogram: cube plans shard by channels"; return RICK_ERR_STATE; }
    static const float2 dummy_vis = {0.f, 0.f};
    int rc = check_inputs(p, n_rows > 0 ? (const void*)&dummy_vis : nullptr, RICK_VIS_C64, uvw_m, chan_freq_hz, n_chan, n_rows);
    if (rc) return rc;
    if (n_rows > 0 && !aligned16(uvw_m)) { p->err = "device pointer not 16-byte aligned (uvw_m)"; return RICK_ERR_INVALID; }
    p->state = 0;
    p->C = n_chan;                  // (no sort scratch: the histogram needs the scales and the w range only)
    p->R = n_rows;
    p->M = n_rows * (int64_t)n_chan;
    p->n_img = 1;
    if ((rc = prepare_scales(p, chan_freq_hz, n_chan))) return rc;
    unsigned long long* hd = nullptr;
    RICK_CUDA(p, cudaMalloc(&hd, sizeof(unsigned long long) * (size_t)p->Nw_total));
    rc = rick_plane_hist(p, uvw_m, hd);
    if (rc == RICK_OK) {
        cudaError_t e = cudaMemcpyAsync(hist_host, hd, sizeof(unsigned long long) * (size_t)p->Nw_total, cudaMemcpyDeviceToHost, p->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
        if (e != cudaSuccess) { p->err = std::string("rick_plane_histogram: ") + cudaGetErrorString(e); p->failed = RICK_ERR_CUDA; rc = RICK_ERR_CUDA; }
    }
    cudaFree(hd);
    return rc;
}

// Linear partition: smallest bottleneck by bisection on the bound, greedy feasibility (a range is closed when
// the next plane would exceed the bound); then the ranges are laid out greedily under the optimal bound, leaving
// at least one plane for every later part.
extern "C" int rick_partition_planes(const int64_t* hist, int32_t n_wplanes, int32_t n_parts, double plane_cost, int32_t* bounds)
{
    if (!hist || !bounds || n_wplanes < 1 || n_parts < 1 || !(plane_cost >= 0.0)) return RICK_ERR_INVALID;
    for (int z = 0; z < n_wplanes; ++z)
        if (hist[z] < 0) return RICK_ERR_INVALID;
    auto cost = [&](int z) { return (double)hist[z] + plane_cost; };
    auto parts_needed = [&](double bound) {
        int parts = 1;
        double acc = 0.0;
        for (int z = 0; z < n_wplanes; ++z) {
            const double c = cost(z);
            if (acc > 0.0 && acc + c > bound) { ++parts; acc = 0.0; }
            acc += c;
        }
        return parts;
    };
    double lo = 0.0, hi = 0.0;
    for (int z = 0; z < n_wplanes; ++z) { hi += cost(z); if (cost(z) > lo) lo = cost(z); }
    for (int it = 0; it < 100 && hi - lo > 1e-9 * (hi > 1.0 ? hi : 1.0); ++it) {
        const double mid = 0.5 * (lo + hi);
        if (parts_needed(mid) <= n_parts) hi = mid; else lo = mid;
    }
    const double bound = hi;
    int z = 0;
    bounds[0] = 0;
    for (int r = 0; r < n_parts; ++r) {
        double acc = 0.0;
        int must_leave = n_wplanes - z - 1;                 // one plane for every later part, as far as the planes go
        if (must_leave < 0) must_leave = 0;
        if (must_leave > n_parts - 1 - r) must_leave = n_parts - 1 - r;
        int taken = 0;
        while (z < n_wplanes - must_leave || (r == n_parts - 1 && z < n_wplanes)) {
            const double c = cost(z);
            if (taken > 0 && acc + c > bound && r < n_parts - 1) break;
            acc += c;
            ++z;
            ++taken;
        }
        bounds[r + 1] = z;
    }
    return RICK_OK;
}

extern "C" int rick_get_image(rick_plan_t* p, double* dst_device)
{
    RICK_ENTER(p);
    if (!dst_device || !aligned16(dst_device)) { p->err = "rick_get_image: null or misaligned destination"; return RICK_ERR_INVALID; }
    if (p->d.cube) { p->err = "rick_get_image: cube plans return their images through image_out"; return RICK_ERR_STATE; }
    if (p->state < 3) { p->err = "no image yet"; return RICK_ERR_STATE; }
    RICK_CUDA(p, cudaMemcpyAsync(dst_device, p->image, sizeof(double) * (size_t)p->N * p->N, cudaMemcpyDeviceToDevice, p->stream));
    return RICK_OK;
}

extern "C" int rick_get_stats(rick_plan_t* p, rick_stats* out)
{
    RICK_ENTER(p);
    if (!out) return RICK_ERR_INVALID;
    DevCounters c;
    WRange w;
    memset(&w, 0, sizeof(w));
    RICK_CUDA(p, cudaStreamSynchronize(p->stream));
    RICK_CUDA(p, cudaMemcpy(&c, p->counters, sizeof(c), cudaMemcpyDeviceToHost));
    if (p->wrange) RICK_CUDA(p, cudaMemcpy(&w, p->wrange, sizeof(w), cudaMemcpyDeviceToHost));
    out->n_vis = p->M;
    out->n_gridded = (int64_t)c.n_gridded;
    out->n_dropped = (int64_t)c.n_dropped;
    out->sum_w = c.sum_w;
    out->w_min = w.w_min;
    out->w_max = w.w_max;
    out->n_launches = p->n_launches;
    // occupancy of the last sort: what the pruned passes move
    out->occ_rows = 0;
    out->occ_tiles = 0;
    out->occ_windows = 0;
    out->n_planes = (int64_t)p->n_img * p->Nw;
    if (p->row_occ && p->tile_occ && p->n_img > 0) {
        const size_t nr = (size_t)p->n_img * p->Nw * p->N, nt = (size_t)p->n_img * p->Nw * p->T * p->T;
        std::vector<unsigned char> h(nr > nt ? nr : nt);
        RICK_CUDA(p, cudaMemcpy(h.data(), p->row_occ, nr, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nr; ++i) out->occ_rows += h[i] != 0;
        const size_t win = (size_t)p->N / 32;
        for (size_t w0 = 0; win && w0 < nr; w0 += win) {
            bool any = false;
            for (size_t i = w0; i < w0 + win; ++i) any |= h[i] != 0;
            out->occ_windows += any;
        }
        RICK_CUDA(p, cudaMemcpy(h.data(), p->tile_occ, nt, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nt; ++i) out->occ_tiles += h[i] != 0;
    }
    if (c.error) {
        p->err = "device-side failure in the radix sort (a tile never saw its predecessor's status)";
        p->failed = RICK_ERR_CUDA;
        return RICK_ERR_CUDA;
    }
    return RICK_OK;
}

extern "C" const uint64_t* rick_debug_items(rick_plan_t* p, int32_t sorted, int32_t* idx_bits, int32_t* key_bits)
{
    if (!p || !p->items) return nullptr;
    if (idx_bits) *idx_bits = p->idx_bits;
    if (key_bits) *key_bits = p->key_bits;
    return (const uint64_t*)(sorted ? p->sorted_items : p->items);
}
extern "C" void* rick_debug_planes(rick_plan_t* p) { return (p && p->state >= 1) ? p->stack : nullptr; }
