// index_sort.cu -- a0 (w range), a1 (cell / plane index + key), a2 (stable LSD radix sort).
//
// a0/a1 follow SURVEY.md 8(c) steps 1-4 / DESIGN.md "Index arithmetic": every floating-point
// operation is individually rounded (__dmul_rn / __dadd_rn / __ddiv_rn, never contracted into
// FMA) and done in the stated order, so cell, plane and key are BIT-EXACT against the oracle.
//   s_c = f_c / c0 (host, IEEE division);  inv_du = N * dl
//   x_u = (u_m * s_c) * inv_du;  i_u = floor(x_u + (N/2 + 0.5))       (nearest cell, ties up; R8)
//   on-grid <=> i_u-h >= 0, i_u+h <= N-1 (same in v)                   (Eq. 5; R10)
//   w_l = w_m * s_c;  dw = (w_max - w_min)/N_w;  i_p = min(N_w-1, floor((w_l - w_min) * (1/dw)))
//                                                                     ("closest w-plane", :48; R4)
//   key = ((((img*N_w + i_p)*T + i_v/B)*T + i_u/B)*B + i_v%B)*B + i_u%B;  dropped -> all ones
//   (image, plane, uv tile, cell inside the tile: DESIGN.md step 4, reading R22)
// a2: the single-GPU analogue of the paper's bucket sort: a stable
// least-significant-digit radix sort of 64-bit items (key << idx_bits) | k over the key bits,
// which equals the oracle's sort by (key, index).
#include "common.cuh"
#include <mutex>

// ------------------------------------------------------------------------------------------
// a0: w range.  min/max over rows of w [m]; multiplication by s_c > 0 is monotone under
// round-to-nearest, so min_{r} fl(w_r s_c) = fl((min_r w_r) s_c) exactly.
// ------------------------------------------------------------------------------------------
__global__ void k_counters_reset(DevCounters* c)
{
    c->wmin_bits = 0xFFFFFFFFFFFFFFFFull;
    c->wmax_bits = 0ull;
    c->n_gridded = 0ull;
    c->n_dropped = 0ull;
    c->sum_w = 0.0;
    c->grid_chunk = 0u;      // (c->error is sticky: cleared at plan creation only)
}

__global__ void k_wrange_rows(const double* __restrict__ uvw, long long R, DevCounters* c, int fold)
{
    unsigned long long lo = 0xFFFFFFFFFFFFFFFFull, hi = 0ull;
    for (long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x; r < R;
         r += (long long)gridDim.x * blockDim.x) {
        double w = uvw[3 * r + 2];
        if (!isfinite(w)) continue;                 // R23: a non-finite w takes no part in the range
        if (fold) w = fabs(w);                      // R24: rows with w < 0 are imaged at -w
        unsigned long long e = rick_ord_encode(w);
        lo = e < lo ? e : lo;
        hi = e > hi ? e : hi;
    }
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long l2 = __shfl_xor_sync(0xffffffffu, lo, o);
        unsigned long long h2 = __shfl_xor_sync(0xffffffffu, hi, o);
        lo = l2 < lo ? l2 : lo;
        hi = h2 > hi ? h2 : hi;
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&c->wmin_bits, lo);
        atomicMax(&c->wmax_bits, hi);
    }
}

__global__ void k_wrange_finish(const DevCounters* c, const double* __restrict__ chan_scale, int C,
                                int cube, int Nw, double w_min_given, double w_max_given,
                                long long R, WRange* __restrict__ out)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    const int n_img = cube ? C : 1;
    if (g >= n_img) return;
    double lo, hi;
    if (R == 0 || c->wmin_bits > c->wmax_bits) {     // no row, or none with a finite w
        lo = 0.0;
        hi = 0.0;
    } else {
        const double wlo_m = rick_ord_decode(c->wmin_bits), whi_m = rick_ord_decode(c->wmax_bits);
        if (cube) {
            const double s = chan_scale[g];
            lo = __dmul_rn(wlo_m, s);
            hi = __dmul_rn(whi_m, s);
        } else {
            lo = INFINITY;
            hi = -INFINITY;
            for (int ch = 0; ch < C; ++ch) {
                const double s = chan_scale[ch];
                lo = fmin(lo, __dmul_rn(wlo_m, s));
                hi = fmax(hi, __dmul_rn(whi_m, s));
            }
        }
    }
    if (w_min_given == w_min_given) lo = w_min_given;
    if (w_max_given == w_max_given) hi = w_max_given;
    WRange w;
    w.w_min = lo;
    w.w_max = hi;
    w.dw = __ddiv_rn(__dsub_rn(hi, lo), (double)Nw);
    w.inv_dw = w.dw > 0.0 ? __ddiv_rn(1.0, w.dw) : 0.0;
    out[g] = w;
}

// Radix passes over the key bits (<= 8-bit digits), shared by a1 (histograms) and a2 (passes).
#define RS_MAXPASS 8
struct RadixPlan {
    int npass;
    int shift[RS_MAXPASS];          // of the KEY (the item shift is idx_bits + shift)
    unsigned int mask[RS_MAXPASS];
};

// Index arithmetic of one visibility (DESIGN.md section 3 steps 2, 3; R24 fold first): centre cell, plane of the WHOLE
// problem, on-grid flag.  Each operation individually rounded, in the normative order.
__device__ __forceinline__ bool vis_index(double um, double vm, double wm, const double s, const WRange& wr, const int N,
                                          const int Nw_total, const int h, const double inv_du, const int fold, int& iu,
                                          int& iv, int& ip)
{
    if (fold && wm < 0.0) {
        um = -um;
        vm = -vm;
        wm = -wm;
    }
    const double shift = (double)(N / 2) + 0.5;
    const double xu = __dmul_rn(__dmul_rn(um, s), inv_du);
    const double xv = __dmul_rn(__dmul_rn(vm, s), inv_du);
    // on-grid test on the doubles, before any cast: floor(x) - h >= 0 <=> x >= h and
    // floor(x) + h <= N-1 <=> x < N-h for integer h, and both are false for NaN / inf (R23: a
    // visibility with a non-finite u, v or w is dropped; (int)floor() of such a value
    // saturated and could pass the integer test)
    const double su = __dadd_rn(xu, shift), sv = __dadd_rn(xv, shift);
    const double wl = __dmul_rn(wm, s);
    const double lo_ok = (double)h, hi_ok = (double)(N - h);
    const bool ok = su >= lo_ok && su < hi_ok && sv >= lo_ok && sv < hi_ok && isfinite(wl);
    iu = ok ? (int)floor(su) : 0;
    iv = ok ? (int)floor(sv) : 0;
    double fp = ok ? floor(__dmul_rn(__dsub_rn(wl, wr.w_min), wr.inv_dw)) : 0.0;
    fp = fp > (double)(Nw_total - 1) ? (double)(Nw_total - 1) : fp;
    fp = fp >= 0.0 ? fp : 0.0;
    ip = (int)fp;
    return ok;
}

// Per-plane counts of the on-grid visibilities of the whole problem (rick_plane_histogram; cube = 0).
__global__ void __launch_bounds__(256)
k_plane_hist(const double* __restrict__ uvw, const double* __restrict__ chan_scale, const WRange* __restrict__ wrange,
             unsigned int M, unsigned int C, int N, int Nw_total, int h, double inv_du, int fold,
             unsigned long long* __restrict__ hist)
{
    extern __shared__ unsigned int s_cnt[];          // [Nw_total] when it fits (<= 8192 planes), else global atomics
    const bool use_s = Nw_total <= 8192;
    if (use_s) {
        for (int i = threadIdx.x; i < Nw_total; i += blockDim.x) s_cnt[i] = 0u;
        __syncthreads();
    }
    const WRange wr = wrange[0];
    for (unsigned long long kk0 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; kk0 < M;
         kk0 += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned int k = (unsigned int)kk0;
        const unsigned int r = k / C, c = k - r * C;
        int iu, iv, ip;
        if (!vis_index(uvw[3ull * r + 0], uvw[3ull * r + 1], uvw[3ull * r + 2], chan_scale[c], wr, N, Nw_total, h, inv_du,
                       fold, iu, iv, ip))
            continue;
        if (use_s) atomicAdd(&s_cnt[ip], 1u); else atomicAdd(&hist[ip], 1ull);
    }
    if (use_s) {
        __syncthreads();
        for (int i = threadIdx.x; i < Nw_total; i += blockDim.x)
            if (s_cnt[i]) atomicAdd(&hist[i], (unsigned long long)s_cnt[i]);
    }
}

// ------------------------------------------------------------------------------------------
// a1: one thread per visibility k = r*C + c.  Writes the sort item (key << idx_bits) | k.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_index_key(const double* __restrict__ uvw, const float* __restrict__ wgt,
            const double* __restrict__ chan_scale, const WRange* __restrict__ wrange,
            unsigned int M, unsigned int C, int N, int Nw, int h, int log2B, int T, int cube,
            double inv_du, int idx_bits, unsigned long long key_dropped,
            unsigned long long* __restrict__ items, DevCounters* cnt, RadixPlan rp,
            unsigned int* __restrict__ ghist, int fold, int z0, int Nw_total)
{
    // digit histograms of ALL radix passes (they do not depend on the order of the items), so that
    // every pass is one read + one write of the items (k_radix_onesweep)
    __shared__ unsigned int s_h[RS_MAXPASS][256];
    for (int i = threadIdx.x; i < RS_MAXPASS * 256; i += blockDim.x) (&s_h[0][0])[i] = 0u;
    __syncthreads();
    // grid-stride: statistics stay in registers, one set of atomics per block (same-address
    // atomics per warp made this kernel atomic-bound)
    unsigned int on = 0, off = 0;
    double sw = 0.0;
    const int Bm = (1 << log2B) - 1;
    for (unsigned long long kk0 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; kk0 < M;
         kk0 += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned int k = (unsigned int)kk0;
        const unsigned int r = k / C, c = k - r * C;
        const int img = cube ? (int)c : 0;
        int iu, iv, ipg;
        const bool ok = vis_index(uvw[3ull * r + 0], uvw[3ull * r + 1], uvw[3ull * r + 2], chan_scale[c], wrange[img], N,
                                  Nw_total, h, inv_du, fold, iu, iv, ipg);
        // this plan's shard of the planes: z0 .. z0 + Nw - 1 (the whole range unless the plan is a shard)
        const int ip = ipg - z0;
        const bool mine = ip >= 0 && ip < Nw;
        unsigned long long key = key_dropped;
        if (ok && mine) {
            unsigned long long kk = (unsigned long long)img * (unsigned)Nw + (unsigned)ip;
            kk = (kk * (unsigned)T + (unsigned)(iv >> log2B)) * (unsigned)T + (unsigned)(iu >> log2B);
            kk = (((kk << log2B) + (unsigned)(iv & Bm)) << log2B) + (unsigned)(iu & Bm);
            key = kk;
            on++;
            sw += wgt ? (double)wgt[k] : 1.0;
        } else if (!ok && z0 == 0) {
            off++;                  // off-grid visibilities are counted once, by the shard that owns plane 0
        }
        items[k] = (key << idx_bits) | (unsigned long long)k;
#pragma unroll
        for (int ps = 0; ps < RS_MAXPASS; ++ps)
            if (ps < rp.npass) atomicAdd(&s_h[ps][(unsigned int)(key >> rp.shift[ps]) & rp.mask[ps]], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < rp.npass * 256; i += blockDim.x) {
        const unsigned int v = (&s_h[0][0])[i];
        if (v) atomicAdd(&ghist[i], v);
    }
    // block-reduced statistics
    __shared__ unsigned int s_on[8], s_off[8];
    __shared__ double s_sw[8];
    for (int o = 16; o > 0; o >>= 1) {
        on += __shfl_xor_sync(0xffffffffu, on, o);
        off += __shfl_xor_sync(0xffffffffu, off, o);
        sw += __shfl_xor_sync(0xffffffffu, sw, o);
    }
    if ((threadIdx.x & 31) == 0) {
        s_on[threadIdx.x >> 5] = on;
        s_off[threadIdx.x >> 5] = off;
        s_sw[threadIdx.x >> 5] = sw;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t_on = 0, t_off = 0;
        double t_sw = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
            t_on += s_on[w];
            t_off += s_off[w];
            t_sw += s_sw[w];
        }
        if (t_on) {
            atomicAdd(&cnt->n_gridded, t_on);
            atomicAdd(&cnt->sum_w, t_sw);
        }
        if (t_off) atomicAdd(&cnt->n_dropped, t_off);
    }
}

// ------------------------------------------------------------------------------------------
// a2: LSD radix sort of the 64-bit items over their key bits, <= 8-bit digits, stable.  The
// visibility index sits in the low idx_bits of an item and is never a digit: stability keeps
// equal keys in index order, so the sorted low parts ARE the permutation.  The digit histograms of
// all passes come from a1 (k_index_key); each pass is then ONE kernel that reads and writes the
// items once (k_radix_onesweep).
// ------------------------------------------------------------------------------------------
#define RS_THREADS 256
#ifndef RS_ITEMS
#define RS_ITEMS 12      // items per thread; 12 x 256 threads x 4 CTAs per SM measured best on B200 (0.59 vs 0.62 ms at 16 x 3)
#endif
#ifndef RS_MINB
#define RS_MINB 4
#endif
#define RS_TILE (RS_THREADS * RS_ITEMS)
typedef unsigned long long u64;

// exclusive scan over the digits of each pass: gbase[ps][d] = number of items whose digit of pass ps is < d
__global__ void __launch_bounds__(256) k_digit_bases(const unsigned int* __restrict__ ghist, int npass,
                                                     unsigned long long* __restrict__ gbase)
{
    __shared__ unsigned long long ws[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int ps = 0; ps < npass; ++ps) {
        const unsigned long long v = ghist[ps * 256 + threadIdx.x];
        unsigned long long x = v;
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) ws[warp] = x;
        __syncthreads();
        unsigned long long off = 0;
        for (int w = 0; w < warp; ++w) off += ws[w];
        gbase[ps * 256 + threadIdx.x] = off + x - v;
        __syncthreads();
    }
}

// One radix pass in one read + one write of the items ("onesweep"): the global digit bases are known
// (k_digit_bases); a tile ranks its items by digit (stable: warp match + per-warp digit counters), publishes
// its digit counts and finds the counts of all EARLIER tiles by decoupled look-back through `status`
// (one 64-bit word per (tile, digit): flag << 62 | count; flag 1 = this tile's count, 2 = inclusive prefix
// over tiles 0..this).  Tiles are taken in order from a ticket counter, so every predecessor of a running
// tile is running or done and the look-back cannot deadlock.  The tile is then reordered by digit in shared
// memory and written out position by position: consecutive threads write consecutive addresses of one
// digit's run, so the stores coalesce.
#define OS_AGG (1ull << 62)
#define OS_INC (2ull << 62)
#define OS_VAL ((1ull << 62) - 1ull)
#ifndef OS_LB
#define OS_LB 8u
#endif
__global__ void __launch_bounds__(RS_THREADS, RS_MINB)
k_radix_onesweep(const u64* __restrict__ in, u64* __restrict__ out, unsigned int M, int shift, uint32_t mask,
                 int nbins, const unsigned long long* __restrict__ gbase, volatile unsigned long long* status,
                 unsigned int* __restrict__ ticket, volatile unsigned int* dev_error)
{
    __shared__ uint32_t cnt[RS_THREADS / 32][256];
    __shared__ u64 buf[RS_TILE];
    __shared__ uint32_t dig_start[256];
    __shared__ long long gofs[256];
    __shared__ uint32_t wsum[RS_THREADS / 32];
    __shared__ unsigned int s_tile;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = threadIdx.x; i < (RS_THREADS / 32) * 256; i += RS_THREADS) (&cnt[0][0])[i] = 0;
    __syncthreads();
    const unsigned int tile = s_tile;
    const unsigned long long tile0 = (unsigned long long)tile * RS_TILE;
    const unsigned long long base = tile0 + (unsigned)warp * (32 * RS_ITEMS);
    u64 it[RS_ITEMS];
    uint32_t rank[RS_ITEMS];
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        const unsigned long long idx = base + (unsigned)i * 32 + lane;
        it[i] = idx < M ? in[idx] : ~0ull;
    }
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        const unsigned long long idx = base + (unsigned)i * 32 + lane;
        const bool valid = idx < M;
        const uint32_t d = (uint32_t)(it[i] >> shift) & mask;
        // lanes with the same digit: eight ballots, one per digit bit (MATCH.ANY costs several times that on
        // sm_100: it was 39 % of this kernel's stall samples, profiles/r1d_ncu_full.md)
        unsigned int m = __ballot_sync(0xffffffffu, valid);
        if (!valid) m = ~m;
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            const bool bit = (d >> b) & 1u;
            const unsigned int bal = __ballot_sync(0xffffffffu, bit);
            m &= bit ? bal : ~bal;
        }
        const int leader = __ffs(m) - 1;
        uint32_t old = 0;
        if (valid && lane == leader) {
            old = cnt[warp][d];
            cnt[warp][d] = old + (uint32_t)__popc(m);
        }
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[i] = old + (uint32_t)__popc(m & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    // digit d = threadIdx.x: exclusive prefix over the warps, then over the digits of the tile
    uint32_t total = 0;
    {
        const int d = threadIdx.x;
#pragma unroll
        for (int w = 0; w < RS_THREADS / 32; ++w) {
            const uint32_t t = cnt[w][d];
            cnt[w][d] = total;
            total += t;
        }
    }
    // publish this tile's count of digit d, then sum the earlier tiles' (look-back)
    volatile unsigned long long* st = status + (size_t)tile * 256 + threadIdx.x;
    unsigned long long excl = 0;
    if ((int)threadIdx.x < nbins) {
        if (tile == 0) {
            *st = OS_INC | (unsigned long long)total;
        } else {
            *st = OS_AGG | (unsigned long long)total;
            // look-back over the preceding tiles, OS_LB status words in flight at a time (a single dependent
            // read per step made every tile wait on a chain of L2 round trips)
            const volatile unsigned long long* q = st - 256;
            bool done = false;
            for (unsigned int back = tile; back > 0 && !done;) {
                const unsigned int n = back < OS_LB ? back : OS_LB;
                unsigned long long v[OS_LB];
#pragma unroll
                for (unsigned int j = 0; j < OS_LB; ++j) v[j] = j < n ? q[-256 * (long long)j] : 0ull;
#pragma unroll
                for (unsigned int j = 0; j < OS_LB; ++j) {
                    if (j < n && !done) {
                        unsigned int spins = 0;
                        while ((v[j] >> 62) == 0ull) {
                            __nanosleep(40);
                            // a lost predecessor: never hang and never trap (a trap would poison the caller's
                            // context across the ABI) -- raise the plan's device error flag, which the next
                            // synchronising call turns into RICK_ERR_CUDA, and let every waiting tile drain
                            if (++spins > (1u << 22) || ((spins & 255u) == 0u && *dev_error != 0u)) {
                                *dev_error = 1u;
                                done = true;
                                break;
                            }
                            v[j] = q[-256 * (long long)j];
                        }
                        if (done) break;
                        excl += v[j] & OS_VAL;
                        if ((v[j] >> 62) == 2ull) done = true;
                    }
                }
                back -= n;
                q -= 256 * (long long)n;
            }
            *st = OS_INC | (excl + (unsigned long long)total);
        }
    }
    uint32_t x = total;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) wsum[warp] = x;
    __syncthreads();
    uint32_t woff = 0;
#pragma unroll
    for (int w = 0; w < RS_THREADS / 32; ++w) woff += (w < warp) ? wsum[w] : 0u;
    const uint32_t start = woff + x - total;
    dig_start[threadIdx.x] = start;
    if ((int)threadIdx.x < nbins)
        gofs[threadIdx.x] = (long long)(gbase[threadIdx.x] + excl) - (long long)start;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        const unsigned long long idx = base + (unsigned)i * 32 + lane;
        if (idx < M) {
            const uint32_t d = (uint32_t)(it[i] >> shift) & mask;
            buf[dig_start[d] + cnt[warp][d] + rank[i]] = it[i];
        }
    }
    __syncthreads();
    const unsigned int n_valid = (unsigned int)((M - tile0) < RS_TILE ? (M - tile0) : RS_TILE);
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        const unsigned int pos = (unsigned)i * RS_THREADS + threadIdx.x;
        if (pos < n_valid) {
            const u64 v = buf[pos];
            const uint32_t d = (uint32_t)(v >> shift) & mask;
            out[gofs[d] + (long long)pos] = v;
        }
    }
}

// plane_start[z] = first sorted position whose key >= z*N*N  (z = 0..n_planes_total)
__global__ void k_plane_starts(const u64* __restrict__ sitems, unsigned int M, int idx_bits,
                               unsigned long long cells_per_plane, int n_planes_total,
                               long long* __restrict__ plane_start)
{
    const int z = blockIdx.x * blockDim.x + threadIdx.x;
    if (z > n_planes_total) return;
    const unsigned long long target = (unsigned long long)z * cells_per_plane;
    unsigned int lo = 0, hi = M;
    while (lo < hi) {
        const unsigned int mid = lo + (hi - lo) / 2;
        if ((sitems[mid] >> idx_bits) < target) lo = mid + 1; else hi = mid;
    }
    plane_start[z] = (long long)lo;
}

// Row occupancy at tile-row granularity.  One thread per (global plane pg, tile row tv): the sorted
// keys of that tile row are the range [lower_bound(prefix), lower_bound(prefix + 1)) with
// prefix = pg * T + tv over key / (N * B); a non-empty range marks the rows tv*B - h .. tv*B + B-1 + h
// (the tile rows plus the kernel halo) of plane pg.  occ is cleared by the caller first.
__global__ void k_row_occupancy(const u64* __restrict__ sitems, unsigned int M, int idx_bits, int N, int B, int T, int h,
                                int n_planes_total, unsigned char* __restrict__ occ)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n_planes_total * T) return;
    const unsigned long long span = (unsigned long long)N * (unsigned long long)B;      // keys per tile row
    const unsigned long long t0 = (unsigned long long)g * span, t1 = t0 + span;
    unsigned int lo = 0, hi = M;
    while (lo < hi) {
        const unsigned int mid = lo + (hi - lo) / 2;
        if ((sitems[mid] >> idx_bits) < t0) lo = mid + 1; else hi = mid;
    }
    if (lo >= M || (sitems[lo] >> idx_bits) >= t1) return;      // empty tile row
    const int pg = g / T, tv = g - pg * T;
    int r0 = tv * B - h, r1 = tv * B + B - 1 + h;
    r0 = r0 < 0 ? 0 : r0;
    r1 = r1 > N - 1 ? N - 1 : r1;
    for (int r = r0; r <= r1; ++r) occ[(size_t)pg * N + r] = 1;
}

// Tile occupancy.  One thread per sorted item; the first item of every run of equal keys (= one
// centre cell, reading R22) marks the B x B tiles its S x S footprint reaches: rows
// (i_v-h)>>log2B .. (i_v+h)>>log2B, columns likewise (on-grid visibilities only, so every tile
// exists).  Plain stores of 1 (idempotent, no atomics).  occ is cleared by the caller first.
__global__ void __launch_bounds__(256)
k_tile_occupancy(const u64* __restrict__ sitems, const long long* __restrict__ plane_start, int n_planes_total,
                 int idx_bits, int log2B, int log2T, int h, unsigned char* __restrict__ tocc)
{
    const long long n_valid = plane_start[n_planes_total];       // dropped visibilities sort last
    const int Bm = (1 << log2B) - 1, Tm = (1 << log2T) - 1;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_valid;
         i += (long long)gridDim.x * blockDim.x) {
        const u64 key = sitems[i] >> idx_bits;
        if (i > 0 && (sitems[i - 1] >> idx_bits) == key) continue;
        const int cu = (int)(key & (u64)Bm), cv = (int)((key >> log2B) & (u64)Bm);
        const u64 tkey = key >> (2 * log2B);
        const int tu = (int)(tkey & (u64)Tm), tv = (int)((tkey >> log2T) & (u64)Tm);
        const u64 pg = tkey >> (2 * log2T);
        const int iu = (tu << log2B) + cu, iv = (tv << log2B) + cv;
        const int u0 = (iu - h) >> log2B, u1 = (iu + h) >> log2B, v0 = (iv - h) >> log2B, v1 = (iv + h) >> log2B;
        unsigned char* o = tocc + ((size_t)pg << (2 * log2T));
        for (int a = v0; a <= v1; ++a)
            for (int b = u0; b <= u1; ++b) o[((size_t)a << log2T) + b] = 1;
    }
}

// ------------------------------------------------------------------------------------------
// a0 alone over n_rows rows: resets the statistics counters and leaves the w range in p->wrange
int rick_wrange_all(rick_plan_t* p, const double* uvw_m, int64_t n_rows)
{
    cudaStream_t st = p->stream;
    RICK_KERNEL(p, RK_RESET, k_counters_reset<<<1, 1, 0, st>>>(p->counters));
    if (n_rows > 0) {
        int nb = (int)((n_rows + 255) / 256);
        if (nb > p->n_sm * 8) nb = p->n_sm * 8;
        RICK_KERNEL(p, RK_WRANGE, k_wrange_rows<<<nb, 256, 0, st>>>(uvw_m, (long long)n_rows, p->counters, p->fold));
    }
    RICK_KERNEL(p, RK_WRANGE, k_wrange_finish<<<(p->n_img + 127) / 128, 128, 0, st>>>(p->counters, p->chan_scale, p->C, p->d.cube,
                                                          p->Nw_total, p->d.w_min, p->d.w_max,
                                                          (long long)n_rows, p->wrange));
    return RICK_OK;
}

// a0 + per-plane counts of the whole problem into hist_dev[Nw_total] (cleared here)
int rick_plane_hist(rick_plan_t* p, const double* uvw_m, unsigned long long* hist_dev)
{
    cudaStream_t st = p->stream;
    const int rc = rick_wrange_all(p, uvw_m, p->R);
    if (rc) return rc;
    RICK_CUDA(p, cudaMemsetAsync(hist_dev, 0, sizeof(unsigned long long) * (size_t)p->Nw_total, st));
    const unsigned int M = (unsigned int)p->M;
    if (M > 0) {
        unsigned int nb = (M + 255) / 256;
        if (nb > (unsigned)p->n_sm * 8u) nb = (unsigned)p->n_sm * 8u;
        const size_t sm = p->Nw_total <= 8192 ? sizeof(unsigned int) * (size_t)p->Nw_total : 0;
        RICK_KERNEL(p, RK_INDEX_KEY, k_plane_hist<<<nb, 256, sm, st>>>(uvw_m, p->chan_scale, p->wrange, M, (unsigned)p->C, p->N,
                                                                      p->Nw_total, p->h, p->inv_du, p->fold, hist_dev));
    }
    return RICK_OK;
}

int rick_index_sort(rick_plan_t* p, const double* uvw_m, const float* weights, int flags)
{
    cudaStream_t st = p->stream;
    const unsigned int M = (unsigned int)p->M;
    const int n_planes_total = p->n_img * p->Nw;

    if (!(flags & RICK_SORT_KEEP_RANGE)) {
        const int rc = rick_wrange_all(p, uvw_m, p->R);
        if (rc) return rc;
    }

    p->sorted_items = p->items;
    if (M > 0) {
        const unsigned long long key_dropped = (1ull << p->key_bits) - 1ull;
        // digits of the passes: the key bits split evenly over ceil(bits / 8) passes
        RadixPlan rp;
        memset(&rp, 0, sizeof(rp));
        const int bits = p->key_bits;
        rp.npass = (bits + 7) / 8;
        int nb_bits[RS_MAXPASS];
        for (int pass = 0, done = 0; pass < rp.npass; ++pass) {
            nb_bits[pass] = (bits - done + (rp.npass - pass) - 1) / (rp.npass - pass);
            rp.shift[pass] = done;
            rp.mask[pass] = (1u << nb_bits[pass]) - 1u;
            done += nb_bits[pass];
        }
        // scratch of the onesweep passes: ghist[8][256] u32 | ticket[8] u32, gbase[8][256] u64,
        // status[npass][nblocks][256] u64 (cleared by every sort)
        const unsigned int nblocks = (M + RS_TILE - 1) / RS_TILE;
        const size_t n_status = (size_t)rp.npass * nblocks * 256;
        if (!p->os_small) {
            RICK_CUDA(p, cudaMalloc(&p->os_small, sizeof(unsigned int) * (RS_MAXPASS * 256 + RS_MAXPASS)));
            RICK_CUDA(p, cudaMalloc(&p->os_gbase, sizeof(unsigned long long) * RS_MAXPASS * 256));
        }
        if (n_status > p->os_status_cap) {
            if (p->os_status) cudaFree(p->os_status);
            p->os_status = nullptr;
            p->os_status_cap = 0;
            RICK_CUDA(p, cudaMalloc(&p->os_status, sizeof(unsigned long long) * n_status));
            p->os_status_cap = n_status;
        }
        RICK_CUDA(p, cudaMemsetAsync(p->os_small, 0, sizeof(unsigned int) * (RS_MAXPASS * 256 + RS_MAXPASS), st));
        RICK_CUDA(p, cudaMemsetAsync(p->os_status, 0, sizeof(unsigned long long) * n_status, st));
        {
            unsigned int nb = (M + 255) / 256;
            if (nb > (unsigned)p->n_sm * 8u) nb = (unsigned)p->n_sm * 8u;
            RICK_KERNEL(p, RK_INDEX_KEY, k_index_key<<<nb, 256, 0, st>>>(uvw_m, weights, p->chan_scale, p->wrange, M,
                                                    (unsigned)p->C, p->N, p->Nw, p->h, p->log2B, p->T,
                                                    p->d.cube, p->inv_du, p->idx_bits, key_dropped, p->items,
                                                    p->counters, rp, p->os_small, p->fold, p->z0, p->Nw_total));
        }
        RICK_KERNEL(p, RK_SCAN, k_digit_bases<<<1, 256, 0, st>>>(p->os_small, rp.npass, p->os_gbase));
        const u64* in = (const u64*)p->items;
        u64* bufs[2] = {(u64*)p->items_a, (u64*)p->items_b};
        for (int pass = 0; pass < rp.npass; ++pass) {
            u64* o = bufs[pass & 1];
            RICK_KERNEL(p, RK_RADIX_SCATTER, k_radix_onesweep<<<nblocks, RS_THREADS, 0, st>>>(
                in, o, M, p->idx_bits + rp.shift[pass], rp.mask[pass], 1 << nb_bits[pass], p->os_gbase + pass * 256,
                p->os_status + (size_t)pass * nblocks * 256, p->os_small + RS_MAXPASS * 256 + pass, &p->counters->error));
            in = o;
        }
        p->sorted_items = (unsigned long long*)in;
    }
    RICK_KERNEL(p, RK_PLANE_STARTS, k_plane_starts<<<(n_planes_total + 1 + 127) / 128, 128, 0, st>>>(
        (const u64*)p->sorted_items, M, p->idx_bits, (unsigned long long)p->N * p->N, n_planes_total,
        (long long*)p->plane_start));
    if (!(flags & RICK_SORT_OCC_ACCUM)) RICK_CUDA(p, cudaMemsetAsync(p->row_occ, 0, (size_t)n_planes_total * p->N, st));
    if (M > 0) {
        const int n = n_planes_total * p->T;
        RICK_KERNEL(p, RK_ROW_OCC, k_row_occupancy<<<(n + 127) / 128, 128, 0, st>>>(
            (const u64*)p->sorted_items, M, p->idx_bits, p->N, p->B, p->T, p->h, n_planes_total, p->row_occ));
    }
    if (!(flags & RICK_SORT_OCC_ACCUM)) RICK_CUDA(p, cudaMemsetAsync(p->tile_occ, 0, (size_t)n_planes_total * p->T * p->T, st));
    if (M > 0) {
        unsigned int nb = (M + 255) / 256;
        if (nb > (unsigned)p->n_sm * 8u) nb = (unsigned)p->n_sm * 8u;
        RICK_KERNEL(p, RK_ROW_OCC, k_tile_occupancy<<<nb, 256, 0, st>>>(
            (const u64*)p->sorted_items, (const long long*)p->plane_start, n_planes_total, p->idx_bits, p->log2B,
            p->log2N - p->log2B, p->h, p->tile_occ));
    }
    return RICK_OK;
}

// ------------------------------------------------------------------------------------------
// rick_plane_histogram_noalloc: the per-plane histogram for callers that must not allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Same kernels as rick_plane_histogram
// (a0: k_counters_reset, k_wrange_rows, k_wrange_finish; then k_plane_hist); what that path keeps in buffers it
// allocates (the histogram accumulators per call, channel scales / w range / a0 counters on the plan) lives here in
// ONE file-scope device array of fixed size.  Every GPU that loads the library holds these 41 216 bytes until exit.
// All calls (of all plans) on a device share the array; it keeps the last call's contents, so what must start at
// zero is cleared by every call; two calls that overlap on the GPU (different streams) race.
// ------------------------------------------------------------------------------------------
constexpr int RICK_NOALLOC_HIST_OFF = 0;                                                   // u64 [MAX_PLANES]
constexpr int RICK_NOALLOC_SCALE_OFF = RICK_NOALLOC_HIST_OFF + 8 * RICK_NOALLOC_MAX_PLANES;  // double [MAX_CHAN]
constexpr int RICK_NOALLOC_WRANGE_OFF = RICK_NOALLOC_SCALE_OFF + 8 * RICK_NOALLOC_MAX_CHAN;  // WRange
constexpr int RICK_NOALLOC_CNT_OFF = RICK_NOALLOC_WRANGE_OFF + 64;                          // DevCounters
static_assert(RICK_NOALLOC_CNT_OFF + 192 == RICK_NOALLOC_SCRATCH_BYTES, "scratch layout vs rick.h");
static_assert(sizeof(WRange) <= 64 && sizeof(DevCounters) <= 192, "scratch layout");
static_assert(RICK_NOALLOC_SCRATCH_BYTES % 256 == 0, "stated size");
static __device__ __align__(256) unsigned char g_noalloc_scratch[RICK_NOALLOC_SCRATCH_BYTES];

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the device address is looked up
// once per device, with that device current, and cached.
static int noalloc_scratch_ptr(rick_plan_t* p, unsigned char** out)
{
    constexpr int MAX_DEV = 64;
    static unsigned char* s_ptr[MAX_DEV] = {};
    static std::mutex s_mu;
    int dev = -1;
    RICK_CUDA(p, cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) { p->err = "rick_plane_histogram_noalloc: device ordinal beyond 63"; return RICK_ERR_STATE; }
    std::lock_guard<std::mutex> lock(s_mu);
    if (!s_ptr[dev]) {
        void* q = nullptr;
        RICK_CUDA(p, cudaGetSymbolAddress(&q, g_noalloc_scratch));
        if (!q) { p->err = "rick_plane_histogram_noalloc: no device address for the scratch array"; return RICK_ERR_CUDA; }
        s_ptr[dev] = static_cast<unsigned char*>(q);
    }
    *out = s_ptr[dev];
    return RICK_OK;
}

extern "C" int rick_plane_histogram_noalloc(rick_plan_t* p, const double* uvw_m, const double* chan_freq_hz, int32_t n_chan,
                                            int64_t n_rows, int64_t* hist_host)
{
    if (!p) return RICK_ERR_INVALID;
    if (p->failed) return p->failed;
    p->err.clear();
    if (!hist_host) { p->err = "null hist_host"; return RICK_ERR_INVALID; }
    if (p->d.cube) { p->err = "rick_plane_histogram_noalloc: cube plans shard by channels"; return RICK_ERR_STATE; }
    if (p->Nw_total > RICK_NOALLOC_MAX_PLANES) {
        p->err = "rick_plane_histogram_noalloc: more than 4096 w-planes (the fixed scratch holds 4096 counters); use rick_plane_histogram";
        return RICK_ERR_INVALID;
    }
    if (n_chan < 1 || !chan_freq_hz) { p->err = "bad channels"; return RICK_ERR_INVALID; }
    if (n_chan > RICK_NOALLOC_MAX_CHAN) {
        p->err = "rick_plane_histogram_noalloc: more than 1024 channels (the fixed scratch holds 1024 scales); use rick_plane_histogram";
        return RICK_ERR_INVALID;
    }
    if (n_rows < 0) { p->err = "negative n_rows"; return RICK_ERR_INVALID; }
    if (n_rows > 0 && !uvw_m) { p->err = "null input"; return RICK_ERR_INVALID; }
    if (n_rows > 0 && (reinterpret_cast<uintptr_t>(uvw_m) & 15u)) { p->err = "device pointer not 16-byte aligned (uvw_m)"; return RICK_ERR_INVALID; }
    for (int c = 0; c < n_chan; ++c)
        if (!(chan_freq_hz[c] > 0.0) || !isfinite(chan_freq_hz[c])) { p->err = "bad frequency"; return RICK_ERR_INVALID; }
    const unsigned long long M64 = (unsigned long long)n_rows * (unsigned long long)n_chan;
    if (M64 >= 0xFFFFFFFFull) { p->err = "too many visibilities for 32-bit indices"; return RICK_ERR_INVALID; }

    unsigned char* scratch = nullptr;
    int rc = noalloc_scratch_ptr(p, &scratch);
    if (rc) return rc;
    unsigned long long* hist = reinterpret_cast<unsigned long long*>(scratch + RICK_NOALLOC_HIST_OFF);
    double* scale = reinterpret_cast<double*>(scratch + RICK_NOALLOC_SCALE_OFF);
    WRange* wr = reinterpret_cast<WRange*>(scratch + RICK_NOALLOC_WRANGE_OFF);
    DevCounters* cnt = reinterpret_cast<DevCounters*>(scratch + RICK_NOALLOC_CNT_OFF);
    cudaStream_t st = p->stream;

    // s_c = f_c / c0 through the plan's pinned staging (exists since plan creation; its previous upload must be done)
    RICK_CUDA(p, cudaEventSynchronize(p->ev_scale));
    for (int c = 0; c < n_chan; ++c) p->h_scale[c] = chan_freq_hz[c] / RICK_C0;
    RICK_CUDA(p, cudaMemcpyAsync(scale, p->h_scale, sizeof(double) * (size_t)n_chan, cudaMemcpyHostToDevice, st));
    RICK_CUDA(p, cudaEventRecord(p->ev_scale, st));
    // (the plan's own device copy of its last scales, p->chan_scale, is untouched)

    // a0 on the scratch counters (reset by k_counters_reset), then the counts (cleared here)
    RICK_KERNEL(p, RK_RESET, k_counters_reset<<<1, 1, 0, st>>>(cnt));
    if (n_rows > 0) {
        int nb = (int)((n_rows + 255) / 256);
        if (nb > p->n_sm * 8) nb = p->n_sm * 8;
        RICK_KERNEL(p, RK_WRANGE, k_wrange_rows<<<nb, 256, 0, st>>>(uvw_m, (long long)n_rows, cnt, p->fold));
    }
    RICK_KERNEL(p, RK_WRANGE, k_wrange_finish<<<1, 128, 0, st>>>(cnt, scale, (int)n_chan, 0, p->Nw_total, p->d.w_min, p->d.w_max,
                                                                 (long long)n_rows, wr));
    RICK_CUDA(p, cudaMemsetAsync(hist, 0, sizeof(unsigned long long) * (size_t)p->Nw_total, st));
    const unsigned int M = (unsigned int)M64;
    if (M > 0) {
        unsigned int nb = (M + 255) / 256;
        if (nb > (unsigned)p->n_sm * 8u) nb = (unsigned)p->n_sm * 8u;
        const size_t sm = sizeof(unsigned int) * (size_t)p->Nw_total;          // (<= 4096 planes: shared-memory counters)
        RICK_KERNEL(p, RK_INDEX_KEY, k_plane_hist<<<nb, 256, sm, st>>>(uvw_m, scale, wr, M, (unsigned)n_chan, p->N, p->Nw_total,
                                                                      p->h, p->inv_du, p->fold, hist));
    }
    RICK_CUDA(p, cudaMemcpyAsync(hist_host, hist, sizeof(unsigned long long) * (size_t)p->Nw_total, cudaMemcpyDeviceToHost, st));
    RICK_CUDA(p, cudaStreamSynchronize(st));
    return RICK_OK;
}
