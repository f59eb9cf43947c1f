// fft_cols12.cu -- the column (v-axis) pass of a4 for the fp64 grid with N = 4096 = 16^3, and its
// fusion with a5/a6 (PAPER.md:53, :68 FFT per w-plane; Eq. 2 :50 and :69 phase screen + plane sum;
// reading R12 taper).
//
// Why a dedicated kernel.  A column of a 4096^2 complex128 plane is 64 KB, so one SM can hold a
// strip of only two columns: the pass touches HBM in 32-byte pieces at a 64 KB stride.  Measured
// on B200 (feed ceilings): 32 B scattered reads run at ~4.7 TB/s through TMA but
// only ~4 TB/s through LSU loads, 32 B scattered WRITES at ~2 TB/s; and the L1 tag stage pays one
// cycle per 128 B line touched (16 lines per warp instruction).  Hence:
//   * the strip is fetched by ONE TMA instruction per (strip, plane): a 5-D tensor map views the
//     rows of a plane as digits row = w + 16 hh + 256 e and delivers the box in the order
//     [e][w][hh][c] that the first radix-16 stage reads conflict-free.  The load of the next item is
//     in flight while the current one is transformed (persistent CTA, one per SM, mbarrier).
//   * k_cols12_wcorrect never writes the transformed plane: it keeps the CTA on one strip, walks
//     the planes from the top down and sums them with Horner's rule in z,
//         S <- P_z + step * S,   step = exp(2 pi i dw (n-1)),
//     then I = Re(exp(2 pi i w_first (n-1)) S) [/ taper] once per strip.  Same mathematics as the
//     geometric phase recurrence of wcorrect.cu, one complex FMA per pixel per plane, two sincospi
//     per pixel per strip.
//   * S and step (2 x 16 complex doubles per thread, 256 KB per SM) do not fit the register file
//     next to the FFT; they live in TENSOR MEMORY, used here as a thread-private accumulator file
//     (tcgen05.ld / tcgen05.st, shape 32x32b) -- the tensor cores themselves are not involved in
//     this kernel.
// Shared memory: 128 KB TMA staging + 68 KB exchange buffer (real / imaginary halves in turn).
#include "common.cuh"
#include "fft_core.cuh"
#include "sm100_ptx.cuh"

namespace {

constexpr int C12_LOG2N = 12, C12_N = 1 << C12_LOG2N, C12_NT = C12_N / 16, C12_WC = 2;
constexpr int C12_THREADS = C12_NT * C12_WC, C12_STRIPS = C12_N / C12_WC;
constexpr uint32_t C12_STAGE_BYTES = (uint32_t)C12_N * C12_WC * 16u;                        // 131072
constexpr size_t C12_EX_BYTES = (size_t)C12_WC * (C12_N + C12_N / 16) * sizeof(double);     // 69632
constexpr size_t C12_SMEM = C12_STAGE_BYTES + C12_EX_BYTES + 64 + 1024;   // + slack for the 1024-byte alignment

struct Roles {
    int w, c, hh, t1, t2, t3;
};
__device__ __forceinline__ Roles roles()
{
    Roles r;
    const int lane = threadIdx.x & 31;
    r.w = threadIdx.x >> 5;
    r.c = lane & 1;
    r.hh = lane >> 1;
    r.t1 = r.w + 16 * r.hh;      // stage 1: rows t1 + 256 e   (exchange 1 stays inside the warp)
    r.t2 = 16 * r.w + r.hh;      // stage 2
    r.t3 = r.t2;                 // stage 3: outputs X[t3 + 256 r]
    return r;
}

// the 4096-point transform of the staged strip; on exit v[r] = X[t3 + 256 r] (uncentred index)
__device__ __forceinline__ void strip_fft(double2 (&v)[16], const Roles& R, const double2* __restrict__ stg,
                                          double* __restrict__ ex, const double2* __restrict__ tw,
                                          unsigned long long* bar, uint32_t& parity, bool issue_next,
                                          const CUtensorMap* tmap, int next_strip, int next_plane)
{
    mbar_wait(bar, parity);
    parity ^= 1u;
    // centring on input = rotation by N/2 = element e <- slot (e + 8) mod 16
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = stg[(((e + 8) & 15) * 256 + R.w * 16 + R.hh) * 2 + R.c];
    bfly16<double, C12_LOG2N, 0>(v, R.t1, tw);
    __syncthreads();             // staging consumed by all; previous item's reads of `ex` are done
    if (threadIdx.x == 0 && issue_next) {
        mbar_arrive_expect_tx(bar, C12_STAGE_BYTES);
        tma_load_5d(const_cast<double2*>(stg), tmap, bar, 4 * next_strip, 0, 0, 0, next_plane);
    }
    xchg16_warp(v, ex + (size_t)R.w * (16 * 17 * 2), R.hh, R.c);
    bfly16<double, C12_LOG2N, 4>(v, R.t2, tw);
    __syncthreads();             // every warp is done with its private region of `ex`
    xchg16_cta(v, ex, R.t2, R.t3, R.c);
    bfly16<double, C12_LOG2N, 8>(v, R.t3, tw);
}

// a4, column pass, in place (staged API).  Stores go straight from registers: 32 B pieces.
__global__ void __launch_bounds__(C12_THREADS, 1)
k_cols12_fft(const __grid_constant__ CUtensorMap tmap, double2* __restrict__ stack,
             const double2* __restrict__ tw, int n_planes)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* stg = reinterpret_cast<double2*>(smem_raw);
    double* ex = reinterpret_cast<double*>(smem_raw + C12_STAGE_BYTES);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem_raw + C12_STAGE_BYTES + C12_EX_BYTES);
    const Roles R = roles();
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int n_items = n_planes * C12_STRIPS;
    int item = blockIdx.x;
    if (threadIdx.x == 0 && item < n_items) {
        mbar_arrive_expect_tx(bar, C12_STAGE_BYTES);
        tma_load_5d(stg, &tmap, bar, 4 * (item % C12_STRIPS), 0, 0, 0, item / C12_STRIPS);
    }
    uint32_t parity = 0;
    for (; item < n_items; item += gridDim.x) {
        const int next = item + gridDim.x;
        double2 v[16];
        strip_fft(v, R, stg, ex, tw, bar, parity, next < n_items, &tmap, next % C12_STRIPS, next / C12_STRIPS);
        const int plane = item / C12_STRIPS, strip = item - plane * C12_STRIPS;
        double2* g = stack + (size_t)plane * C12_N * C12_N + (size_t)strip * C12_WC + R.c;
#pragma unroll
        for (int e = 0; e < 16; ++e) g[(size_t)(R.t3 + C12_NT * ((e + 8) & 15)) * C12_N] = v[e];
    }
}

// ---------------------------------------------------------------------------------------------------
// a4 column pass fused with a5 (+ a6 when taper != nullptr).
//
// The CTA is two COLUMN GROUPS of 256 threads: group g (warps 8g .. 8g+7) owns column g of the strip,
// thread role (w, hh) = (tg >> 4, tg & 15).  The groups share the TMA staging of the item but run out of
// phase: group 1 may read the staging only after group 0 has (named barrier 3), and from there on each
// group synchronises only with itself (named barrier 1 + g), so one group's shared-memory exchange runs
// under the other group's butterflies (with one 512-thread lock step the item time was the SUM of its
// fp64 time and its shared-memory time, profiles/r1b_ncu_full.md).  The staging is 32-byte swizzled by
// the tensor map (16-byte chunk ^= bit 7 of the byte offset) so that a group's 16-byte reads at a
// 32-byte pitch are bank-conflict free.  `full` = TMA landed; `empty` = all 16 warps have read the
// staging, waited for by the one thread that issues the next load.
struct RolesG {
    int g, w, hh, wl, t1, t2;
};
__device__ __forceinline__ RolesG roles_g()
{
    RolesG r;
    const int tg = threadIdx.x & 255;
    r.g = threadIdx.x >> 8;
    r.w = tg >> 4;
    r.hh = tg & 15;
    r.wl = (threadIdx.x >> 4) & 1;
    r.t1 = r.w + 16 * r.hh;      // stage 1: rows t1 + 256 e
    r.t2 = 16 * r.w + r.hh;      // stages 2 and 3; outputs X[t2 + 256 r]
    return r;
}

__device__ __forceinline__ void strip_fft_g(double2 (&v)[16], const RolesG& R, const double2* __restrict__ stg,
                                            double* __restrict__ ex, const double2* __restrict__ tw,
                                            unsigned long long* full, unsigned long long* empty, uint32_t& parity,
                                            bool issue_next, const CUtensorMap* tmap, int next_strip, int next_plane)
{
    if (R.g == 1) named_bar_sync(3, 512);        // group 0 has read the staging of this item
    mbar_wait(full, parity);
    // centring on input = rotation by N/2 = element e <- slot (e + 8) mod 16; swizzled chunk of column g
    const int sw = R.g ^ ((R.hh >> 2) & 1);
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = stg[(((e + 8) & 15) * 256 + R.w * 16 + R.hh) * 2 + sw];
    if (R.g == 0) named_bar_arrive(3, 512);
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(empty);
    if (threadIdx.x == 256 && issue_next) {
        mbar_wait(empty, parity);
        mbar_arrive_expect_tx(full, C12_STAGE_BYTES);
        tma_load_5d(const_cast<double2*>(stg), tmap, full, 4 * next_strip, 0, 0, 0, next_plane);
    }
    parity ^= 1u;
    bfly16<double, C12_LOG2N, 0>(v, R.t1, tw);
    // the base twiddles of stages 2 and 3 are fetched before the exchanges they follow
    const double2 w1_s2 = tw[bfly16_tw_index<C12_LOG2N, 4>(R.t2)];
    named_bar_sync(1 + R.g, 256);                // the group's reads of the previous item's exchange are done
    xchg16_warp_grp(v, ex + (size_t)(threadIdx.x >> 5) * (2 * 16 * 17), R.wl, R.hh);
    bfly16<double, C12_LOG2N, 4>(v, R.t2, tw, &w1_s2);
    const double2 w1_s3 = tw[bfly16_tw_index<C12_LOG2N, 8>(R.t2)];
    named_bar_sync(1 + R.g, 256);                // every warp of the group is done with its private region
    xchg16_grp(v, ex + (size_t)R.g * (C12_N + C12_N / 16), R.t2, 1 + R.g);
    bfly16<double, C12_LOG2N, 8>(v, R.t2, tw, &w1_s3);
}

__global__ void __launch_bounds__(C12_THREADS, 1)
k_cols12_wcorrect(const __grid_constant__ CUtensorMap tmap, const double2* __restrict__ tw, int n_planes,
                  int z_first, double dl, const WRange* __restrict__ wr, double* __restrict__ image,
                  int accumulate, const double* __restrict__ taper, int strip_begin, int strip_end, int slot_first)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // the swizzle pattern is a function of the shared-memory ADDRESS: staging on a 1024-byte boundary
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    double2* stg = reinterpret_cast<double2*>(smem);
    double* ex = reinterpret_cast<double*>(smem + C12_STAGE_BYTES);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + C12_STAGE_BYTES + C12_EX_BYTES);
    unsigned long long* empty = full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C12_STAGE_BYTES + C12_EX_BYTES + 16);
    const RolesG R = roles_g();
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        mbar_init(full, 1);
        mbar_init(empty, C12_THREADS / 32);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc_all(tmem_slot);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tmem_slot;
    // warps w, w+4, w+8, w+12 share the TMEM lanes 32 (w%4) ..; 128 columns each: S | step
    const uint32_t tS = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 128);
    const uint32_t tStep = tS + 64;

    int strip = strip_begin + (int)blockIdx.x;
    if (threadIdx.x == 0 && strip < strip_end) {
        mbar_arrive_expect_tx(full, C12_STAGE_BYTES);
        tma_load_5d(stg, &tmap, full, 4 * strip, 0, 0, 0, slot_first + n_planes - 1);
    }
    uint32_t parity = 0;
    const double dw = wr->dw;
    const double w_first = wr->w_min + ((double)z_first + 0.5) * dw;
    for (; strip < strip_end; strip += gridDim.x) {
        const int p = strip * C12_WC + R.g;
        const double l = (double)(p - C12_N / 2) * dl;
        const double itp = taper ? taper[C12_N + p] : 1.0;       // 1 / c(nu_p): taper[N ..) holds the reciprocals
        // step = exp(2 pi i dw (n-1)) of this thread's 16 pixels (rows t2 + 256 ((e+8)&15)) -> TMEM
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double2 st[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int q = R.t2 + C12_NT * ((4 * k + i + 8) & 15);
                const double m = (double)(q - C12_N / 2) * dl;
                const double r2 = l * l + m * m;
                double xs = 0.0;
                if (r2 < 1.0) xs = dw * nm1_of(r2);
                xs -= rint(xs);
                sincospi(2.0 * xs, &st[i].y, &st[i].x);
            }
            uint32_t r[16];
            pack4(st, r);
            tmem_st16(tStep + 16 * k, r);
        }
        tmem_wait_st();
        for (int plane = n_planes - 1; plane >= 0; --plane) {
            const bool more = plane > 0 || strip + (int)gridDim.x < strip_end;
            double2 v[16];
            strip_fft_g(v, R, stg, ex, tw, full, empty, parity, more, &tmap, plane > 0 ? strip : strip + (int)gridDim.x,
                        slot_first + (plane > 0 ? plane - 1 : n_planes - 1));
            // Horner in z: S <- P_z + step S
            if (plane == n_planes - 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double2 s4[4] = {v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]};
                    uint32_t r[16];
                    pack4(s4, r);
                    tmem_st16(tS + 16 * k, r);
                }
            } else {
                tmem_wait_st();      // the previous plane's stores of S (their latency ran under this item's transform)
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint32_t rs[16], rt[16];
                    tmem_ld16(tS + 16 * k, rs);
                    tmem_ld16(tStep + 16 * k, rt);
                    tmem_wait_ld();
                    double2 s4[4], st[4];
                    unpack4(rs, s4);
                    unpack4(rt, st);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double2 a = v[4 * k + i];
                        double2 o;
                        o.x = fma(st[i].x, s4[i].x, fma(-st[i].y, s4[i].y, a.x));
                        o.y = fma(st[i].x, s4[i].y, fma(st[i].y, s4[i].x, a.y));
                        s4[i] = o;
                    }
                    pack4(s4, rs);
                    tmem_st16(tS + 16 * k, rs);
                }
            }
        }
        // I = Re(exp(2 pi i w_first (n-1)) S)  [+ previous batches]  [/ taper]
        tmem_wait_st();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t rs[16];
            tmem_ld16(tS + 16 * k, rs);
            tmem_wait_ld();
            double2 s4[4];
            unpack4(rs, s4);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int q = R.t2 + C12_NT * ((4 * k + i + 8) & 15);
                const double m = (double)(q - C12_N / 2) * dl;
                const double r2 = l * l + m * m;
                double val = 0.0;
                if (r2 < 1.0) {
                    double x0 = w_first * nm1_of(r2);
                    x0 -= rint(x0);
                    double pr, pi;
                    sincospi(2.0 * x0, &pi, &pr);
                    val = pr * s4[i].x - pi * s4[i].y;
                }
                const size_t pix = (size_t)q * C12_N + p;
                if (accumulate) val += image[pix];
                if (taper) val *= itp * taper[C12_N + q];
                image[pix] = val;
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc_all(tbase);
}


// ---------------------------------------------------------------------------------------------------
// N = 8192 = 2 * 4096 (fp64): the same fused single pass for a column of 128 KB.  One SM holds ONE column
// (staging 128 KB, the transform in registers, S and step in tensor memory), fetched by one TMA instruction
// per (column, plane) in 16-byte pieces.  The two column groups of the N = 4096 kernel become the two halves
// of a decimation-in-frequency split that needs no exchange between the groups: with x'[n] = G[(n + N/2) mod N]
// (centring on input) and H = N/2,
//     X[2 kk]     = FFT_H( x'[n] + x'[n + H] )            = FFT_H( G[n + H] + G[n] )              group 0
//     X[2 kk + 1] = FFT_H( (x'[n] - x'[n + H]) W_N^n )    = FFT_H( (G[n + H] - G[n]) W_N^n )      group 1
// both groups read the whole staging (rows n and n + H of the thread's 16 values of n), run their own
// 4096-point transform exactly as in k_cols12_wcorrect, and keep the outputs k = 2 (t2 + 256 r) + g, i.e. the
// pixel rows q = (k + N/2) mod N = 2 t2 + g + 512 ((r + 8) & 15).  Against the two-pass path (fft.cu) the stack
// is read ONCE and never written: 68.7 GB instead of 170 GB at configs[2].
constexpr int C13_N = 2 * C12_N;
constexpr uint32_t C13_STAGE_BYTES = (uint32_t)C13_N * 16u;          // 131072: one column

constexpr uint32_t C13_WIN_BYTES = C13_STAGE_BYTES / 32;            // a window of 256 rows of one column: 4 KB

// Pacing.  A 16-byte piece of a column sits in a 128-byte line with the pieces of the seven neighbouring columns,
// which seven other SMs fetch, and an L2 miss on this access pattern fills far more than the piece from DRAM (measured
// with the copies alone: 126 bytes of DRAM traffic per 16-byte piece when every SM walks a plane of its own, 1.03 x the
// useful bytes when all walk the same plane).  The stack is read once only as long as the CTAs work
// on the same plane at about the same time.  While the pass was bound by its feed they did by themselves (a CTA that
// ran ahead missed in L2 and fell back); with the known-zero windows skipped most planes are bound by their arithmetic,
// nothing couples the CTAs any more, they drift apart by whole planes and DRAM delivered 2.5 x the bytes.  So the CTAs
// pace each other: arrivals[i] counts the CTAs that have issued their item number i (one RED per CTA and item), and a
// CTA issues its item i only once every CTA that has an item i - C13_PACE_SLACK has issued it.  One word is polled, and
// it is fetched at the top of the item, long before the copy it gates.  The wait is bounded (0.3 ms): if the others do
// not show up (CTAs of the grid not resident) the warp stops pacing for good -- the result does not depend on it.
constexpr int C13_PACE_SLACK = 2;
constexpr unsigned long long C13_PACE_TIMEOUT_NS = 300000ull;
struct Pace {
    uint32_t* arrivals;               // [items per CTA], zeroed before the launch; null = no pacing
    int n_planes, n_cols;             // of the launch: item i belongs to column round i / n_planes
    bool on;
};
__device__ __forceinline__ uint32_t pace_load(const Pace& pc, int item)            // arrivals of the item that gates `item`
{
    return pc.on && item >= C13_PACE_SLACK ? *(volatile uint32_t*)(pc.arrivals + (item - C13_PACE_SLACK)) : 0u;
}
__device__ __forceinline__ void pace_wait(Pace& pc, int item, uint32_t seen)
{
    if (!pc.on || item < C13_PACE_SLACK) return;
    const int round = (item - C13_PACE_SLACK) / pc.n_planes, full = pc.n_cols / (int)gridDim.x;
    const uint32_t need = round < full ? gridDim.x : (round == full ? (uint32_t)(pc.n_cols % (int)gridDim.x) : 0u);
    if (seen >= need) return;
    // (rare path) bounded in TIME: ~40 item periods.  CTAs of the grid that are not resident yet -- another kernel holds
    // their SMs -- must not stall the ones that are.
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do {
        seen = pace_load(pc, item);
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    } while (seen < need && t - t0 < C13_PACE_TIMEOUT_NS);
    if (seen < need) pc.on = false;
}

// Fetch the occupied windows of (column, plane) into the staging: called by the EIGHT warps first_warp .. first_warp + 7,
// lanes 0 .. 3 of each issue one window (32 copies issued by one warp held that warp, and its group, up).  mask bit
// k = e + 16 e2 <-> rows 256 k .. 256 k + 255 <-> staging bytes [4096 k, 4096 (k + 1)).  Windows with no occupied
// row are zero in HBM and are neither fetched nor read.  (A copy may complete before the
// expect_tx of the one arriving thread: the barrier's pending arrival keeps the phase open.)  `item` = the number of
// this item among the CTA's items, `seen` = pace_load(pc, item) fetched earlier.
__device__ __forceinline__ void col13_issue(const double2* stg, unsigned long long* full, const CUtensorMap* tmap_all,
                                            const CUtensorMap* tmap_win, uint32_t mask, int col, int slot, int first_warp,
                                            Pace& pc, int item, uint32_t seen)
{
    const int lane = threadIdx.x & 31, wq = (int)(threadIdx.x >> 5) - first_warp;
    pace_wait(pc, item, seen);
    if (pc.arrivals && wq == 0 && lane == 0) atomicAdd(pc.arrivals + item, 1u);
    if (mask == 0xffffffffu) {
        if (wq == 0 && lane == 0) {
            mbar_arrive_expect_tx(full, C13_STAGE_BYTES);
            tma_load_5d(const_cast<double2*>(stg), tmap_all, full, 2 * col, 0, 0, 0, 2 * slot);
        }
        return;
    }
    if (wq == 0 && lane == 0) mbar_arrive_expect_tx(full, (uint32_t)__popc(mask) * C13_WIN_BYTES);
    const int k = 4 * wq + lane;
    if (lane < 4 && ((mask >> k) & 1u))
        tma_load_5d(const_cast<double2*>(stg) + k * (int)(C13_WIN_BYTES / 16), tmap_win, full, 2 * col, 0, 0, k & 15,
                    2 * slot + (k >> 4));
}

__device__ __forceinline__ void col13_fft_g(double2 (&v)[16], const RolesG& R, const double2* __restrict__ stg,
                                            double* __restrict__ ex, const double2* __restrict__ twN,
                                            unsigned long long* full, unsigned long long* empty, uint32_t& parity,
                                            bool issue_next, const CUtensorMap* tmap, const CUtensorMap* tmap_win,
                                            uint32_t mask, uint32_t mask_next, int next_col, int next_plane, Pace& pc,
                                            int next_item)
{
    // group 1: W_N^n for n = t1 + 256 e is W_N^t1 times the constant e^{2 pi i e / 32}
    double2 wb;
    uint32_t seen = 0;
    if (R.g == 1) {
        if (issue_next) seen = pace_load(pc, next_item);       // (consumed after the staging read)
        wb = twN[R.t1];
        named_bar_sync(3, 512);                  // group 0 has read the staging of this item
    }
    mbar_wait(full, parity);
    // staging order [e2][e][w][hh] (16-byte elements): row = w + 16 hh + 256 e + 4096 e2; windows the mask leaves
    // out were not fetched and count as zero
    const double2* s0 = stg + R.w * 16 + R.hh;
    const double2 zero = make_double2(0.0, 0.0);
    if (R.g == 0) {
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const double2 hi = (mask >> (16 + e)) & 1u ? s0[(16 + e) * 256] : zero;
            const double2 lo = (mask >> e) & 1u ? s0[e * 256] : zero;
            v[e] = cadd(hi, lo);
        }
    } else {
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const double2 hi = (mask >> (16 + e)) & 1u ? s0[(16 + e) * 256] : zero;
            const double2 lo = (mask >> e) & 1u ? s0[e * 256] : zero;
            v[e] = csub(hi, lo);
        }
    }
    if (R.g == 0) named_bar_arrive(3, 512);
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(empty);
    if (R.g == 1 && issue_next) {                     // group 1 is the last to read the staging
        mbar_wait(empty, parity);
        col13_issue(stg, full, tmap, tmap_win, mask_next, next_col, next_plane, 8, pc, next_item, seen);
    }
    parity ^= 1u;
    if (R.g == 1) {
        // e^{2 pi i e / 32}, e = 1 .. 15
        constexpr double c32[16] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                                    0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                                    0.19509032201612826785, 0.0, -0.19509032201612826785, -0.38268343236508977173,
                                    -0.55557023301960222474, -0.70710678118654752440, -0.83146961230254523708,
                                    -0.92387953251128675613, -0.98078528040323044913};
        v[0] = cmul(v[0], wb);
#pragma unroll
        for (int e = 1; e < 16; ++e) {
            double2 c;
            c.x = c32[e];
            c.y = c32[e < 8 ? 8 - e : e - 8];                             // sin(pi e/16) = cos(pi (e - 8)/16)
            v[e] = cmul(v[e], cmul(wb, c));
        }
    }
    bfly16<double, C12_LOG2N, 0>(v, R.t1, twN);
    // the 4096-point twiddles are every second entry of the N = 8192 table
    const double2 w1_s2 = twN[2 * bfly16_tw_index<C12_LOG2N, 4>(R.t2)];
    named_bar_sync(1 + R.g, 256);                // the group's reads of the previous item's exchange are done
    xchg16_warp_grp(v, ex + (size_t)(threadIdx.x >> 5) * (2 * 16 * 17), R.wl, R.hh);
    bfly16<double, C12_LOG2N, 4>(v, R.t2, twN, &w1_s2);
    const double2 w1_s3 = twN[2 * bfly16_tw_index<C12_LOG2N, 8>(R.t2)];
    named_bar_sync(1 + R.g, 256);                // every warp of the group is done with its private region
    xchg16_grp(v, ex + (size_t)R.g * (C12_N + C12_N / 16), R.t2, 1 + R.g);
    bfly16<double, C12_LOG2N, 8>(v, R.t2, twN, &w1_s3);
}

__global__ void __launch_bounds__(C12_THREADS, 1)
k_cols13_wcorrect(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_win,
                  const uint32_t* __restrict__ wmask, const double2* __restrict__ twN, int n_planes,
                  int z_first, double dl, const WRange* __restrict__ wr, double* __restrict__ image,
                  int accumulate, const double* __restrict__ taper, int col_begin, int col_end, int slot_first,
                  uint32_t* arrivals)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    double2* stg = reinterpret_cast<double2*>(smem);
    double* ex = reinterpret_cast<double*>(smem + C13_STAGE_BYTES);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + C13_STAGE_BYTES + C12_EX_BYTES);
    unsigned long long* empty = full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C13_STAGE_BYTES + C12_EX_BYTES + 16);
    const RolesG R = roles_g();
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        mbar_init(full, 1);
        mbar_init(empty, C12_THREADS / 32);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc_all(tmem_slot);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tmem_slot;
    const uint32_t tS = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 128);
    const uint32_t tStep = tS + 64;

    int col = col_begin + (int)blockIdx.x;
    // wmask[plane]: the occupied 256-row windows of the batch's planes (k_window_mask, fft.cu)
    const uint32_t mask_top = wmask[n_planes - 1];
    uint32_t mask = mask_top;
    Pace pc = {arrivals, n_planes, col_end - col_begin, arrivals != nullptr};
    int item = 0;                                // items this CTA has issued
    if (col < col_end) {
        if (warp < 8) col13_issue(stg, full, &tmap, &tmap_win, mask, col, slot_first + n_planes - 1, 0, pc, 0, 0u);
        item = 1;
    }
    uint32_t parity = 0;
    const double dw = wr->dw;
    const double w_first = wr->w_min + ((double)z_first + 0.5) * dw;
    const int q0 = 2 * R.t2 + R.g;               // pixel rows of this thread: q0 + 512 ((r + 8) & 15)
    for (; col < col_end; col += gridDim.x) {
        const double l = (double)(col - C13_N / 2) * dl;
        const double itp = taper ? taper[C13_N + col] : 1.0;     // 1 / c(nu_p)
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double2 st[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int q = q0 + 512 * ((4 * k + i + 8) & 15);
                const double m = (double)(q - C13_N / 2) * dl;
                const double r2 = l * l + m * m;
                double xs = 0.0;
                if (r2 < 1.0) xs = dw * nm1_of(r2);
                xs -= rint(xs);
                sincospi(2.0 * xs, &st[i].y, &st[i].x);
            }
            uint32_t r[16];
            pack4(st, r);
            tmem_st16(tStep + 16 * k, r);
        }
        tmem_wait_st();
        for (int plane = n_planes - 1; plane >= 0; --plane) {
            const bool more = plane > 0 || col + (int)gridDim.x < col_end;
            const uint32_t mask_next = plane > 0 ? wmask[plane - 1] : mask_top;
            double2 v[16];
            col13_fft_g(v, R, stg, ex, twN, full, empty, parity, more, &tmap, &tmap_win, mask, mask_next,
                        plane > 0 ? col : col + (int)gridDim.x, slot_first + (plane > 0 ? plane - 1 : n_planes - 1), pc, item);
            item += more;
            mask = mask_next;
            if (plane == n_planes - 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double2 s4[4] = {v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]};
                    uint32_t r[16];
                    pack4(s4, r);
                    tmem_st16(tS + 16 * k, r);
                }
            } else {
                tmem_wait_st();
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint32_t rs[16], rt[16];
                    tmem_ld16(tS + 16 * k, rs);
                    tmem_ld16(tStep + 16 * k, rt);
                    tmem_wait_ld();
                    double2 s4[4], st[4];
                    unpack4(rs, s4);
                    unpack4(rt, st);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double2 a = v[4 * k + i];
                        double2 o;
                        o.x = fma(st[i].x, s4[i].x, fma(-st[i].y, s4[i].y, a.x));
                        o.y = fma(st[i].x, s4[i].y, fma(st[i].y, s4[i].x, a.y));
                        s4[i] = o;
                    }
                    pack4(s4, rs);
                    tmem_st16(tS + 16 * k, rs);
                }
            }
        }
        tmem_wait_st();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t rs[16];
            tmem_ld16(tS + 16 * k, rs);
            tmem_wait_ld();
            double2 s4[4];
            unpack4(rs, s4);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int q = q0 + 512 * ((4 * k + i + 8) & 15);
                const double m = (double)(q - C13_N / 2) * dl;
                const double r2 = l * l + m * m;
                double val = 0.0;
                if (r2 < 1.0) {
                    double x0 = w_first * nm1_of(r2);
                    x0 -= rint(x0);
                    double pr, pi;
                    sincospi(2.0 * x0, &pi, &pr);
                    val = pr * s4[i].x - pi * s4[i].y;
                }
                const size_t pix = (size_t)q * C13_N + col;
                if (accumulate) val += image[pix];
                if (taper) val *= itp * taper[C13_N + q];
                image[pix] = val;
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc_all(tbase);
}

}   // namespace

// Build the 5-D tensor maps over the plan's resident stack (once, at plan creation).
static int encode_map(rick_plan_t* p, void* out, const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box,
                      CUtensorMapSwizzle sw, CUtensorMapL2promotion promo)
{
    rick_encode_tiled_fn enc = rick_get_encode_tiled();
    if (!enc) {
        p->err = "cuTensorMapEncodeTiled is not available from this driver";
        return RICK_ERR_CUDA;
    }
    const cuuint32_t es[5] = {1, 1, 1, 1, 1};
    const CUresult r = enc(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, p->stack, dims, strides,
                           box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, sw, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        p->err = "cuTensorMapEncodeTiled failed";
        return RICK_ERR_CUDA;
    }
    return RICK_OK;
}

int rick_cols12_init(rick_plan_t* p)
{
    p->cols12_ok = 0;
    p->cols13_ok = 0;
    if (p->f32 || (p->N != C12_N && p->N != C13_N)) return RICK_OK;
    static_assert(sizeof(CUtensorMap) <= sizeof(p->cols12_tmap), "tensor map storage");
    static_assert(sizeof(CUtensorMap) <= sizeof(p->cols12_tmap_sw), "tensor map storage");
    const cuuint64_t rowB = (cuuint64_t)p->N * 16;
    int rc;
    if (p->N == C13_N) {
        // dims: (re/im of one column as doubles, hh, w, e, e2 + 2 plane) with row = w + 16 hh + 256 e + 4096 e2
        const cuuint64_t dims[5] = {(cuuint64_t)2 * C13_N, 16, 16, 16, (cuuint64_t)2 * p->slots};
        const cuuint64_t strides[4] = {16 * rowB, rowB, 256 * rowB, 4096 * rowB};
        const cuuint32_t box[5] = {2, 16, 16, 16, 2};
        if ((rc = encode_map(p, p->cols12_tmap_sw, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE))) return rc;
        // the same view with a box of ONE window of 256 rows (e, e2 fixed): planes with empty windows are fetched window by window
        const cuuint32_t box_win[5] = {2, 16, 16, 1, 1};
        if ((rc = encode_map(p, p->cols12_tmap, dims, strides, box_win, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE))) return rc;
        RICK_CUDA(p, cudaFuncSetAttribute(k_cols13_wcorrect, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C12_SMEM));
        // pacing counters (k_cols13_wcorrect, "Pacing"): one per item of a CTA, at most ceil(N / n_sm) columns x the
        // resident planes of one launch
        if (!p->cols_arrivals) {
            const size_t cap = (size_t)((C13_N + p->n_sm - 1) / p->n_sm) * (size_t)p->slots;
            RICK_CUDA(p, cudaMalloc(&p->cols_arrivals, sizeof(uint32_t) * cap));
            p->cols_arrivals_cap = cap;
        }
        p->cols13_ok = 1;
        return RICK_OK;
    }
    // dims: (re/im/column pair as doubles, hh, w, e, plane) with row = w + 16 hh + 256 e
    const cuuint64_t dims[5] = {(cuuint64_t)2 * C12_N, 16, 16, 16, (cuuint64_t)p->slots};
    const cuuint64_t strides[4] = {16 * rowB, rowB, 256 * rowB, (cuuint64_t)C12_N * rowB};
    const cuuint32_t box[5] = {4, 16, 16, 16, 1};
    if ((rc = encode_map(p, p->cols12_tmap, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE))) return rc;
    if ((rc = encode_map(p, p->cols12_tmap_sw, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_NONE))) return rc;
    RICK_CUDA(p, cudaFuncSetAttribute(k_cols12_fft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C12_SMEM));
    RICK_CUDA(p, cudaFuncSetAttribute(k_cols12_wcorrect, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C12_SMEM));
    p->cols12_ok = 1;
    return RICK_OK;
}

int rick_cols12_fft(rick_plan_t* p, int n_planes)
{
    const CUtensorMap tm = *reinterpret_cast<const CUtensorMap*>(p->cols12_tmap);
    RICK_KERNEL(p, RK_FFT_COLS, k_cols12_fft<<<p->n_sm, C12_THREADS, C12_SMEM, p->stream>>>(
        tm, (double2*)p->stack, (const double2*)p->twiddle, n_planes));
    return RICK_OK;
}

// units [strip_begin, strip_end) only.  N = 4096: a unit is a strip of two columns (2048 units); N = 8192: one
// column (8192 units).  rick_image_host launches the pass in a few parts (each a whole number of rounds of the
// persistent grid) so that the device -> host copy of one part runs under the next part's kernel.
int rick_cols12_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image, int accumulate,
                         int fuse_taper, int strip_begin, int strip_end, int slot_first)
{
    if (strip_end <= strip_begin) return RICK_OK;
    const CUtensorMap tm = *reinterpret_cast<const CUtensorMap*>(p->cols12_tmap_sw);
    const int n = strip_end - strip_begin;
    if (p->cols13_ok) {
        const CUtensorMap tm_win = *reinterpret_cast<const CUtensorMap*>(p->cols12_tmap);
        // (the row pass of these planes has just written their window masks)
        // the pacing counters of this launch: one per item of a CTA
        const int grid = n < p->n_sm ? n : p->n_sm;
        const size_t n_items = (size_t)((n + grid - 1) / grid) * (size_t)n_planes;
        if (n_items > p->cols_arrivals_cap) { p->err = "k_cols13_wcorrect: pacing counters too small"; return RICK_ERR_STATE; }
        RICK_CUDA(p, cudaMemsetAsync(p->cols_arrivals, 0, sizeof(uint32_t) * n_items, p->stream));
        RICK_KERNEL(p, RK_COLS_WCORRECT, k_cols13_wcorrect<<<grid, C12_THREADS, C12_SMEM, p->stream>>>(
            tm, tm_win, p->win_mask + (size_t)img * p->Nw + z_first, (const double2*)p->twiddle, n_planes, p->z0 + z_first, p->dl,
            p->wrange + img, image, accumulate, fuse_taper ? p->taper : nullptr, strip_begin, strip_end, slot_first,
            p->cols_arrivals));
        return RICK_OK;
    }
    RICK_KERNEL(p, RK_COLS_WCORRECT, k_cols12_wcorrect<<<n < p->n_sm ? n : p->n_sm, C12_THREADS, C12_SMEM, p->stream>>>(
        tm, (const double2*)p->twiddle, n_planes, p->z0 + z_first, p->dl, p->wrange + img, image, accumulate,
        fuse_taper ? p->taper : nullptr, strip_begin, strip_end, slot_first));
    return RICK_OK;
}

int rick_cols12_strips(const rick_plan_t* p) { return p->cols13_ok ? C13_N : C12_STRIPS; }
int rick_cols12_unit_cols(const rick_plan_t* p) { return p->cols13_ok ? 1 : C12_WC; }
int rick_cols_fused(const rick_plan_t* p) { return p->cols12_ok || p->cols13_ok; }
