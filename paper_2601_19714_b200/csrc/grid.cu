// grid.cu -- a3: convolutional gridding with a separable Kaiser-Bessel kernel
// (Eq. 3; kernel :62; halo = (S-1)/2 cells, Eq. 5 :129).
//
//   G[i_p][i_v+b][i_u+a] += (w V) g(d_a) g(d_b),  a,b in [-h,h],
//   d_a = (i_u - N/2 + a) - x_u,  g(t) = I0(beta sqrt(1-(2t/S)^2)) / I0(beta)
//
// Design (B200): the visibilities arrive sorted by (image, plane, uv tile of B x B cells, cell
// inside the tile) -- DESIGN.md step 4.  Each WARP takes fixed-size chunks of the sorted order from
// a dynamic counter (perfect balance in visibilities, whatever the skew of the uv coverage) and
// owns a PRIVATE shared-memory accumulation tile of (B+S-1)^2 cells -- the tile plus the kernel
// halo, the single-GPU analogue of the paper's ghost region.  Per batch of 32 visibilities every
// lane evaluates the 2S kernel values of its own visibility and stages them in shared memory
// (the u-axis values already multiplied by w V); then the warp walks the batch run by run.
//   * Run accumulation: consecutive visibilities of the SAME centre cell (reading R22; 5.5 per run in
//     config 2) share one footprint, and their sum is sum_k g_v(k) (x) [g_u(k) wV_re(k), g_u(k) wV_im(k)]:
//     an (S x K)(K x 2S) product over the K visibilities of the run.  The warp accumulates it as rank-4
//     updates with the fp64 mma.sync m8n8k4 (fragment rows = footprint rows, fragment columns =
//     (footprint column, re | im): a lane's two accumulators are the (re, im) of one cell).  The
//     accumulators are loaded from the tile when a run starts and stored back when it ends: the
//     shared-memory tile is read-modified-written once per run, not once per visibility.
//   * When the tile changes, the tile is flushed to HBM with fire-and-forget RED atomics
//     (non-zero cells only, scanned linearly with four cells per lane in flight) and re-zeroed.
//
// Kernel values.  d_a = (a-h) - delta with delta = x_u - (i_u - N/2) in [-1/2, 1/2): tap a sees g
// only on one unit interval, where it is a degree-KB_DEG polynomial f_a(s), s = 2 delta, to < 2e-16
// (tables.cu fits and checks it at plan time).  g is even, so the mirror tap is f_{S-1-a}(s) =
// f_a(-s): with f_a = E(s^2) + s O(s^2) one even and one odd Horner chain give BOTH taps, and the
// centre tap has O = 0 -- (S-1)/2 (KB_DEG+1) + KB_DEG/2 DFMA per axis instead of S KB_DEG.  The
// coefficients travel as kernel parameters, so every Horner step is one DFMA with a constant-bank
// operand and no load.
//
// The tile row pitch is odd (and > B+S-1, the pad column takes the zero-weight partner of the last
// cell of a footprint row), so the lanes of a quarter warp hit distinct 16-byte bank groups.
#include "common.cuh"

struct GridParams {
    const void* vis;
    const float* wgt;
    const double* uvw;
    const double* chan_scale;
    const unsigned long long* sitems;    // sorted items (key << idx_bits) | k
    const long long* plane_start;
    int idx_bits;
    int plane_first, n_planes;
    void* stack;
    int N, h, B, log2B, T, TWp, TH, C;
    int vis_c128;
    int fold;                            // RICK_FLAG_FOLD_W: rows with w < 0 are gridded at (-u, -v) with conj V (R24)
    double inv_du;
    unsigned int* chunk_counter;
};
template <int S> struct GridParamsS {
    GridParams g;
    double poly[(S + 1) / 2][RICK_KB_DEG + 1];     // poly[a][k]: coefficient of s^k of tap a <= h
};

#define GRID_WARPS 8
#define GRID_CHUNK 512

__host__ __device__ inline int grid_pitch(int B, int S)
{
    int tw = B + S;                      // one pad column
    if ((tw & 1) == 0) ++tw;
    return tw;
}

template <typename GT> struct cell_t;
template <> struct cell_t<double> { typedef double2 type; };
template <> struct cell_t<float> { typedef float2 type; };

__device__ __forceinline__ void red_add(double2* a, double2 v)
{
    atomicAdd(&a->x, v.x);
    atomicAdd(&a->y, v.y);
}
__device__ __forceinline__ void red_add(float2* a, float2 v) { atomicAdd(a, v); }

__global__ void k_chunk_reset(unsigned int* c) { *c = 0u; }

// shared-window (32-bit) addressing of the walk
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ double2 lds_d2(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_d(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
// D (8 x 8) += A (8 x 4, row) B (4 x 8, col) in fp64: lane l holds A[l>>2][l&3], B[l&3][l>>2],
// D[l>>2][2(l&3)], D[l>>2][2(l&3)+1]
__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
// one tile cell <-> the (re, im) register pair of an accumulator fragment
template <typename GT> __device__ __forceinline__ void tile_load(uint32_t a, double (&c)[2]);
template <typename GT> __device__ __forceinline__ void tile_store(uint32_t a, const double (&c)[2]);
template <> __device__ __forceinline__ void tile_load<double>(uint32_t a, double (&c)[2])
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(c[0]), "=d"(c[1]) : "r"(a));
}
template <> __device__ __forceinline__ void tile_store<double>(uint32_t a, const double (&c)[2])
{
    asm volatile("st.shared.v2.f64 [%2], {%0, %1};" :: "d"(c[0]), "d"(c[1]), "r"(a) : "memory");
}
template <> __device__ __forceinline__ void tile_load<float>(uint32_t a, double (&c)[2])
{
    float t0, t1;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(t0), "=f"(t1) : "r"(a));
    c[0] = (double)t0;
    c[1] = (double)t1;
}
template <> __device__ __forceinline__ void tile_store<float>(uint32_t a, const double (&c)[2])
{
    const float t0 = (float)c[0], t1 = (float)c[1];
    asm volatile("st.shared.v2.f32 [%2], {%0, %1};" :: "f"(t0), "f"(t1), "r"(a) : "memory");
}

#define GRID_KS 36      // staging row stride in visibilities (32 + the overhang of the last group of 4)

template <int S> __host__ __device__ constexpr size_t grid_stage_bytes()
{
    // kb[2S][KS] double | ka[S][KS] double | run[34] uint2
    return (size_t)2 * S * GRID_KS * 8 + (size_t)S * GRID_KS * 8 + 34 * 8;
}

template <typename GT, int S>
__global__ void __launch_bounds__(GRID_WARPS * 32, 2) k_grid(const __grid_constant__ GridParamsS<S> PS)
{
    typedef typename cell_t<GT>::type cell;
    typedef unsigned long long u64;
    constexpr int H = (S - 1) / 2;
    constexpr int MT = (S + 7) / 8;                 // 8-row fragments of the footprint
    constexpr int NT = (2 * S + 7) / 8;             // 8-column fragments: columns are (cell a, re | im)
    constexpr int KS = GRID_KS;
    constexpr int DEG = RICK_KB_DEG;
    static_assert(DEG % 2 == 0, "even/odd Horner split assumes an even degree");
    const GridParams& P = PS.g;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int TWp = P.TWp, TH = P.TH, N = P.N, h = P.h, B = P.B, T = P.T, log2B = P.log2B;
    const int tile_cells = TH * TWp;
    const int sub_bits = 2 * log2B, idx_bits = P.idx_bits;
    const u64 idx_mask = (1ull << idx_bits) - 1ull;

    // shared layout per warp: tile | kb[2S][KS] | ka[S][KS] | run[34]
    const size_t tile_bytes = ((size_t)tile_cells * sizeof(cell) + 15) & ~(size_t)15;
    const size_t per_warp = tile_bytes + grid_stage_bytes<S>();
    unsigned char* wbase = smem_raw + (size_t)warp * per_warp;
    cell* tile = reinterpret_cast<cell*>(wbase);
    double* s_kb = reinterpret_cast<double*>(wbase + tile_bytes);      // [2 a + c][k] = g_u[a] (w V)_c of visibility k
    double* s_ka = s_kb + 2 * S * KS;                                  // [b][k] = g_v[b] of visibility k
    uint2* s_run = reinterpret_cast<uint2*>(s_ka + S * KS);

    cell zero;
    zero.x = 0;
    zero.y = 0;
    for (int i = lane; i < tile_cells; i += 32) tile[i] = zero;
    for (int i = lane; i < 3 * S * KS; i += 32) s_kb[i] = 0.0;      // kb and ka
    __syncwarp();

    // Fragment roles (DMMA m8n8k4; M = footprint row b, N = (footprint column a, re | im), K = visibility):
    // lane = 4 g + q feeds A[g][q] = g_v[b = g + 8 mt] of visibility jj + q and B[q][g] = g_u[a] (w V)_c,
    // 2 a + c = g + 8 nt, of the same visibility; its two accumulators of fragment (mt, nt) are the (re, im)
    // of footprint cell (b = g + 8 mt, a = 4 nt + q) -- the register pair a 16-byte tile access moves.
    const int g = lane >> 2, q = lane & 3;
    bool has[MT][NT], row_ok[MT], col_ok[NT];
    uint32_t a_tile[MT][NT], a_ka[MT], a_kb[NT];
    double c[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        row_ok[mt] = g + 8 * mt < S;
        a_ka[mt] = smem_u32(s_ka + (row_ok[mt] ? g + 8 * mt : 0) * KS + q);
    }
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        col_ok[nt] = g + 8 * nt < 2 * S;
        a_kb[nt] = smem_u32(s_kb + (col_ok[nt] ? g + 8 * nt : 0) * KS + q);
    }
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            has[mt][nt] = row_ok[mt] && (4 * nt + q < S);
            a_tile[mt][nt] = smem_u32(tile + (has[mt][nt] ? (g + 8 * mt) * TWp + 4 * nt + q : 0));
            c[mt][nt][0] = c[mt][nt][1] = 0.0;
        }
    const uint32_t a_run = smem_u32(s_run);

    const long long v_begin = P.plane_start[P.plane_first];
    const long long v_end = P.plane_start[P.plane_first + P.n_planes];
    const long long n_chunks = (v_end - v_begin + GRID_CHUNK - 1) / GRID_CHUNK;
    const unsigned int TT = (unsigned)T * (unsigned)T;
    const double shift = (double)(N / 2) + 0.5;
    const unsigned int C = (unsigned)P.C;

    const u64 NOKEY = ~0ull;
    u64 last_key = NOKEY;          // key of the visibility before this batch (NOKEY: nothing pending)
    u64 cur_tile = 0;              // (image, plane, tile) of the run held in the accumulators
    uint32_t cur_off = 0;          // byte offset of its top-left footprint cell inside the tile
    bool have_run = false;

    // accumulators <-> tile: a run starts FROM the tile's cells and is stored back when it ends
    auto run_load = [&]() {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
                if (has[mt][nt]) tile_load<GT>(a_tile[mt][nt] + cur_off, c[mt][nt]);
    };
    auto run_store = [&]() {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
                if (has[mt][nt]) tile_store<GT>(a_tile[mt][nt] + cur_off, c[mt][nt]);
    };
    // tile -> HBM, once per (tile, chunk): the TH x TH cells scanned linearly, four cells per lane in flight
    const float inv_TH = 1.0f / (float)TH;
    const int n_cells = TH * TH;
    auto flush_tile = [&](u64 tkey) {
        __syncwarp();
        const unsigned int pz = (unsigned int)(tkey / TT), rem = (unsigned int)(tkey - (u64)pz * TT);
        const int tv = (int)(rem / (unsigned)T), tu = (int)(rem - (unsigned)tv * (unsigned)T);
        cell* plane = reinterpret_cast<cell*>(P.stack) + (size_t)(pz - (unsigned)P.plane_first) * N * N;
        const long long g0 = (long long)(tv * B - h) * N + (tu * B - h);     // may be < 0 on the grid edge
        for (int i0 = lane; i0 < n_cells; i0 += 128) {
            cell v[4];
            int t[4];
            long long gofs[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = i0 + 32 * u;
                const int row = __float2int_rd(((float)i + 0.5f) * inv_TH), col = i - row * TH;   // exact: i < 2^11
                t[u] = row * TWp + col;
                gofs[u] = g0 + (long long)row * N + col;
                v[u] = zero;
                if (i < n_cells) v[u] = tile[t[u]];
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (v[u].x != 0 || v[u].y != 0) {
                    red_add(plane + gofs[u], v[u]);
                    tile[t[u]] = zero;
                }
        }
        __syncwarp();
    };

    // inputs of one visibility, loaded one batch ahead of their use
    struct VisIn {
        u64 key;
        double um, vm, wm, s, vr, vi;  // vr, vi: raw value as loaded (complex128), else see raw
        float2 raw;                    // complex64 as loaded
        float om;                      // weight as loaded
    };
    auto load_item = [&](long long ks, long long c_end) -> u64 { return ks < c_end ? P.sitems[ks] : NOKEY; };
    // loads only: nothing here depends on a loaded value, so the whole batch of loads stays in flight
    // while the previous batch is accumulated (conversions and the weight product happen in finish_vis)
    auto load_vis = [&](u64 item, VisIn& in) {
        in.key = NOKEY;
        if (item == NOKEY) return;
        in.key = item >> idx_bits;
        const unsigned int idx = (unsigned int)(item & idx_mask);
        const unsigned int r = idx / C, c = idx - r * C;
        in.s = P.chan_scale[c];
        in.um = P.uvw[3ull * r + 0];
        in.vm = P.uvw[3ull * r + 1];
        in.wm = P.fold ? P.uvw[3ull * r + 2] : 0.0;
        if (P.vis_c128) {
            const double2 v = reinterpret_cast<const double2*>(P.vis)[idx];
            in.vr = v.x;
            in.vi = v.y;
        } else {
            in.raw = reinterpret_cast<const float2*>(P.vis)[idx];
        }
        in.om = 1.0f;
        if (P.wgt) in.om = P.wgt[idx];
    };
    auto finish_vis = [&](VisIn& in) {
        if (!P.vis_c128) {
            in.vr = (double)in.raw.x;
            in.vi = (double)in.raw.y;
        }
        if (in.wm < 0.0) {              // folded row (R24): (u, v) -> (-u, -v), V -> conj V
            in.um = -in.um;
            in.vm = -in.vm;
            in.vi = -in.vi;
        }
        if (P.wgt) {
            const double om = (double)in.om;
            in.vr *= om;
            in.vi *= om;
        }
    };

    long long chunk = 0;
    if (lane == 0) chunk = (long long)atomicAdd(P.chunk_counter, 1u);
    chunk = __shfl_sync(0xffffffffu, chunk, 0);
    while (chunk < n_chunks) {
        long long next_chunk = 0;
        if (lane == 0) next_chunk = (long long)atomicAdd(P.chunk_counter, 1u);      // in flight during this chunk
        const long long c_begin = v_begin + chunk * GRID_CHUNK;
        const long long c_end = (c_begin + GRID_CHUNK < v_end) ? c_begin + GRID_CHUNK : v_end;

        VisIn cur;
        load_vis(load_item(c_begin + lane, c_end), cur);
        u64 item_next = load_item(c_begin + 32 + lane, c_end);
        for (long long b0 = c_begin; b0 < c_end; b0 += 32) {
            // ---- stage this batch: kernel values of the lane's own visibility, run descriptors ----
            const int nb = (int)((c_end - b0) < 32 ? (c_end - b0) : 32);
            const u64 key = cur.key;
            const bool valid = key != NOKEY;
            // a run starts where the key differs from the previous visibility's; a tile where its
            // (image, plane, tile) part does
            u64 prev = __shfl_up_sync(0xffffffffu, key, 1);
            if (lane == 0) prev = last_key;
            const unsigned int run_mask = __ballot_sync(0xffffffffu, valid && key != prev);
            const unsigned int tile_mask = __ballot_sync(0xffffffffu, valid && (key >> sub_bits) != (prev >> sub_bits));
            last_key = __shfl_sync(0xffffffffu, key, 31);      // NOKEY after a short (= last) batch
            // descriptor r: x = first visibility | count << 8 | new tile << 16 | continuation << 17, y = byte
            // offset of the footprint in the tile.  A batch that opens inside a run gets a continuation first.
            const unsigned int cont = (run_mask & 1u) ? 0u : 1u;
            const int n_runs = __popc(run_mask) + (int)cont;
            if (valid && (((run_mask >> lane) & 1u) || lane == 0)) {
                const unsigned int above = lane < 31 ? (run_mask >> (lane + 1)) : 0u;
                int end = above ? lane + __ffs(above) : nb;
                end = end < nb ? end : nb;
                const int sub = (int)(key & ((1ull << sub_bits) - 1ull));
                const unsigned int r = (unsigned)__popc(run_mask & ((1u << lane) - 1u)) + (((run_mask >> lane) & 1u) ? cont : 0u);
                uint2 d;
                d.x = (unsigned)lane | ((unsigned)(end - lane) << 8) | (((tile_mask >> lane) & 1u) << 16) |
                      ((((run_mask >> lane) & 1u) ^ 1u) << 17);
                d.y = (uint32_t)(((sub >> log2B) * TWp + (sub & (B - 1))) * (int)sizeof(cell));
                s_run[r] = d;
            }
            if (valid) {
                finish_vis(cur);
                const double xu = __dmul_rn(__dmul_rn(cur.um, cur.s), P.inv_du);
                const double xv = __dmul_rn(__dmul_rn(cur.vm, cur.s), P.inv_du);
                const int iu = (int)floor(__dadd_rn(xu, shift));
                const int iv = (int)floor(__dadd_rn(xv, shift));
                // tap a at d_a = (a-h) - s/2, s = 2 (x - (i - N/2)); mirror taps share E, O
                const double su = 2.0 * (xu - (double)(iu - N / 2));
                const double sv = 2.0 * (xv - (double)(iv - N / 2));
                const double su2 = su * su, sv2 = sv * sv;
                double fu[S], fv[S];
#pragma unroll
                for (int a = 0; a <= H; ++a) {
                    double eu = PS.poly[a][DEG], ev = PS.poly[a][DEG];
                    double ou = PS.poly[a][DEG - 1], ov = PS.poly[a][DEG - 1];
#pragma unroll
                    for (int k = DEG - 2; k >= 0; k -= 2) {
                        eu = fma(eu, su2, PS.poly[a][k]);
                        ev = fma(ev, sv2, PS.poly[a][k]);
                        if (k >= 2 && a < H) {
                            ou = fma(ou, su2, PS.poly[a][k - 1]);
                            ov = fma(ov, sv2, PS.poly[a][k - 1]);
                        }
                    }
                    if (a < H) {
                        fu[a] = fma(su, ou, eu);
                        fu[S - 1 - a] = fma(-su, ou, eu);
                        fv[a] = fma(sv, ov, ev);
                        fv[S - 1 - a] = fma(-sv, ov, ev);
                    } else {
                        fu[a] = eu;
                        fv[a] = ev;
                    }
                }
#pragma unroll
                for (int a = 0; a < S; ++a) {
                    s_ka[a * KS + lane] = fv[a];
                    s_kb[(2 * a) * KS + lane] = cur.vr * fu[a];
                    s_kb[(2 * a + 1) * KS + lane] = cur.vi * fu[a];
                }
            }
            __syncwarp();
            // ---- next batch's inputs: in flight while this batch is accumulated ----
            load_vis(item_next, cur);
            item_next = load_item(b0 + 64 + lane, c_end);

            // ---- walk the batch run by run: rank-4 updates of the footprint on the fp64 tensor pipe ----
            uint2 d = lds_u2(a_run);
            for (int r = 0; r < n_runs; ++r) {
                const uint2 dn = lds_u2(a_run + 8u * (uint32_t)(r + 1));      // next descriptor (slot 33 exists)
                const int j = (int)(d.x & 255u), end = j + (int)((d.x >> 8) & 255u);
                if (!((d.x >> 17) & 1u)) {
                    const bool new_tile = (d.x >> 16) & 1u;
                    if (have_run) {
                        run_store();
                        if (new_tile) flush_tile(cur_tile);
                    }
                    have_run = true;
                    cur_off = d.y;
                    if (new_tile) cur_tile = __shfl_sync(0xffffffffu, key, j) >> sub_bits;
                    run_load();
                }
                for (int jj = j; jj < end; jj += 4) {
                    const bool live = jj + q < end;
                    double av[MT], bv[NT];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        av[mt] = 0.0;
                        if (live && row_ok[mt]) av[mt] = lds_d(a_ka[mt] + (uint32_t)jj * 8u);
                    }
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        bv[nt] = 0.0;
                        if (live && col_ok[nt]) bv[nt] = lds_d(a_kb[nt] + (uint32_t)jj * 8u);
                    }
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) dmma884(c[mt][nt], av[mt], bv[nt]);
                }
                d = dn;
            }
            __syncwarp();
        }
        if (have_run) {
            run_store();
            flush_tile(cur_tile);
            have_run = false;
        }
        last_key = NOKEY;
        chunk = __shfl_sync(0xffffffffu, next_chunk, 0);
    }
}

// Zero-fill.  The gridder accumulates with atomics into a stack that must start from zero, but only
// rows that were written since they were last cleared can be non-zero: the plan keeps one "dirty" byte
// per (resident slot, row) and this kernel clears exactly those rows.
// A small persistent grid walks the (slot, row) pairs -- a clean row costs one byte read -- so the
// kernel, which runs on the low-priority side stream, never floods the block scheduler in front of
// the index / sort kernels of the main stream.  16-byte stores; a row is N * E bytes.
__global__ void __launch_bounds__(256) k_zero_dirty_rows(uint4* __restrict__ stack, unsigned char* __restrict__ dirty,
                                                         size_t n_rows, size_t row16)
{
    const uint4 z = make_uint4(0, 0, 0, 0);
    for (size_t r = blockIdx.x; r < n_rows; r += gridDim.x) {      // slot-major row index
        const bool d = dirty[r] != 0;
        __syncthreads();                          // every thread has read the flag before it is cleared
        if (!d) continue;
        uint4* dst = stack + r * row16;
        for (size_t i = threadIdx.x; i < row16; i += 256) dst[i] = z;
        if (threadIdx.x == 0) dirty[r] = 0;      // only this CTA ever looks at row r
    }
}

// Zero-fill of rick_image ("known-zero tiles").  One warp per (slot, row) of the resident batch:
//   dirty, not occupied now  -> the row holds stale data the column pass would read: cleared whole;
//   dirty and occupied now   -> the row pass reads only the tiles some footprint reaches (tile_occ) and
//                               overwrites the whole row, so only those tiles are cleared for the gridder;
//   not dirty                -> already zero.
// unit16 = 16-byte units per tile row (B * E / 16), row16 = units per row.
__global__ void __launch_bounds__(256) k_zero_sparse(uint4* __restrict__ stack, unsigned char* __restrict__ dirty,
                                                     const unsigned char* __restrict__ occ,
                                                     const unsigned char* __restrict__ tocc, size_t n_rows, int N,
                                                     int log2B, int T, size_t row16, int unit16, int keep_stale)
{
    const uint4 z = make_uint4(0, 0, 0, 0);
    const int lane = threadIdx.x & 31;
    const size_t warp = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const size_t n_warps = ((size_t)gridDim.x * blockDim.x) >> 5;
    for (size_t r = warp; r < n_rows; r += n_warps) {            // slot-major row index
        if (!dirty[r]) continue;
        uint4* dst = stack + r * row16;
        if (!occ[r]) {
            if (keep_stale) continue;      // nobody reads this row before it is written again; it stays dirty
            for (size_t i = lane; i < row16; i += 32) dst[i] = z;
            __syncwarp();
            if (lane == 0) dirty[r] = 0;
            continue;
        }
        const size_t slot = r / (size_t)N;
        const int row = (int)(r - slot * (size_t)N);
        const unsigned char* to = tocc + (slot * (size_t)T + (size_t)(row >> log2B)) * (size_t)T;
        for (int t0 = 0; t0 < T; t0 += 32) {
            const int ti = t0 + lane;
            unsigned int m = __ballot_sync(0xffffffffu, ti < T && to[ti] != 0);
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                uint4* d = dst + (size_t)(t0 + b) * unit16;
                for (int i = lane; i < unit16; i += 32) d[i] = z;
            }
        }
    }
}

__global__ void __launch_bounds__(256) k_mark_dirty(unsigned char* __restrict__ dirty, const unsigned char* __restrict__ occ,
                                                    size_t n)
{
    const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (i < n && occ[i]) dirty[i] = 1;
}

int rick_zero_dirty(rick_plan_t* p, int n_slots, cudaStream_t st)
{
    const size_t row16 = p->plane_bytes / 16 / (size_t)p->N;
    RICK_KERNEL_ON(p, st, RK_ZERO, k_zero_dirty_rows<<<p->n_sm * 4, 256, 0, st>>>(
        reinterpret_cast<uint4*>(p->stack), p->row_dirty, (size_t)n_slots * p->N, row16));
    return RICK_OK;
}

// slots 0..n_slots-1 are about to receive global planes plane_first.. (occupancy of the current sort)
int rick_zero_sparse(rick_plan_t* p, int plane_first, int n_slots, int keep_stale)
{
    const size_t cell = p->f32 ? 8 : 16;
    const size_t row16 = p->plane_bytes / 16 / (size_t)p->N;
    const int unit16 = (int)((size_t)p->B * cell / 16);
    RICK_KERNEL(p, RK_ZERO, k_zero_sparse<<<p->n_sm * 8, 256, 0, p->stream>>>(
        reinterpret_cast<uint4*>(p->stack), p->row_dirty, p->row_occ + (size_t)plane_first * p->N,
        p->tile_occ + (size_t)plane_first * p->T * p->T, (size_t)n_slots * p->N, p->N, p->log2B, p->T, row16, unit16, keep_stale));
    return RICK_OK;
}

// rows of the batch [plane_first, plane_first + n_planes) that the gridder / row pass will write
int rick_mark_dirty(rick_plan_t* p, int plane_first, int n_planes)
{
    const size_t n = (size_t)n_planes * p->N;
    RICK_KERNEL(p, RK_ROW_OCC, k_mark_dirty<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>(
        p->row_dirty, p->row_occ + (size_t)plane_first * p->N, n));
    return RICK_OK;
}

// an in-place column pass writes every row of the slots it transformed
int rick_all_dirty(rick_plan_t* p, int n_slots)
{
    RICK_CUDA(p, cudaMemsetAsync(p->row_dirty, 1, (size_t)n_slots * p->N, p->stream));
    return RICK_OK;
}

template <typename GT, int S>
static int launch_grid(rick_plan_t* p, const GridParams& P)
{
    typedef typename cell_t<GT>::type cell;
    GridParamsS<S> PS;
    PS.g = P;
    for (int a = 0; a < (S + 1) / 2; ++a)
        for (int k = 0; k <= RICK_KB_DEG; ++k) PS.poly[a][k] = p->kb_poly[a * (RICK_KB_DEG + 1) + k];
    const size_t tile_bytes = ((size_t)P.TH * P.TWp * sizeof(cell) + 15) & ~(size_t)15;
    const size_t per_warp = tile_bytes + grid_stage_bytes<S>();
    int warps = GRID_WARPS;                     // fewer warps per CTA when the tile is large
    while (warps > 1 && warps * per_warp > 227 * 1024) warps >>= 1;
    const size_t smem = warps * per_warp;
    if (smem > 227 * 1024) {
        p->err = "tile/support too large for the gridder's shared memory";
        return RICK_ERR_INVALID;
    }
    RICK_CUDA(p, cudaFuncSetAttribute(k_grid<GT, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    RICK_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_grid<GT, S>, warps * 32, smem));
    if (per_sm < 1) per_sm = 1;
    RICK_KERNEL(p, RK_RESET, k_chunk_reset<<<1, 1, 0, p->stream>>>(P.chunk_counter));
    RICK_KERNEL(p, RK_GRID, k_grid<GT, S><<<p->n_sm * per_sm, warps * 32, smem, p->stream>>>(PS));
    return RICK_OK;
}

template <typename GT>
static int launch_grid_s(rick_plan_t* p, const GridParams& P)
{
    switch (p->S) {
        case 3: return launch_grid<GT, 3>(p, P);
        case 5: return launch_grid<GT, 5>(p, P);
        case 7: return launch_grid<GT, 7>(p, P);
        case 9: return launch_grid<GT, 9>(p, P);
        case 11: return launch_grid<GT, 11>(p, P);
        case 13: return launch_grid<GT, 13>(p, P);
        case 15: return launch_grid<GT, 15>(p, P);
    }
    p->err = "unsupported support";
    return RICK_ERR_INVALID;
}

int rick_grid_planes(rick_plan_t* p, const void* vis, int vis_dtype, const double* uvw_m,
                     const float* weights, int plane_first, int n_planes)
{
    GridParams P;
    P.vis = vis;
    P.wgt = weights;
    P.uvw = uvw_m;
    P.chan_scale = p->chan_scale;
    P.sitems = p->sorted_items;
    P.idx_bits = p->idx_bits;
    P.plane_start = (const long long*)p->plane_start;
    P.plane_first = plane_first;
    P.n_planes = n_planes;
    P.stack = p->stack;
    P.N = p->N;
    P.h = p->h;
    P.B = p->B;
    P.log2B = p->log2B;
    P.T = p->T;
    P.TH = p->B + p->S - 1;
    P.TWp = grid_pitch(p->B, p->S);
    P.C = p->C;
    P.vis_c128 = vis_dtype == RICK_VIS_C128;
    P.fold = p->fold;
    P.inv_du = p->inv_du;
    P.chunk_counter = &p->counters->grid_chunk;
    if (p->M == 0) return RICK_OK;
    return p->f32 ? launch_grid_s<float>(p, P) : launch_grid_s<double>(p, P);
}
