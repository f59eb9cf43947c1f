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
// (the v-axis values already multiplied by w V); then the warp walks the 32 visibilities one by one
// with its lanes spread over the footprint, each lane owning two horizontally adjacent cells.
//   * Run accumulation: consecutive visibilities of the SAME centre cell have the same footprint,
//     so their contributions are summed in REGISTERS (4 DFMA per lane per visibility, operands by
//     two broadcast LDS.128); the shared-memory tile is read-modified-written once per run, when
//     the centre cell changes (core-dense uv coverage: 5.5 visibilities per run in config 2).
//     Before, every visibility paid the 2 x 49-cell RMW and the gridder ran at the shared-memory
//     bandwidth.
//   * When the tile changes, the tile is flushed to HBM with fire-and-forget RED atomics
//     (non-zero cells only) and re-zeroed.
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

template <int S> __host__ __device__ constexpr size_t grid_stage_bytes()
{
    // ku[32][SP] doubles | kw[32][S] double2 | key[32] u64
    return (size_t)32 * (2 * ((S + 1) / 2)) * 8 + (size_t)32 * S * 16 + 32 * 8;
}

template <typename GT, int S>
__global__ void __launch_bounds__(GRID_WARPS * 32) k_grid(const __grid_constant__ GridParamsS<S> PS)
{
    typedef typename cell_t<GT>::type cell;
    typedef unsigned long long u64;
    constexpr int H = (S - 1) / 2;
    constexpr int PW = (S + 1) / 2;                 // cell pairs per footprint row
    constexpr int SP = 2 * PW;                      // padded footprint width (even)
    constexpr int NPAIR = S * PW, ROUNDS = (NPAIR + 31) / 32;
    constexpr int DEG = RICK_KB_DEG;
    static_assert(DEG % 2 == 0, "even/odd Horner split assumes an even degree");
    const GridParams& P = PS.g;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int TWp = P.TWp, TH = P.TH, N = P.N, h = P.h, B = P.B, T = P.T, log2B = P.log2B;
    const int tile_cells = TH * TWp;
    const int sub_bits = 2 * log2B, idx_bits = P.idx_bits;
    const u64 idx_mask = (1ull << idx_bits) - 1ull;

    // shared layout per warp: tile | ku[32][SP] | kw[32][S] | key[32]
    const size_t tile_bytes = ((size_t)tile_cells * sizeof(cell) + 15) & ~(size_t)15;
    const size_t per_warp = tile_bytes + grid_stage_bytes<S>();
    unsigned char* wbase = smem_raw + (size_t)warp * per_warp;
    cell* tile = reinterpret_cast<cell*>(wbase);
    double* s_ku = reinterpret_cast<double*>(wbase + tile_bytes);
    double2* s_kw = reinterpret_cast<double2*>(s_ku + 32 * SP);
    u64* s_key = reinterpret_cast<u64*>(s_kw + 32 * S);

    cell zero;
    zero.x = 0;
    zero.y = 0;
    for (int i = lane; i < tile_cells; i += 32) tile[i] = zero;
    for (int i = lane; i < 32 * SP; i += 32) s_ku[i] = 0.0;      // also the zero weight of the pad column
    __syncwarp();

    // cell pair(s) of this lane: pair = lane + 32*rr -> row b, cells (b, 2 a2), (b, 2 a2 + 1).
    // Lanes without a pair read valid staging addresses (pair 0) and are masked at the flush only,
    // so the accumulation loop has no per-lane branch.
    int foff[ROUNDS];
    bool has[ROUNDS];
    const double2* pku[ROUNDS];
    const double2* pkw[ROUNDS];
    double acc[ROUNDS][4];
#pragma unroll
    for (int rr = 0; rr < ROUNDS; ++rr) {
        const int pi = lane + 32 * rr;
        has[rr] = pi < NPAIR;
        const int b = has[rr] ? pi / PW : 0;
        const int a2 = has[rr] ? 2 * (pi - b * PW) : 0;
        foff[rr] = b * TWp + a2;
        pku[rr] = reinterpret_cast<const double2*>(s_ku + a2);
        pkw[rr] = s_kw + b;
        acc[rr][0] = acc[rr][1] = acc[rr][2] = acc[rr][3] = 0.0;
    }

    const long long v_begin = P.plane_start[P.plane_first];
    const long long v_end = P.plane_start[P.plane_first + P.n_planes];
    const long long n_chunks = (v_end - v_begin + GRID_CHUNK - 1) / GRID_CHUNK;
    const unsigned int TT = (unsigned)T * (unsigned)T;
    const double shift = (double)(N / 2) + 0.5;
    const unsigned int C = (unsigned)P.C;

    const u64 NOKEY = ~0ull;
    u64 cur_cell = NOKEY;          // key of the run being summed in registers
    int cur_base = 0;              // its top-left footprint cell, local to the tile

    // registers -> tile, once per run
    auto flush_run = [&]() {
#pragma unroll
        for (int rr = 0; rr < ROUNDS; ++rr) {
            if (has[rr]) {
                cell* tp = tile + cur_base + foff[rr];
                cell t0 = tp[0], t1 = tp[1];
                t0.x += (GT)acc[rr][0];
                t0.y += (GT)acc[rr][1];
                t1.x += (GT)acc[rr][2];
                t1.y += (GT)acc[rr][3];
                tp[0] = t0;
                tp[1] = t1;
            }
            acc[rr][0] = acc[rr][1] = acc[rr][2] = acc[rr][3] = 0.0;
        }
    };
    // tile -> HBM, once per (tile, chunk)
    auto flush_tile = [&](u64 tkey) {
        __syncwarp();
        const unsigned int pz = (unsigned int)(tkey / TT), rem = (unsigned int)(tkey - (u64)pz * TT);
        const int tv = (int)(rem / (unsigned)T), tu = (int)(rem - (unsigned)tv * (unsigned)T);
        cell* plane = reinterpret_cast<cell*>(P.stack) + (size_t)(pz - (unsigned)P.plane_first) * N * N;
        for (int row = 0; row < TH; ++row) {
            for (int col = lane; col < TH; col += 32) {
                cell v = tile[row * TWp + col];
                if (v.x != 0 || v.y != 0) {
                    const int gv = tv * B - h + row, gu = tu * B - h + col;
                    red_add(plane + ((size_t)gv * N + gu), v);
                    tile[row * TWp + col] = zero;
                }
            }
        }
        __syncwarp();
    };

    // inputs of one visibility, loaded one batch ahead of their use
    struct VisIn {
        u64 key;
        double um, vm, s, vr, vi;
    };
    auto load_item = [&](long long ks, long long c_end) -> u64 { return ks < c_end ? P.sitems[ks] : NOKEY; };
    auto load_vis = [&](u64 item, VisIn& in) {
        in.key = NOKEY;
        if (item == NOKEY) return;
        in.key = item >> idx_bits;
        const unsigned int idx = (unsigned int)(item & idx_mask);
        const unsigned int r = idx / C, c = idx - r * C;
        in.s = P.chan_scale[c];
        in.um = P.uvw[3ull * r + 0];
        in.vm = P.uvw[3ull * r + 1];
        if (P.vis_c128) {
            const double2 v = reinterpret_cast<const double2*>(P.vis)[idx];
            in.vr = v.x;
            in.vi = v.y;
        } else {
            const float2 v = reinterpret_cast<const float2*>(P.vis)[idx];
            in.vr = (double)v.x;
            in.vi = (double)v.y;
        }
        if (P.wgt) {
            const double om = (double)P.wgt[idx];
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
            // ---- stage this batch: kernel values of the lane's own visibility ----
            const bool valid = cur.key != NOKEY;
            // a run starts where the key differs from the previous visibility's (lane 0: from the run in registers)
            u64 prev = __shfl_up_sync(0xffffffffu, cur.key, 1);
            if (lane == 0) prev = cur_cell;
            const unsigned int run_mask = __ballot_sync(0xffffffffu, valid && cur.key != prev);
            if (valid) {
                s_key[lane] = cur.key;
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
                    s_ku[lane * SP + a] = fu[a];
                    s_kw[lane * S + a] = make_double2(cur.vr * fv[a], cur.vi * fv[a]);
                }
            }
            __syncwarp();
            // ---- next batch's inputs: in flight while this batch is accumulated ----
            load_vis(item_next, cur);
            item_next = load_item(b0 + 64 + lane, c_end);

            // ---- walk the batch run by run (run_mask is warp-uniform) ----
            const int nb = (int)((c_end - b0) < 32 ? (c_end - b0) : 32);
            int j = 0;
            while (j < nb) {
                if ((run_mask >> j) & 1u) {
                    const u64 kj = s_key[j];
                    if (cur_cell != NOKEY) {
                        flush_run();
                        if ((kj >> sub_bits) != (cur_cell >> sub_bits)) flush_tile(cur_cell >> sub_bits);
                    }
                    cur_cell = kj;
                    const int sub = (int)(kj & ((1ull << sub_bits) - 1ull));
                    cur_base = (sub >> log2B) * TWp + (sub & (B - 1));
                }
                const unsigned int rest = j < 31 ? (run_mask >> (j + 1)) : 0u;
                int end = rest ? j + __ffs(rest) : nb;
                end = end < nb ? end : nb;
#pragma unroll 4
                for (int jj = j; jj < end; ++jj) {
#pragma unroll
                    for (int rr = 0; rr < ROUNDS; ++rr) {
                        const double2 k2 = pku[rr][jj * PW];
                        const double2 w2 = pkw[rr][jj * S];
                        acc[rr][0] = fma(w2.x, k2.x, acc[rr][0]);
                        acc[rr][1] = fma(w2.y, k2.x, acc[rr][1]);
                        acc[rr][2] = fma(w2.x, k2.y, acc[rr][2]);
                        acc[rr][3] = fma(w2.y, k2.y, acc[rr][3]);
                    }
                }
                j = end;
            }
            __syncwarp();
        }
        if (cur_cell != NOKEY) {
            flush_run();
            flush_tile(cur_cell >> sub_bits);
            cur_cell = NOKEY;
        }
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
                                                     int log2B, int T, size_t row16, int unit16)
{
    const uint4 z = make_uint4(0, 0, 0, 0);
    const int lane = threadIdx.x & 31;
    const size_t warp = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const size_t n_warps = ((size_t)gridDim.x * blockDim.x) >> 5;
    for (size_t r = warp; r < n_rows; r += n_warps) {            // slot-major row index
        if (!dirty[r]) continue;
        uint4* dst = stack + r * row16;
        if (!occ[r]) {
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
int rick_zero_sparse(rick_plan_t* p, int plane_first, int n_slots)
{
    const size_t cell = p->f32 ? 8 : 16;
    const size_t row16 = p->plane_bytes / 16 / (size_t)p->N;
    const int unit16 = (int)((size_t)p->B * cell / 16);
    RICK_KERNEL(p, RK_ZERO, k_zero_sparse<<<p->n_sm * 8, 256, 0, p->stream>>>(
        reinterpret_cast<uint4*>(p->stack), p->row_dirty, p->row_occ + (size_t)plane_first * p->N,
        p->tile_occ + (size_t)plane_first * p->T * p->T, (size_t)n_slots * p->N, p->N, p->log2B, p->T, row16, unit16));
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
    P.inv_du = p->inv_du;
    P.chunk_counter = &p->counters->grid_chunk;
    if (p->M == 0) return RICK_OK;
    return p->f32 ? launch_grid_s<float>(p, P) : launch_grid_s<double>(p, P);
}
