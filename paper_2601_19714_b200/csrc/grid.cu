// grid.cu -- a3: convolutional gridding with a separable Kaiser-Bessel kernel
// (Eq. 3; kernel :62; halo = (S-1)/2 cells, Eq. 5 :129).
//
//   G[i_p][i_v+b][i_u+a] += (w V) g(d_a) g(d_b),  a,b in [-h,h],
//   d_a = (i_u - N/2 + a) - x_u,  g(t) = I0(beta sqrt(1-(2t/S)^2)) / I0(beta)
//
// Design (B200): the visibilities arrive sorted by (image, plane, uv tile of B x B cells).
// Each WARP takes fixed-size chunks of the sorted order from a dynamic counter (perfect
// balance in visibilities, whatever the skew of the uv coverage) and owns a PRIVATE
// shared-memory accumulation tile of (B+S-1)^2 cells -- the tile plus the kernel halo, the
// single-GPU analogue of the paper's ghost region.  Per batch of 32 visibilities every lane
// evaluates the 2S kernel values of its own visibility, stages them in shared memory, then the
// warp walks the 32 visibilities one by one with its lanes spread over the footprint, each lane
// owning two horizontally adjacent cells: plain read-modify-write, no shared-memory atomics
// (cells of one footprint are distinct, and successive visibilities are ordered by __syncwarp).
// When the tile key changes, the tile is flushed to HBM with fire-and-forget RED atomics
// (non-zero cells only) and re-zeroed.
//
// Kernel values.  d_a = (a-h) - delta with delta = x_u - (i_u - N/2) in [-1/2, 1/2): tap a sees g
// only on one unit interval, where it is a degree-KB_DEG polynomial in s = 2 delta to < 2e-16
// (tables.cu fits and checks it at plan time).  The coefficients travel as kernel parameters, so
// every Horner step is one DFMA with a constant-bank operand: 2 S (KB_DEG+1) DFMA per visibility
// and no load -- against ~45 terms of the I0 power series per tap before.
//
// The tile row pitch is odd (and > B+S-1, the pad column takes the zero-weight partner of the last
// cell of a footprint row), so the lanes of a quarter warp hit distinct 16-byte bank groups.
#include "common.cuh"

struct GridParams {
    const void* vis;
    const float* wgt;
    const double* uvw;
    const double* chan_scale;
    const uint32_t* skeys;
    const uint32_t* sperm;
    const long long* plane_start;
    int plane_first, n_planes;
    void* stack;
    int N, h, B, T, TWp, TH, C;
    int vis_c128;
    double inv_du;
    unsigned int* chunk_counter;
};
template <int S> struct GridParamsS {
    GridParams g;
    double poly[S][RICK_KB_DEG + 1];     // poly[a][k]: coefficient of s^k of tap a
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

template <typename GT, int S>
__global__ void __launch_bounds__(GRID_WARPS * 32) k_grid(const __grid_constant__ GridParamsS<S> PS)
{
    typedef typename cell_t<GT>::type cell;
    constexpr int PW = (S + 1) / 2;                 // cell pairs per footprint row
    constexpr int SP = 2 * PW;                      // padded footprint width (even)
    constexpr int NPAIR = S * PW, ROUNDS = (NPAIR + 31) / 32;
    constexpr int DEG = RICK_KB_DEG;
    const GridParams& P = PS.g;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int TWp = P.TWp, TH = P.TH, N = P.N, h = P.h, B = P.B, T = P.T;
    const int tile_cells = TH * TWp;

    // shared layout per warp: tile | ku[32][SP] | kv[32][SP] | vr[32] | vi[32] | base[32]
    const size_t tile_bytes = ((size_t)tile_cells * sizeof(cell) + 15) & ~(size_t)15;
    const size_t per_warp = tile_bytes + (size_t)(2 * 32 * SP + 64) * sizeof(double) + 32 * sizeof(int);
    unsigned char* wbase = smem_raw + (size_t)warp * per_warp;
    cell* tile = reinterpret_cast<cell*>(wbase);
    double* s_ku = reinterpret_cast<double*>(wbase + tile_bytes);
    double* s_kv = s_ku + 32 * SP;
    double* s_vr = s_kv + 32 * SP;
    double* s_vi = s_vr + 32;
    int* s_base = reinterpret_cast<int*>(s_vi + 32);

    cell zero;
    zero.x = 0;
    zero.y = 0;
    for (int i = lane; i < tile_cells; i += 32) tile[i] = zero;
    for (int i = lane; i < 2 * 32 * SP; i += 32) s_ku[i] = 0.0;      // also the zero weight of the pad column
    __syncwarp();

    // cell pair(s) of this lane: pair = lane + 32*rr -> row b, cells (b, 2 a2), (b, 2 a2 + 1)
    int fb[ROUNDS], fa[ROUNDS], foff[ROUNDS];
#pragma unroll
    for (int rr = 0; rr < ROUNDS; ++rr) {
        const int pi = lane + 32 * rr;
        fb[rr] = pi / PW;
        fa[rr] = 2 * (pi - fb[rr] * PW);
        foff[rr] = fb[rr] * TWp + fa[rr];
    }

    const long long v_begin = P.plane_start[P.plane_first];
    const long long v_end = P.plane_start[P.plane_first + P.n_planes];
    const long long n_chunks = (v_end - v_begin + GRID_CHUNK - 1) / GRID_CHUNK;
    const unsigned int TT = (unsigned)T * (unsigned)T;
    const double shift = (double)(N / 2) + 0.5;

    uint32_t cur_key = RICK_KEY_DROPPED;

    auto flush = [&](uint32_t key) {
        const unsigned int pz = key / TT, rem = key - pz * TT;
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

    for (;;) {
        long long chunk = 0;
        if (lane == 0) chunk = (long long)atomicAdd(P.chunk_counter, 1u);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk >= n_chunks) break;
        const long long c_begin = v_begin + chunk * GRID_CHUNK;
        const long long c_end = (c_begin + GRID_CHUNK < v_end) ? c_begin + GRID_CHUNK : v_end;

        for (long long b0 = c_begin; b0 < c_end; b0 += 32) {
            const long long ks = b0 + lane;
            const bool valid = ks < c_end;
            uint32_t key = RICK_KEY_DROPPED;
            if (valid) {
                key = P.skeys[ks];
                const unsigned int idx = P.sperm[ks];
                const unsigned int r = idx / (unsigned)P.C, c = idx - r * (unsigned)P.C;
                const double s = P.chan_scale[c];
                const double xu = __dmul_rn(__dmul_rn(P.uvw[3ull * r + 0], s), P.inv_du);
                const double xv = __dmul_rn(__dmul_rn(P.uvw[3ull * r + 1], s), P.inv_du);
                const int iu = (int)floor(__dadd_rn(xu, shift));
                const int iv = (int)floor(__dadd_rn(xv, shift));
                double vr, vi;
                if (P.vis_c128) {
                    const double2 v = reinterpret_cast<const double2*>(P.vis)[idx];
                    vr = v.x;
                    vi = v.y;
                } else {
                    const float2 v = reinterpret_cast<const float2*>(P.vis)[idx];
                    vr = (double)v.x;
                    vi = (double)v.y;
                }
                if (P.wgt) {
                    const double om = (double)P.wgt[idx];
                    vr *= om;
                    vi *= om;
                }
                s_vr[lane] = vr;
                s_vi[lane] = vi;
                // top-left footprint cell, local to the tile: (i_u - h) - (tu*B - h) = i_u mod B
                s_base[lane] = (iv - (iv / B) * B) * TWp + (iu - (iu / B) * B);
                // kernel values: tap a at d_a = (a-h) - s/2, s = 2 (x - (i - N/2)); 2S Horner chains
                const double su = 2.0 * (xu - (double)(iu - N / 2));
                const double sv = 2.0 * (xv - (double)(iv - N / 2));
                double au[S], av[S];
#pragma unroll
                for (int a = 0; a < S; ++a) {
                    au[a] = PS.poly[a][DEG];
                    av[a] = PS.poly[a][DEG];
                }
#pragma unroll
                for (int k = DEG - 1; k >= 0; --k) {
#pragma unroll
                    for (int a = 0; a < S; ++a) {
                        au[a] = fma(au[a], su, PS.poly[a][k]);
                        av[a] = fma(av[a], sv, PS.poly[a][k]);
                    }
                }
#pragma unroll
                for (int a = 0; a < S; ++a) {
                    s_ku[lane * SP + a] = au[a];
                    s_kv[lane * SP + a] = av[a];
                }
            }
            __syncwarp();
            const int nb = (int)((c_end - b0) < 32 ? (c_end - b0) : 32);
            for (int j = 0; j < nb; ++j) {
                const uint32_t kj = __shfl_sync(0xffffffffu, key, j);
                if (kj != cur_key) {
                    if (cur_key != RICK_KEY_DROPPED) flush(cur_key);
                    cur_key = kj;
                }
                const int base = s_base[j];
                const double vr = s_vr[j], vi = s_vi[j];
#pragma unroll
                for (int rr = 0; rr < ROUNDS; ++rr) {
                    if (lane + 32 * rr < NPAIR) {
                        const double2 k2 = *reinterpret_cast<const double2*>(&s_ku[j * SP + fa[rr]]);
                        const double kvb = s_kv[j * SP + fb[rr]];
                        const double wr = vr * kvb, wi = vi * kvb;
                        cell* tp = tile + base + foff[rr];
                        cell t0 = tp[0], t1 = tp[1];
                        t0.x += (GT)(wr * k2.x);
                        t0.y += (GT)(wi * k2.x);
                        t1.x += (GT)(wr * k2.y);
                        t1.y += (GT)(wi * k2.y);
                        tp[0] = t0;
                        tp[1] = t1;
                    }
                }
                __syncwarp();
            }
        }
        if (cur_key != RICK_KEY_DROPPED) flush(cur_key);
        cur_key = RICK_KEY_DROPPED;
    }
}

// zero-fill of the resident planes (the gridder accumulates with atomics)
__global__ void __launch_bounds__(256) k_zero(uint4* __restrict__ dst, size_t n16)
{
    const uint4 z = make_uint4(0, 0, 0, 0);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16;
         i += (size_t)gridDim.x * blockDim.x)
        dst[i] = z;
}

int rick_zero_planes(rick_plan_t* p, int n_planes)
{
    const size_t n16 = p->plane_bytes / 16 * (size_t)n_planes;
    RICK_KERNEL(p, RK_ZERO, k_zero<<<p->n_sm * 8, 256, 0, p->stream>>>(reinterpret_cast<uint4*>(p->stack), n16));
    return RICK_OK;
}

template <typename GT, int S>
static int launch_grid(rick_plan_t* p, const GridParams& P)
{
    typedef typename cell_t<GT>::type cell;
    constexpr int SP = 2 * ((S + 1) / 2);
    GridParamsS<S> PS;
    PS.g = P;
    for (int a = 0; a < S; ++a)
        for (int k = 0; k <= RICK_KB_DEG; ++k) PS.poly[a][k] = p->kb_poly[a * (RICK_KB_DEG + 1) + k];
    const size_t tile_bytes = ((size_t)P.TH * P.TWp * sizeof(cell) + 15) & ~(size_t)15;
    const size_t per_warp = tile_bytes + (size_t)(2 * 32 * SP + 64) * sizeof(double) + 32 * sizeof(int);
    const size_t smem = GRID_WARPS * per_warp;
    if (smem > 227 * 1024) {
        p->err = "tile/support too large for the gridder's shared memory";
        return RICK_ERR_INVALID;
    }
    RICK_CUDA(p, cudaFuncSetAttribute(k_grid<GT, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    RICK_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_grid<GT, S>, GRID_WARPS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    RICK_KERNEL(p, RK_RESET, k_chunk_reset<<<1, 1, 0, p->stream>>>(P.chunk_counter));
    RICK_KERNEL(p, RK_GRID, k_grid<GT, S><<<p->n_sm * per_sm, GRID_WARPS * 32, smem, p->stream>>>(PS));
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
    P.skeys = p->sorted_keys;
    P.sperm = p->sorted_perm;
    P.plane_start = (const long long*)p->plane_start;
    P.plane_first = plane_first;
    P.n_planes = n_planes;
    P.stack = p->stack;
    P.N = p->N;
    P.h = p->h;
    P.B = p->B;
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
