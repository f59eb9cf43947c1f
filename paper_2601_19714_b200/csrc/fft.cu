// fft.cu -- a4: centred, unnormalised, + sign 2-D complex FFT of every resident w-plane, in
// place (PAPER.md:53 "each w-plane is Fourier transformed separately", :68):
//   P_z[q][p] = sum_{j,i} G_z[j][i] exp(+2 pi i ((i-N/2)(p-N/2) + (j-N/2)(q-N/2)) / N)
// Two passes over the stack (the HBM floor for a plane that does not fit L2: 4 * N^2 * E
// bytes): k_fft_rows transforms the contiguous u axis, one row per CTA held in registers
// (16 elements per thread) with shared-memory exchanges between radix-16 stages;
// k_fft_cols transforms the strided v axis on column strips WC columns wide.
// Centring = index rotation by N/2 = register renaming e -> (e+8) mod 16 (fft_core.cuh).
#include "common.cuh"
#include "fft_core.cuh"
#include "sm100_ptx.cuh"

template <typename T, int LOG2N> struct RowCfg {
    static constexpr int N = 1 << LOG2N, NT = N / 16;
    static constexpr int THREADS = NT >= 256 ? NT : 256;
    static constexpr int RPC = THREADS / NT;                       // rows per CTA
    static constexpr size_t SMEM_EX = (size_t)RPC * (N + N / 16) * 2 * sizeof(T);
    // one row per CTA and one CTA per SM anyway (512 threads and more): a second buffer for 5/8 of the output row
    // (what fits beside the exchange buffer)
    static constexpr bool HALF_OUT = RPC == 1 && THREADS >= 512;
    static constexpr int N_OWN = 5 * N / 8;                          // elements of the row that leave from the buffer of their own
    static constexpr size_t SMEM = SMEM_EX + (HALF_OUT ? (size_t)N_OWN * 2 * sizeof(T) : 0);
};

// Work list of the row pass: the groups of RPC consecutive rows (slot-major) with at least one occupied row.
__global__ void __launch_bounds__(256) k_row_list(const unsigned char* __restrict__ occ, unsigned int n_groups, int rpc,
                                                  unsigned int* __restrict__ list, unsigned int* __restrict__ count)
{
    const unsigned int gidx = blockIdx.x * 256u + threadIdx.x;
    bool any = false;
    if (gidx < n_groups)
        for (int i = 0; i < rpc; ++i) any |= occ[(size_t)gidx * rpc + i] != 0;
    // warp-aggregated append (the order of the list does not matter)
    const unsigned int m = __ballot_sync(0xffffffffu, any);
    if (!m) return;
    const int lane = threadIdx.x & 31;
    unsigned int base = 0;
    if (lane == __ffs(m) - 1) base = atomicAdd(count, (unsigned)__popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (any) list[base + __popc(m & ((1u << lane) - 1u))] = gidx;
}

// win_mask[plane]: bit k = some row of rows [k N/32, (k+1) N/32) is occupied.  One CTA of 32 warps per plane.
__global__ void __launch_bounds__(1024) k_window_mask(const unsigned char* __restrict__ occ, int N, uint32_t* __restrict__ mask)
{
    __shared__ uint32_t s_mask;
    if (threadIdx.x == 0) s_mask = 0;
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, win = N >> 5;
    const unsigned char* o = occ + (size_t)blockIdx.x * N + (size_t)warp * win;
    bool any = false;
    for (int i = lane; i < win; i += 32) any |= o[i] != 0;
    if (__any_sync(0xffffffffu, any) && lane == 0) atomicOr(&s_mask, 1u << warp);
    __syncthreads();
    if (threadIdx.x == 0) mask[blockIdx.x] = s_mask;
}

template <typename T, int LOG2N>
__global__ void __launch_bounds__(RowCfg<T, LOG2N>::THREADS, (RowCfg<T, LOG2N>::THREADS <= 256 ? 3 : 1))
k_fft_rows(typename cplx_of<T>::type* __restrict__ stack,
           const typename cplx_of<T>::type* __restrict__ tw, const unsigned int* __restrict__ list,
           const unsigned int* __restrict__ count, const unsigned char* __restrict__ tocc, int log2B)
{
    typedef typename cplx_of<T>::type C;
    typedef RowCfg<T, LOG2N> K;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // Rows no visibility touches are zero in HBM and their transform is zero: they are not on the list.
    // Persistent CTAs walk the list of occupied row groups.
    const int rl = threadIdx.x / K::NT, t = threadIdx.x - rl * K::NT;
    C* sm = reinterpret_cast<C*>(smem_raw) + (size_t)rl * (K::N + K::N / 16);
    __shared__ unsigned char s_to[2][K::RPC][K::N / 8];
    const int Tn = K::N >> log2B;
    const unsigned int n_work = *count;
    // only the tiles some footprint reaches hold gridded data (tile_occ); whatever else the row holds
    // (rick_image leaves the previous transform there) is not read and counts as zero.  The flags of the
    // NEXT group are fetched (list entry, then flag bytes) while this group is transformed: at most two
    // bytes per thread (RPC * Tn = THREADS * 16 / B, B >= 8), parked in registers across the transform.
    auto flag_addr = [&](size_t grp, int i) -> const unsigned char* {
        const int a = i / Tn, ti = i - a * Tn;
        const size_t R = grp * K::RPC + a;          // slot-major row
        const size_t slot = R / K::N;
        const int row = (int)(R - slot * K::N);
        return tocc + (slot * Tn + (size_t)(row >> log2B)) * Tn + ti;
    };
    const int n_flags = K::RPC * Tn;
    unsigned int w = blockIdx.x;
    size_t grp = w < n_work ? list[w] : 0;
    if (w < n_work)
        for (int i = threadIdx.x; i < n_flags; i += K::THREADS) (&s_to[0][0][0])[(i / Tn) * (K::N / 8) + (i % Tn)] = *flag_addr(grp, i);
    __syncthreads();
    for (int it = 0; w < n_work; w += gridDim.x, ++it) {
        const int cur = it & 1;
        const unsigned int w_next = w + gridDim.x;
        const bool has_next = w_next < n_work;
        const size_t grp_next = has_next ? list[w_next] : 0;
        C* g = stack + (grp * K::RPC + rl) * K::N;
        C v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int i = t + K::NT * ((e + 8) & 15);
            C x;
            x.x = 0;
            x.y = 0;
            if (s_to[cur][rl][i >> log2B]) x = g[i];
            v[e] = x;
        }
        unsigned char f0 = 0, f1 = 0;
        if (has_next) {
            if ((int)threadIdx.x < n_flags) f0 = *flag_addr(grp_next, threadIdx.x);
            if ((int)threadIdx.x + K::THREADS < n_flags) f1 = *flag_addr(grp_next, threadIdx.x + K::THREADS);
        }
        // BULK (one row per CTA, N >= 4096): the transformed row is assembled in shared memory and leaves by bulk stores
        // of the TMA unit while the CTA goes on to the next row (the 16 direct stores per thread came in a burst that
        // filled the store queue with every warp waiting behind it).  With three CTAs per SM (N = 4096) the row is
        // assembled in the exchange buffer, free after the last exchange, and the next row's first exchange waits
        // until the store has read it (the other CTAs run meanwhile).  With one CTA per SM that wait was 16 % of the
        // kernel (the store drains at the SM's share of the HBM write rate): there the first 5/8 of the row go to
        // a buffer of their own, which nothing touches for a whole row, and only the rest to the exchange buffer.
        constexpr bool BULK = K::RPC == 1 && LOG2N >= 12;
        if (BULK && it > 0) {
            if (threadIdx.x == 0) { if (K::HALF_OUT) bulk_wait_read_but_last(); else bulk_wait_read(); }
            __syncthreads();
        }
        fft_thread<T, LOG2N>(v, t, sm, 1, 0, tw);
        if constexpr (BULK && K::HALF_OUT) {
            C* out_lo = reinterpret_cast<C*>(smem_raw + K::SMEM_EX);
            if (it > 0) {
                if (threadIdx.x == 0) bulk_wait_read();      // (long done: issued a whole row ago)
                __syncthreads();
            }
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int i = t + K::NT * ((e + 8) & 15);
                if (i < K::N_OWN) out_lo[i] = v[e]; else sm[i - K::N_OWN] = v[e];
            }
            fence_proxy_async_smem();
            __syncthreads();
            if (threadIdx.x == 0) {
                bulk_store(g + K::N_OWN, sm, (uint32_t)((K::N - K::N_OWN) * sizeof(C)));      // first: the one the next row waits for
                bulk_store(g, out_lo, (uint32_t)(K::N_OWN * sizeof(C)));
            }
        } else if constexpr (BULK) {
#pragma unroll
            for (int e = 0; e < 16; ++e) sm[t + K::NT * ((e + 8) & 15)] = v[e];
            fence_proxy_async_smem();
            __syncthreads();
            if (threadIdx.x == 0) bulk_store(g, sm, (uint32_t)(K::N * sizeof(C)));
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) g[t + K::NT * ((e + 8) & 15)] = v[e];
        }
        if (has_next) {
            unsigned char* nx = &s_to[cur ^ 1][0][0];
            const int i0 = threadIdx.x, i1 = threadIdx.x + K::THREADS;
            if (i0 < n_flags) nx[(i0 / Tn) * (K::N / 8) + (i0 % Tn)] = f0;
            if (i1 < n_flags) nx[(i1 / Tn) * (K::N / 8) + (i1 % Tn)] = f1;
        }
        __syncthreads();
        grp = grp_next;
    }
    if (K::RPC == 1 && LOG2N >= 12 && threadIdx.x == 0) bulk_wait_read();      // shared memory stays valid until the last store has read it
}

template <typename T, int LOG2N> struct ColCfg {
    static constexpr int N = 1 << LOG2N, NT = N / 16;
    static constexpr int MAXT = sizeof(T) == 8 ? 512 : 1024;       // register budget
    static constexpr int WANT = 32 / (2 * (int)sizeof(T));          // one 32-byte sector
    static constexpr int W0 = NT * WANT <= MAXT ? WANT : (MAXT / NT >= 1 ? MAXT / NT : 1);
    static constexpr int WC = NT * W0 >= 256 ? W0 : 256 / NT;       // columns per CTA
    static constexpr int THREADS = NT * WC;
    static constexpr size_t SMEM = (size_t)WC * (N + N / 16) * 2 * sizeof(T);
};

template <typename T, int LOG2N>
__global__ void __launch_bounds__(ColCfg<T, LOG2N>::THREADS)
k_fft_cols(typename cplx_of<T>::type* __restrict__ stack,
           const typename cplx_of<T>::type* __restrict__ tw)
{
    typedef typename cplx_of<T>::type C;
    typedef ColCfg<T, LOG2N> K;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* sm = reinterpret_cast<C*>(smem_raw);
    constexpr int STRIPS = K::N / K::WC;
    const int plane = blockIdx.x / STRIPS, strip = blockIdx.x - plane * STRIPS;
    const int c = threadIdx.x % K::WC, t = threadIdx.x / K::WC;
    C* g = stack + (size_t)plane * K::N * K::N + (size_t)strip * K::WC + c;
    C v[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = g[(size_t)(t + K::NT * ((e + 8) & 15)) * K::N];
    fft_thread<T, LOG2N>(v, t, sm, K::WC, c, tw);
#pragma unroll
    for (int e = 0; e < 16; ++e) g[(size_t)(t + K::NT * ((e + 8) & 15)) * K::N] = v[e];
}

template <typename T, int LOG2N>
static int launch_fft(rick_plan_t* p, int plane_first, int n_planes, int which)   // which: 1 rows, 2 columns, 3 both
{
    typedef typename cplx_of<T>::type C;
    typedef RowCfg<T, LOG2N> KR;
    typedef ColCfg<T, LOG2N> KC;
    if (which & 1) {
        RICK_CUDA(p, cudaFuncSetAttribute(k_fft_rows<T, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)KR::SMEM));
        const unsigned int n_groups = (unsigned int)((size_t)n_planes * KR::N / KR::RPC);
        if (n_groups > p->row_list_cap) {
            if (p->row_list) cudaFree(p->row_list);
            p->row_list = nullptr;
            p->row_list_cap = 0;
            RICK_CUDA(p, cudaMalloc(&p->row_list, sizeof(unsigned int) * ((size_t)n_groups + 1)));
            p->row_list_cap = n_groups;
        }
        unsigned int* count = p->row_list + p->row_list_cap;
        RICK_CUDA(p, cudaMemsetAsync(count, 0, sizeof(unsigned int), p->stream));
        RICK_KERNEL(p, RK_ROW_OCC, k_row_list<<<(n_groups + 255) / 256, 256, 0, p->stream>>>(
            p->row_occ + (size_t)plane_first * p->N, n_groups, KR::RPC, p->row_list, count));
        if (p->cols13_ok)      // the fused N = 8192 column pass fetches occupied windows of 256 rows only
            RICK_KERNEL(p, RK_ROW_OCC, k_window_mask<<<n_planes, 1024, 0, p->stream>>>(
                p->row_occ + (size_t)plane_first * p->N, p->N, p->win_mask + plane_first));
        int per_sm = 1;
        RICK_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fft_rows<T, LOG2N>, KR::THREADS, KR::SMEM));
        if (per_sm < 1) per_sm = 1;
        unsigned int row_blocks = (unsigned int)(p->n_sm * per_sm);
        if (row_blocks > n_groups) row_blocks = n_groups;
        RICK_KERNEL(p, RK_FFT_ROWS, k_fft_rows<T, LOG2N><<<row_blocks, KR::THREADS, KR::SMEM, p->stream>>>(
            (C*)p->stack, (const C*)p->twiddle, p->row_list, count,
            p->tile_occ + (size_t)plane_first * p->T * p->T, p->log2B));
    }
    if (which & 2) {
        // the in-place column passes write every row of the slots they transform
        const int rcd = rick_all_dirty(p, n_planes);
        if (rcd) return rcd;
        if (!p->f32 && p->cols12_ok) return rick_cols12_fft(p, n_planes);
        RICK_CUDA(p, cudaFuncSetAttribute(k_fft_cols<T, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)KC::SMEM));
        const unsigned int col_blocks = (unsigned int)((size_t)n_planes * (KC::N / KC::WC));
        RICK_KERNEL(p, RK_FFT_COLS, k_fft_cols<T, LOG2N><<<col_blocks, KC::THREADS, KC::SMEM, p->stream>>>((C*)p->stack, (const C*)p->twiddle));
    }
    return RICK_OK;
}


// ------------------------------------------------------------------------------------------
// Long columns (N >= 8192: a column is 128 KB and one SM can hold a single one, so the strided pass above
// touches HBM in 16-byte pieces with nothing in flight while it transforms: 1.8 TB/s at N = 8192 fp64,
// 1.1 TB/s at N = 16384 fp32).  rick_image transforms them in TWO passes at full line width instead
// ("four-step", N = 16 N2, n = n1 + 16 n2, m = m2 + N2 m1):
//     X[m2 + N2 m1] = sum_n1 W16^(n1 m1) [ W_N^(n1 m2) sum_n2 x[n1 + 16 n2] W_N2^(n2 m2) ]
//   pass A (k_fft_cols_a): for each n1 the N2-point transform over rows n1 + 16 n2 of a strip of 8 columns
//     (128-byte pieces in fp64, the same in-register Stockham core as the row pass), times W_N^(n1 m2), stored at
//     row n1 + 16 m2;
//   pass B (k_cols_b_wcorrect, below): for each m2 one THREAD transforms the 16 consecutive rows 16 m2 + n1 of
//     its column in registers (no exchange at all; lanes run along the columns), fused with the w-correction.
// Pass A reads and writes the stack once more than a single pass would, at full line width; pass B replaces
// the read of the correction pass.  The centring is the rotation by N2/2 in n2 (pass A input, e -> (e+8) mod
// 16) and by 8 in m1 (pass B output).  The staged API keeps the single-pass kernel (its planes are complete
// transforms in natural order).
#ifndef C2_MINB
#define C2_MINB 512
#endif
template <typename T, int LOG2N> struct Col2Cfg {
    static constexpr int N = 1 << LOG2N, LOG2N2 = LOG2N - 4, N2 = N / 16, NT2 = N2 / 16;
    static constexpr int W = 8;      // 128-byte (fp64) / 64-byte (fp32) row pieces; 16 fp32 columns measured no faster
    static constexpr int THREADS = NT2 * W;
    static constexpr size_t SMEM = (size_t)W * (N2 + N2 / 16) * 2 * sizeof(T);
};

template <typename T, int LOG2N>
__global__ void __launch_bounds__(Col2Cfg<T, LOG2N>::THREADS, C2_MINB / Col2Cfg<T, LOG2N>::THREADS)
k_fft_cols_a(typename cplx_of<T>::type* __restrict__ stack, const typename cplx_of<T>::type* __restrict__ tw2,
             const typename cplx_of<T>::type* __restrict__ twN, const unsigned char* __restrict__ occ,
             const int* __restrict__ sparse_max, int sparse_cap, unsigned int n_units)
{
    typedef typename cplx_of<T>::type C;
    typedef Col2Cfg<T, LOG2N> K;
    if (sparse_max && *sparse_max <= sparse_cap) return;      // the sparse fused pass (fft_cols_sparse.cu) serves this image
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* sm = reinterpret_cast<C*>(smem_raw);
    constexpr int STRIPS = K::N / K::W;
    const int c = threadIdx.x % K::W, t = threadIdx.x / K::W;
    // persistent CTAs over the (plane, strip, n1) units: a launch that returns at once (above) costs nothing
    for (unsigned int unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
        const int n1 = unit & 15;                    // the 16 units of a strip are taken by neighbouring CTAs
        const unsigned int rest = unit >> 4;
        const int strip = (int)(rest % STRIPS), plane = (int)(rest / STRIPS);
        C* g = stack + (size_t)plane * K::N * K::N + (size_t)n1 * K::N + (size_t)strip * K::W + c;
        // rows no footprint reaches were never transformed by the row pass and count as zero: they are not read
        // (and rick_image does not clear them, rick_zero_sparse keep_stale); the pass writes every row
        const unsigned char* oc = occ + (size_t)plane * K::N + n1;
        C v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int n2 = t + K::NT2 * ((e + 8) & 15);
            C x;
            x.x = 0;
            x.y = 0;
            if (oc[16 * n2]) x = g[(size_t)16 * n2 * K::N];
            v[e] = x;
        }
        fft_thread<T, K::LOG2N2>(v, t, sm, K::W, c, tw2);
        // four outputs at a time: their twiddle loads are not hoisted above the transform (register budget)
#pragma unroll
        for (int e0 = 0; e0 < 16; e0 += 4) {
            asm volatile("" ::: "memory");
            C w[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) w[i] = twN[n1 * (t + K::NT2 * (e0 + i))];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int m2 = t + K::NT2 * (e0 + i);
                g[(size_t)16 * m2 * K::N] = cmul(v[e0 + i], w[i]);      // twN[0] = 1 when n1 = 0
            }
        }
        __syncthreads();                             // the exchange buffer is free for the next unit
    }
}

template <typename T, int LOG2N> static int launch_cols2(rick_plan_t* p, int plane_first, int n_planes)
{
    typedef typename cplx_of<T>::type C;
    typedef Col2Cfg<T, LOG2N> K;
    const int rcd = rick_all_dirty(p, n_planes);       // the pass writes every row of the slots
    if (rcd) return rcd;
    RICK_CUDA(p, cudaFuncSetAttribute(k_fft_cols_a<T, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM));
    const unsigned int n_units = (unsigned int)((size_t)n_planes * (K::N / K::W) * 16);
    int per_sm = 1;
    RICK_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fft_cols_a<T, LOG2N>, K::THREADS, K::SMEM));
    if (per_sm < 1) per_sm = 1;
    unsigned int blocks_a = (unsigned int)(p->n_sm * per_sm);
    if (blocks_a > n_units) blocks_a = n_units;
    RICK_KERNEL(p, RK_FFT_COLS, k_fft_cols_a<T, LOG2N><<<blocks_a, K::THREADS, K::SMEM, p->stream>>>(
        (C*)p->stack, (const C*)p->twiddle2, (const C*)p->twiddle, p->row_occ + (size_t)plane_first * p->N,
        rick_sparse_maxcount(p), rick_sparse_cap(p), n_units));
    return RICK_OK;
}

int rick_cols2_on(const rick_plan_t* p) { return p->log2N >= 13 && !p->cols13_ok; }

int rick_fft_cols2(rick_plan_t* p, int plane_first, int n_planes)
{
    if (n_planes <= 0) return RICK_OK;
    if (p->f32) {
        if (p->log2N == 13) return launch_cols2<float, 13>(p, plane_first, n_planes);
        if (p->log2N == 14) return launch_cols2<float, 14>(p, plane_first, n_planes);
    } else if (p->log2N == 13) {
        return launch_cols2<double, 13>(p, plane_first, n_planes);
    }
    p->err = "two-pass column transform: grid edge not supported";
    return RICK_ERR_INVALID;
}

static int fft_dispatch(rick_plan_t* p, int plane_first, int n_planes, int which)
{
    if (n_planes <= 0) return RICK_OK;
    if (p->f32) {
        switch (p->log2N) {
            case 6: return launch_fft<float, 6>(p, plane_first, n_planes, which);
            case 7: return launch_fft<float, 7>(p, plane_first, n_planes, which);
            case 8: return launch_fft<float, 8>(p, plane_first, n_planes, which);
            case 9: return launch_fft<float, 9>(p, plane_first, n_planes, which);
            case 10: return launch_fft<float, 10>(p, plane_first, n_planes, which);
            case 11: return launch_fft<float, 11>(p, plane_first, n_planes, which);
            case 12: return launch_fft<float, 12>(p, plane_first, n_planes, which);
            case 13: return launch_fft<float, 13>(p, plane_first, n_planes, which);
            case 14: return launch_fft<float, 14>(p, plane_first, n_planes, which);
        }
    } else {
        switch (p->log2N) {
            case 6: return launch_fft<double, 6>(p, plane_first, n_planes, which);
            case 7: return launch_fft<double, 7>(p, plane_first, n_planes, which);
            case 8: return launch_fft<double, 8>(p, plane_first, n_planes, which);
            case 9: return launch_fft<double, 9>(p, plane_first, n_planes, which);
            case 10: return launch_fft<double, 10>(p, plane_first, n_planes, which);
            case 11: return launch_fft<double, 11>(p, plane_first, n_planes, which);
            case 12: return launch_fft<double, 12>(p, plane_first, n_planes, which);
            case 13: return launch_fft<double, 13>(p, plane_first, n_planes, which);
        }
    }
    p->err = "grid edge not supported by the FFT at this precision";
    return RICK_ERR_INVALID;
}

int rick_fft_planes(rick_plan_t* p, int plane_first, int n_planes) { return fft_dispatch(p, plane_first, n_planes, 3); }
int rick_fft_rows(rick_plan_t* p, int plane_first, int n_planes) { return fft_dispatch(p, plane_first, n_planes, 1); }
int rick_fft_cols(rick_plan_t* p, int n_planes) { return fft_dispatch(p, 0, n_planes, 2); }

// ------------------------------------------------------------------------------------------
// Pass B of the long-column transform FUSED with a5 (+ a6): the 16-point transforms of pass B need no
// exchange, so a thread can keep transforming the same 16 rows of its column plane after plane and sum the
// planes with Horner's rule in z (S <- P_z + step S, step = exp(2 pi i dw (n-1)); Eq. 2) --
// the transformed planes are never written and never read back: two transfers of the stack less.
// Two threads (h = 0, 1) share one (column p, block m2): both transform the 16 rows, each keeps the 8
// outputs of its half (pixel rows q = m2 + N2 (8 h + i)) -- 8 x (S, step) complex doubles fit the
// register file next to the transform, 16 do not.  A warp = 16 consecutive columns x 2 halves.
template <typename T, int LOG2N>
__global__ void __launch_bounds__(256, 2)
k_cols_b_wcorrect(const typename cplx_of<T>::type* __restrict__ stack, int n_planes, int z_first, double dl,
                  const WRange* __restrict__ wr, double* __restrict__ image, int accumulate,
                  const double* __restrict__ taper, int col_begin, int n_col16, const int* __restrict__ sparse_max, int sparse_cap)
{
    typedef typename cplx_of<T>::type C;
    constexpr int N = 1 << LOG2N, N2 = N / 16;
    if (sparse_max && *sparse_max <= sparse_cap) return;      // the sparse fused pass serves this image
    // columns col_begin .. col_begin + 16 n_col16 - 1 only (the host-buffer entry launches the pass in parts)
    const size_t gid = (size_t)blockIdx.x * 256 + threadIdx.x;       // < 16 n_col16 * N2 * 2 by construction of the grid
    const int pl = (int)(gid & 15), h = (int)((gid >> 4) & 1);
    const size_t rest = gid >> 5;
    const int p = col_begin + (int)(rest % (size_t)n_col16) * 16 + pl, m2 = (int)(rest / (size_t)n_col16);
    const double dw = wr->dw;
    const double l = (double)(p - N / 2) * dl;
    double2 S[8], st[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int q = m2 + N2 * (8 * h + i);
        const double m = (double)(q - N / 2) * dl;
        const double r2 = l * l + m * m;
        double xs = 0.0;
        if (r2 < 1.0) xs = dw * (-r2 / (1.0 + sqrt(1.0 - r2)));
        xs -= rint(xs);
        sincospi(2.0 * xs, &st[i].y, &st[i].x);
        S[i].x = 0.0;
        S[i].y = 0.0;
    }
    const C* g = stack + (size_t)(16 * m2) * N + p;
    for (int plane = n_planes - 1; plane >= 0; --plane) {
        const C* gp = g + (size_t)plane * N * N;
        C b[16];
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) b[n1] = gp[(size_t)n1 * N];
        fft16<T>(b);
        // memory slot s = (m1 + 8) & 15 holds pixel row m2 + N2 s: half h keeps outputs m1 = 8 (1 - h) + i
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const C lo = b[leg_reg<16>(i)], hi = b[leg_reg<16>(8 + i)];
            const double xr = (double)(h ? lo.x : hi.x), xi = (double)(h ? lo.y : hi.y);
            const double2 s = S[i];
            S[i].x = fma(st[i].x, s.x, fma(-st[i].y, s.y, xr));
            S[i].y = fma(st[i].x, s.y, fma(st[i].y, s.x, xi));
        }
    }
    const double w_first = wr->w_min + ((double)z_first + 0.5) * dw;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int q = m2 + N2 * (8 * h + i);
        const double m = (double)(q - N / 2) * dl;
        const double r2 = l * l + m * m;
        double val = 0.0;
        if (r2 < 1.0) {
            double x0 = w_first * (-r2 / (1.0 + sqrt(1.0 - r2)));
            x0 -= rint(x0);
            double pr, pi;
            sincospi(2.0 * x0, &pi, &pr);
            val = pr * S[i].x - pi * S[i].y;
        }
        const size_t pix = (size_t)q * N + p;
        if (accumulate) val += image[pix];
        if (taper) val /= (taper[p] * taper[q]);
        image[pix] = val;
    }
}

template <typename T, int LOG2N>
static int launch_cols_b_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image, int accumulate,
                                  int fuse_taper, int slot_first, int col_begin, int col_end)
{
    typedef typename cplx_of<T>::type C;
    constexpr int N = 1 << LOG2N;
    const int n_col16 = (col_end - col_begin) / 16;                   // both multiples of 16
    if (n_col16 <= 0) return RICK_OK;
    const size_t n_threads = (size_t)n_col16 * 16 * (N / 16) * 2;     // a multiple of 256
    RICK_KERNEL(p, RK_WCORRECT, k_cols_b_wcorrect<T, LOG2N><<<(unsigned int)(n_threads / 256), 256, 0, p->stream>>>(
        (const C*)p->stack + (size_t)slot_first * N * N, n_planes, p->z0 + z_first, p->dl, p->wrange + img, image, accumulate,
        fuse_taper ? p->taper : nullptr, col_begin, n_col16, rick_sparse_maxcount(p), rick_sparse_cap(p)));
    return RICK_OK;
}

int rick_cols2_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image, int accumulate,
                        int fuse_taper, int slot_first, int col_begin, int col_end)
{
    if (n_planes <= 0) return RICK_OK;
    if (col_end < 0) col_end = p->N;
    if (p->f32) {
        if (p->log2N == 13) return launch_cols_b_wcorrect<float, 13>(p, img, z_first, n_planes, image, accumulate, fuse_taper, slot_first, col_begin, col_end);
        if (p->log2N == 14) return launch_cols_b_wcorrect<float, 14>(p, img, z_first, n_planes, image, accumulate, fuse_taper, slot_first, col_begin, col_end);
    } else if (p->log2N == 13) {
        return launch_cols_b_wcorrect<double, 13>(p, img, z_first, n_planes, image, accumulate, fuse_taper, slot_first, col_begin, col_end);
    }
    p->err = "two-pass column transform: grid edge not supported";
    return RICK_ERR_INVALID;
}
