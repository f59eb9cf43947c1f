// fft_cols_sparse.cu -- the column pass of a4 fused with a5 (+ a6) for the fp32 grid with long columns
// (N = 8192, 16384: configs[3]), in ONE pass that reads only the OCCUPIED rows of the stack
// (PAPER.md:53, :68 FFT per w-plane; Eq. 2 :50 and :69 phase screen + plane sum; reading R12 taper).
//
// Why.  A column of a 16384^2 complex64 plane is 128 KB: one SM holds one column, and a column touches HBM in
// 8-byte pieces -- too small for TMA (16-byte minimum) and, read densely, 1.1 TB/s.  The
// two-pass path (fft.cu) therefore moved the stack three times at full line width.  But with the core-dense uv
// coverage of the paper's arrays (:81, :108) most ROWS of a plane are never touched (configs[3]: 12 % are
// occupied), every column of a plane has the same occupied rows, and the row pass left the others untouched --
// they count as zero.  So, per plane, the sort's row occupancy is compacted into a row list + a bitmap with
// word prefix sums (k_row_compact), and the column kernel
//   * gathers the occupied rows of its column with 8-byte cp.async into a compact staging buffer (the copies
//     of the next item run under the transform of the current one),
//   * expands them into the 16 registers per thread through the bitmap (position = prefix + popcount),
//   * runs the in-register Stockham transform of fft_core.cuh (one 1024-thread CTA per column),
//   * and keeps the column's Horner state S, step (complex fp32, 16 B per pixel = 256 KB per column) in TENSOR
//     MEMORY, exactly as the fp64 kernels of fft_cols12.cu do: S <- P_z + step S per plane, I += Re(ph0 S).
// Lanes of this kernel run along the ROWS of one column, so it accumulates into a TRANSPOSED image ([p][q]:
// contiguous 128 KB per column); k_image_transpose_taper turns it into the [q][p] image (and divides by the
// taper) after the last plane batch.  The stack is read once, where occupied, and never written.
// The compact staging holds N/2 rows.  Whether every plane of the image fits is decided ON THE DEVICE
// (max_count): when one does not, these kernels return at once and the two-pass kernels of fft.cu, which
// return at once in the other case, do the work -- no host synchronisation either way.
#include "common.cuh"
#include "fft_core.cuh"
#include "sm100_ptx.cuh"

namespace {

// ---------------------------------------------------------------------------------------------------
// Row compaction.  One CTA per plane, thread i = word i of the bitmap (rows 32 i .. 32 i + 31).
__global__ void __launch_bounds__(512) k_row_compact(const unsigned char* __restrict__ occ, int N, unsigned int* __restrict__ bits,
                                                     unsigned int* __restrict__ prefix, unsigned short* __restrict__ list,
                                                     int* __restrict__ count, int* __restrict__ max_count)
{
    __shared__ unsigned int s_scan[512];
    const int z = blockIdx.x, nw = N / 32, i = threadIdx.x;
    unsigned int word = 0;
    if (i < nw) {
        const uint4* o = reinterpret_cast<const uint4*>(occ + (size_t)z * N + (size_t)i * 32);
        const uint4 a = o[0], b = o[1];
        const unsigned int w8[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 8; ++k)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((w8[k] >> (8 * j)) & 0xffu) word |= 1u << (4 * k + j);
    }
    const unsigned int c = __popc(word);
    s_scan[i] = c;
    __syncthreads();
    for (int d = 1; d < 512; d <<= 1) {          // inclusive Hillis-Steele scan
        const unsigned int v = i >= d ? s_scan[i - d] : 0u;
        __syncthreads();
        s_scan[i] += v;
        __syncthreads();
    }
    const unsigned int excl = s_scan[i] - c;
    if (i < nw) {
        bits[(size_t)z * nw + i] = word;
        prefix[(size_t)z * nw + i] = excl;
        unsigned int pos = excl, w = word;
        while (w) {
            const int b = __ffs(w) - 1;
            w &= w - 1;
            list[(size_t)z * N + pos++] = (unsigned short)(i * 32 + b);
        }
    }
    if (i == 511) {
        count[z] = (int)s_scan[511];
        atomicMax(max_count, (int)s_scan[511]);
    }
}

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// exp(2 pi i w (n-1)) as complex fp32: the argument and its reduction to one turn in fp64, the sine and cosine in fp32
__device__ __forceinline__ float2 phase32(double w, double r2)
{
    double x = w * nm1_of(r2);
    x -= rint(x);
    float2 ph;
    sincospif(2.0f * (float)x, &ph.y, &ph.x);
    return ph;
}

template <int LOG2N> struct SparseCfg {
    static constexpr int N = 1 << LOG2N, NT = N / 16, CAP = N / 2, NW = N / 32;
    static constexpr size_t EX_BYTES = (size_t)(N + N / 16) * sizeof(float2);
    static constexpr size_t STG_BYTES = (size_t)CAP * sizeof(float2);
    static constexpr size_t SMEM = EX_BYTES + STG_BYTES + 2 * NW * sizeof(unsigned int) + 64;
};

__device__ __forceinline__ void tmem_ld8c(uint32_t taddr, float2 (&a)[8])
{
    uint32_t r[16];
    tmem_ld16(taddr, r);
    tmem_wait_ld();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i].x = __uint_as_float(r[2 * i]);
        a[i].y = __uint_as_float(r[2 * i + 1]);
    }
}
__device__ __forceinline__ void tmem_st8c(uint32_t taddr, const float2 (&a)[8])
{
    uint32_t r[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r[2 * i] = __float_as_uint(a[i].x);
        r[2 * i + 1] = __float_as_uint(a[i].y);
    }
    tmem_st16(taddr, r);
}

template <int LOG2N>
__global__ void __launch_bounds__(SparseCfg<LOG2N>::NT, 1)
k_cols_sparse_wcorrect(const float2* __restrict__ stack, const float2* __restrict__ tw, const int* __restrict__ max_count,
                       const unsigned int* __restrict__ bits, const unsigned int* __restrict__ prefix,
                       const unsigned short* __restrict__ list, const int* __restrict__ count, int plane_first, int n_planes,
                       int z_first, double dl, const WRange* __restrict__ wr, double* __restrict__ imageT, int accumulate,
                       int col_begin, int col_end)
{
    typedef SparseCfg<LOG2N> K;
    if (*max_count > K::CAP) return;            // some plane is too dense for the staging: the two-pass kernels run instead
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    float2* stg = reinterpret_cast<float2*>(smem_raw + K::EX_BYTES);
    unsigned int* s_bits = reinterpret_cast<unsigned int*>(smem_raw + K::EX_BYTES + K::STG_BYTES);
    unsigned int* s_pref = s_bits + K::NW;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(s_pref + K::NW);
    const int t = threadIdx.x, warp = t >> 5;
    if (warp == 0) tmem_alloc_all(tmem_slot);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tmem_slot;
    // 64 columns per thread: S (16 complex fp32) | step (16 complex fp32); warps w, w+4, ... share the lanes 32 (w % 4) ..
    const uint32_t tS = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 64);
    const uint32_t tStep = tS + 32;

    // gather of one item: the occupied rows of column `col` of the plane in slot `slot`, and that plane's maps
    auto issue = [&](int col, int slot) {
        const int z = plane_first + slot;
        const int n = count[z];
        const unsigned short* li = list + (size_t)z * K::N;
        const float2* src = stack + (size_t)slot * K::N * K::N + col;
        for (int i = t; i < n; i += K::NT) cp_async8(stg + i, src + (size_t)li[i] * K::N);
        for (int i = t; i < K::NW; i += K::NT) {
            cp_async4(s_bits + i, bits + (size_t)z * K::NW + i);
            cp_async4(s_pref + i, prefix + (size_t)z * K::NW + i);
        }
    };

    int col = col_begin + (int)blockIdx.x;       // columns [col_begin, col_end) of the image
    if (col < col_end) issue(col, n_planes - 1);
    const double dw = wr->dw;
    const double w_first = wr->w_min + ((double)z_first + 0.5) * dw;
    for (; col < col_end; col += gridDim.x) {
        const double l = (double)(col - K::N / 2) * dl;
        // pixel rows of this thread: q_e = t + NT ((e + 8) & 15), for the input rows and the outputs alike
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            float2 st[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int q = t + K::NT * ((8 * k + i + 8) & 15);
                const double m = (double)(q - K::N / 2) * dl;
                const double r2 = l * l + m * m;
                st[i] = r2 < 1.0 ? phase32(dw, r2) : make_float2(1.f, 0.f);
            }
            tmem_st8c(tStep + 16 * k, st);
        }
        tmem_wait_st();
        for (int plane = n_planes - 1; plane >= 0; --plane) {
            cp_async_wait_all();
            __syncthreads();
            float2 v[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int r = t + K::NT * ((e + 8) & 15);
                const unsigned int word = s_bits[r >> 5], bit = 1u << (r & 31);
                float2 x = make_float2(0.f, 0.f);
                if (word & bit) x = stg[s_pref[r >> 5] + __popc(word & (bit - 1u))];
                v[e] = x;
            }
            __syncthreads();                       // staging and maps consumed: the next item may land
            if (plane > 0) issue(col, plane - 1);
            else if (col + (int)gridDim.x < col_end) issue(col + (int)gridDim.x, n_planes - 1);
            fft_thread<float, LOG2N>(v, t, sm, 1, 0, tw);
            // Horner in z: S <- P_z + step S
            if (plane == n_planes - 1) {
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const float2 s8[8] = {v[8 * k], v[8 * k + 1], v[8 * k + 2], v[8 * k + 3], v[8 * k + 4], v[8 * k + 5],
                                          v[8 * k + 6], v[8 * k + 7]};
                    tmem_st8c(tS + 16 * k, s8);
                }
            } else {
                tmem_wait_st();
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    float2 s8[8], st[8];
                    tmem_ld8c(tS + 16 * k, s8);
                    tmem_ld8c(tStep + 16 * k, st);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float2 a = v[8 * k + i];
                        float2 o;
                        o.x = fmaf(st[i].x, s8[i].x, fmaf(-st[i].y, s8[i].y, a.x));
                        o.y = fmaf(st[i].x, s8[i].y, fmaf(st[i].y, s8[i].x, a.y));
                        s8[i] = o;
                    }
                    tmem_st8c(tS + 16 * k, s8);
                }
            }
        }
        // I^T[p][q] (+)= Re(exp(2 pi i w_first (n-1)) S)
        tmem_wait_st();
        double* out = imageT + (size_t)col * K::N;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            float2 s8[8];
            tmem_ld8c(tS + 16 * k, s8);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int q = t + K::NT * ((8 * k + i + 8) & 15);
                const double m = (double)(q - K::N / 2) * dl;
                const double r2 = l * l + m * m;
                double val = 0.0;
                if (r2 < 1.0) {
                    const float2 ph = phase32(w_first, r2);
                    val = (double)(ph.x * s8[i].x - ph.y * s8[i].y);
                }
                if (accumulate) val += out[q];
                out[q] = val;
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc_all(tbase);
}

// image[q][p] = imageT[p][q] (/ (taper[p] taper[q])): 32 x 32 tiles through shared memory
__global__ void __launch_bounds__(256) k_image_transpose_taper(const double* __restrict__ imageT, double* __restrict__ image, int N,
                                                               const double* __restrict__ taper, const int* __restrict__ max_count,
                                                               int cap, int p_begin)
{
    if (*max_count > cap) return;
    __shared__ double tile[32][33];
    const int p0 = p_begin + blockIdx.x * 32, q0 = blockIdx.y * 32;      // image columns p_begin + 32 blockIdx.x ..
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int j = ty; j < 32; j += 8) tile[j][tx] = imageT[(size_t)(p0 + j) * N + q0 + tx];      // [p][q]
    __syncthreads();
    for (int j = ty; j < 32; j += 8) {
        const int q = q0 + j, p = p0 + tx;
        double v = tile[tx][j];
        if (taper) v /= (taper[p] * taper[q]);
        image[(size_t)q * N + p] = v;
    }
}

}   // namespace

// ---------------------------------------------------------------------------------------------------
int rick_sparse_init(rick_plan_t* p)
{
    p->sp_ok = 0;
    if (!p->f32 || p->log2N < 13 || p->d.cube) return RICK_OK;
    const size_t nz = (size_t)p->Nw, N = (size_t)p->N;
    // without room for the transposed image and the maps the plan keeps the two-pass path
    if (cudaMalloc(&p->sp_imageT, sizeof(double) * N * N) != cudaSuccess) {
        cudaGetLastError();
        p->sp_imageT = nullptr;
        return RICK_OK;
    }
    RICK_CUDA(p, cudaMalloc(&p->sp_bits, sizeof(unsigned int) * nz * (N / 32)));
    RICK_CUDA(p, cudaMalloc(&p->sp_prefix, sizeof(unsigned int) * nz * (N / 32)));
    RICK_CUDA(p, cudaMalloc(&p->sp_list, sizeof(unsigned short) * nz * N));
    RICK_CUDA(p, cudaMalloc(&p->sp_count, sizeof(int) * (nz + 1)));
    if (p->log2N == 13)
        RICK_CUDA(p, cudaFuncSetAttribute(k_cols_sparse_wcorrect<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SparseCfg<13>::SMEM));
    else
        RICK_CUDA(p, cudaFuncSetAttribute(k_cols_sparse_wcorrect<14>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SparseCfg<14>::SMEM));
    p->sp_ok = 1;
    return RICK_OK;
}

void rick_sparse_free(rick_plan_t* p)
{
    if (p->sp_imageT) cudaFree(p->sp_imageT);
    if (p->sp_bits) cudaFree(p->sp_bits);
    if (p->sp_prefix) cudaFree(p->sp_prefix);
    if (p->sp_list) cudaFree(p->sp_list);
    if (p->sp_count) cudaFree(p->sp_count);
}

const int* rick_sparse_maxcount(const rick_plan_t* p) { return p->sp_ok ? p->sp_count + p->Nw : nullptr; }
int rick_sparse_cap(const rick_plan_t* p) { return p->N / 2; }

// once per image, after the sort: row lists, bitmaps and prefix sums of all its planes; the largest count
int rick_sparse_prepare(rick_plan_t* p)
{
    int* maxc = p->sp_count + p->Nw;
    RICK_CUDA(p, cudaMemsetAsync(maxc, 0, sizeof(int), p->stream));
    RICK_KERNEL(p, RK_ROW_OCC, k_row_compact<<<p->Nw, 512, 0, p->stream>>>(p->row_occ, p->N, p->sp_bits, p->sp_prefix, p->sp_list,
                                                                         p->sp_count, maxc));
    return RICK_OK;
}

// planes z_first .. z_first + n_planes - 1 of the image, resident in slots 0 .. n_planes - 1
int rick_sparse_wcorrect(rick_plan_t* p, int z_first, int n_planes, int accumulate, int col_begin, int col_end)
{
    if (col_end < 0) col_end = p->N;
    if (n_planes <= 0 || col_end <= col_begin) return RICK_OK;
    const int* maxc = p->sp_count + p->Nw;
    if (p->log2N == 13) {
        RICK_KERNEL(p, RK_COLS_WCORRECT, k_cols_sparse_wcorrect<13><<<p->n_sm, SparseCfg<13>::NT, SparseCfg<13>::SMEM, p->stream>>>(
            (const float2*)p->stack, (const float2*)p->twiddle, maxc, p->sp_bits, p->sp_prefix, p->sp_list, p->sp_count, z_first,
            n_planes, p->z0 + z_first, p->dl, p->wrange, p->sp_imageT, accumulate, col_begin, col_end));
    } else {
        RICK_KERNEL(p, RK_COLS_WCORRECT, k_cols_sparse_wcorrect<14><<<p->n_sm, SparseCfg<14>::NT, SparseCfg<14>::SMEM, p->stream>>>(
            (const float2*)p->stack, (const float2*)p->twiddle, maxc, p->sp_bits, p->sp_prefix, p->sp_list, p->sp_count, z_first,
            n_planes, p->z0 + z_first, p->dl, p->wrange, p->sp_imageT, accumulate, col_begin, col_end));
    }
    return RICK_OK;
}

// after the last batch: the transposed image becomes the image (divided by the taper when fuse_taper)
// (image columns [col_begin, col_end), multiples of 32; col_end < 0: to the last column)
int rick_sparse_finish(rick_plan_t* p, double* image, int fuse_taper, int col_begin, int col_end)
{
    if (col_end < 0) col_end = p->N;
    if (col_end <= col_begin) return RICK_OK;
    dim3 grid((unsigned)((col_end - col_begin) / 32), (unsigned)(p->N / 32));
    RICK_KERNEL(p, RK_TAPER, k_image_transpose_taper<<<grid, 256, 0, p->stream>>>(p->sp_imageT, image, p->N,
                                                                                 fuse_taper ? p->taper : nullptr,
                                                                                 p->sp_count + p->Nw, p->N / 2, col_begin));
    return RICK_OK;
}
