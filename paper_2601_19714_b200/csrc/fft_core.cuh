// fft_core.cuh -- in-register Stockham FFT building blocks (a4).
//
// Transform: X[k] = sum_n x[n] e^{+2 pi i n k / N}  (unnormalised, + sign; reading R11).
// N = 16^A * 2^REM: A radix-16 stages then one radix-2^REM stage.  Every thread of a
// transform holds E = 16 elements, x[t + NT*e] (NT = N/16), in registers in EVERY stage
// (Stockham autosort: a stage reads positions t + NT*e and writes positions
// (j/Ns)*Ns*R + (j mod Ns) + r*Ns), so global loads / stores are coalesced and only the
// inter-stage exchanges go through shared memory.  Twiddles: one table load w1 = tw[...] per
// butterfly, the powers w1^r by <= 4-deep multiplication.
// The centring of the transform (origin at cell N/2; readings R9, R11) is an index ROTATION by
// N/2 on input and output, which in this layout is the register renaming e -> (e+8) mod 16
// (see fft.cu) -- no checkerboard multiplications.
#pragma once
#include <cuda_runtime.h>

// n - 1 = sqrt(1 - r2) - 1 without cancellation, r2 = l^2 + m^2 < 1 (the w-term of Eq. 2).  Small
// fields take the binomial series (no square root, no division): its first neglected term is 2e-19 relative at
// r2 = 1/128; beyond that the closed form -r2 / (1 + sqrt(1 - r2)).
__device__ __forceinline__ double nm1_of(double r2)
{
    if (r2 < 0.0078125) {
        double s = 429.0 / 32768.0;
        s = fma(s, r2, 33.0 / 2048.0);
        s = fma(s, r2, 21.0 / 1024.0);
        s = fma(s, r2, 7.0 / 256.0);
        s = fma(s, r2, 5.0 / 128.0);
        s = fma(s, r2, 1.0 / 16.0);
        s = fma(s, r2, 1.0 / 8.0);
        s = fma(s, r2, 0.5);
        return -(s * r2);
    }
    return -r2 / (1.0 + sqrt(1.0 - r2));
}

template <typename T> struct cplx_of;
template <> struct cplx_of<double> { typedef double2 type; };
template <> struct cplx_of<float> { typedef float2 type; };

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b)
{
    C r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
// multiply by +i
template <typename C> __device__ __forceinline__ C cmuli(C a) { C r; r.x = -a.y; r.y = a.x; return r; }

template <typename C> __device__ __forceinline__ void fft2(C& a0, C& a1)
{
    C t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}

// 4-point, + sign, natural order in and out
template <typename C> __device__ __forceinline__ void fft4(C& a0, C& a1, C& a2, C& a3)
{
    C t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = cmuli(csub(a1, a3));
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, t3);
    a3 = csub(t1, t3);
}

// (a + i b) * e^{+i pi/4} and * e^{+3 i pi/4}
template <typename T, typename C> __device__ __forceinline__ C cmul_w8_1(C a)
{
    const T s = (T)0.70710678118654752440;
    C r; r.x = (a.x - a.y) * s; r.y = (a.x + a.y) * s; return r;
}
template <typename T, typename C> __device__ __forceinline__ C cmul_w8_3(C a)
{
    const T s = (T)0.70710678118654752440;
    C r; r.x = -(a.x + a.y) * s; r.y = (a.x - a.y) * s; return r;
}

// 8-point: on exit b[2*k1 + k2] = X[k1 + 4*k2]
template <typename T, typename C> __device__ __forceinline__ void fft8(C (&b)[8])
{
    fft4(b[0], b[2], b[4], b[6]);     // n2 = 0 -> y[0][k1] in b[2*k1]
    fft4(b[1], b[3], b[5], b[7]);     // n2 = 1 -> y[1][k1] in b[2*k1+1]
    b[3] = cmul_w8_1<T>(b[3]);        // W8^1
    b[5] = cmuli(b[5]);               // W8^2 = i
    b[7] = cmul_w8_3<T>(b[7]);        // W8^3
    fft2(b[0], b[1]);
    fft2(b[2], b[3]);
    fft2(b[4], b[5]);
    fft2(b[6], b[7]);
}

// 16-point: on exit b[4*k1 + k2] = X[k1 + 4*k2]
template <typename T, typename C> __device__ __forceinline__ void fft16(C (&b)[16])
{
    const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173;
    fft4(b[0], b[4], b[8], b[12]);    // n2 = 0: y[0][k1] -> b[4*k1 + 0]
    fft4(b[1], b[5], b[9], b[13]);
    fft4(b[2], b[6], b[10], b[14]);
    fft4(b[3], b[7], b[11], b[15]);
    // b[4*k1 + n2] *= W16^{n2*k1}
    C w;
    w.x = c1; w.y = s1;   b[5] = cmul(b[5], w);        // W16^1
    b[6] = cmul_w8_1<T>(b[6]);                          // W16^2
    w.x = s1; w.y = c1;   b[7] = cmul(b[7], w);        // W16^3
    b[9] = cmul_w8_1<T>(b[9]);                          // W16^2
    b[10] = cmuli(b[10]);                               // W16^4
    b[11] = cmul_w8_3<T>(b[11]);                        // W16^6
    w.x = s1; w.y = c1;   b[13] = cmul(b[13], w);      // W16^3
    b[14] = cmul_w8_3<T>(b[14]);                        // W16^6
    w.x = -c1; w.y = -s1; b[15] = cmul(b[15], w);      // W16^9
    fft4(b[0], b[1], b[2], b[3]);
    fft4(b[4], b[5], b[6], b[7]);
    fft4(b[8], b[9], b[10], b[11]);
    fft4(b[12], b[13], b[14], b[15]);
}

// register of leg r (= output index X[r]) after fftR
template <int R> __device__ __forceinline__ constexpr int leg_reg(int r)
{
    return R == 16 ? 4 * (r & 3) + (r >> 2) : (R == 8 ? 2 * (r & 3) + (r >> 2) : r);
}

template <typename T, int R, typename C> __device__ __forceinline__ void fftR(C (&b)[R])
{
    if constexpr (R == 16) fft16<T>(b);
    else if constexpr (R == 8) fft8<T>(b);
    else if constexpr (R == 4) fft4(b[0], b[1], b[2], b[3]);
    else fft2(b[0], b[1]);
}

__device__ __forceinline__ int fft_pad(int i) { return i + (i >> 4); }

// One Stockham stage.  v[e] = x[t + NT*e] on entry.  WC = columns interleaved in shared
// memory (element stride), c = this thread's column.  LAST: results stay in registers with
// v[e] = X[t + NT*e]; otherwise they go through shared memory and v[e] is reloaded.
template <typename T, int LOG2N, int R, int LOG2NS, bool LAST>
__device__ __forceinline__ void fft_stage(typename cplx_of<T>::type (&v)[16], const int t,
                                          typename cplx_of<T>::type* __restrict__ sm, const int WC,
                                          const int c,
                                          const typename cplx_of<T>::type* __restrict__ tw)
{
    typedef typename cplx_of<T>::type C;
    constexpr int N = 1 << LOG2N, NT = N / 16, NB = 16 / R, NS = 1 << LOG2NS;
    constexpr int LOG2R = R == 16 ? 4 : (R == 8 ? 3 : (R == 4 ? 2 : 1));
#pragma unroll
    for (int m = 0; m < NB; ++m) {
        C b[R];
#pragma unroll
        for (int r = 0; r < R; ++r) b[r] = v[m + r * NB];
        const int j = t + NT * m;
        const int jm = j & (NS - 1);
        if constexpr (LOG2NS > 0) {
            const C w1 = tw[jm * (N / (NS * R))];
            b[1] = cmul(b[1], w1);
            if constexpr (R >= 4) {
                const C w2 = cmul(w1, w1);
                const C w3 = cmul(w2, w1);
                b[2] = cmul(b[2], w2);
                b[3] = cmul(b[3], w3);
                if constexpr (R >= 8) {
                    const C w4 = cmul(w2, w2);
                    b[4] = cmul(b[4], w4);
                    b[5] = cmul(b[5], cmul(w4, w1));
                    b[6] = cmul(b[6], cmul(w4, w2));
                    const C w7 = cmul(w4, w3);
                    b[7] = cmul(b[7], w7);
                    if constexpr (R >= 16) {
                        const C w8 = cmul(w4, w4);
                        b[8] = cmul(b[8], w8);
                        b[9] = cmul(b[9], cmul(w8, w1));
                        b[10] = cmul(b[10], cmul(w8, w2));
                        b[11] = cmul(b[11], cmul(w8, w3));
                        const C w12 = cmul(w8, w4);
                        b[12] = cmul(b[12], w12);
                        b[13] = cmul(b[13], cmul(w12, w1));
                        b[14] = cmul(b[14], cmul(w12, w2));
                        b[15] = cmul(b[15], cmul(w8, w7));
                    }
                }
            }
        }
        fftR<T, R>(b);
        if constexpr (LAST) {
#pragma unroll
            for (int r = 0; r < R; ++r) v[m + r * NB] = b[leg_reg<R>(r)];
        } else {
            const int pos0 = ((j >> LOG2NS) << (LOG2NS + LOG2R)) + jm;
#pragma unroll
            for (int r = 0; r < R; ++r) sm[fft_pad(pos0 + r * NS) * WC + c] = b[leg_reg<R>(r)];
        }
    }
    if constexpr (!LAST) {
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = sm[fft_pad(t + NT * e) * WC + c];
        __syncthreads();
    }
}

// Whole length-N transform of the 16 elements per thread.
template <typename T, int LOG2N>
__device__ __forceinline__ void fft_thread(typename cplx_of<T>::type (&v)[16], const int t,
                                           typename cplx_of<T>::type* __restrict__ sm, const int WC,
                                           const int c,
                                           const typename cplx_of<T>::type* __restrict__ tw)
{
    constexpr int A = LOG2N / 4, REM = LOG2N % 4;
    static_assert(A >= 1 && A <= 3, "supported N: 16 .. 32768");
    if constexpr (A == 1) {
        if constexpr (REM == 0) fft_stage<T, LOG2N, 16, 0, true>(v, t, sm, WC, c, tw);
        else {
            fft_stage<T, LOG2N, 16, 0, false>(v, t, sm, WC, c, tw);
            fft_stage<T, LOG2N, (1 << REM), 4, true>(v, t, sm, WC, c, tw);
        }
    } else if constexpr (A == 2) {
        fft_stage<T, LOG2N, 16, 0, false>(v, t, sm, WC, c, tw);
        if constexpr (REM == 0) fft_stage<T, LOG2N, 16, 4, true>(v, t, sm, WC, c, tw);
        else {
            fft_stage<T, LOG2N, 16, 4, false>(v, t, sm, WC, c, tw);
            fft_stage<T, LOG2N, (1 << REM), 8, true>(v, t, sm, WC, c, tw);
        }
    } else {
        fft_stage<T, LOG2N, 16, 0, false>(v, t, sm, WC, c, tw);
        fft_stage<T, LOG2N, 16, 4, false>(v, t, sm, WC, c, tw);
        if constexpr (REM == 0) fft_stage<T, LOG2N, 16, 8, true>(v, t, sm, WC, c, tw);
        else {
            fft_stage<T, LOG2N, 16, 8, false>(v, t, sm, WC, c, tw);
            fft_stage<T, LOG2N, (1 << REM), 12, true>(v, t, sm, WC, c, tw);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Building blocks of the N = 4096 = 16^3 column kernels (fft_cols12.cu): one radix-16 stage on
// the 16 registers of a thread, and the two inter-stage exchanges through a DOUBLE buffer
// (real parts, then imaginary parts: half the shared memory of a complex exchange).
// ------------------------------------------------------------------------------------------

// twiddle (NS = 2^LOG2NS butterflies already combined) + radix-16 butterfly over v[e] = x[t + (N/16) e];
// on exit v[r] = leg r in natural order.
// index of the thread's base twiddle w1 of the stage with NS = 2^LOG2NS butterflies combined
template <int LOG2N, int LOG2NS> __device__ __forceinline__ int bfly16_tw_index(const int t)
{
    constexpr int N = 1 << LOG2N, NS = 1 << LOG2NS;
    return (t & (NS - 1)) * (N / (NS * 16));
}

template <typename T, int LOG2N, int LOG2NS>
__device__ __forceinline__ void bfly16(typename cplx_of<T>::type (&v)[16], const int t,
                                       const typename cplx_of<T>::type* __restrict__ tw,
                                       const typename cplx_of<T>::type* w1_pre = nullptr)
{
    typedef typename cplx_of<T>::type C;
    if constexpr (LOG2NS > 0) {
        // w1_pre: the base twiddle already fetched by the caller (before an exchange, whose barriers the
        // load cannot be hoisted over)
        const C w1 = w1_pre ? *w1_pre : tw[bfly16_tw_index<LOG2N, LOG2NS>(t)];
        v[1] = cmul(v[1], w1);
        const C w2 = cmul(w1, w1);
        const C w3 = cmul(w2, w1);
        v[2] = cmul(v[2], w2);
        v[3] = cmul(v[3], w3);
        const C w4 = cmul(w2, w2);
        v[4] = cmul(v[4], w4);
        v[5] = cmul(v[5], cmul(w4, w1));
        v[6] = cmul(v[6], cmul(w4, w2));
        const C w7 = cmul(w4, w3);
        v[7] = cmul(v[7], w7);
        const C w8 = cmul(w4, w4);
        v[8] = cmul(v[8], w8);
        v[9] = cmul(v[9], cmul(w8, w1));
        v[10] = cmul(v[10], cmul(w8, w2));
        v[11] = cmul(v[11], cmul(w8, w3));
        const C w12 = cmul(w8, w4);
        v[12] = cmul(v[12], w12);
        v[13] = cmul(v[13], cmul(w12, w1));
        v[14] = cmul(v[14], cmul(w12, w2));
        v[15] = cmul(v[15], cmul(w8, w7));
    }
    fft16<T>(v);
    C o[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) o[r] = v[leg_reg<16>(r)];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = o[r];
}

// Exchange after stage 1 when a warp holds the roles t1 = w + 16 hh (hh = 0..15, two columns c
// interleaved): the Stockham permutation closes inside the warp -- a 16 x 16 transpose per column,
// writer hh leg r -> reader hh' = r element e = hh.  wb: this warp's 16*17*2 doubles.  No CTA barrier.
__device__ __forceinline__ void xchg16_warp(double2 (&v)[16], double* __restrict__ wb, const int hh, const int c)
{
#pragma unroll
    for (int r = 0; r < 16; ++r) wb[(hh * 17 + r) * 2 + c] = v[r].x;
    __syncwarp();
    double re[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) re[e] = wb[(e * 17 + hh) * 2 + c];
    __syncwarp();
#pragma unroll
    for (int r = 0; r < 16; ++r) wb[(hh * 17 + r) * 2 + c] = v[r].y;
    __syncwarp();
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        v[e].y = wb[(e * 17 + hh) * 2 + c];
        v[e].x = re[e];
    }
    __syncwarp();
}

// Exchange after stage 2 (NS = 16), CTA-wide: writer role t2 leg r -> position pos0 + 16 r;
// reader role t3 element e <- position t3 + 256 e.  sm: 2 * (4096 + 256) doubles.
__device__ __forceinline__ void xchg16_cta(double2 (&v)[16], double* __restrict__ sm, const int t2, const int t3,
                                           const int c)
{
    const int pos0 = ((t2 >> 4) << 8) + (t2 & 15);
#pragma unroll
    for (int r = 0; r < 16; ++r) sm[fft_pad(pos0 + r * 16) * 2 + c] = v[r].x;
    __syncthreads();
    double re[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) re[e] = sm[fft_pad(t3 + 256 * e) * 2 + c];
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 16; ++r) sm[fft_pad(pos0 + r * 16) * 2 + c] = v[r].y;
    __syncthreads();
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        v[e].y = sm[fft_pad(t3 + 256 * e) * 2 + c];
        v[e].x = re[e];
    }
}

// ------------------------------------------------------------------------------------------
// The same two exchanges for a CTA split into two COLUMN GROUPS of 256 threads (k_cols12_wcorrect):
// a group owns one column of the strip, role (w, hh) = (tg >> 4, tg & 15), so a warp holds two
// values of w (wl = lane >> 4) and all 16 hh.  Only group-wide named barriers (`bar_id`, 256
// threads): the two groups run out of phase, one in its butterflies while the other exchanges.
// ------------------------------------------------------------------------------------------

// after stage 1: 16 x 16 transpose among the hh of one w, inside the warp.  wb: this warp's 2*16*17 doubles.
__device__ __forceinline__ void xchg16_warp_grp(double2 (&v)[16], double* __restrict__ wb, const int wl, const int hh)
{
    double* b = wb + wl * (16 * 17);
#pragma unroll
    for (int r = 0; r < 16; ++r) b[hh * 17 + r] = v[r].x;
    __syncwarp();
    double re[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) re[e] = b[e * 17 + hh];
    __syncwarp();
#pragma unroll
    for (int r = 0; r < 16; ++r) b[hh * 17 + r] = v[r].y;
    __syncwarp();
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        v[e].y = b[e * 17 + hh];
        v[e].x = re[e];
    }
    __syncwarp();
}

// after stage 2, group-wide: writer role t2 leg r -> position pos0 + 16 r; reader element e <- position
// t2 + 256 e.  gb: the group's 4096 + 256 doubles.
__device__ __forceinline__ void xchg16_grp(double2 (&v)[16], double* __restrict__ gb, const int t2, const int bar_id)
{
    const int pos0 = ((t2 >> 4) << 8) + (t2 & 15);
#pragma unroll
    for (int r = 0; r < 16; ++r) gb[fft_pad(pos0 + r * 16)] = v[r].x;
    asm volatile("bar.sync %0, 256;\n" ::"r"(bar_id) : "memory");
    double re[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) re[e] = gb[fft_pad(t2 + 256 * e)];
    asm volatile("bar.sync %0, 256;\n" ::"r"(bar_id) : "memory");
#pragma unroll
    for (int r = 0; r < 16; ++r) gb[fft_pad(pos0 + r * 16)] = v[r].y;
    asm volatile("bar.sync %0, 256;\n" ::"r"(bar_id) : "memory");
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        v[e].y = gb[fft_pad(t2 + 256 * e)];
        v[e].x = re[e];
    }
}
