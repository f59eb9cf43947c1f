// tables.cu -- plan-time tables: FFT twiddles, taper vector, Kaiser-Bessel tap polynomials.
//
// Kaiser-Bessel kernel (reading R5):
//   g(t) = I0(beta sqrt(y)) / I0(beta),  y = 1 - (2t/S)^2,   I0(x) = sum_k (x^2/4)^k / (k!)^2.
// The gridder needs g only at d_a = (a-h) - delta, |delta| <= 1/2, i.e. tap a sees one unit interval
// of t.  On it g is fitted here (host, long double) by Chebyshev interpolation of degree RICK_KB_DEG in
// s = 2 delta, converted to monomial coefficients, and CHECKED against the series at 257 points: a
// plan whose fit is worse than 1e-14 (beta far above ~4 S) is refused.
// Taper (reading R12): closed-form transform of g,
//   c(nu) = (S / I0(beta)) sinh(sqrt(a)) / sqrt(a),  a = beta^2 - (pi S nu)^2.
#include "common.cuh"

#include <math.h>
#include <vector>

template <typename T2>
__global__ void k_twiddle(T2* __restrict__ tw, int N)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    double s, c;
    sincospi(2.0 * (double)k / (double)N, &s, &c);
    T2 v;
    v.x = c;
    v.y = s;
    tw[k] = v;
}

__global__ void k_taper(double* __restrict__ taper, int N, int S, double beta, double i0_beta)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const double PI = 3.14159265358979323846;
    double nu = (double)(p - N / 2) / (double)N;
    double x = PI * (double)S * nu;
    double a = beta * beta - x * x;
    double f;
    if (fabs(a) < 1e-6) {
        f = 1.0 + a / 6.0;
    } else if (a > 0.0) {
        double r = sqrt(a);
        f = sinh(r) / r;
    } else {
        double r = sqrt(-a);
        f = sin(r) / r;
    }
    taper[p] = (double)S / i0_beta * f;
    taper[N + p] = 1.0 / taper[p];          // [N .. 2N): the reciprocals (the fused column kernels multiply)
}

static long double i0_series(long double x)
{
    const long double q = 0.25L * x * x;
    long double term = 1.0L, sum = 1.0L;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((long double)k * (long double)k);
        sum += term;
        if (term < 1e-22L * sum) break;
    }
    return sum;
}

static long double kb_exact(long double t, int S, long double beta, long double i0_beta)
{
    const long double r = 2.0L * t / (long double)S;
    long double y = 1.0L - r * r;
    if (y < 0.0L) y = 0.0L;
    return i0_series(beta * sqrtl(y)) / i0_beta;
}

int rick_tables_build(rick_plan_t* p)
{
    const int N = p->N, S = p->S, h = p->h;
    constexpr int D = RICK_KB_DEG, NN = D + 1;
    const long double PI = 3.14159265358979323846264338327950288L;
    const long double beta = (long double)p->beta;
    const long double i0 = i0_series(beta);
    long double worst = 0.0L;
    for (int a = 0; a < S; ++a) {
        // Chebyshev coefficients of f(s) = g((a-h) - s/2) on [-1,1] from its values at the nodes
        long double fv[NN], cheb[NN], mono[NN], Tm[NN], Tc[NN], Tn[NN];
        for (int k = 0; k < NN; ++k) {
            const long double sk = cosl(PI * (2.0L * k + 1.0L) / (2.0L * NN));
            fv[k] = kb_exact((long double)(a - h) - 0.5L * sk, S, beta, i0);
        }
        for (int j = 0; j < NN; ++j) {
            long double acc = 0.0L;
            for (int k = 0; k < NN; ++k) acc += fv[k] * cosl(PI * j * (2.0L * k + 1.0L) / (2.0L * NN));
            cheb[j] = acc * (j == 0 ? 1.0L : 2.0L) / (long double)NN;
        }
        // sum_j cheb[j] T_j(s) -> monomials, T_{j+1} = 2 s T_j - T_{j-1}
        for (int k = 0; k < NN; ++k) { mono[k] = 0.0L; Tm[k] = 0.0L; Tc[k] = 0.0L; }
        Tm[0] = 1.0L;                     // T_0
        Tc[1] = 1.0L;                     // T_1
        mono[0] += cheb[0];
        if (NN > 1) mono[1] += cheb[1];
        for (int j = 2; j < NN; ++j) {
            for (int k = 0; k < NN; ++k) Tn[k] = (k > 0 ? 2.0L * Tc[k - 1] : 0.0L) - Tm[k];
            for (int k = 0; k < NN; ++k) { mono[k] += cheb[j] * Tn[k]; Tm[k] = Tc[k]; Tc[k] = Tn[k]; }
        }
        for (int k = 0; k < NN; ++k) p->kb_poly[a * NN + k] = (double)mono[k];
        // g is even: the mirror tap is f_{S-1-a}(s) = f_a(-s) and the centre tap is an even function.
        // The gridder evaluates only the taps a <= h and uses exactly this symmetry, so impose it on
        // the table the check below runs on.
        if (a > h)
            for (int k = 0; k < NN; ++k) p->kb_poly[a * NN + k] = ((k & 1) ? -1.0 : 1.0) * p->kb_poly[(S - 1 - a) * NN + k];
        if (a == h)
            for (int k = 1; k < NN; k += 2) p->kb_poly[a * NN + k] = 0.0;
        // check the double-precision Horner evaluation against the series
        for (int i = 0; i <= 256; ++i) {
            const double sd = -1.0 + (double)i / 128.0;
            double acc = p->kb_poly[a * NN + D];
            for (int k = D - 1; k >= 0; --k) acc = fma(acc, sd, p->kb_poly[a * NN + k]);
            const long double ex = kb_exact((long double)(a - h) - 0.5L * (long double)sd, S, beta, i0);
            const long double e = fabsl((long double)acc - ex);
            if (e > worst) worst = e;
        }
    }
    if (!(worst < 1e-14L)) {
        p->err = "kb_beta too large for this support: the per-tap polynomial fit of the kernel is not accurate";
        return RICK_ERR_INVALID;
    }

    RICK_CUDA(p, cudaMalloc(&p->taper, sizeof(double) * 2 * N));
    RICK_KERNEL(p, RK_TABLES, k_taper<<<(N + 255) / 256, 256, 0, p->stream>>>(p->taper, N, p->S, p->beta, (double)i0));

    RICK_CUDA(p, cudaMalloc(&p->twiddle, (p->f32 ? sizeof(float2) : sizeof(double2)) * (size_t)N));
    if (p->f32) {
        RICK_KERNEL(p, RK_TABLES, k_twiddle<float2><<<(N + 255) / 256, 256, 0, p->stream>>>((float2*)p->twiddle, N));
    } else {
        RICK_KERNEL(p, RK_TABLES, k_twiddle<double2><<<(N + 255) / 256, 256, 0, p->stream>>>((double2*)p->twiddle, N));
    }
    if (rick_cols2_on(p)) {      // table of the length-N/16 sub-transforms of the two-pass column pass
        const int N2 = N / 16;
        RICK_CUDA(p, cudaMalloc(&p->twiddle2, (p->f32 ? sizeof(float2) : sizeof(double2)) * (size_t)N2));
        if (p->f32) {
            RICK_KERNEL(p, RK_TABLES, k_twiddle<float2><<<(N2 + 255) / 256, 256, 0, p->stream>>>((float2*)p->twiddle2, N2));
        } else {
            RICK_KERNEL(p, RK_TABLES, k_twiddle<double2><<<(N2 + 255) / 256, 256, 0, p->stream>>>((double2*)p->twiddle2, N2));
        }
    }
    return RICK_OK;
}
