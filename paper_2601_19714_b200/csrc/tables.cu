// tables.cu -- plan-time tables: FFT twiddles, taper vector, Kaiser-Bessel series.
//
// Kaiser-Bessel kernel (reading R5):
//   g(t) = I0(beta sqrt(y)) / I0(beta),  y = 1 - (2t/S)^2,
// and I0(beta sqrt(y)) = sum_k (beta^2/4)^k y^k / (k!)^2 is a power series in y with positive
// coefficients, so g is evaluated by Horner in y on the device (kb_coef[k] = c_k / I0(beta)).
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
}

int rick_tables_build(rick_plan_t* p)
{
    const int N = p->N;
    // series coefficients on the host in long double (<= RICK_MAX_KB_TERMS numbers)
    std::vector<long double> c;
    long double q = 0.25L * (long double)p->beta * (long double)p->beta, term = 1.0L, i0 = 1.0L;
    c.push_back(1.0L);
    for (int k = 1; k < 400; ++k) {
        term *= q / ((long double)k * (long double)k);
        c.push_back(term);
        i0 += term;
        if (term < 1e-21L * i0) break;
    }
    if ((int)c.size() > RICK_MAX_KB_TERMS) {
        p->err = "kb_beta too large for the kernel series";
        return RICK_ERR_INVALID;
    }
    p->kb_terms = (int)c.size();
    std::vector<double> cd(c.size());
    for (size_t k = 0; k < c.size(); ++k) cd[k] = (double)(c[k] / i0);
    RICK_CUDA(p, cudaMalloc(&p->kb_coef, sizeof(double) * RICK_MAX_KB_TERMS));
    RICK_CUDA(p, cudaMemcpyAsync(p->kb_coef, cd.data(), sizeof(double) * cd.size(),
                                 cudaMemcpyHostToDevice, p->stream));
    RICK_CUDA(p, cudaStreamSynchronize(p->stream));   // cd is a local

    RICK_CUDA(p, cudaMalloc(&p->taper, sizeof(double) * N));
    RICK_KERNEL(p, RK_TABLES, k_taper<<<(N + 255) / 256, 256, 0, p->stream>>>(p->taper, N, p->S, p->beta, (double)i0));

    RICK_CUDA(p, cudaMalloc(&p->twiddle, (p->f32 ? sizeof(float2) : sizeof(double2)) * (size_t)N));
    if (p->f32) {
        RICK_KERNEL(p, RK_TABLES, k_twiddle<float2><<<(N + 255) / 256, 256, 0, p->stream>>>((float2*)p->twiddle, N));
    } else {
        RICK_KERNEL(p, RK_TABLES, k_twiddle<double2><<<(N + 255) / 256, 256, 0, p->stream>>>((double2*)p->twiddle, N));
    }
    return RICK_OK;
}
