// wcorrect.cu -- a5: w-term phase screen + sum over w-planes (Eq. 2, PAPER.md:50; :69;
// reading R2), a6: grid correction (reading R12).
//
//   I_raw[q][p] = sum_z Re( P_z[q][p] * exp(+2 pi i w_z (n-1)) ),  n-1 = -r2 / (1 + sqrt(1-r2)),
//   r2 = l^2 + m^2, l = (p-N/2) dl, m = (q-N/2) dl, w_z = w_min + (z + 0.5) dw;  r2 >= 1 -> 0.
//   I = I_raw / (c(nu_p) c(nu_q))
//
// One coalesced pass over the stack: a thread owns one pixel and walks the planes.  The
// planes are equally spaced in w, so the screen is a geometric sequence in z:
// phase_z = phase_0 * step^z -- two sincospi per pixel, then one complex multiply per plane
// instead of a sincos per pixel per plane (which would make the pass ALU-bound in fp64).
#include "common.cuh"

template <typename C>
__global__ void __launch_bounds__(256)
k_wcorrect(const C* __restrict__ stack, int n_planes, int z_first, int N, double dl,
           const WRange* __restrict__ wr, double* __restrict__ image, int accumulate,
           const double* __restrict__ taper)
{
    const size_t NN = (size_t)N * N;
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= NN) return;
    const int q = (int)(pix / N), p = (int)(pix - (size_t)q * N);
    const double l = (double)(p - N / 2) * dl, m = (double)(q - N / 2) * dl;
    const double r2 = l * l + m * m;
    double acc = 0.0;
    if (r2 < 1.0) {
        const double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
        const double w0 = wr->w_min + ((double)z_first + 0.5) * wr->dw;
        double x0 = w0 * nm1, xs = wr->dw * nm1;
        x0 -= rint(x0);
        xs -= rint(xs);
        double pr, pi, sr, si;
        sincospi(2.0 * x0, &pi, &pr);
        sincospi(2.0 * xs, &si, &sr);
        const C* g = stack + pix;
        int z = 0;
        for (; z + 4 <= n_planes; z += 4) {
            const C a0 = g[(size_t)(z + 0) * NN], a1 = g[(size_t)(z + 1) * NN];
            const C a2 = g[(size_t)(z + 2) * NN], a3 = g[(size_t)(z + 3) * NN];
            double t;
            acc += (double)a0.x * pr - (double)a0.y * pi;
            t = pr * sr - pi * si; pi = pr * si + pi * sr; pr = t;
            acc += (double)a1.x * pr - (double)a1.y * pi;
            t = pr * sr - pi * si; pi = pr * si + pi * sr; pr = t;
            acc += (double)a2.x * pr - (double)a2.y * pi;
            t = pr * sr - pi * si; pi = pr * si + pi * sr; pr = t;
            acc += (double)a3.x * pr - (double)a3.y * pi;
            t = pr * sr - pi * si; pi = pr * si + pi * sr; pr = t;
        }
        for (; z < n_planes; ++z) {
            const C a = g[(size_t)z * NN];
            acc += (double)a.x * pr - (double)a.y * pi;
            const double t = pr * sr - pi * si;
            pi = pr * si + pi * sr;
            pr = t;
        }
    }
    if (accumulate) acc += image[pix];
    if (taper) acc /= (taper[p] * taper[q]);
    image[pix] = acc;
}

__global__ void __launch_bounds__(256)
k_taper_divide(double* __restrict__ image, int N, const double* __restrict__ taper)
{
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= (size_t)N * N) return;
    const int q = (int)(pix / N), p = (int)(pix - (size_t)q * N);
    image[pix] = image[pix] / (taper[p] * taper[q]);
}

int rick_wcorrect(rick_plan_t* p, int img, int z_first, int n_planes, double* image, int accumulate,
                  int fuse_taper, int slot_first)
{
    const size_t NN = (size_t)p->N * p->N;
    const unsigned int blocks = (unsigned int)((NN + 255) / 256);
    const double* tp = fuse_taper ? p->taper : nullptr;
    if (p->f32) {
        RICK_KERNEL(p, RK_WCORRECT, k_wcorrect<float2><<<blocks, 256, 0, p->stream>>>(
            (const float2*)p->stack + (size_t)slot_first * p->N * p->N, n_planes, p->z0 + z_first, p->N, p->dl, p->wrange + img, image, accumulate, tp));
    } else {
        RICK_KERNEL(p, RK_WCORRECT, k_wcorrect<double2><<<blocks, 256, 0, p->stream>>>(
            (const double2*)p->stack + (size_t)slot_first * p->N * p->N, n_planes, p->z0 + z_first, p->N, p->dl, p->wrange + img, image, accumulate, tp));
    }
    return RICK_OK;
}

int rick_taper_divide(rick_plan_t* p, double* image)
{
    const size_t NN = (size_t)p->N * p->N;
    RICK_KERNEL(p, RK_TAPER, k_taper_divide<<<(unsigned int)((NN + 255) / 256), 256, 0, p->stream>>>(image, p->N, p->taper));
    return RICK_OK;
}
