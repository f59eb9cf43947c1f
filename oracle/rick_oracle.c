/*
 * rick_oracle.c -- CPU ORACLE for the w-stacking imaging hot path of RICK 2.0
 * (arxiv/paper_2601_19714).  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product
 * (paper_2601_19714_b200/, librick_b200.so) never does, shares no code,
 * header, table or constant generator with it, and neither imports the other.
 *
 * Plain, slow, obviously correct: fp64 throughout, the algorithm step by step
 * in the paper's order (the method is an APPROXIMATION of the direct sum --
 * nearest-w-plane quantisation and a finite-support kernel -- so the oracle is
 * the algorithm, and rko_dft below is the plain definition it is pinned to):
 *
 *   Eq. 1  PAPER.md:45   measurement equation (signs)         -> rko_dft
 *   :48                  "mapped to the closest w-plane"      -> rko_index
 *   Eq. 3  PAPER.md:64   V~(u_i,v_j,w_k) = sum_m V_m G(...)    -> rko_grid_plane
 *   :62                  G = Kaiser-Bessel                    -> rko_kb
 *   Eq. 5  PAPER.md:129  halo = (Kernel-1)/2 cells            -> on-grid rule
 *   :53 / :68            each w-plane Fourier transformed     -> rko_fft2_centered
 *   Eq. 2  PAPER.md:50   e^{+2 pi i w (n-1)} screen, plane sum -> rko_wcorrect_accumulate
 *   (paper silent)       division by the kernel's transform   -> rko_taper / rko_gridcorrect
 *
 * Every reading of a silent / garbled passage is DESIGN.md's "Readings" list
 * (R1..R21, the same numbers as SURVEY.md 8(c)).  No blocking, fusion or
 * reordering beyond those statements.  OpenMP only splits independent rows /
 * pixels / grid-row bands; every sum keeps visibility-index order, so results
 * do not depend on the thread count.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): direct DFT on tiny inputs,
 * closed forms, mass invariant, Parseval, numpy.fft, scipy.special.i0, the
 * O(N^4) DFT definition, hand-computed index cases.  Nothing is "parity
 * unpinned".
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define RKO_C0 299792458.0
#define RKO_PI 3.14159265358979323846264338327950288
#define RKO_KEY_DROPPED 0xFFFFFFFFFFFFFFFFull

/* ------------------------------------------------------------------------ */
/* Kaiser-Bessel kernel (reading R5: exact evaluation, g(0)=1)  */
/* ------------------------------------------------------------------------ */

/* I0(x) = sum_k ((x/2)^2)^k / (k!)^2 ; all terms positive, no cancellation. */
double rko_bessel_i0(double x)
{
    double q = 0.25 * x * x, term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-20 * sum) break;
    }
    return sum;
}

/* g(t) = I0(beta sqrt(1-(2t/S)^2)) / I0(beta), |t| <= S/2 ; 0 outside. */
double rko_kb(double t, int S, double beta)
{
    double r = 2.0 * t / (double)S;
    double y = 1.0 - r * r;
    if (y < 0.0) {
        if (y < -1e-12) return 0.0;
        y = 0.0;
    }
    return rko_bessel_i0(beta * sqrt(y)) / rko_bessel_i0(beta);
}

/* Gauss-Legendre nodes/weights on [-1,1] by Newton iteration on P_n. */
static void gauss_legendre(int n, double *x, double *w)
{
    for (int i = 0; i < n; ++i) {
        double z = cos(RKO_PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double z1 = z;
            z = z1 - p1 / pp;
            if (fabs(z - z1) < 1e-16) break;
        }
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* c(nu) = int_{-S/2}^{S/2} g(t) cos(2 pi nu t) dt, by quadrature (reading R12).
 * Deliberately NOT the closed form the CUDA path uses. */
double rko_taper(double nu, int S, double beta)
{
    enum { NQ = 160 };
    static double x[NQ], w[NQ];
    static int ready = 0;
#pragma omp critical(rko_gl)
    {
        if (!ready) { gauss_legendre(NQ, x, w); ready = 1; }
    }
    double half = 0.5 * (double)S, acc = 0.0;
    for (int i = 0; i < NQ; ++i) {
        double t = half * x[i];
        acc += w[i] * rko_kb(t, S, beta) * cos(2.0 * RKO_PI * nu * t);
    }
    return half * acc;
}

/* ------------------------------------------------------------------------ */
/* Steps 1-4: scales, index, plane, key              */
/* ------------------------------------------------------------------------ */

/* Visibility k = r*C + c.  Outputs per visibility: iu, iv (centre cell), ip
 * (plane of its image), key (64-bit; all ones when dropped), xu, xv (cell
 * coordinates from the grid centre).
 * key = ((((img*N_w + i_p)*T + i_v/B)*T + i_u/B)*B + i_v%B)*B + i_u%B
 * (image, plane, uv tile of B x B cells, cell inside the tile: DESIGN.md
 * step 4 / reading R22 -- the paper's bucket sort, leaves
 * the order inside a bucket open).  w_min/w_max: [n_img] (n_img = C when
 * cube, else 1); on input NaN -> derived from ALL visibilities of that image
 * (on-grid or not).  Each operation individually rounded (no FMA; build with
 * -ffp-contract=off), in exactly this order. */
int rko_index(int64_t n_rows, int32_t n_chan, const double *uvw_m, const double *freq_hz,
              int32_t N, int32_t Nw, int32_t S, double dl, int32_t B, int32_t cube,
              double *w_min, double *w_max,
              int32_t *iu, int32_t *iv, int32_t *ip, uint64_t *key, double *xu, double *xv)
{
    const int32_t h = (S - 1) / 2, T = N / B;
    const double inv_du = (double)N * dl;
    const double shift = (double)(N / 2) + 0.5;
    const int32_t n_img = cube ? n_chan : 1;
    double *s = (double *)malloc(sizeof(double) * (size_t)n_chan);
    for (int32_t c = 0; c < n_chan; ++c) s[c] = freq_hz[c] / RKO_C0;

    /* w range per image over all (r,c) of that image */
    for (int32_t g = 0; g < n_img; ++g) {
        if (w_min[g] == w_min[g] && w_max[g] == w_max[g]) continue; /* given */
        double lo = INFINITY, hi = -INFINITY;
        for (int64_t r = 0; r < n_rows; ++r)
            for (int32_t c = 0; c < n_chan; ++c) {
                if (cube && c != g) continue;
                double wl = uvw_m[3 * r + 2] * s[c];
                if (!isfinite(wl)) continue;   /* R23: a non-finite w takes no part in the range */
                if (wl < lo) lo = wl;
                if (wl > hi) hi = wl;
            }
        if (!(lo <= hi)) { lo = 0.0; hi = 0.0; }   /* no (finite) row at all */
        w_min[g] = lo;
        w_max[g] = hi;
    }

#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n_rows; ++r) {
        for (int32_t c = 0; c < n_chan; ++c) {
            const int64_t k = r * n_chan + c;
            const int32_t img = cube ? c : 0;
            double t, x_u, x_v;
            t = uvw_m[3 * r + 0] * s[c];
            x_u = t * inv_du;
            t = uvw_m[3 * r + 1] * s[c];
            x_v = t * inv_du;
            const double dw = (w_max[img] - w_min[img]) / (double)Nw;
            const double inv_dw = dw > 0.0 ? 1.0 / dw : 0.0;
            double wl = uvw_m[3 * r + 2] * s[c];
            /* R23: a visibility with a non-finite u, v or w cannot lie on the grid -> dropped
             * (R10); coordinates beyond the int range likewise (the casts below stay defined). */
            const double f_u = floor(x_u + shift), f_v = floor(x_v + shift);
            const int fin = isfinite(x_u) && isfinite(x_v) && isfinite(wl) &&
                            fabs(f_u) < 2147483000.0 && fabs(f_v) < 2147483000.0;
            int32_t i_u = fin ? (int32_t)f_u : 0;
            int32_t i_v = fin ? (int32_t)f_v : 0;
            double f_p = fin ? floor((wl - w_min[img]) * inv_dw) : 0.0;
            if (f_p > (double)(Nw - 1)) f_p = (double)(Nw - 1);
            if (!(f_p >= 0.0)) f_p = 0.0; /* only reachable with a caller-given w_min */
            int32_t i_p = (int32_t)f_p;
            int on = fin && (i_u - h >= 0) && (i_u + h <= N - 1) && (i_v - h >= 0) && (i_v + h <= N - 1);
            iu[k] = i_u; iv[k] = i_v; ip[k] = i_p;
            if (xu) xu[k] = x_u;
            if (xv) xv[k] = x_v;
            if (on) {
                uint64_t kk = (uint64_t)img * (uint64_t)Nw + (uint64_t)i_p;
                kk = (kk * (uint64_t)T + (uint64_t)(i_v / B)) * (uint64_t)T + (uint64_t)(i_u / B);
                kk = (kk * (uint64_t)B + (uint64_t)(i_v % B)) * (uint64_t)B + (uint64_t)(i_u % B);
                key[k] = kk;
            } else {
                key[k] = RKO_KEY_DROPPED;
            }
        }
    }
    free(s);
    return 0;
}

/* Reading R24 (not in the paper): conjugate-symmetry FOLDING of the
 * rows with w < 0.  A real sky gives V(-u,-v,-w) = conj V(u,v,w) (Eq. 1), and the dirty
 * image keeps only the real part (R13), so replacing a row (u,v,w) with w < 0 by (-u,-v,-w) and the
 * visibilities of that row by their conjugates changes no term of the direct sum
 *   Re[ V e^{+2 pi i (u l + v m + w (n-1))} ] = Re[ conj(V) e^{-2 pi i (...)} ],
 * while every w becomes >= 0: the w range the N_w planes have to cover halves.  Applied to the inputs
 * IN PLACE, before step 1; everything after it is the unchanged path.  uvw_m [R][3] metres, vis [R][C]
 * complex128 interleaved.  A row with w == 0 (either sign) or a non-finite w is left alone.
 * Returns the number of rows folded. */
int64_t rko_fold_w(int64_t n_rows, int32_t n_chan, double *uvw_m, double *vis)
{
    int64_t n = 0;
    for (int64_t r = 0; r < n_rows; ++r) {
        if (!(uvw_m[3 * r + 2] < 0.0)) continue;
        uvw_m[3 * r + 0] = -uvw_m[3 * r + 0];
        uvw_m[3 * r + 1] = -uvw_m[3 * r + 1];
        uvw_m[3 * r + 2] = -uvw_m[3 * r + 2];
        for (int32_t c = 0; c < n_chan; ++c) {
            double *v = vis + 2 * (r * (int64_t)n_chan + c);
            v[1] = -v[1];
        }
        ++n;
    }
    return n;
}

/* Stable sort by key == sort by (key, original index): perm[q] = index of the
 * visibility at sorted position q. */
typedef struct { uint64_t key; uint64_t idx; } rko_pair;

static int cmp_pair(const void *a, const void *b)
{
    const rko_pair *x = (const rko_pair *)a, *y = (const rko_pair *)b;
    if (x->key != y->key) return (x->key > y->key) - (x->key < y->key);
    return (x->idx > y->idx) - (x->idx < y->idx);
}

int rko_sort(int64_t M, const uint64_t *key, uint32_t *perm)
{
    rko_pair *c = (rko_pair *)malloc(sizeof(rko_pair) * (size_t)(M > 0 ? M : 1));
    for (int64_t k = 0; k < M; ++k) { c[k].key = key[k]; c[k].idx = (uint64_t)k; }
    qsort(c, (size_t)M, sizeof(rko_pair), cmp_pair);
    for (int64_t k = 0; k < M; ++k) perm[k] = (uint32_t)c[k].idx;
    free(c);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Steps 5-6: convolutional gridding, Eq. 3                    */
/* ------------------------------------------------------------------------ */

/* Scatter the visibilities listed in `list` (visibility indices, ascending)
 * onto ONE plane [N][N] complex (interleaved re,im; row = v, column = u).
 * vis: complex128 interleaved [M]; wgt: float [M] or NULL.  */
int rko_grid_plane(int64_t n_list, const int64_t *list, const double *vis, const float *wgt,
                   const int32_t *iu, const int32_t *iv, const double *xu, const double *xv,
                   int32_t N, int32_t S, double beta, double *plane)
{
    const int32_t h = (S - 1) / 2;
#pragma omp parallel
    {
        int nt = 1, tid = 0;
#ifdef _OPENMP
        nt = omp_get_num_threads();
        tid = omp_get_thread_num();
#endif
        const int32_t j0 = (int32_t)((int64_t)N * tid / nt), j1 = (int32_t)((int64_t)N * (tid + 1) / nt);
        double ku[32], kv[32];
        for (int64_t q = 0; q < n_list; ++q) {
            const int64_t k = list[q];
            const int32_t cu = iu[k], cv = iv[k];
            if (cv + h < j0 || cv - h >= j1) continue;
            const double om = wgt ? (double)wgt[k] : 1.0;
            const double vr = om * vis[2 * k], vi = om * vis[2 * k + 1];
            for (int32_t a = -h; a <= h; ++a) {
                double d_a = (double)(cu - N / 2 + a) - xu[k];
                double d_b = (double)(cv - N / 2 + a) - xv[k];
                ku[a + h] = rko_kb(d_a, S, beta);
                kv[a + h] = rko_kb(d_b, S, beta);
            }
            for (int32_t b = -h; b <= h; ++b) {
                const int32_t j = cv + b;
                if (j < j0 || j >= j1) continue;
                for (int32_t a = -h; a <= h; ++a) {
                    const double kk = ku[a + h] * kv[b + h];
                    double *cell = plane + 2 * ((int64_t)j * N + (cu + a));
                    cell[0] += vr * kk;
                    cell[1] += vi * kk;
                }
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Step 7: centred, unnormalised, + sign 2-D transform of one plane          */
/* P[q][p] = sum_{j,i} G[j][i] e^{+2 pi i ((i-N/2)(p-N/2)+(j-N/2)(q-N/2))/N} */
/* ------------------------------------------------------------------------ */

/* textbook iterative radix-2 Cooley-Tukey, + sign, unnormalised, length n=2^m,
 * on a contiguous interleaved complex vector; tw[k] = e^{+2 pi i k/n}, k<n/2. */
static void fft1d_pos(double *x, int32_t n, const double *tw)
{
    for (int32_t i = 1, j = 0; i < n; ++i) {           /* bit reversal */
        int32_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * j]; x[2 * i + 1] = x[2 * j + 1];
            x[2 * j] = tr; x[2 * j + 1] = ti;
        }
    }
    for (int32_t len = 2; len <= n; len <<= 1) {
        const int32_t half = len >> 1, step = n / len;
        for (int32_t i = 0; i < n; i += len)
            for (int32_t k = 0; k < half; ++k) {
                const double wr = tw[2 * (k * step)], wi = tw[2 * (k * step) + 1];
                double *a = x + 2 * (i + k), *b = x + 2 * (i + k + half);
                const double br = b[0] * wr - b[1] * wi, bi = b[0] * wi + b[1] * wr;
                b[0] = a[0] - br; b[1] = a[1] - bi;
                a[0] = a[0] + br; a[1] = a[1] + bi;
            }
    }
}

int rko_fft2_centered(double *plane, int32_t N)
{
    if (N < 4 || (N & (N - 1)) || (N % 4)) return -1;
    double *tw = (double *)malloc(sizeof(double) * (size_t)N);
    for (int32_t k = 0; k < N / 2; ++k) {
        long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)N;
        tw[2 * k] = (double)cosl(a);
        tw[2 * k + 1] = (double)sinl(a);
    }
    /* input checkerboard (-1)^(i+j): moves the origin to cell (N/2, N/2) */
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < N; ++j)
        for (int32_t i = 0; i < N; ++i)
            if ((i + j) & 1) {
                plane[2 * ((int64_t)j * N + i)] = -plane[2 * ((int64_t)j * N + i)];
                plane[2 * ((int64_t)j * N + i) + 1] = -plane[2 * ((int64_t)j * N + i) + 1];
            }
    /* rows */
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < N; ++j) fft1d_pos(plane + 2 * (int64_t)j * N, N, tw);
    /* columns */
#pragma omp parallel
    {
        double *col = (double *)malloc(sizeof(double) * 2 * (size_t)N);
#pragma omp for schedule(static)
        for (int32_t i = 0; i < N; ++i) {
            for (int32_t j = 0; j < N; ++j) {
                col[2 * j] = plane[2 * ((int64_t)j * N + i)];
                col[2 * j + 1] = plane[2 * ((int64_t)j * N + i) + 1];
            }
            fft1d_pos(col, N, tw);
            for (int32_t j = 0; j < N; ++j) {
                plane[2 * ((int64_t)j * N + i)] = col[2 * j];
                plane[2 * ((int64_t)j * N + i) + 1] = col[2 * j + 1];
            }
        }
        free(col);
    }
    /* output checkerboard (-1)^(p+q): origin of the image at pixel (N/2, N/2)
     * (exact for N = 0 mod 4: e^{i pi N/2} = 1 per axis) */
#pragma omp parallel for schedule(static)
    for (int32_t q = 0; q < N; ++q)
        for (int32_t p = 0; p < N; ++p)
            if ((p + q) & 1) {
                plane[2 * ((int64_t)q * N + p)] = -plane[2 * ((int64_t)q * N + p)];
                plane[2 * ((int64_t)q * N + p) + 1] = -plane[2 * ((int64_t)q * N + p) + 1];
            }
    free(tw);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Step 8: w-correction + plane sum (Eq. 2; reading R2)          */
/* ------------------------------------------------------------------------ */

/* image[q][p] += Re( P[q][p] * exp(+2 pi i w_z (n-1)) ),  n-1 = -r2/(1+sqrt(1-r2)) */
int rko_wcorrect_accumulate(const double *plane, int32_t N, double dl, double w_z, double *image)
{
#pragma omp parallel for schedule(static)
    for (int32_t q = 0; q < N; ++q) {
        const double m = (double)(q - N / 2) * dl;
        for (int32_t p = 0; p < N; ++p) {
            const double l = (double)(p - N / 2) * dl;
            const double r2 = l * l + m * m;
            if (r2 >= 1.0) continue;                       /* reading R18: stays 0 */
            const double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
            double x = w_z * nm1;
            x = x - rint(x);                               /* phase in cycles, reduced */
            const double c = cos(2.0 * RKO_PI * x), s = sin(2.0 * RKO_PI * x);
            const double pr = plane[2 * ((int64_t)q * N + p)], pi = plane[2 * ((int64_t)q * N + p) + 1];
            image[(int64_t)q * N + p] += pr * c - pi * s;
        }
    }
    return 0;
}

/* Step 9: I = I_raw / (c(nu_p) c(nu_q)), nu = (p - N/2)/N (reading R12). */
int rko_gridcorrect(double *image, int32_t N, int32_t S, double beta)
{
    double *c = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp parallel for schedule(static)
    for (int32_t p = 0; p < N; ++p) c[p] = rko_taper((double)(p - N / 2) / (double)N, S, beta);
#pragma omp parallel for schedule(static)
    for (int32_t q = 0; q < N; ++q)
        for (int32_t p = 0; p < N; ++p) image[(int64_t)q * N + p] /= (c[p] * c[q]);
    free(c);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Whole path, plane-streamed (never holds more than one plane + the image)   */
/* ------------------------------------------------------------------------ */

/* vis: complex128 interleaved [R*C].  image: [n_img][N][N] f64, overwritten.
 * Optional outputs (NULL to skip): stack_grid / stack_fft [n_img*Nw][N][N]
 * complex interleaved (planes after a3 / after a4); raw_image [n_img][N][N]
 * (after a5, before the taper); stats[6] = n_vis, n_gridded, n_dropped,
 * sum_w (over gridded), w_min, w_max (image 0).
 * stage_mask: bit0 grid, bit1 fft, bit2 wcorrect, bit3 taper (for timing a
 * subset; normal use 15).  timings[4]: seconds per stage (NULL to skip). */
int rko_image(int64_t n_rows, int32_t n_chan, const double *uvw_m, const double *freq_hz,
              const double *vis, const float *wgt,
              int32_t N, int32_t Nw, int32_t S, double dl, double beta, int32_t B, int32_t cube,
              double w_min_in, double w_max_in, int32_t stage_mask,
              double *image, double *raw_image, double *stack_grid, double *stack_fft,
              double *stats, double *timings)
{
    const int64_t M = n_rows * n_chan;
    const int32_t n_img = cube ? n_chan : 1;
    if (beta <= 0.0) beta = 2.34 * (double)S;
    int32_t *iu = (int32_t *)malloc(sizeof(int32_t) * (size_t)(M + 1));
    int32_t *iv = (int32_t *)malloc(sizeof(int32_t) * (size_t)(M + 1));
    int32_t *ip = (int32_t *)malloc(sizeof(int32_t) * (size_t)(M + 1));
    uint64_t *key = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(M + 1));
    double *xu = (double *)malloc(sizeof(double) * (size_t)(M + 1));
    double *xv = (double *)malloc(sizeof(double) * (size_t)(M + 1));
    double *wmin = (double *)malloc(sizeof(double) * (size_t)n_img);
    double *wmax = (double *)malloc(sizeof(double) * (size_t)n_img);
    for (int32_t g = 0; g < n_img; ++g) { wmin[g] = w_min_in; wmax[g] = w_max_in; }
    rko_index(n_rows, n_chan, uvw_m, freq_hz, N, Nw, S, dl, B, cube, wmin, wmax, iu, iv, ip, key, xu, xv);

    /* per (image, plane) lists of on-grid visibilities in index order */
    const int64_t n_pl = (int64_t)n_img * Nw;
    int64_t *cnt = (int64_t *)calloc((size_t)(n_pl + 1), sizeof(int64_t));
    int64_t n_gridded = 0;
    double sum_w = 0.0;
    for (int64_t k = 0; k < M; ++k)
        if (key[k] != RKO_KEY_DROPPED) {
            const int32_t img = cube ? (int32_t)(k % n_chan) : 0;
            cnt[(int64_t)img * Nw + ip[k] + 1]++;
            n_gridded++;
            sum_w += wgt ? (double)wgt[k] : 1.0;
        }
    for (int64_t z = 0; z < n_pl; ++z) cnt[z + 1] += cnt[z];
    int64_t *list = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_gridded + 1));
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_pl + 1));
    memcpy(fill, cnt, sizeof(int64_t) * (size_t)(n_pl + 1));
    for (int64_t k = 0; k < M; ++k)
        if (key[k] != RKO_KEY_DROPPED) {
            const int32_t img = cube ? (int32_t)(k % n_chan) : 0;
            list[fill[(int64_t)img * Nw + ip[k]]++] = k;
        }
    if (stats) {
        stats[0] = (double)M; stats[1] = (double)n_gridded; stats[2] = (double)(M - n_gridded);
        stats[3] = sum_w; stats[4] = wmin[0]; stats[5] = wmax[0];
    }

    const int64_t NN = (int64_t)N * N;
    double *plane = (double *)malloc(sizeof(double) * 2 * (size_t)NN);
    double t_stage[4] = {0, 0, 0, 0};
    for (int32_t g = 0; g < n_img; ++g) {
        double *img_out = image + (int64_t)g * NN;
        memset(img_out, 0, sizeof(double) * (size_t)NN);
        const double dw = (wmax[g] - wmin[g]) / (double)Nw;
        for (int32_t z = 0; z < Nw; ++z) {
            const int64_t pz = (int64_t)g * Nw + z;
            double t0 = 0, t1 = 0, t2 = 0, t3 = 0;
#ifdef _OPENMP
            t0 = omp_get_wtime();
#endif
            memset(plane, 0, sizeof(double) * 2 * (size_t)NN);
            if (stage_mask & 1)
                rko_grid_plane(cnt[pz + 1] - cnt[pz], list + cnt[pz], vis, wgt, iu, iv, xu, xv, N, S, beta, plane);
            if (stack_grid) memcpy(stack_grid + 2 * pz * NN, plane, sizeof(double) * 2 * (size_t)NN);
#ifdef _OPENMP
            t1 = omp_get_wtime();
#endif
            if (stage_mask & 2) rko_fft2_centered(plane, N);
            if (stack_fft) memcpy(stack_fft + 2 * pz * NN, plane, sizeof(double) * 2 * (size_t)NN);
#ifdef _OPENMP
            t2 = omp_get_wtime();
#endif
            const double w_z = wmin[g] + ((double)z + 0.5) * dw;   /* plane centre, reading R4 */
            if (stage_mask & 4) rko_wcorrect_accumulate(plane, N, dl, w_z, img_out);
#ifdef _OPENMP
            t3 = omp_get_wtime();
#endif
            t_stage[0] += t1 - t0; t_stage[1] += t2 - t1; t_stage[2] += t3 - t2;
        }
        if (raw_image) memcpy(raw_image + (int64_t)g * NN, img_out, sizeof(double) * (size_t)NN);
        double t4 = 0, t5 = 0;
#ifdef _OPENMP
        t4 = omp_get_wtime();
#endif
        if (stage_mask & 8) rko_gridcorrect(img_out, N, S, beta);
#ifdef _OPENMP
        t5 = omp_get_wtime();
#endif
        t_stage[3] += t5 - t4;
    }
    if (timings) memcpy(timings, t_stage, sizeof(t_stage));
    free(plane); free(list); free(fill); free(cnt);
    free(iu); free(iv); free(ip); free(key); free(xu); free(xv); free(wmin); free(wmax);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Direct DFT (the plain definition the method approximates; tiny inputs)     */
/* D[q][p] = Re sum_k om_k V_k exp(+2 pi i (u_k l + v_k m + w_k (n-1)))        */
/* keep[k] != 0 selects the visibilities (the on-grid ones); w_use[k] is the  */
/* w in wavelengths to use (exact w, or the plane centre for the "w-snapped"  */
/* twin).  u_l, v_l in wavelengths.                                           */
/* ------------------------------------------------------------------------ */
int rko_dft(int64_t M, const double *u_l, const double *v_l, const double *w_use,
            const double *vis, const float *wgt, const uint8_t *keep,
            int32_t N, double dl, double *image)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t q = 0; q < N; ++q) {
        const double m = (double)(q - N / 2) * dl;
        for (int32_t p = 0; p < N; ++p) {
            const double l = (double)(p - N / 2) * dl;
            const double r2 = l * l + m * m;
            double acc = 0.0;
            if (r2 < 1.0) {
                const double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
                for (int64_t k = 0; k < M; ++k) {
                    if (keep && !keep[k]) continue;
                    double x = u_l[k] * l + v_l[k] * m + w_use[k] * nm1;
                    x = x - rint(x);
                    const double c = cos(2.0 * RKO_PI * x), s = sin(2.0 * RKO_PI * x);
                    const double om = wgt ? (double)wgt[k] : 1.0;
                    acc += om * (vis[2 * k] * c - vis[2 * k + 1] * s);
                }
            }
            image[(int64_t)q * N + p] = acc;
        }
    }
    return 0;
}

int rko_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
