/*
 * cm_oracle.c — ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the hot path of
 * arXiv 2301.06763 ("Computing the gravitational potential on nested meshes
 * using the convolution method") computes, written from PAPER.md only.
 * It shares no code, header, table or constant with the CUDA library under
 * paper_2301_06763_b200/csrc/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may build, load or call it.
 *
 * Everything is fp64 (accumulation of the direct sum in long double).  There is
 * no blocking, pruning, real-symmetry trick or fusion: each function is the
 * definition written out.
 *
 * Conventions:
 *   - a level is an N^3 array, index ((k*N + j)*N + i), i = x fastest;
 *   - level l+1 covers coarse indices [N/4, 3N/4) of level l in every axis
 *     (Fig. 1; the offset N/4 is PAPER.md:L76);
 *   - offsets between cell centres are measured in cells: the inverse distance
 *     of Eq. 10 is g(o)/dx with g(o) = 1/|o|, and the mass is rho*dx^3, so
 *     Phi = -G dx^2 sum_s rho[s] g(t-s)
 *   - g(0) = I0 = int_{[-1/2,1/2]^3} d^3u/|u| = 3 ln(2+sqrt 3) - pi/2
 *     (Eq. 13: potential of a uniform cube at its centre).
 *
 * Pins (tests/test_oracle_*.py): I0 against a smooth 2-D quadrature; single
 * source cell = -G rho dx^2 / |t-s| exactly; direct sum == this file's FFT path
 * == numpy/scipy fftconvolve (L=1 is the textbook Hockney-Eastwood isolated
 * convolution); restriction conserves mass; prolongation is exact on affine
 * fields; homogeneous sphere / ellipsoid closed forms; far field -GM/r;
 * linearity; mirror symmetry; Table 3 of the paper (soft pin).
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define IDX(N, k, j, i) ((((size_t)(k)) * (size_t)(N) + (size_t)(j)) * (size_t)(N) + (size_t)(i))

/* ---- Eq. 13: the zero-offset value of the dimensionless kernel ------------ */
double orc_I0(void)
{
    return (double)(3.0L * logl(2.0L + sqrtl(3.0L)) - acosl(-1.0L) / 2.0L);
}

/* g(o) for an integer cell offset o: Eq. 10 (1/|o|) with Eq. 13 at o = 0. */
static double g_of(long ox, long oy, long oz)
{
    if (ox == 0 && oy == 0 && oz == 0) return orc_I0();
    return 1.0 / sqrt((double)(ox * ox + oy * oy + oz * oz));
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int in_cavity(int N, int k, int j, int i)
{
    const int lo = N / 4, hi = 3 * N / 4;
    return k >= lo && k < hi && j >= lo && j < hi && i >= lo && i < hi;
}

/* ---- a1: restriction cascade ("projected from the fine to
 * the coarse grid"; reading: arithmetic mean of the 8 children's density =
 * sum of their masses; readings 9, 10).  rho, rhobar: [L][N^3]. ---- */
void orc_restrict(int N, int L, const double *rho, double *rhobar)
{
    const size_t n3 = (size_t)N * N * N;
    memcpy(rhobar, rho, sizeof(double) * n3 * (size_t)L);
    for (int l = L - 2; l >= 0; --l) {
        double *c = rhobar + n3 * (size_t)l;
        const double *f = rhobar + n3 * (size_t)(l + 1);
        for (int pk = N / 4; pk < 3 * N / 4; ++pk)
            for (int pj = N / 4; pj < 3 * N / 4; ++pj)
                for (int pi = N / 4; pi < 3 * N / 4; ++pi) {
                    double s = 0.0;
                    for (int c3 = 0; c3 < 2; ++c3)
                        for (int b = 0; b < 2; ++b)
                            for (int a = 0; a < 2; ++a)
                                s += f[IDX(N, 2 * (pk - N / 4) + c3, 2 * (pj - N / 4) + b, 2 * (pi - N / 4) + a)];
                    c[IDX(N, pk, pj, pi)] = 0.125 * s;
                }
    }
}

/* ---- Eq. 10 by brute force on one level (O(N^6)); hole != 0 zeroes the
 * cavity first ("the density in the cavity is set equal to zero").
 * phi[t] = -G dx^2 sum_s rho[s] g(t - s). ----------------------------------- */
void orc_field_direct(int N, const double *rho, int hole, double G, double dx, double *phi)
{
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int tk = 0; tk < N; ++tk)
        for (int tj = 0; tj < N; ++tj)
            for (int ti = 0; ti < N; ++ti) {
                long double acc = 0.0L;
                for (int sk = 0; sk < N; ++sk)
                    for (int sj = 0; sj < N; ++sj)
                        for (int si = 0; si < N; ++si) {
                            if (hole && in_cavity(N, sk, sj, si)) continue;
                            const double m = rho[IDX(N, sk, sj, si)];
                            if (m == 0.0) continue;
                            acc += (long double)m * (long double)g_of(ti - si, tj - sj, tk - sk);
                        }
                phi[IDX(N, tk, tj, ti)] = (double)(-(long double)G * (long double)dx * (long double)dx * acc);
            }
}

/* Same sum, only at the listed targets (tgt = nt triples (k, j, i)); used to
 * check full-size GPU results on sampled outputs. */
void orc_field_direct_at(int N, const double *rho, int hole, double G, double dx,
                         int nt, const int *tgt, double *out)
{
    for (int t = 0; t < nt; ++t) {
        const int tk = tgt[3 * t + 0], tj = tgt[3 * t + 1], ti = tgt[3 * t + 2];
        long double acc = 0.0L;
#pragma omp parallel
        {
            long double part = 0.0L;
#pragma omp for schedule(static) nowait
            for (int sk = 0; sk < N; ++sk)
                for (int sj = 0; sj < N; ++sj)
                    for (int si = 0; si < N; ++si) {
                        if (hole && in_cavity(N, sk, sj, si)) continue;
                        const double m = rho[IDX(N, sk, sj, si)];
                        if (m == 0.0) continue;
                        part += (long double)m * (long double)g_of(ti - si, tj - sj, tk - sk);
                    }
#pragma omp critical
            acc += part;
        }
        out[t] = (double)(-(long double)G * (long double)dx * (long double)dx * acc);
    }
}

/* ---- the oracle's own naive FFT: iterative radix-2, in place, unnormalised,
 * sign = -1 forward / +1 inverse (Eq. 11; reading 5). --- */
static void fft1d(double complex *a, long n, int sign, const double complex *w /* n/2 roots, forward */)
{
    /* bit reversal */
    for (long i = 1, j = 0; i < n; ++i) {
        long bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { double complex t = a[i]; a[i] = a[j]; a[j] = t; }
    }
    for (long len = 2; len <= n; len <<= 1) {
        const long step = n / len;
        for (long i = 0; i < n; i += len)
            for (long k = 0; k < len / 2; ++k) {
                double complex tw = w[k * step];
                if (sign > 0) tw = conj(tw);
                const double complex u = a[i + k], v = a[i + k + len / 2] * tw;
                a[i + k] = u + v;
                a[i + k + len / 2] = u - v;
            }
    }
}

/* plain O(n^2) DFT of one sequence: exported only so a test can pin fft1d. */
void orc_dft_naive(long n, const double *in_re, const double *in_im, int sign, double *out_re, double *out_im)
{
    const long double tau = 2.0L * acosl(-1.0L);
    for (long k = 0; k < n; ++k) {
        long double sr = 0.0L, si = 0.0L;
        for (long j = 0; j < n; ++j) {
            const long double ang = (long double)sign * tau * (long double)((j * k) % n) / (long double)n;
            const long double c = cosl(ang), s = sinl(ang);
            sr += in_re[j] * c - in_im[j] * s;
            si += in_re[j] * s + in_im[j] * c;
        }
        out_re[k] = (double)sr;
        out_im[k] = (double)si;
    }
}

void orc_fft1d(long n, double *re_im_interleaved, int sign)
{
    double complex *w = (double complex *)malloc(sizeof(double complex) * (size_t)(n / 2 + 1));
    const long double tau = 2.0L * acosl(-1.0L);
    for (long k = 0; k < n / 2; ++k)
        w[k] = (double)cosl(-tau * k / n) + I * (double)sinl(-tau * k / n);
    fft1d((double complex *)re_im_interleaved, n, sign, w);
    free(w);
}

/* 3-D transform of an n^3 complex array, one axis after the other. */
static void fft3d(double complex *a, long n, int sign)
{
    double complex *w = (double complex *)malloc(sizeof(double complex) * (size_t)(n / 2 + 1));
    const long double tau = 2.0L * acosl(-1.0L);
    for (long k = 0; k < n / 2; ++k)
        w[k] = (double)cosl(-tau * k / n) + I * (double)sinl(-tau * k / n);
    for (int axis = 0; axis < 3; ++axis) {
        const size_t stride = axis == 0 ? 1 : (axis == 1 ? (size_t)n : (size_t)n * n);
#pragma omp parallel
        {
            double complex *buf = (double complex *)malloc(sizeof(double complex) * (size_t)n);
#pragma omp for schedule(static)
            for (long p = 0; p < n * n; ++p) {
                const size_t u = (size_t)(p / n), v = (size_t)(p % n);
                size_t base;
                if (axis == 0) base = (u * n + v) * n;          /* (k=u, j=v) */
                else if (axis == 1) base = u * n * n + v;       /* (k=u, i=v) */
                else base = u * n + v;                          /* (j=u, i=v) */
                for (long q = 0; q < n; ++q) buf[q] = a[base + (size_t)q * stride];
                fft1d(buf, n, sign, w);
                for (long q = 0; q < n; ++q) a[base + (size_t)q * stride] = buf[q];
            }
            free(buf);
        }
    }
    free(w);
}

/* Transform of the kernel on the doubled, rearranged mesh (PAPER.md:L143-L147,
 * Fig. 4): array index a maps to offset a (a <= N) or a - 2N (a > N).
 * ghat: (2N)^3 complex, interleaved re/im, caller-allocated. */
void orc_green_hat(int N, double *ghat_interleaved)
{
    const long n = 2L * N;
    double complex *g = (double complex *)ghat_interleaved;
#pragma omp parallel for collapse(2)
    for (long c = 0; c < n; ++c)
        for (long b = 0; b < n; ++b)
            for (long a = 0; a < n; ++a) {
                const long oz = c <= N ? c : c - n, oy = b <= N ? b : b - n, ox = a <= N ? a : a - n;
                g[((size_t)c * n + b) * n + a] = g_of(ox, oy, oz);
            }
    fft3d(g, n, -1);
}

/* One field by the convolution theorem on the zero-padded (2N)^3 mesh:
 * pad, transform, multiply (Eq. 11), inverse, crop the
 * "original active region 1" (Fig. 4), scale by -G dx^2 / (2N)^3.
 * work: caller-allocated (2N)^3 complex scratch. */
void orc_field_fft(int N, const double *rho, int hole, double G, double dx,
                   const double *ghat_interleaved, double *work_interleaved, double *phi)
{
    const long n = 2L * N;
    double complex *a = (double complex *)work_interleaved;
    const double complex *gh = (const double complex *)ghat_interleaved;
    memset(a, 0, sizeof(double complex) * (size_t)n * n * n);
    for (int k = 0; k < N; ++k)
        for (int j = 0; j < N; ++j)
            for (int i = 0; i < N; ++i) {
                if (hole && in_cavity(N, k, j, i)) continue;
                a[((size_t)k * n + j) * n + i] = rho[IDX(N, k, j, i)];
            }
    fft3d(a, n, -1);
    const size_t tot = (size_t)n * n * n;
#pragma omp parallel for
    for (size_t q = 0; q < tot; ++q) a[q] *= gh[q];
    fft3d(a, n, +1);
    const double scale = -G * dx * dx / ((double)n * (double)n * (double)n);
    for (int k = 0; k < N; ++k)
        for (int j = 0; j < N; ++j)
            for (int i = 0; i < N; ++i)
                phi[IDX(N, k, j, i)] = scale * creal(a[((size_t)k * n + j) * n + i]);
}

/* ---- coarse -> fine operator (the tilde of Eq. 14): the paper's only printed
 * interpolation, Eq. 3-6, applied to every fine cell
 * (reading 6): fine cell f has parent p = N/4 + f/2 per axis and child-offset
 * sign s = +1 (f odd) / -1 (f even) per axis; value = 3/4 C[p] + 1/4 C[p+s]. - */
void orc_prolong(int N, const double *coarse, double *fine)
{
    for (int fk = 0; fk < N; ++fk)
        for (int fj = 0; fj < N; ++fj)
            for (int fi = 0; fi < N; ++fi) {
                const int pk = N / 4 + fk / 2, pj = N / 4 + fj / 2, pi = N / 4 + fi / 2;
                const int sk = (fk & 1) ? 1 : -1, sj = (fj & 1) ? 1 : -1, si = (fi & 1) ? 1 : -1;
                fine[IDX(N, fk, fj, fi)] = 0.75 * coarse[IDX(N, pk, pj, pi)] +
                                           0.25 * coarse[IDX(N, pk + sk, pj + sj, pi + si)];
            }
}

/* ---- Oracle-B (physical cross-check, NOT the parity oracle): direct sum over
 * the leaf cells of all levels with true centre-to-centre distances
 * (north_star: "direct triple sum over all cells of all levels").  Bounds the
 * METHOD's error, not the implementation's.  half0 = half-width of level 0.
 * Targets: every cell of level lt. ----------------------------------------- */
void orc_leaf_direct(int N, int L, double half0, double G, const double *rho, int lt, double *phi)
{
    const size_t n3 = (size_t)N * N * N;
    const double dxt = 2.0 * half0 / N / (double)(1 << lt);
    const double lot = -half0 / (double)(1 << lt);
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int tk = 0; tk < N; ++tk)
        for (int tj = 0; tj < N; ++tj)
            for (int ti = 0; ti < N; ++ti) {
                const double tx = lot + (ti + 0.5) * dxt, ty = lot + (tj + 0.5) * dxt, tz = lot + (tk + 0.5) * dxt;
                long double acc = 0.0L;
                for (int l = 0; l < L; ++l) {
                    const double dx = 2.0 * half0 / N / (double)(1 << l);
                    const double lo = -half0 / (double)(1 << l);
                    const double *r = rho + n3 * (size_t)l;
                    for (int sk = 0; sk < N; ++sk)
                        for (int sj = 0; sj < N; ++sj)
                            for (int si = 0; si < N; ++si) {
                                if (l < L - 1 && in_cavity(N, sk, sj, si)) continue; /* not a leaf */
                                const double m = r[IDX(N, sk, sj, si)] * dx * dx * dx;
                                if (m == 0.0) continue;
                                const double ex = tx - (lo + (si + 0.5) * dx), ey = ty - (lo + (sj + 0.5) * dx),
                                             ez = tz - (lo + (sk + 0.5) * dx);
                                const double d2 = ex * ex + ey * ey + ez * ez;
                                if (d2 < 1e-24 * dx * dx + 1e-300) acc += (long double)m * (long double)(orc_I0() / dx);
                                else acc += (long double)m / (long double)sqrt(d2);
                            }
                }
                phi[IDX(N, tk, tj, ti)] = (double)(-(long double)G * acc);
            }
}
