// Host-side unit test of the register DFT blocks in csrc/cm_fft.cuh against a naive
// long-double DFT (test-only; compiled with g++ by tests/test_host_logic.py).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include "../paper_2301_06763_b200/csrc/cm_fft.cuh"

template <int M, int DIR>
static double check()
{
    double2 x[M], ref[M];
    for (int i = 0; i < M; ++i) x[i] = make_double2(std::sin(1.0 + 0.7 * i * i), std::cos(2.0 + 1.3 * i));
    const long double tau = 2.0L * acosl(-1.0L);
    for (int k = 0; k < M; ++k) {
        long double sr = 0, si = 0;
        for (int n = 0; n < M; ++n) {
            const long double a = DIR * tau * ((n * k) % M) / M;
            sr += x[n].x * cosl(a) - x[n].y * sinl(a);
            si += x[n].x * sinl(a) + x[n].y * cosl(a);
        }
        ref[k] = make_double2((double)sr, (double)si);
    }
    cmfft::Dft<M, DIR>::run(x);
    double e = 0;
    for (int k = 0; k < M; ++k) e = std::fmax(e, std::fmax(std::fabs(x[k].x - ref[k].x), std::fabs(x[k].y - ref[k].y)));
    return e;
}

// DftK: DFT of k[i] x[i]; Dft16Mod: DFT16 of x[r] w32^{DIR r}; Dft16ModAcc: acc[r] += w32^{DIR r} DFT16(x)[r]
template <int M, int DIR>
static double check_k()
{
    double2 x[M], y[M];
    double k[M];
    for (int i = 0; i < M; ++i) {
        x[i] = make_double2(std::sin(0.3 + 0.9 * i * i), std::cos(1.0 + 0.37 * i));
        k[i] = 0.5 + std::sin(2.0 + i);
        y[i] = make_double2(k[i] * x[i].x, k[i] * x[i].y);
    }
    cmfft::Dft<M, DIR>::run(y);            // checked above against the naive DFT
    cmfft::DftK<M, DIR>::run(x, k);
    double e = 0;
    for (int i = 0; i < M; ++i) e = std::fmax(e, std::fmax(std::fabs(x[i].x - y[i].x), std::fabs(x[i].y - y[i].y)));
    return e;
}

template <int DIR>
static double check_mod()
{
    const long double tau = 2.0L * acosl(-1.0L);
    double2 x[16], acc[16], acc0[16], xa[16];
    long double rr[16], ri[16];
    for (int i = 0; i < 16; ++i) {
        x[i] = xa[i] = make_double2(std::sin(0.1 + 0.77 * i * i), std::cos(1.5 + 0.21 * i * i));
        acc[i] = acc0[i] = make_double2(0.25 * i - 1.0, std::sin(3.0 * i));
    }
    double e = 0;
    // modulated input
    for (int k = 0; k < 16; ++k) {
        long double sr = 0, si = 0;
        for (int n = 0; n < 16; ++n) {
            const long double a = DIR * tau * (n / 32.0L + (long double)((n * k) % 16) / 16.0L);
            sr += x[n].x * cosl(a) - x[n].y * sinl(a);
            si += x[n].x * sinl(a) + x[n].y * cosl(a);
        }
        rr[k] = sr; ri[k] = si;
    }
    cmfft::Dft16Mod<DIR>::run(x);
    for (int k = 0; k < 16; ++k) e = std::fmax(e, std::fmax(std::fabs(x[k].x - (double)rr[k]), std::fabs(x[k].y - (double)ri[k])));
    // modulated output, accumulated
    for (int k = 0; k < 16; ++k) {
        long double sr = 0, si = 0;
        for (int n = 0; n < 16; ++n) {
            const long double a = DIR * tau * (k / 32.0L + (long double)((n * k) % 16) / 16.0L);
            sr += xa[n].x * cosl(a) - xa[n].y * sinl(a);
            si += xa[n].x * sinl(a) + xa[n].y * cosl(a);
        }
        rr[k] = acc0[k].x + sr; ri[k] = acc0[k].y + si;
    }
    cmfft::Dft16ModAcc<DIR>::run(xa, acc);
    for (int k = 0; k < 16; ++k) e = std::fmax(e, std::fmax(std::fabs(acc[k].x - (double)rr[k]), std::fabs(acc[k].y - (double)ri[k])));
    return e;
}

template <int M>
static double check_w()
{
    const long double tau = 2.0L * acosl(-1.0L);
    double2 a = make_double2(0.3, -1.1);
    double e = 0;
    double2 f = cmfft::mulw32<M, -1>(a), b = cmfft::mulw32<M, +1>(a);
    long double c = cosl(tau * M / 32), s = sinl(tau * M / 32);
    e = std::fmax(e, std::fabs(f.x - (double)(a.x * c + a.y * s)));
    e = std::fmax(e, std::fabs(f.y - (double)(-a.x * s + a.y * c)));
    e = std::fmax(e, std::fabs(b.x - (double)(a.x * c - a.y * s)));
    e = std::fmax(e, std::fabs(b.y - (double)(a.x * s + a.y * c)));
    return e;
}

template <int M> struct WLoop { static double run() { return std::fmax(check_w<M>(), WLoop<M - 1>::run()); } };
template <> struct WLoop<-1> { static double run() { return 0; } };

int main()
{
    double e = 0;
    e = std::fmax(e, check<2, -1>());  e = std::fmax(e, check<2, 1>());
    e = std::fmax(e, check<4, -1>());  e = std::fmax(e, check<4, 1>());
    e = std::fmax(e, check<8, -1>());  e = std::fmax(e, check<8, 1>());
    e = std::fmax(e, check<16, -1>()); e = std::fmax(e, check<16, 1>());
    e = std::fmax(e, check_k<1, 1>());  e = std::fmax(e, check_k<2, 1>());  e = std::fmax(e, check_k<4, 1>());
    e = std::fmax(e, check_k<8, 1>());  e = std::fmax(e, check_k<16, 1>()); e = std::fmax(e, check_k<16, -1>());
    e = std::fmax(e, check_mod<-1>());  e = std::fmax(e, check_mod<1>());
    double ew = WLoop<40>::run();
    // slot <-> frequency is a bijection
    int bad = 0;
    for (int N = 16; N <= 256; N *= 2) {
        int *seen = (int *)calloc(2 * N, sizeof(int));
        for (int s = 0; s < 2 * N; ++s) seen[cmfft::slot_to_freq(s, N)]++;
        for (int k = 0; k < 2 * N; ++k) bad += seen[k] != 1;
        free(seen);
    }
    std::printf("dft_err %.3e w_err %.3e slot_bad %d\n", e, ew, bad);
    return (e < 1e-14 && ew < 1e-15 && bad == 0) ? 0 : 1;
}
