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
