// cm_fft.cuh — register-resident fp64 DFT building blocks for the pruned pencil FFT.
//
// The (2N)-point transform of a zero-padded length-N pencil (Fig. 4:
// "doubling the computational domain ... assigning zero values to M") is taken as
//     n = j + T r   (j < T, r < 32, a[n] = 0 for r >= 16),     2N = 32 T,
//     k = kp + 32 k2,  kp = 2 k1 + p  (k1 < 16, p in {0,1}, k2 < T)
//     X[k] = sum_j w_T^{j k2} w_2N^{j kp} [ sum_{r<16} a[j+Tr] w_32^{r kp} ]
// i.e. a pruned radix-32 first stage done in the registers of thread j as two radix-16
// DFTs (p = 0: plain, p = 1: inputs pre-multiplied by w_32^r), a twiddle, one exchange
// through shared memory and a radix-T stage.  The inverse runs the same graph backwards
// and only forms the N outputs that survive the crop ("original active region 1",
// PAPER.md:L147).  Everything here is host+device so the butterflies can be unit-tested
// on the CPU box (tests/test_host_fft_blocks.py compiles this header with g++).
#pragma once

#if defined(__CUDACC__)
#define CM_HD __host__ __device__ __forceinline__
#else
#include <cmath>
#define CM_HD inline
struct double2 { double x, y; };
static inline double2 make_double2(double x, double y) { double2 r; r.x = x; r.y = y; return r; }
#endif

namespace cmfft {

constexpr int E = 16;  // elements a thread holds; first-stage radix (per parity)

// cos(2 pi q / 32), q = 0..8
CM_HD constexpr double cos32_base(int q)
{
    return q == 0 ? 1.0
         : q == 1 ? 0.9807852804032304491261822
         : q == 2 ? 0.9238795325112867561281832
         : q == 3 ? 0.8314696123025452370787884
         : q == 4 ? 0.7071067811865475244008444
         : q == 5 ? 0.5555702330196022247428308
         : q == 6 ? 0.3826834323650897717284600
         : q == 7 ? 0.1950903220161282678482849
         : 0.0;
}
CM_HD constexpr double cos32(int r)
{
    int q = r & 31;
    if (q > 16) q = 32 - q;
    return q <= 8 ? cos32_base(q) : -cos32_base(16 - q);
}
CM_HD constexpr double sin32(int r) { return cos32(r - 8); }

// a + k b and a - k b as one FMA per component (written with fma(): the compiler does not contract a product that
// has two uses, and every product below feeds a sum AND a difference)
CM_HD double2 cfma(double k, double2 b, double2 a) { return make_double2(fma(k, b.x, a.x), fma(k, b.y, a.y)); }
CM_HD double2 cfms(double k, double2 b, double2 a) { return make_double2(fma(-k, b.x, a.x), fma(-k, b.y, a.y)); }
CM_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
CM_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
CM_HD double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
CM_HD double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }

// a * exp(DIR * 2 pi i M / 32), M a compile-time constant; DIR = -1 forward, +1 inverse.
template <int M, int DIR>
CM_HD double2 mulw32(double2 a)
{
    constexpr int m = ((M % 32) + 32) % 32;
    if (m == 0) return a;
    if (m == 16) return make_double2(-a.x, -a.y);
    if (m == 8) return DIR < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);     // -+ i
    if (m == 24) return DIR < 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    constexpr double c = cos32(m);
    constexpr double s = (DIR < 0 ? -1.0 : 1.0) * sin32(m);
    return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
}

template <int DIR>
CM_HD void radix2(double2 &a0, double2 &a1)
{
    const double2 t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}

// 4-point DFT, natural order in and out.
template <int DIR>
CM_HD void radix4(double2 &a0, double2 &a1, double2 &a2, double2 &a3)
{
    const double2 s02 = cadd(a0, a2), d02 = csub(a0, a2);
    const double2 s13 = cadd(a1, a3), d13 = csub(a1, a3);
    // forward: X1 = d02 - i d13, X3 = d02 + i d13 ; inverse swaps them
    const double2 id13 = make_double2(-d13.y, d13.x);  // i * d13
    a0 = cadd(s02, s13);
    a2 = csub(s02, s13);
    if (DIR < 0) { a1 = csub(d02, id13); a3 = cadd(d02, id13); }
    else         { a1 = cadd(d02, id13); a3 = csub(d02, id13); }
}

// ---- twiddle constants in tangent form (FMA-fused butterflies) -----------------------
// exp(DIR 2 pi i M / 32) = i^Q * G * (1 + i TN) with |TN| <= 1, G > 0: the product a * (1 + i TN) costs two FMAs,
// the quarter turn i^Q is a swap, and the real factor G rides on the multiplier of the FMA that consumes the
// value in the next butterfly (Linzer-Feig form) — a twiddled radix-4 butterfly takes 22 fp64 instructions
// instead of 28, and the adds of the butterflies become FMAs at no cost.
template <int M, int DIR> struct W32 {
    static constexpr int mp = (((DIR * M) % 32) + 32) % 32;     // counter-clockwise angle in units of 2 pi / 32
    static constexpr int Q = ((mp + 4) / 8) % 4;
    static constexpr int R = mp - 8 * ((mp + 4) / 8);           // residual angle, -4 .. 3
    static constexpr double G = cos32(R);
    static constexpr double TN = sin32(R) / cos32(R);
};

// a * i^Q * (1 + i TN): the twiddle without its real factor G
template <int M, int DIR>
CM_HD double2 twpre(double2 a)
{
    using W = W32<M, DIR>;
    const double2 u = (W::R == 0) ? a : make_double2(fma(-W::TN, a.y, a.x), fma(W::TN, a.x, a.y));
    if (W::Q == 0) return u;
    if (W::Q == 1) return make_double2(-u.y, u.x);
    if (W::Q == 2) return make_double2(-u.x, -u.y);
    return make_double2(u.y, -u.x);
}

// radix-4 DFT (direction DIR) of a_i * exp(DIR 2 pi i M_i / 32), i = 0..3, natural order in and out.  The results
// come out divided by G0 = W32<M0, DIR>::G (1 when M0 = 0); the caller folds G0 into what follows.
template <int DIR, int M0, int M1, int M2, int M3>
CM_HD void radix4_tw(double2 &a0, double2 &a1, double2 &a2, double2 &a3)
{
    constexpr double g0 = W32<M0, DIR>::G, g1 = W32<M1, DIR>::G, g2 = W32<M2, DIR>::G, g3 = W32<M3, DIR>::G;
    constexpr double r2 = g2 / g0, r3 = g3 / g1, r1 = g1 / g0;
    const double2 u0 = twpre<M0, DIR>(a0), u1 = twpre<M1, DIR>(a1), u2 = twpre<M2, DIR>(a2), u3 = twpre<M3, DIR>(a3);
    const double2 s02 = cfma(r2, u2, u0), d02 = cfms(r2, u2, u0);
    const double2 s13 = cfma(r3, u3, u1), d13 = cfms(r3, u3, u1);
    a0 = cfma(r1, s13, s02);
    a2 = cfms(r1, s13, s02);
    // forward: X1 = d02 - i d13, X3 = d02 + i d13 ; inverse swaps them   (i d13 = (-d13.y, d13.x))
    if (DIR < 0) {
        a1 = make_double2(fma(r1, d13.y, d02.x), fma(-r1, d13.x, d02.y));
        a3 = make_double2(fma(-r1, d13.y, d02.x), fma(r1, d13.x, d02.y));
    } else {
        a1 = make_double2(fma(-r1, d13.y, d02.x), fma(r1, d13.x, d02.y));
        a3 = make_double2(fma(r1, d13.y, d02.x), fma(-r1, d13.x, d02.y));
    }
}

// radix-2 butterfly of (a0, a1 * exp(DIR 2 pi i M / 32))
template <int DIR, int M>
CM_HD void radix2_tw(double2 &a0, double2 &a1)
{
    constexpr double g = W32<M, DIR>::G;
    const double2 u = twpre<M, DIR>(a1), t = a0;
    a0 = cfma(g, u, t);
    a1 = cfms(g, u, t);
}

// radix-4 DFT of (k0 a0, k1 a1, k2 a2, k3 a3), k real (the K-hat product of Eq. 11 folded into the first butterflies
// of the inverse transform: one multiply and two FMAs per pair instead of two multiplies and two adds)
template <int DIR>
CM_HD void radix4_k(double2 &a0, double2 &a1, double2 &a2, double2 &a3, double k0, double k1, double k2, double k3)
{
    const double2 p0 = make_double2(k0 * a0.x, k0 * a0.y), p1 = make_double2(k1 * a1.x, k1 * a1.y);
    const double2 s02 = cfma(k2, a2, p0), d02 = cfms(k2, a2, p0);
    const double2 s13 = cfma(k3, a3, p1), d13 = cfms(k3, a3, p1);
    const double2 id13 = make_double2(-d13.y, d13.x);
    a0 = cadd(s02, s13);
    a2 = csub(s02, s13);
    if (DIR < 0) { a1 = csub(d02, id13); a3 = cadd(d02, id13); }
    else         { a1 = cadd(d02, id13); a3 = csub(d02, id13); }
}

// M-point DFT of x[0..M), natural order in and out, in registers.
template <int M, int DIR> struct Dft;

template <int DIR> struct Dft<1, DIR> { CM_HD static void run(double2 *) {} };
template <int DIR> struct Dft<2, DIR> { CM_HD static void run(double2 *x) { radix2<DIR>(x[0], x[1]); } };
template <int DIR> struct Dft<4, DIR> { CM_HD static void run(double2 *x) { radix4<DIR>(x[0], x[1], x[2], x[3]); } };

// second halves of the 8- and 16-point transforms (after the first radix-4 stage), shared by the plain and the
// K-scaled variants
template <int DIR> CM_HD void dft8_tail(double2 *x)
{
    // y[0][k1] at x[2 k1], y[1][k1] at x[1 + 2 k1];  X[k1 + 4 k2] = y[0][k1] + (-1)^k2 w8^{k1} y[1][k1]
    radix2<DIR>(x[0], x[1]);               // X[0], X[4]
    radix2_tw<DIR, 4>(x[2], x[3]);         // X[1], X[5]
    radix2_tw<DIR, 8>(x[4], x[5]);         // X[2], X[6]
    radix2_tw<DIR, 12>(x[6], x[7]);        // X[3], X[7]
    const double2 t1 = x[1], t2 = x[2], t3 = x[3], t4 = x[4], t5 = x[5], t6 = x[6];
    x[1] = t2; x[2] = t4; x[3] = t6; x[4] = t1; x[5] = t3; x[6] = t5;
}
CM_HD void transpose4x4(double2 *x)
{
    double2 t;
    t = x[1];  x[1] = x[4];   x[4] = t;
    t = x[2];  x[2] = x[8];   x[8] = t;
    t = x[3];  x[3] = x[12];  x[12] = t;
    t = x[6];  x[6] = x[9];   x[9] = t;
    t = x[7];  x[7] = x[13];  x[13] = t;
    t = x[11]; x[11] = x[14]; x[14] = t;
}
template <int DIR> CM_HD void dft16_tail(double2 *x)
{
    // y[n1][k1] at x[n1 + 4 k1];  X[k1 + 4 k2] = sum_n1 w4^{n1 k2} w16^{n1 k1} y[n1][k1],  w16 = w32^2
    radix4<DIR>(x[0], x[1], x[2], x[3]);                 // X[0 + 4 k2] at x[k2]
    radix4_tw<DIR, 0, 2, 4, 6>(x[4], x[5], x[6], x[7]);  // X[1 + 4 k2] at x[4 + k2]
    radix4_tw<DIR, 0, 4, 8, 12>(x[8], x[9], x[10], x[11]);
    radix4_tw<DIR, 0, 6, 12, 18>(x[12], x[13], x[14], x[15]);
    transpose4x4(x);                                     // natural[k1 + 4 k2] = x[4 k1 + k2]
}

template <int DIR> struct Dft<8, DIR> {
    // n = n1 + 2 n2, k = k1 + 4 k2:  X = sum_n1 w8^{n1 k1} (-1)^{n1 k2} [sum_n2 x[n1+2n2] w4^{n2 k1}]
    CM_HD static void run(double2 *x)
    {
        radix4<DIR>(x[0], x[2], x[4], x[6]);   // y[0][k1] at x[2 k1]
        radix4<DIR>(x[1], x[3], x[5], x[7]);   // y[1][k1] at x[1 + 2 k1]
        dft8_tail<DIR>(x);
    }
};

template <int DIR> struct Dft<16, DIR> {
    // n = n1 + 4 n2, k = k1 + 4 k2:  X = sum_n1 w16^{n1 k1} w4^{n1 k2} [sum_n2 x[n1+4n2] w4^{n2 k1}]
    CM_HD static void run(double2 *x)
    {
        radix4<DIR>(x[0], x[4], x[8], x[12]);  // y[n1][k1] at x[n1 + 4 k1]
        radix4<DIR>(x[1], x[5], x[9], x[13]);
        radix4<DIR>(x[2], x[6], x[10], x[14]);
        radix4<DIR>(x[3], x[7], x[11], x[15]);
        dft16_tail<DIR>(x);
    }
};

// M-point DFT of (k[0] x[0], ..., k[M-1] x[M-1]) with real k: the scaling rides on the first butterflies.
template <int M, int DIR> struct DftK;
template <int DIR> struct DftK<1, DIR> {
    CM_HD static void run(double2 *x, const double *k) { x[0] = make_double2(k[0] * x[0].x, k[0] * x[0].y); }
};
template <int DIR> struct DftK<2, DIR> {
    CM_HD static void run(double2 *x, const double *k)
    {
        const double2 p = make_double2(k[0] * x[0].x, k[0] * x[0].y), q = x[1];
        x[0] = cfma(k[1], q, p);
        x[1] = cfms(k[1], q, p);
    }
};
template <int DIR> struct DftK<4, DIR> {
    CM_HD static void run(double2 *x, const double *k) { radix4_k<DIR>(x[0], x[1], x[2], x[3], k[0], k[1], k[2], k[3]); }
};
template <int DIR> struct DftK<8, DIR> {
    CM_HD static void run(double2 *x, const double *k)
    {
        radix4_k<DIR>(x[0], x[2], x[4], x[6], k[0], k[2], k[4], k[6]);
        radix4_k<DIR>(x[1], x[3], x[5], x[7], k[1], k[3], k[5], k[7]);
        dft8_tail<DIR>(x);
    }
};
template <int DIR> struct DftK<16, DIR> {
    CM_HD static void run(double2 *x, const double *k)
    {
        radix4_k<DIR>(x[0], x[4], x[8], x[12], k[0], k[4], k[8], k[12]);
        radix4_k<DIR>(x[1], x[5], x[9], x[13], k[1], k[5], k[9], k[13]);
        radix4_k<DIR>(x[2], x[6], x[10], x[14], k[2], k[6], k[10], k[14]);
        radix4_k<DIR>(x[3], x[7], x[11], x[15], k[3], k[7], k[11], k[15]);
        dft16_tail<DIR>(x);
    }
};

// 16-point DFT of x[r] * exp(DIR 2 pi i r / 32) — the odd half of the pruned 32-point first stage.  The modulation
// w32^r = w32^{n1} w8^{n2} (r = n1 + 4 n2) is split: w8^{n2} goes into the first butterflies, w32^{n1} is common to
// the four outputs of butterfly n1 and merges with the inter-stage twiddle w16^{n1 k1} into w32^{n1 (2 k1 + 1)}.
template <int DIR> struct Dft16Mod {
    CM_HD static void run(double2 *x)
    {
        radix4_tw<DIR, 0, 4, 8, 12>(x[0], x[4], x[8], x[12]);
        radix4_tw<DIR, 0, 4, 8, 12>(x[1], x[5], x[9], x[13]);
        radix4_tw<DIR, 0, 4, 8, 12>(x[2], x[6], x[10], x[14]);
        radix4_tw<DIR, 0, 4, 8, 12>(x[3], x[7], x[11], x[15]);
        radix4_tw<DIR, 0, 1, 2, 3>(x[0], x[1], x[2], x[3]);
        radix4_tw<DIR, 0, 3, 6, 9>(x[4], x[5], x[6], x[7]);
        radix4_tw<DIR, 0, 5, 10, 15>(x[8], x[9], x[10], x[11]);
        radix4_tw<DIR, 0, 7, 14, 21>(x[12], x[13], x[14], x[15]);
        transpose4x4(x);
    }
};

// acc[r] += exp(DIR 2 pi i r / 32) * DFT16(x)[r] — the odd half of the pruned 32-point last stage of the inverse,
// added to the even half.  The output modulation w32^{k1} w8^{k2} (r = k1 + 4 k2) is split the same way: w32^{k1}
// moves to the inputs of the second butterfly k1 (with w16^{n1 k1}: w32^{k1 (2 n1 + 1)}), w8^{k2} and the real
// factor left over from the tangent form ride on the FMA that adds the result to acc.
template <int DIR, int K1> CM_HD void dft16modacc_row(double2 *x, double2 *acc)
{
    radix4_tw<DIR, K1, 3 * K1, 5 * K1, 7 * K1>(x[4 * K1], x[4 * K1 + 1], x[4 * K1 + 2], x[4 * K1 + 3]);
    constexpr double g0 = W32<K1, DIR>::G;
    {
        const double2 z = x[4 * K1];
        acc[K1] = cfma(g0, z, acc[K1]);
    }
    {
        constexpr double g = g0 * W32<4, DIR>::G;
        const double2 z = twpre<4, DIR>(x[4 * K1 + 1]);
        acc[K1 + 4] = cfma(g, z, acc[K1 + 4]);
    }
    {
        const double2 z = twpre<8, DIR>(x[4 * K1 + 2]);
        acc[K1 + 8] = cfma(g0, z, acc[K1 + 8]);
    }
    {
        constexpr double g = g0 * W32<12, DIR>::G;
        const double2 z = twpre<12, DIR>(x[4 * K1 + 3]);
        acc[K1 + 12] = cfma(g, z, acc[K1 + 12]);
    }
}
template <int DIR> struct Dft16ModAcc {
    CM_HD static void run(double2 *x, double2 *acc)
    {
        radix4<DIR>(x[0], x[4], x[8], x[12]);  // y[n1][k1] at x[n1 + 4 k1]
        radix4<DIR>(x[1], x[5], x[9], x[13]);
        radix4<DIR>(x[2], x[6], x[10], x[14]);
        radix4<DIR>(x[3], x[7], x[11], x[15]);
        dft16modacc_row<DIR, 0>(x, acc);
        dft16modacc_row<DIR, 1>(x, acc);
        dft16modacc_row<DIR, 2>(x, acc);
        dft16modacc_row<DIR, 3>(x, acc);
    }
};

// storage slot <-> frequency along a transformed axis (2N slots):
//   slot s = p N + 16 k2 + k1   holds frequency   k = 2 k1 + p + 32 k2.
CM_HD int slot_to_freq(int s, int N)
{
    const int p = s / N, rem = s % N;
    return 2 * (rem % E) + p + 2 * E * (rem / E);
}

}  // namespace cmfft
