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

// M-point DFT of x[0..M), natural order in and out, in registers.
template <int M, int DIR> struct Dft;

template <int DIR> struct Dft<1, DIR> { CM_HD static void run(double2 *) {} };
template <int DIR> struct Dft<2, DIR> { CM_HD static void run(double2 *x) { radix2<DIR>(x[0], x[1]); } };
template <int DIR> struct Dft<4, DIR> { CM_HD static void run(double2 *x) { radix4<DIR>(x[0], x[1], x[2], x[3]); } };

template <int DIR> struct Dft<8, DIR> {
    // n = n1 + 2 n2, k = k1 + 4 k2:  X = sum_n1 w8^{n1 k1} (-1)^{n1 k2} [sum_n2 x[n1+2n2] w4^{n2 k1}]
    CM_HD static void run(double2 *x)
    {
        radix4<DIR>(x[0], x[2], x[4], x[6]);   // y[0][k1] at x[2 k1]
        radix4<DIR>(x[1], x[3], x[5], x[7]);   // y[1][k1] at x[1 + 2 k1]
        x[3] = mulw32<4, DIR>(x[3]);
        x[5] = mulw32<8, DIR>(x[5]);
        x[7] = mulw32<12, DIR>(x[7]);
        radix2<DIR>(x[0], x[1]);               // X[0], X[4]
        radix2<DIR>(x[2], x[3]);               // X[1], X[5]
        radix2<DIR>(x[4], x[5]);               // X[2], X[6]
        radix2<DIR>(x[6], x[7]);               // X[3], X[7]
        const double2 t1 = x[1], t2 = x[2], t3 = x[3], t4 = x[4], t5 = x[5], t6 = x[6];
        x[1] = t2; x[2] = t4; x[3] = t6; x[4] = t1; x[5] = t3; x[6] = t5;
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
        // w16^{n1 k1} = w32^{2 n1 k1}
        x[5] = mulw32<2, DIR>(x[5]);   x[6] = mulw32<4, DIR>(x[6]);    x[7] = mulw32<6, DIR>(x[7]);
        x[9] = mulw32<4, DIR>(x[9]);   x[10] = mulw32<8, DIR>(x[10]);  x[11] = mulw32<12, DIR>(x[11]);
        x[13] = mulw32<6, DIR>(x[13]); x[14] = mulw32<12, DIR>(x[14]); x[15] = mulw32<18, DIR>(x[15]);
        radix4<DIR>(x[0], x[1], x[2], x[3]);      // X[0 + 4 k2] at x[k2]
        radix4<DIR>(x[4], x[5], x[6], x[7]);      // X[1 + 4 k2] at x[4 + k2]
        radix4<DIR>(x[8], x[9], x[10], x[11]);
        radix4<DIR>(x[12], x[13], x[14], x[15]);
        // transpose 4x4: natural[k1 + 4 k2] = x[4 k1 + k2]
        double2 t;
        t = x[1];  x[1] = x[4];   x[4] = t;
        t = x[2];  x[2] = x[8];   x[8] = t;
        t = x[3];  x[3] = x[12];  x[12] = t;
        t = x[6];  x[6] = x[9];   x[9] = t;
        t = x[7];  x[7] = x[13];  x[13] = t;
        t = x[11]; x[11] = x[14]; x[14] = t;
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
