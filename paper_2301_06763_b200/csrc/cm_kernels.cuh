// cm_kernels.cuh — the CUDA kernels of libcm (sm_100a, fp64).
//
// Data flow of one solve (steps a1-a8 of SURVEY.md §8):
//
//   rho --k_restrict* (fine->coarse cascade)--> rc       projected cavity density (L280-L282)
//   per level b one COMPLEX field  c_b = rho_full + i rho_hole  (K-hat is real, so the
//   real/imaginary parts of the convolution are Phi_full and Phi_hole: L174-L176)
//   P1 k_x_fwd : rho,rc      -> W1[b][z<N][y<N][sx<2N]     x transform of [N data, N zeros]
//   P2 k_y_fwd : W1          -> W2[b][z<N][sy<2N][sx<2N]
//   P3 k_z_conv: W2 in place    z transform, * K-hat (Eq. 11), inverse z, keep z < N
//   P4 k_y_inv : W2          -> W1[b][z<N][y<N][sx<2N]
//   P5 k_x_inv : W1          -> phi (Re) and hole (Im), scaled by -G dx_b^2, x < N kept; one launch per level,
//                coarse -> fine, adding the prolonged ext_b = P[ext_{b-1} + Phi_hole^{b-1}] (Eq. 3-6 + Eq. 14, step a8)
//
// "sx, sy, sz" are storage slots, not frequencies: slot s = p N + 16 k2 + k1 holds
// frequency 2 k1 + p + 32 k2 (cm_fft.cuh).  The order is whatever makes every global
// access a full 128-byte segment; K-hat is stored in the same slot order.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "cm_fft.cuh"

namespace cmk {

using cmfft::cadd;
using cmfft::cmul;
using cmfft::cmulc;
using cmfft::Dft;

constexpr int kThreads = 128;
// threads of a CTA in the batch-fastest mapping (8 pencils x T threads, at least 128) and pencils it covers
template <int T> __host__ __device__ constexpr int batch_threads() { return 8 * T > kThreads ? 8 * T : kThreads; }
template <int T> __host__ __device__ constexpr int batch_pencils() { return batch_threads<T>() / T; }

// Which slot (within one parity block of N slots) register i of thread j holds after the forward radix-T stage.
//   T <= 16: i = cc T + k2, row k1 = cc T + j            -> slot 16 k2 + k1
//   T = 32 (N = 512): the 32-point stage is split between two threads (below): thread j = (q, c) = (j / 16, j % 16)
//            holds the outputs k2 = 2 i + q of row k1 = c  -> slot 16 (2 i + q) + c
template <int T> __host__ __device__ __forceinline__ constexpr int vslot(int i, int j)
{
    return T <= 16 ? 16 * (i % (T <= 16 ? T : 1)) + (i / (T <= 16 ? T : 1)) * T + j : 16 * (2 * i + (j >> 4)) + (j & 15);
}

// ---- shared-memory exchange layouts ----------------------------------------------
// One pencil's exchange buffer is a [16 (k1)][T (j)] matrix of complex, row stride RS,
// pencil stride PS (in complex elements).  16-byte accesses: a quarter-warp (8 lanes)
// must hit 8 distinct 16-byte columns modulo 128 B.
//  * batch-fastest mapping (y/z passes): the 8 lanes of a quarter-warp are 8 adjacent
//    pencils with the same j  ->  PS odd.
//  * j-fastest mapping (x passes): lanes are consecutive j of one row (and, for T < 8,
//    several rows)  ->  RS odd; PS = 4 (T=4) or 2 (T=2) modulo 8.
template <int T> struct LayBatch {
    static constexpr int RS = T;
    static constexpr int PS = 16 * T + 1;
};
template <int T> struct LayRow {
    static constexpr int RS = T + 1;
    static constexpr int PS = 16 * (T + 1) + (T == 4 ? 4 : (T == 2 ? 2 : 0));
};

struct SyncBlock { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
struct SyncWarp  { __device__ __forceinline__ void operator()() const { __syncwarp(); } };

// ---- twiddle sources ------------------------------------------------------------------
// w_2N^{j (2 k1 + P)}: from the global table (read-only path) or from a per-CTA shared copy
// laid out [2 k1 + P][j] so that consecutive j are consecutive 16-byte words.
struct TwGlobal {
    const double2 *__restrict__ tw;
    int j;
    static constexpr bool RECUR = false;
    template <int P> __device__ __forceinline__ double2 get(int k1) const { return __ldg(&tw[j * (2 * k1 + P)]); }
};
// P3 is bound by the shared-memory data pipe as much as by fp64 (profiles/): only every ANCH-th twiddle (k1 = 0, ANCH, ...)
// is read from the table.  The ones between follow from the three-term recurrence of a geometric sequence,
//     t[k+1] = 2 cos(phi) t[k] - t[k-1],   phi = arg of the ratio rho = w_2N^{2 j},
// one FMA per component (a complex multiply by rho would be four).  Its rounding error is ~1e-14 of a twiddle whatever the
// anchor spacing (it is set by the cancellation in 2 cos(phi) at small phi, not by the step count: 1.1e-14 / 1.6e-14 /
// 1.0e-14 at ANCH = 4 / 8 / 16), three orders below the parity bar.  ANCH is chosen per kernel by measurement
// (profiles/r02_p3_experiments.md): 16 in the CTA-wide TMA kernel (one table read per exchange), 8 in the warp-autonomous
// one (16 spills registers there).
template <int T, int ANCH_ = 16> struct TwShared {
    const double2 *base;   // table + j
    double2 rho;           // w_2N^{2 j}
    static constexpr bool RECUR = true;
    static constexpr int ANCH = ANCH_;
    template <int P> __device__ __forceinline__ double2 get(int k1) const { return base[(2 * k1 + P) * T]; }
};

// twiddle w_2N^{j (2 k1 + P)} for k1 = 0..15 in turn; p1 / p2 carry the two values before it
struct TwCarry { double2 p1, p2; };
template <int P, class Tw> __device__ __forceinline__ double2 tw_next(const Tw &tw, int k1, TwCarry &c)
{
    double2 t;
    if constexpr (Tw::RECUR) {
        if ((k1 & (Tw::ANCH - 1)) == 0) t = (P == 0 && k1 == 0) ? make_double2(1.0, 0.0) : tw.template get<P>(k1);
        else if (k1 == 1) t = (P == 0) ? tw.rho : cmul(c.p1, tw.rho);
        else {
            const double c2 = 2.0 * tw.rho.x;
            t = make_double2(fma(c2, c.p1.x, -c.p2.x), fma(c2, c.p1.y, -c.p2.y));
        }
    } else {
        t = tw.template get<P>(k1);
    }
    c.p2 = c.p1;
    c.p1 = t;
    return t;
}

// ---- half transforms ---------------------------------------------------------------
// element (row, col) of a pencil's exchange matrix
template <class Lay> __device__ __forceinline__ double2 &ex_at(double2 *sm, int row, int col) { return sm[row * Lay::RS + col]; }
// K-hat of a slot: a pencil's parity block as it lies in memory, or an accessor (cm_expand.cuh keeps only the half that
// the evenness of K-hat in the z frequency leaves)
__device__ __forceinline__ double kh_at(const double *kh, int slot) { return kh[slot]; }
template <class KH> __device__ __forceinline__ double kh_at(const KH &kh, int slot) { return kh(slot); }

// Forward, parity P: a[r] = input element n = j + T r (r < 16).  On return
// v[cc*T + k2] is the spectrum value of slot  P*N + 16*k2 + cc*T + j.
// PRE: synchronise before writing the exchange buffer (needed when one buffer serves
// consecutive exchanges).
template <int T, int P, class Lay, bool PRE = false, class Sync, class Tw>
__device__ __forceinline__ void fwd_half(const double2 (&a)[16], double2 (&v)[16], int j, double2 *sm, Tw tw, Sync sync)
{
    double2 b[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) b[r] = a[r];
    if (P) cmfft::Dft16Mod<-1>::run(b);     // inputs times w_32^r, folded into the butterflies
    else Dft<16, -1>::run(b);
    if (T > 1) {
        if (PRE) sync();
        TwCarry twc{make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) {
            const double2 t = tw_next<P>(tw, k1, twc);
            if (k1 > 0 || P) b[k1] = cmul(b[k1], t);
            ex_at<Lay>(sm, k1, j) = b[k1];
        }
        sync();
        if constexpr (T <= 16) {
#pragma unroll
            for (int cc = 0; cc < 16 / T; ++cc) {
#pragma unroll
                for (int jj = 0; jj < T; ++jj) v[cc * T + jj] = ex_at<Lay>(sm, cc * T + j, jj);
                Dft<T, -1>::run(&v[cc * T]);
            }
        } else {
            // 32-point stage over the threads, decimated in frequency and split between two threads: thread (q, c)
            // forms the outputs k2 = 2 m + q of row c:  X[2m+q] = sum_jj w16^{jj m} w32^{jj q} (x[jj] + (-1)^q x[jj+16])
            static_assert(T == 32, "radix-T stage: T <= 16 or T = 32");
            const int q = j >> 4, c = j & 15;
            const double sg = q ? -1.0 : 1.0;
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) v[jj] = cmfft::cfma(sg, ex_at<Lay>(sm, c, jj + 16), ex_at<Lay>(sm, c, jj));
            if (q) cmfft::Dft16Mod<-1>::run(v);
            else Dft<16, -1>::run(v);
        }
    } else {
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) v[k1] = b[k1];
    }
}

// cos / sin of 2 pi n / 32, n = 0 .. 15 (the modulation of the odd half of a 32-point stage, folded variant)
__host__ __device__ constexpr double cos32(int n)
{
    constexpr double t[9] = {1.0, 0.98078528040323043, 0.92387953251128674, 0.83146961230254524, 0.70710678118654757,
                             0.55557023301960218, 0.38268343236508978, 0.19509032201612825, 0.0};
    return n <= 8 ? t[n] : -t[16 - n];
}
__host__ __device__ constexpr double sin32(int n) { return n <= 8 ? cos32(8 - n) : cos32(n - 8); }

// Inverse, parity P: v as above (consumed).  P = 0: on return o[r] is the even half's contribution to output
// element n = j + T r, r < 16 (the cropped half).  P = 1: the odd half's contribution, times conj(w_32^r), is ADDED
// to o[r] (the caller passes the even half's result).  KM: v is first multiplied by the real
// kh[16*k2 + cc*T] (K-hat of this thread's slots, Eq. 11), folded into the first butterflies.
// DEC > 1 (cm_expand.cuh): only the threads with j % DEC == 0 run the last stage — their outputs n = j + T r are the
// multiples of DEC, all a decimated inverse keeps; the others only take part in the exchange.
template <int T, int P, class Lay, bool PRE = false, bool KM = false, int DEC = 1, class Sync, class Tw, class KH = const double *>
__device__ __forceinline__ void inv_half(double2 (&v)[16], double2 (&o)[16], int j, double2 *sm, Tw tw, Sync sync, KH kh = nullptr)
{
    static_assert(DEC == 1 || (T > 1 && T % DEC == 0), "decimation needs the radix-T stage");
    double2 w[16];
    if (T > 1) {
        if (PRE) sync();
        if constexpr (T <= 16 && DEC > 1) {
            // Decimated: only the outputs jj = DEC jj' of the T-point stage are ever read (by the threads j % DEC == 0), and
            //     y[DEC jj'] = sum_{m < T/DEC} ( sum_{q < DEC} V[m + (T/DEC) q] ) w_{T/DEC}^{m jj'}:
            // fold the inputs (the K-hat product rides on the fold as FMAs), transform T/DEC points, write T/DEC columns.
            constexpr int TD = T / DEC;
#pragma unroll
            for (int cc = 0; cc < 16 / T; ++cc) {
                double2 f[TD];
#pragma unroll
                for (int m = 0; m < TD; ++m) {
#pragma unroll
                    for (int q = 0; q < DEC; ++q) {
                        const int i = cc * T + m + TD * q;
                        if (KM) {
                            const double k = kh_at(kh, vslot<T>(i, j));
                            f[m] = q ? make_double2(fma(k, v[i].x, f[m].x), fma(k, v[i].y, f[m].y)) : make_double2(k * v[i].x, k * v[i].y);
                        } else {
                            f[m] = q ? make_double2(f[m].x + v[i].x, f[m].y + v[i].y) : v[i];
                        }
                    }
                }
                Dft<TD, +1>::run(f);
#pragma unroll
                for (int jj = 0; jj < TD; ++jj) ex_at<Lay>(sm, cc * T + j, DEC * jj) = f[jj];
            }
            sync();
        } else if constexpr (T <= 16) {
#pragma unroll
            for (int cc = 0; cc < 16 / T; ++cc) {
                if (KM) {
                    double k[T];
#pragma unroll
                    for (int k2 = 0; k2 < T; ++k2) k[k2] = kh_at(kh, vslot<T>(cc * T + k2, j));
                    cmfft::DftK<T, +1>::run(&v[cc * T], k);
                } else {
                    Dft<T, +1>::run(&v[cc * T]);
                }
#pragma unroll
                for (int jj = 0; jj < T; ++jj) ex_at<Lay>(sm, cc * T + j, jj) = v[cc * T + jj];
            }
            sync();
        } else {
            // the 32-point stage backwards: thread (q, c) turns its outputs k2 = 2 m + q of row c into
            // y_q[jj] = w32^{-q jj} sum_m V[2m+q] w16^{-m jj}; the owner of column jj + 16 h then takes y_0 + (-1)^h y_1
            const int q = j >> 4, c = j & 15;
            if constexpr (DEC > 1) {
                // Decimated (see the T <= 16 branch): only the columns jj = DEC jj' are read, and for those
                //     y_q[DEC jj'] = w32^{-q DEC jj'} sum_{m' < 16/DEC} ( sum_p V[2 (m' + (16/DEC) p) + q] ) w_{16/DEC}^{-m' jj'}
                constexpr int TD = 16 / DEC;
                double2 f[TD];
#pragma unroll
                for (int m = 0; m < TD; ++m) {
#pragma unroll
                    for (int p = 0; p < DEC; ++p) {
                        const int i = m + TD * p;
                        if (KM) {
                            const double k = kh_at(kh, vslot<T>(i, j));
                            f[m] = p ? make_double2(fma(k, v[i].x, f[m].x), fma(k, v[i].y, f[m].y)) : make_double2(k * v[i].x, k * v[i].y);
                        } else {
                            f[m] = p ? make_double2(f[m].x + v[i].x, f[m].y + v[i].y) : v[i];
                        }
                    }
                }
                Dft<TD, +1>::run(f);
#pragma unroll
                for (int jj = 0; jj < TD; ++jj) {
                    // conj(w32)^{DEC jj}, applied by the odd-k2 thread only
                    const double2 m32 = make_double2(cos32(DEC * jj), sin32(DEC * jj));
                    ex_at<Lay>(sm, c, 16 * q + DEC * jj) = q ? cmul(f[jj], m32) : f[jj];
                }
                sync();
            } else {
            double2 y[16];
            if (q) {
                if (KM) {
#pragma unroll
                    for (int m = 0; m < 16; ++m) {
                        const double k = kh_at(kh, vslot<T>(m, j));
                        v[m].x *= k;
                        v[m].y *= k;
                    }
                }
#pragma unroll
                for (int m = 0; m < 16; ++m) y[m] = make_double2(0.0, 0.0);
                cmfft::Dft16ModAcc<+1>::run(v, y);
            } else {
                if (KM) {
                    double k[16];
#pragma unroll
                    for (int m = 0; m < 16; ++m) k[m] = kh_at(kh, vslot<T>(m, j));
                    cmfft::DftK<16, +1>::run(v, k);
                } else {
                    Dft<16, +1>::run(v);
                }
#pragma unroll
                for (int m = 0; m < 16; ++m) y[m] = v[m];
            }
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) ex_at<Lay>(sm, c, 16 * q + jj) = y[jj];
            sync();
            }
        }
        if (DEC > 1 && (j % DEC) != 0) return;
        TwCarry twc{make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) {
            if constexpr (T <= 16) w[k1] = ex_at<Lay>(sm, k1, j);
            else w[k1] = cmfft::cfma((j >> 4) ? -1.0 : 1.0, ex_at<Lay>(sm, k1, 16 + (j & 15)), ex_at<Lay>(sm, k1, j & 15));
            const double2 t = tw_next<P>(tw, k1, twc);
            if (k1 > 0 || P) w[k1] = cmulc(w[k1], t);
        }
    } else {
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) {
            w[k1] = v[k1];
            if (KM) { const double k = kh_at(kh, vslot<T>(k1, j)); w[k1].x *= k; w[k1].y *= k; }
        }
    }
    if (P) {
        cmfft::Dft16ModAcc<+1>::run(w, o);
    } else {
        Dft<16, +1>::run(w);
#pragma unroll
        for (int r = 0; r < 16; ++r) o[r] = w[r];
    }
}

__device__ __forceinline__ bool in_cavity1(int v, int N) { return v >= N / 4 && v < 3 * N / 4; }
__device__ __forceinline__ bool in_ring1(int v, int N) { return v >= N / 4 - 1 && v <= 3 * N / 4; }

// ================================ P1: x forward ====================================
// One row (b, z, y) per group of T threads (j fastest).  Reads N reals, forms the complex
// pair field (step a2, never materialised), writes 2N complex slots.
// body: thread (rowl, j) of a CTA transforms global row `row` (b, z, y) and writes its 2N slots to `dst`
// GEN (general sizes): the level has nd <= N cells per axis (nd % 4 == 0) and is transformed at the next power
// of two N = 16 T — the rows, the cavity geometry and the arrays of the caller follow nd, the spectra follow N; cells
// x >= nd are zero like the padding.  GEN = false: nd = N at compile time (the code of the power-of-two sizes).
template <int T, bool GEN = false>
__device__ __forceinline__ void x_fwd_body(const double *__restrict__ rho, const double *__restrict__ rc, double2 *dst,
                                           const double2 *__restrict__ tw, int L, size_t row, double2 *smem, int nd_arg = 0,
                                           bool valid = true)
{
    constexpr int N = 16 * T, ROWS = kThreads / T;
    const int nd = GEN ? nd_arg : N, H = nd / 2, Q = nd / 4;
    using Lay = LayRow<T>;
    const int tid = threadIdx.x, j = tid % T, rowl = tid / T;
    const int y = (int)(row % nd), z = (int)((row / nd) % nd), b = (int)(row / ((size_t)nd * nd));
    const bool finest = (b == L - 1);
    const bool rowcav = !finest && in_cavity1(z, nd) && in_cavity1(y, nd);
    const double *src = rho + row * nd;
    const double *srcc = rowcav ? rc + (((size_t)b * H + (z - Q)) * H + (y - Q)) * H - Q : rho;

    double2 a[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int x = j + T * r;
        const bool cav = rowcav && in_cavity1(x, nd);
        double re = 0.0;
        if (!GEN || x < nd) re = cav ? __ldg(srcc + x) : __ldg(src + x);
        a[r] = make_double2(re, (finest || cav) ? 0.0 : re);
    }
    double2 *bufA = smem + rowl * Lay::PS, *bufB = bufA + ROWS * Lay::PS;
    {
        double2 v[16];
        fwd_half<T, 0, Lay>(a, v, j, bufA, TwGlobal{tw, j}, SyncWarp());
        if (!GEN || valid) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dst[vslot<T>(i, j)] = v[i];
        }
    }
    {
        double2 v[16];
        fwd_half<T, 1, Lay>(a, v, j, bufB, TwGlobal{tw, j}, SyncWarp());
        if (!GEN || valid) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dst[N + vslot<T>(i, j)] = v[i];
        }
    }
}

template <int T, bool GEN = false>
__global__ void __launch_bounds__(kThreads) k_x_fwd(const double *__restrict__ rho, const double *__restrict__ rc,
                                                    double2 *__restrict__ W1, const double2 *__restrict__ tw, int L,
                                                    size_t row0, int nd = 0, size_t row_end = 0)
{
    // row0: first global row (b, z, y) of this launch; GEN: rows at and beyond row_end do not exist (the last CTA is ragged:
    // its surplus threads redo the last row without storing, so that every warp stays whole for the exchanges)
    constexpr int NN = 32 * T, ROWS = kThreads / T;
    extern __shared__ double2 smem[];
    size_t row = row0 + (size_t)blockIdx.x * ROWS + threadIdx.x / T;
    const bool valid = !GEN || row < row_end;
    if (GEN && !valid) row = row_end - 1;
    x_fwd_body<T, GEN>(rho, rc, W1 + row * NN, tw, L, row, smem, nd, valid);
}

// P1 split by output parity (see k_y_fwd_split): 256 threads, warps 0-3 the even slots, warps 4-7 the odd ones
// of the SAME rows.
template <int T>
__global__ void __launch_bounds__(2 * kThreads, 2) k_x_fwd_split(const double *__restrict__ rho, const double *__restrict__ rc,
                                                                 double2 *__restrict__ W1, const double2 *__restrict__ tw, int L)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, H = N / 2, Q = N / 4;
    using Lay = LayRow<T>;
    extern __shared__ double2 smem[];
    const int P = threadIdx.x / kThreads, tid = threadIdx.x % kThreads, j = tid % T, rowl = tid / T;
    const size_t row = (size_t)blockIdx.x * ROWS + rowl;
    const int y = (int)(row % N), z = (int)((row / N) % N), b = (int)(row / ((size_t)N * N));
    const bool finest = (b == L - 1);
    const bool rowcav = !finest && in_cavity1(z, N) && in_cavity1(y, N);
    const double *src = rho + row * N;
    const double *srcc = rowcav ? rc + (((size_t)b * H + (z - Q)) * H + (y - Q)) * H - Q : rho;
    double2 a[16], v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int x = j + T * r;
        const bool cav = rowcav && in_cavity1(x, N);
        const double re = cav ? __ldg(srcc + x) : __ldg(src + x);
        a[r] = make_double2(re, (finest || cav) ? 0.0 : re);
    }
    double2 *buf = smem + (P * ROWS + rowl) * Lay::PS;
    if (P == 0) fwd_half<T, 0, Lay>(a, v, j, buf, TwGlobal{tw, j}, SyncWarp());
    else fwd_half<T, 1, Lay>(a, v, j, buf, TwGlobal{tw, j}, SyncWarp());
    double2 *dst = W1 + row * NN + P * N;
#pragma unroll
    for (int i = 0; i < 16; ++i) dst[vslot<T>(i, j)] = v[i];
}

// ====================== P5: x inverse + a8 (prolongation, Eq. 14) ==================
// One launch per level b, coarse -> fine (row0 = b N^2): the level's rows are transformed back,
// cropped to x < N and scaled by -G dx_b^2; then the contribution of the coarser levels is added
// on the spot (step a8): with Hc = ext_{b-1} + Phi_hole^{b-1} on the parent grid (valid on the
// cavity grown by one cell, written by the previous launch), a fine cell f with parent
// p = N/4 + f/2 and sign s = +1 (f odd) / -1 (f even) gets
//     ext_b(f) = 3/4 Hc[p] + 1/4 Hc[p+s]        (Eq. 3-6)
//     Phi(Omega_b) = Phi^b + ext_b               (Eq. 14)
// and hole_b = Phi_hole^b + ext_b is kept where the next level will read it (on every cell if hole_all:
// the modified method, Eq. B.1, builds Phi(Omega_b) from it).
//
// The L launches are chained by programmatic dependent launch: a level's CTAs let the next level start as soon as
// they are all resident (griddepcontrol.launch_dependents at the top), and only the fetch of Hc — the one thing that
// needs the level before — sits behind griddepcontrol.wait.  So level b+1 loads its spectrum and runs its inverse
// transforms under the tail of level b instead of after it (at N <= 128 a level is a wave or less: without this
// the levels ran one after the other on a partly empty GPU).  W1 is complete before level 0 starts (a normal launch).
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// LATE (N <= 128): fetch Hc after the transforms, behind griddepcontrol.wait — the level overlaps the one before it.
// N = 256 (a level is 28 waves, the overlap is worth little): wait first and fetch Hc at the top, so that its latency
// hides behind the transforms as before (measured: late fetch there 1.68 -> 2.18 ms).
template <int T, bool GEN = false>
__global__ void __launch_bounds__(kThreads, 2) k_x_inv(const double2 *__restrict__ W1, double *__restrict__ phi,
                                                    double *__restrict__ hole, const double *__restrict__ hole_c,
                                                    const double2 *__restrict__ tw, int L, double scale0 /* -G dx0^2 */,
                                                    size_t row0, int hole_all, int nd_arg = 0)
{
    // GEN: nd <= N cells per axis (see x_fwd_body); a level has nd^2 rows, the last CTA may be ragged
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T;
    const int nd = GEN ? nd_arg : N, Q = nd / 4;
    constexpr bool LATE = (T <= 8);
    using Lay = LayRow<T>;
    extern __shared__ double2 smem[];
    pdl_launch_dependents();
    const int tid = threadIdx.x, j = tid % T, rowl = tid / T;
    size_t rowc = (size_t)blockIdx.x * ROWS + rowl;
    const bool valid = !GEN || rowc < (size_t)nd * nd;
    if (GEN && !valid) rowc = (size_t)nd * nd - 1;
    const size_t row = row0 + rowc;
    const int y = (int)(row % nd), z = (int)((row / nd) % nd), b = (int)(row / ((size_t)nd * nd));
    const double2 *src = W1 + row * NN;
    double2 *bufA = smem + rowl * Lay::PS, *bufB = bufA + ROWS * Lay::PS;

    // a8: the prolonged contribution of the coarser levels (L2 hits: the launch before this one wrote it)
    double ext[16];
    auto fetch_ext = [&]() {
        if (b > 0) {
            pdl_wait();
            const double *Hc = hole_c + (size_t)(b - 1) * nd * nd * nd;
            const int pk = Q + z / 2, pj = Q + y / 2, sk = (z & 1) ? 1 : -1, sj = (y & 1) ? 1 : -1;
            const double *h0 = Hc + ((size_t)pk * nd + pj) * nd, *h1 = Hc + ((size_t)(pk + sk) * nd + (pj + sj)) * nd;
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int x = j + T * r, pi = Q + x / 2, si = (x & 1) ? 1 : -1;
                ext[r] = (!GEN || x < nd) ? 0.75 * __ldcg(h0 + pi) + 0.25 * __ldcg(h1 + pi + si) : 0.0;
            }
        } else {
#pragma unroll
            for (int r = 0; r < 16; ++r) ext[r] = 0.0;
        }
    };

    double2 v0[16], v1[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        v0[i] = src[vslot<T>(i, j)];
        v1[i] = src[N + vslot<T>(i, j)];
    }
    if (!LATE) fetch_ext();
    double2 e[16];
    inv_half<T, 0, Lay>(v0, e, j, bufA, TwGlobal{tw, j}, SyncWarp());
    inv_half<T, 1, Lay>(v1, e, j, bufB, TwGlobal{tw, j}, SyncWarp());     // adds the odd half
    if (LATE) fetch_ext();
    if (GEN && !valid) return;

    const bool rowring = (b < L - 1) && in_ring1(z, nd) && in_ring1(y, nd);
    const double scale = scale0 * exp2(-2.0 * b);   // dx_b^2 = dx0^2 / 4^b, exact
    double *dphi = phi + row * nd, *dh = hole + row * nd;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int x = j + T * r;
        if (GEN && x >= nd) continue;
        const double re = scale * e[r].x, im = scale * e[r].y;
        dphi[x] = b > 0 ? re + ext[r] : re;
        if (hole_all ? (b < L - 1) : (rowring && in_ring1(x, nd))) dh[x] = b > 0 ? im + ext[r] : im;
    }
}

// ======================= batch-fastest mapping (y and z passes) ====================
// tid -> px = tid & 7 (8 adjacent slots = one 128-byte segment), j = (tid >> 3) % T,
// g = tid / (8 T).  A CTA covers batch_pencils<T>() adjacent batch positions (128 threads; 256 at T = 32).

// ================================ P2: y forward ====================================
// (min-blocks choices are measured, DESIGN.md §6 / profiles/r02_pass_variants.md: with the FMA-fused butterflies every
// pass is best with a floor of 2 CTAs per SM, which lets ptxas use up to 255 registers — capping P4 or P5 at 168
// registers for a third CTA costs 25-45 %; P2 at N <= 128 is left to ptxas (178 registers))
// body: the CTA transforms PEN = 8 * (16/T) adjacent sx columns of one (b, z) plane; src/dst point at
// this thread's column (sx) of the plane's W1 rows / W2 rows.  [ylo, yhi): the rows that hold data (the rest of the
// column is taken as zero without being read: the expanded grids of cm_expand.cuh); the whole column by default.
template <int T, class Sync = SyncBlock>
__device__ __forceinline__ void y_fwd_body(const double2 *src, double2 *dst, const double2 *__restrict__ tw, double2 *smem,
                                           int ylo = 0, int yhi = 16 * T)
{
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    using Lay = LayBatch<T>;
    const int tid = threadIdx.x, px = tid & 7, j = (tid >> 3) % T, g = tid / (8 * T);
    double2 *bufA = smem + (g * 8 + px) * Lay::PS, *bufB = bufA + PEN * Lay::PS;

    double2 a[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int y = j + T * r;
        a[r] = (y >= ylo && y < yhi) ? src[(size_t)y * NN] : make_double2(0.0, 0.0);
    }
    {
        double2 v[16];
        fwd_half<T, 0, Lay>(a, v, j, bufA, TwGlobal{tw, j}, Sync());
#pragma unroll
        for (int i = 0; i < 16; ++i) dst[(size_t)vslot<T>(i, j) * NN] = v[i];
    }
    {
        double2 v[16];
        fwd_half<T, 1, Lay>(a, v, j, bufB, TwGlobal{tw, j}, Sync());
#pragma unroll
        for (int i = 0; i < 16; ++i) dst[(size_t)(N + vslot<T>(i, j)) * NN] = v[i];
    }
}

template <int T, bool GEN = false, bool PF = false>
__global__ void __launch_bounds__(batch_threads<T>()) k_y_fwd(const double2 *__restrict__ W1, double2 *__restrict__ W2,
                                                    const double2 *__restrict__ tw, int nd_arg = 0, int ahead = 0)
{
    // GEN: a plane has nd <= N rows of data (see x_fwd_body); bz counts the nd planes of every level
    // PF (one or two CTAs per SM and register loads: nothing else hides the load latency): pull the columns of the CTA `ahead`
    // places later into L2.  A template flag: the code without it is untouched.
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    const int nd = GEN ? nd_arg : N;
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, px = tid & 7, g = tid / (8 * T);
    const size_t q = (size_t)blockIdx.x * PEN + g * 8 + px;      // (b*nd + z) * 2N + sx
    const size_t bz = q / NN;
    const int sx = (int)(q % NN);
    if (PF && px == 0 && blockIdx.x + ahead < gridDim.x) {
        const size_t q2 = (size_t)(blockIdx.x + ahead) * PEN + g * 8;
        const double2 *s2 = W1 + (q2 / NN) * nd * NN + (q2 % NN);
        const int j = (tid >> 3) % T;
#pragma unroll
        for (int r = 0; r < 16; ++r)
            if (j + T * r < nd) asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)(j + T * r) * NN));
    }
    y_fwd_body<T>(W1 + bz * nd * NN + sx, W2 + bz * NN * NN + sx, tw, smem, 0, nd);
}

// P2 split by output parity: 256 threads, warps 0-3 form the even slots (P = 0), warps 4-7 the odd ones
// (P = 1) of the SAME columns.  The two halves of a forward transform share nothing but their input, so
// each thread carries one half only: about half the registers, twice the warps per SM (latency hiding),
// at the price of reading the input twice (the second read is an L1/L2 hit).
struct SyncParity {
    int id;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }
};
template <int T>
__global__ void __launch_bounds__(2 * kThreads, 2) k_y_fwd_split(const double2 *__restrict__ W1, double2 *__restrict__ W2,
                                                                 const double2 *__restrict__ tw, int ahead)
{
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    using Lay = LayBatch<T>;
    extern __shared__ double2 smem[];
    const int P = threadIdx.x / kThreads, tid = threadIdx.x % kThreads;
    const int px = tid & 7, j = (tid >> 3) % T, g = tid / (8 * T);
    const size_t q = (size_t)blockIdx.x * PEN + g * 8 + px;      // (b*N + z) * 2N + sx
    const size_t bz = q / NN;
    const int sx = (int)(q % NN);
    const double2 *src = W1 + bz * N * NN + sx;
    double2 *dst = W2 + bz * NN * NN + sx + (size_t)P * N * NN;
    double2 *buf = smem + (P * PEN + g * 8 + px) * Lay::PS;
    double2 a[16], v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) a[r] = src[(size_t)(j + T * r) * NN];
    {   // Pull the input of the tile `ahead` CTAs later into L2 (one lane per 128-byte line).  ncu: 55 % of this kernel's
        // stall samples sit on the load scoreboard and it moves 5.8 TB/s where P4 — the same bytes the other way round, twice
        // the unique loads per CTA in flight — reaches the copy peak; registers (128 x 512 threads = the whole file) leave no
        // room for a second tile.  With the next wave's columns already in L2 the load phase shrinks: 2.78 -> 2.59 ms at
        // 10 x 256^3 (ahead = 148 = half a wave of CTAs; 74 ... 444 within 3 %; profiles/r02_pass_variants.md).
        if (ahead > 0 && P == 0 && px == 0 && blockIdx.x + ahead < gridDim.x) {
            const size_t q2 = (size_t)(blockIdx.x + ahead) * PEN + g * 8;
            const double2 *s2 = W1 + (q2 / NN) * N * NN + (q2 % NN);
#pragma unroll
            for (int r = 0; r < 16; ++r) asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)(j + T * r) * NN));
        }
    }
    if (P == 0) fwd_half<T, 0, Lay>(a, v, j, buf, TwGlobal{tw, j}, SyncParity{1});
    else fwd_half<T, 1, Lay>(a, v, j, buf, TwGlobal{tw, j}, SyncParity{2});
#pragma unroll
    for (int i = 0; i < 16; ++i) dst[(size_t)vslot<T>(i, j) * NN] = v[i];
}

// ================================ P4: y inverse ====================================
template <int T, bool GEN = false, bool PF = false>
__global__ void __launch_bounds__(batch_threads<T>(), T == 32 ? 1 : 2) k_y_inv(const double2 *__restrict__ W2, double2 *__restrict__ W1,
                                                    const double2 *__restrict__ tw, int nd_arg = 0, int ahead = 0)
{
    // GEN: only the nd <= N rows of data are kept (see x_fwd_body); ahead: as in k_y_fwd
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    const int nd = GEN ? nd_arg : N;
    using Lay = LayBatch<T>;
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, px = tid & 7, j = (tid >> 3) % T, g = tid / (8 * T);
    const size_t q = (size_t)blockIdx.x * PEN + g * 8 + px;
    const size_t bz = q / NN;
    const int sx = (int)(q % NN);
    if (PF && px == 0 && blockIdx.x + ahead < gridDim.x) {
        const size_t q2 = (size_t)(blockIdx.x + ahead) * PEN + g * 8;
        const double2 *s2 = W2 + (q2 / NN) * NN * NN + (q2 % NN);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)vslot<T>(i, j) * NN));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)(N + vslot<T>(i, j)) * NN));
        }
    }
    const double2 *src = W2 + bz * NN * NN + sx;
    double2 *dst = W1 + bz * nd * NN + sx;
    double2 *bufA = smem + (g * 8 + px) * Lay::PS, *bufB = bufA + PEN * Lay::PS;

    double2 v0[16], v1[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        v0[i] = src[(size_t)vslot<T>(i, j) * NN];
        v1[i] = src[(size_t)(N + vslot<T>(i, j)) * NN];
    }
    double2 e[16];
    inv_half<T, 0, Lay>(v0, e, j, bufA, TwGlobal{tw, j}, SyncBlock());
    inv_half<T, 1, Lay>(v1, e, j, bufB, TwGlobal{tw, j}, SyncBlock());   // adds the odd half
#pragma unroll
    for (int r = 0; r < 16; ++r)
        if (!GEN || j + T * r < nd) dst[(size_t)(j + T * r) * NN] = e[r];
}

// ============================ a1: restriction cascade ==============================
// rc[lf-1][ck][cj][ci] = mean of the 8 children of fine level lf, where a child that lies
// under level lf+1 takes the already projected value rc[lf] (L280-L282; readings 9, 10).
__device__ __forceinline__ double restrict_cell(int N, bool use_rc, const double *__restrict__ rho_f, const double *__restrict__ rc_f,
                                                int ci, int cj, int ck)
{
    const int H = N / 2, Q = N / 4;
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int bb = 0; bb < 2; ++bb)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int k = 2 * ck + c, jx = 2 * cj + bb, i = 2 * ci + a;
                const bool cav = use_rc && in_cavity1(k, N) && in_cavity1(jx, N) && in_cavity1(i, N);
                s += cav ? rc_f[((size_t)(k - Q) * H + (jx - Q)) * H + (i - Q)]
                         : rho_f[((size_t)k * N + jx) * N + i];
            }
    return 0.125 * s;
}
static __global__ void k_restrict(int N, int lf, int L, const double *__restrict__ rho_f, const double *__restrict__ rc_f,
                                  double *__restrict__ rc_out)
{
    const int H = N / 2;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= H * H * H) return;
    rc_out[idx] = restrict_cell(N, lf < L - 1, rho_f, rc_f, idx % H, (idx / H) % H, idx / (H * H));
}
// The cascade is sequential only where a parent has a child under the next finer grid: the box [I0, I1)^3 of parents,
// I0 = N/8 (rounded down), I1 = 3N/8 (rounded up) — 1/8 of a level's outputs.  cm_potential therefore runs a1 as ONE launch
// over every level for the parents outside that box (all parents of the finest level), which read rho only, and then
// fine -> coarse one small launch per level for the box.  Same per-cell sum in the same order as k_restrict: same bits.
__device__ __forceinline__ int restrict_box_lo(int N) { return (N / 4) / 2; }
__device__ __forceinline__ int restrict_box_hi(int N) { return (3 * (N / 4) + 1) / 2; }
static __global__ void k_restrict_outer(int N, int L, const double *__restrict__ rho, double *__restrict__ rc)
{
    const int H = N / 2, lf = blockIdx.y + 1;                      // level lf projects onto level lf - 1
    const size_t n3 = (size_t)N * N * N, h3 = n3 / 8;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= H * H * H) return;
    const int ci = idx % H, cj = (idx / H) % H, ck = idx / (H * H), lo = restrict_box_lo(N), hi = restrict_box_hi(N);
    if (lf < L - 1 && ci >= lo && ci < hi && cj >= lo && cj < hi && ck >= lo && ck < hi) return;   // the cascade's
    // rho only: the two x-children of a parent are one aligned 16-byte word; summed in restrict_cell's order
    const double *rho_f = rho + n3 * lf;
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int bb = 0; bb < 2; ++bb) {
            const double2 v = __ldg(reinterpret_cast<const double2 *>(rho_f + ((size_t)(2 * ck + c) * N + (2 * cj + bb)) * N + 2 * ci));
            s += v.x;
            s += v.y;
        }
    rc[h3 * (lf - 1) + idx] = 0.125 * s;
}
static __global__ void k_restrict_inner(int N, int lf, const double *__restrict__ rho_f, const double *__restrict__ rc_f,
                                        double *__restrict__ rc_out)
{
    const int H = N / 2, lo = restrict_box_lo(N), B = restrict_box_hi(N) - lo;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= B * B * B) return;
    const int ci = lo + idx % B, cj = lo + (idx / B) % B, ck = lo + idx / (B * B);
    rc_out[((size_t)ck * H + cj) * H + ci] = restrict_cell(N, true, rho_f, rc_f, ci, cj, ck);
}

// Level sharding across GPUs: all that a8 of level b reads of level b-1 is H = ext + Phi_hole on the
// cavity grown by one cell, the box [N/4 - 1, 3N/4 + 1)^3.  Pack it into (N/2 + 2)^3 contiguous doubles for the
// exchange, or unpack a received box into the level's slot of the hole buffer.
static __global__ void k_ring_box(int N, double *__restrict__ level, double *__restrict__ box, int unpack)
{
    const int B = N / 2 + 2, Q1 = N / 4 - 1;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)B * B * B) return;
    const int x = (int)(i % B), y = (int)((i / B) % B), z = (int)(i / ((size_t)B * B));
    double *c = level + ((size_t)(Q1 + z) * N + (Q1 + y)) * N + (Q1 + x);
    if (unpack) *c = box[i];
    else box[i] = *c;
}

// ============================ a0: Green's function ================================
// g on the rearranged doubled mesh (Fig. 4): index a -> offset a (a <= N) or a - 2N.
static __global__ void k_green_sample(double2 *__restrict__ Gm, int N, double I0)
{
    const int n = 2 * N;
    const size_t tot = (size_t)n * n * n;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += (size_t)gridDim.x * blockDim.x) {
        const int a = (int)(q % n), bb = (int)((q / n) % n), c = (int)(q / ((size_t)n * n));
        const double ox = a <= N ? a : a - n, oy = bb <= N ? bb : bb - n, oz = c <= N ? c : c - n;
        const double d2 = ox * ox + oy * oy + oz * oz;
        Gm[q] = make_double2(d2 == 0.0 ? I0 : 1.0 / sqrt(d2), 0.0);
    }
}

// Plain in-place radix-2 transform of one pencil per CTA (one-time set-up, not the hot
// path): n = 2N points, n/2 threads, natural order in and out.
static __global__ void k_fft_simple(double2 *__restrict__ data, int n, int log2n, int axis, const double2 *__restrict__ tw)
{
    extern __shared__ double2 sm[];
    const size_t u = blockIdx.x / n, v = blockIdx.x % n;
    size_t base, stride;
    if (axis == 0) { base = (u * n + v) * n; stride = 1; }
    else if (axis == 1) { base = u * n * n + v; stride = n; }
    else { base = u * n + v; stride = (size_t)n * n; }
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int rev = (int)(__brev((unsigned)i) >> (32 - log2n));
        sm[rev] = data[base + (size_t)i * stride];
    }
    __syncthreads();
    for (int len = 2; len <= n; len <<= 1) {
        const int half = len >> 1, step = n / len;
        for (int t = threadIdx.x; t < n / 2; t += blockDim.x) {
            const int grp = t / half, k = t % half;
            const int i0 = grp * len + k, i1 = i0 + half;
            const double2 w = tw[k * step];
            const double2 x0 = sm[i0], x1 = cmul(sm[i1], w);
            sm[i0] = cadd(x0, x1);
            sm[i1] = cmfft::csub(x0, x1);
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) data[base + (size_t)i * stride] = sm[i];
}

// Row stride (in doubles) of one pencil of K-hat: 2N slots + a pad that makes P3's shared-memory reads
// conflict-free (a half-warp = T lanes j x 16/T pencils must hit 16 distinct 8-byte bank pairs: RSK = T mod 16).
__host__ __device__ constexpr int khat_row_stride(int N) { return 2 * N + (N / 16 < 16 ? N / 16 : 0); }

// K-hat, pencil-major: Kt[(sy 2N + sx) RSK + sz] = Re Ghat[f(sz)][f(sy)][f(sx)] / (2N)^3, f = slot_to_freq.  The PEN
// pencils of one P3 tile are one contiguous block, fetched by a single bulk copy and read as it lies.
static __global__ void k_green_permute(const double2 *__restrict__ Gm, double *__restrict__ Kt, int N)
{
    const int n = 2 * N, RSK = khat_row_stride(N);
    const size_t tot = (size_t)n * n * n;
    const double inv = 1.0 / ((double)n * (double)n * (double)n);
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += (size_t)gridDim.x * blockDim.x) {
        const int sz = (int)(q % n), sx = (int)((q / n) % n), sy = (int)(q / ((size_t)n * n));
        const size_t fx = cmfft::slot_to_freq(sx, N), fy = cmfft::slot_to_freq(sy, N), fz = cmfft::slot_to_freq(sz, N);
        Kt[((size_t)sy * n + sx) * RSK + sz] = Gm[(fz * n + fy) * n + fx].x * inv;
    }
}
// test access: the same values as [sz][sy][sx]
static __global__ void k_khat_export(const double *__restrict__ Kt, double *__restrict__ out, int N)
{
    const int n = 2 * N, RSK = khat_row_stride(N);
    const size_t tot = (size_t)n * n * n;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += (size_t)gridDim.x * blockDim.x) {
        const int sx = (int)(q % n), sy = (int)((q / n) % n), sz = (int)(q / ((size_t)n * n));
        out[q] = Kt[((size_t)sy * n + sx) * RSK + sz];
    }
}

// ===================== f-1: gravitational acceleration on the nested mesh ==================
// g = -grad Phi by the six-point stencil (Eq. 8); a neighbour the level cannot
// supply comes from the parent level through Eq. 3-6 (method A, Eq. A.1), a neighbour
// that lies under the finer grid is the mean of its 8 children (method B, Eq. A.2),
// and the outer boundary of level 0 uses the second-order one-sided difference.

// pbar[l][ck][cj][ci] = mean of the 8 children (level l+1) of cavity cell (N/4 + c*) of level l.
static __global__ void k_child_mean(int N, int L, const double *__restrict__ phi, double *__restrict__ pbar)
{
    const int H = N / 2;
    const size_t h3 = (size_t)H * H * H, n3 = (size_t)N * N * N;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)(L - 1) * h3) return;
    const int l = (int)(idx / h3);
    const size_t r = idx - (size_t)l * h3;
    const int ci = (int)(r % H), cj = (int)((r / H) % H), ck = (int)(r / ((size_t)H * H));
    const double *f = phi + (size_t)(l + 1) * n3;
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const double2 v = *reinterpret_cast<const double2 *>(f + ((size_t)(2 * ck + c) * N + (2 * cj + b)) * N + 2 * ci);
            s += v.x;
            s += v.y;
        }
    pbar[idx] = s / 8.0;
}

// value of level l at (k, j, i), any ONE of which may be -1 or N
struct AccelField {
    const double *phi_l, *phi_c, *pbar_l;   // this level, its parent (nullptr on level 0), children means (nullptr on the finest)
    int N;
    __device__ __forceinline__ double core(int k, int j, int i) const
    {
        const int Q = N / 4, H = N / 2;
        if (pbar_l && in_cavity1(k, N) && in_cavity1(j, N) && in_cavity1(i, N))
            return pbar_l[((size_t)(k - Q) * H + (j - Q)) * H + (i - Q)];
        return phi_l[((size_t)k * N + j) * N + i];
    }
    // ghost beyond the face: along axis `ax` the index f is -1 or N
    __device__ __forceinline__ double ghost(int k, int j, int i, int ax) const
    {
        if (!phi_c) {   // level 0: 3 Phi[0] - 3 Phi[1] + Phi[2] makes the central formula the one-sided one
            const int f = ax == 0 ? i : (ax == 1 ? j : k);
            const int d = f < 0 ? 1 : -1, e0 = f + d;
            const int di = ax == 0 ? d : 0, dj = ax == 1 ? d : 0, dk = ax == 2 ? d : 0;
            const int i0 = ax == 0 ? e0 : i, j0 = ax == 1 ? e0 : j, k0 = ax == 2 ? e0 : k;
            return (3.0 * core(k0, j0, i0) - 3.0 * core(k0 + dk, j0 + dj, i0 + di)) + core(k0 + 2 * dk, j0 + 2 * dj, i0 + 2 * di);
        }
        const int Q = N / 4;
        // floor(f/2) and parity for f = -1: parent Q-1, odd
        const int pk = Q + ((k + 2) >> 1) - 1, pj = Q + ((j + 2) >> 1) - 1, pi = Q + ((i + 2) >> 1) - 1;
        const int sk = (k & 1) ? 1 : -1, sj = (j & 1) ? 1 : -1, si = (i & 1) ? 1 : -1;
        return 0.75 * phi_c[((size_t)pk * N + pj) * N + pi] + 0.25 * phi_c[((size_t)(pk + sk) * N + (pj + sj)) * N + (pi + si)];
    }
    __device__ __forceinline__ double at(int k, int j, int i, int ax) const
    {
        const int f = ax == 0 ? i : (ax == 1 ? j : k);
        return (f < 0 || f >= N) ? ghost(k, j, i, ax) : core(k, j, i);
    }
};

// Two x-adjacent cells per thread, marching ZCH planes in z with the z-neighbours kept in
// registers; a CTA is a (TY rows) x (TX pairs) tile so that the y- and x-neighbours are L1 hits.
// g layout [L][3][N][N][N] (component x, y, z).  A step whose stencil touches neither a face of
// the grid nor the cavity takes the fast path; the others go through AccelField.  HBM-bound:
// 8 B read + 24 B written per cell.

// the general (face / cavity) case of one pair of cells, kept out of line so that the streaming
// loop of k_accel stays small in registers
// the one ghost value beyond an x face, out of line as well
static __device__ __noinline__ double accel_ghost_x(const AccelField F, int k, int j, int i) { return F.ghost(k, j, i, 0); }

static __device__ __noinline__ void accel_pair_general(const AccelField F, int k, int j, int i, double inv, double2 &gx,
                                                double2 &gy, double2 &gz)
{
    const double c0 = F.at(k, j, i, 0), c1 = F.at(k, j, i + 1, 0);
    gx = make_double2(-(c1 - F.at(k, j, i - 1, 0)) * inv, -(F.at(k, j, i + 2, 0) - c0) * inv);
    gy = make_double2(-(F.at(k, j + 1, i, 1) - F.at(k, j - 1, i, 1)) * inv,
                      -(F.at(k, j + 1, i + 1, 1) - F.at(k, j - 1, i + 1, 1)) * inv);
    gz = make_double2(-(F.at(k + 1, j, i, 2) - F.at(k - 1, j, i, 2)) * inv,
                      -(F.at(k + 1, j, i + 1, 2) - F.at(k - 1, j, i + 1, 2)) * inv);
}

static __global__ void __launch_bounds__(256, 4) k_accel(int N, int L, int TX, int TY, int ZCH, double dx0, const double *__restrict__ phi,
                                               const double *__restrict__ pbar, double *__restrict__ g)
{
    const size_t n3 = (size_t)N * N * N, h3 = n3 / 8, nn = (size_t)N * N;
    const int Q = N / 4;
    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    const int ntx = (N / 2) / TX, nty = N / TY, nz = N / ZCH;
    int bid = blockIdx.x;
    const int bx = bid % ntx; bid /= ntx;
    const int by = bid % nty; bid /= nty;
    const int bz = bid % nz;
    const int l = bid / nz;
    const int i = 2 * (bx * TX + tx), j = by * TY + ty, k0 = bz * ZCH;
    const double inv = 1.0 / (2.0 * (dx0 * exp2(-(double)l)));
    const double *pl = phi + (size_t)l * n3;
    const bool has_cav = l < L - 1;
    const AccelField F{pl, l > 0 ? phi + (size_t)(l - 1) * n3 : nullptr, has_cav ? pbar + (size_t)l * h3 : nullptr, N};
    // fast path: every y/z neighbour inside the grid and nothing under the finer grid; at the two x ends of a row only
    // the one missing x neighbour is a ghost (a row is 1-4 warps: sending those warps down the general path for one
    // lane each cost half of the kernel's time)
    const bool inner_ji = j >= 1 && j <= N - 2;
    const bool cav_ji = has_cav && j >= Q - 1 && j <= 3 * Q && i >= Q - 2 && i <= 3 * Q;
    const size_t rji = (size_t)j * N + i;
    double2 zm = make_double2(0.0, 0.0), c = *reinterpret_cast<const double2 *>(pl + (size_t)k0 * nn + rji);
    if (k0 > 0) zm = *reinterpret_cast<const double2 *>(pl + (size_t)(k0 - 1) * nn + rji);
#pragma unroll 2
    for (int kk = 0; kk < ZCH; ++kk) {
        const int k = k0 + kk;
        const size_t r = (size_t)k * nn + rji;
        double2 zp = make_double2(0.0, 0.0);
        if (k + 1 < N) zp = *reinterpret_cast<const double2 *>(pl + r + nn);
        double2 gx, gy, gz;
        if (inner_ji && k >= 1 && k <= N - 2 && !(cav_ji && k >= Q - 1 && k <= 3 * Q)) {
            const double xm = i > 0 ? pl[r - 1] : accel_ghost_x(F, k, j, -1), xp = i + 2 < N ? pl[r + 2] : accel_ghost_x(F, k, j, N);
            const double2 ym = *reinterpret_cast<const double2 *>(pl + r - N), yp = *reinterpret_cast<const double2 *>(pl + r + N);
            gx = make_double2(-(c.y - xm) * inv, -(xp - c.x) * inv);
            gy = make_double2(-(yp.x - ym.x) * inv, -(yp.y - ym.y) * inv);
            gz = make_double2(-(zp.x - zm.x) * inv, -(zp.y - zm.y) * inv);
        } else {
            accel_pair_general(F, k, j, i, inv, gx, gy, gz);
        }
        double *gl = g + (size_t)l * 3 * n3 + r;
        __stcs(reinterpret_cast<double2 *>(gl), gx);
        __stcs(reinterpret_cast<double2 *>(gl + n3), gy);
        __stcs(reinterpret_cast<double2 *>(gl + 2 * n3), gz);
        zm = c;
        c = zp;
    }
}

// ========================= f-2: modified method, Eq. 15 / B.1-B.6 — sources and sums ==========================
// rho-bar of level l1 as a compact N^3 array: the level's density with the finer levels projected onto it (rc);
// `hole`: its own cavity zeroed (the doubled grid "with a central hole" of the triplet scheme, so that grid l1+1's
// mass is not counted twice).  The expanded grid around it is never materialised (cm_expand.cuh).
static __global__ void k_level_density(int N, int hole, int l1, int L, const double *__restrict__ rho, const double *__restrict__ rc,
                                double *__restrict__ out)
{
    const int H = N / 2, Q = N / 4;
    const size_t n3 = (size_t)N * N * N;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n3) return;
    const int i = (int)(idx % N), j = (int)((idx / N) % N), k = (int)(idx / ((size_t)N * N));
    const bool cav = in_cavity1(k, N) && in_cavity1(j, N) && in_cavity1(i, N);
    double v = 0.0;
    if (!(cav && hole))
        v = (cav && l1 < L - 1) ? rc[(size_t)l1 * (n3 / 8) + ((size_t)(k - Q) * H + (j - Q)) * H + (i - Q)] : rho[(size_t)l1 * n3 + idx];
    out[idx] = v;
}

// phi_n = base + scale * add   (the "reduce" of B.1 / B.3: `add` holds the block sums the decimated passes formed)
static __global__ void k_add_scaled(size_t n, const double *base, const double *__restrict__ add, double scale, double *phi_n)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < n) phi_n[idx] = base[idx] + scale * add[idx];
}

// ================= f-3: direct fine -> coarse summation, Eq. B.7 =================
// Phi_ds(t) = -G sum_s M_s / |r_t - r_s| over all N^3 cells s of the source (finer) grid, for every cell t of
// the coarser target grid; M_s = rho_s dx_s^3, distances between cell centres (never zero: a coarse centre is a
// corner of fine cells).  One thread per target, the sources stream through shared memory as (x, y, z, M)
// in tiles of 256.  fp64 ALU-bound: N^6 inverse square roots; the paper uses it for N <= 32 only.
// gridDim.y source chunks (so that small grids still fill the GPU): chunk c sums sources [c, c+1) * n3 / gridDim.y
// into part[c][t]; k_direct_reduce adds the chunks in a fixed order (deterministic).
static __global__ void __launch_bounds__(256) k_direct_sum(int N, double dxs, double dxd, const double *__restrict__ rho_src,
                                                    double *__restrict__ part)
{
    __shared__ double4 src[256];
    const size_t n3 = (size_t)N * N * N;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int ti = (int)(t % N), tj = (int)((t / N) % N), tk = (int)((t / ((size_t)N * N)) % N);
    const double half = 0.5 - 0.5 * N;
    const double tx = (ti + half) * dxd, ty = (tj + half) * dxd, tz = (tk + half) * dxd;
    const double m3 = dxs * dxs * dxs;
    double acc = 0.0;
    const size_t s_lo = n3 * blockIdx.y / gridDim.y, s_hi = n3 * (blockIdx.y + 1) / gridDim.y;
    for (size_t base = s_lo; base < s_hi; base += 256) {
        const size_t s = base + threadIdx.x;
        if (s < s_hi) {
            const int si = (int)(s % N), sj = (int)((s / N) % N), sk = (int)(s / ((size_t)N * N));
            src[threadIdx.x] = make_double4((si + half) * dxs, (sj + half) * dxs, (sk + half) * dxs, rho_src[s] * m3);
        } else {
            src[threadIdx.x] = make_double4(0.0, 0.0, 0.0, 0.0);   // zero mass at the origin: distance > 0 for every target
        }
        __syncthreads();
#pragma unroll 8
        for (int q = 0; q < 256; ++q) {
            const double4 v = src[q];
            const double ex = tx - v.x, ey = ty - v.y, ez = tz - v.z;
            acc += v.w / sqrt(ex * ex + ey * ey + ez * ez);
        }
        __syncthreads();
    }
    if (t < n3) part[(size_t)blockIdx.y * n3 + t] = acc;
}
static __global__ void k_direct_reduce(size_t n3, int chunks, double G, const double *__restrict__ part, double *__restrict__ phi_dst)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n3) return;
    double acc = 0.0;
    for (int c = 0; c < chunks; ++c) acc += part[(size_t)c * n3 + t];
    phi_dst[t] = -G * acc;
}

}  // namespace cmk
