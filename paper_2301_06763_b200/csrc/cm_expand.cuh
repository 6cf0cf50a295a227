// cm_expand.cuh — the expanded grids of the modified method (Eq. 15, Appendix B Eq. B.1-B.6)
// without their zeros and without the cells nobody asks for.
//
// The doubled (F = 2) or quadrupled (F = 4) grid of a fine level is (F N)^3 cells of the fine size of which only
// the central N^3 carry mass, and its potential is wanted only as the mean over the F^3 cells that make up a cell
// of the coarse grid ("reduced to the coarse grid", L288).  Run as an ordinary single-level problem of size
// N' = F N it moves (and transforms) F^3 times the data of a level.  Here instead, on the same plan of size N':
//
//   * forward passes are PRUNED to the block: P1 runs on the N^2 rows of the block only and reads the compact N^3
//     source; P2 runs on its N z-planes and reads N of the N' rows of a column; P3 reads N of the N' z-rows;
//   * inverse passes are DECIMATED.  With M = 2 N' the transform length and phi(t) = sum_k Z(k) e^{2 pi i k t / M},
//         sum_{q<F} phi(F a + q) = sum_k Z(k) E(k) e^{2 pi i k F a / M} = phi_E(F a),   E(k) = sum_{q<F} e^{2 pi i k q / M}:
//     the block sum is every F-th output of the inverse transform of the spectrum multiplied by E.  In the
//     radix-16 x radix-T inverse the outputs of thread j are n = j + T r, so the multiples of F are exactly the
//     outputs of the threads with j % F == 0: the others stop after the exchange (inv_half<..., DEC>), and each
//     pass writes 1/F of the rows: P3 -> N coarse z-planes, P4 -> N x N coarse (z, y) rows, P5 -> N^3 block sums.
//     E is Hermitian (E(-k) = conj E(k)) and K-hat real and even, so a second real field still rides as the
//     imaginary part (two expanded grids per complex solve).
//
// Bytes of one expanded solve, in units of N'^3 x 16 B: 29 as a plain single-level solve, about 8.5 (F = 4) here,
// of which 4 are the K-hat read of P3.
#pragma once

#include "cm_kernels.cuh"
#include "cm_zconv.cuh"

namespace cmk {

// Thread -> j in the decimated passes (batch-fastest mapping, u = (tid >> 3) % T): the T / DEC values of j that are
// multiples of DEC come first, so the threads that run the last stage of the inverse fill whole warps
// (8 T / DEC >= 32 threads when T / DEC >= 4) instead of a quarter of every warp.
template <int T, int DEC> __device__ __forceinline__ int dec_j(int u) { return (u % (T / DEC)) * DEC + u / (T / DEC); }

// v[i] *= E[slot of v[i]]  (E in slot order, one parity block)
template <int T> __device__ __forceinline__ void mul_E(double2 (&v)[16], const double2 *Ep, int j)
{
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], Ep[vslot<T>(i, j)]);
}

// P1 on the block: compact row rc = zc Nc + yc of the Nc^3 source sits at row (c0 + zc, c0 + yc) of the big grid, its
// cells at x = c0 + xc.  src_im (optional): the second real field.
template <int T>
__global__ void __launch_bounds__(kThreads) k_x_fwd_blk(const double *__restrict__ src_re, const double *__restrict__ src_im,
                                                        double2 *__restrict__ W1, const double2 *__restrict__ tw, int Nc, int c0)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T;
    using Lay = LayRow<T>;
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, j = tid % T, rowl = tid / T;
    size_t rc = (size_t)blockIdx.x * ROWS + rowl;
    const bool valid = rc < (size_t)Nc * Nc;       // the last CTA may be ragged: surplus threads redo the last row, storing nothing
    if (!valid) rc = (size_t)Nc * Nc - 1;
    const int zc = (int)(rc / Nc), yc = (int)(rc % Nc);
    const int nbig = 2 * c0 + Nc;                  // rows per plane of the expanded grid as W1 holds it
    double2 *dst = W1 + ((size_t)(c0 + zc) * nbig + (c0 + yc)) * NN;
    double2 a[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int xc = j + T * r - c0;
        const bool in = xc >= 0 && xc < Nc;
        a[r] = make_double2(in ? __ldg(src_re + rc * Nc + xc) : 0.0, (in && src_im) ? __ldg(src_im + rc * Nc + xc) : 0.0);
    }
    double2 *bufA = smem + rowl * Lay::PS, *bufB = bufA + ROWS * Lay::PS;
    {
        double2 v[16];
        fwd_half<T, 0, Lay>(a, v, j, bufA, TwGlobal{tw, j}, SyncWarp());
        if (valid) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dst[vslot<T>(i, j)] = v[i];
        }
    }
    {
        double2 v[16];
        fwd_half<T, 1, Lay>(a, v, j, bufB, TwGlobal{tw, j}, SyncWarp());
        if (valid) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dst[N + vslot<T>(i, j)] = v[i];
        }
    }
}

// P2 on the block's z-planes: plane zc -> z = c0 + zc; rows outside [c0, c0 + Nc) are zero and not read.
template <int T>
__global__ void __launch_bounds__(batch_threads<T>()) k_y_fwd_blk(const double2 *__restrict__ W1, double2 *__restrict__ W2,
                                                                  const double2 *__restrict__ tw, int Nc, int c0, int ahead = 0)
{
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, px = tid & 7, g = tid / (8 * T);
    const size_t q = (size_t)blockIdx.x * PEN + g * 8 + px;      // zc * 2N + sx
    const size_t z = c0 + q / NN;
    const int sx = (int)(q % NN);
    const size_t nbig = 2 * (size_t)c0 + Nc;       // rows per plane of the expanded grid as W1 holds it
    if (ahead > 0 && px == 0 && blockIdx.x + ahead < gridDim.x) {     // the next resident CTA's columns into L2 (see k_y_fwd)
        const size_t q2 = (size_t)(blockIdx.x + ahead) * PEN + g * 8;
        const double2 *s2 = W1 + (c0 + q2 / NN) * nbig * NN + (q2 % NN);
        const int j = (tid >> 3) % T;
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int y = j + T * r;
            if (y >= c0 && y < c0 + Nc) asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)y * NN));
        }
    }
    y_fwd_body<T>(W1 + z * nbig * NN + sx, W2 + z * NN * NN + sx, tw, smem, c0, c0 + Nc);
}

// P3 on an expanded grid, batch-fastest mapping (lane = 8 adjacent pencils x 4 values of j; loads and stores straight
// from/to registers in whole 128-byte lines): the z-rows outside [zlo, zhi) are zero and not read; the spectrum is
// multiplied by K-hat and E; the inverse is decimated (the threads with j % DEC == 0 write the N / DEC coarse rows
// a = (j + T r) / DEC).  K-hat is the largest stream of this pass (8 B x (2N')^3 against 2 x 16 B x (N / DEC) x (2N')^2 of
// W2), so a CTA fetches the K-hat tile of its 8 (or 16) pencils once, by bulk copies into shared memory that fly
// under the loads and the first forward half, and uses it twice: for the pencils at (fy, sx) and for those at the
// mirror frequency (-fy, sx), where K-hat is the same (it is even in every frequency).
template <int T> struct ZDecCfg {
    static constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    static constexpr int RSK = khat_row_stride(N);   // doubles per pencil of K-hat in global memory
    // K-hat is even in the z frequency; in slot order the mirror of slot m of the even block is slot N - m and of the odd
    // block N - 1 - m, so the first N/2 + 1 (even) and N/2 (odd) slots of a pencil are all of it.  Row stride N + 2: the
    // 8 pencils x 2 j of a half-warp hit 16 distinct 8-byte words.
    static constexpr int KE = N / 2 + 2, RSKH = N + 2;
    static constexpr uint32_t EX_BYTES = 2 * PEN * LayBatch<T>::PS * 16, KH_BYTES = PEN * RSKH * 8, TW_BYTES = 32 * T * 16,
                              E_BYTES = NN * 16;
    static constexpr uint32_t OFF_KH = EX_BYTES, OFF_TW = OFF_KH + KH_BYTES, OFF_E = OFF_TW + TW_BYTES, OFF_BAR = OFF_E + E_BYTES,
                              SMEM = OFF_BAR + 16;
};

template <int N> struct KhHalf {     // K-hat of slot m of a parity block from the stored half
    const double *blk;               // the block's stored slots
    int odd;
    __device__ __forceinline__ double operator()(int m) const { return blk[m <= (N - odd) / 2 ? m : N - odd - m]; }
};

// every twiddle w_2N^{j (2 k1 + P)} from a shared-memory copy of the table laid out [2 k1 + P][j]
template <int T> struct TwAllShared {
    const double2 *base;   // table + j
    static constexpr bool RECUR = false;
    template <int P> __device__ __forceinline__ double2 get(int k1) const { return base[(2 * k1 + P) * T]; }
};

__host__ __device__ __forceinline__ constexpr int freq_to_slot(int k, int N)   // inverse of cmfft::slot_to_freq
{
    return (k & 1) * N + 16 * (k >> 5) + ((k >> 1) & 15);
}

// DEC = 1 is the plain P3 of N = 512 plans (cm_lib.cu: no decimation, no E, every row read): levels b0 .. b0 + L - 1 of W2
// (nd planes each) share the CTA's K-hat tile like the two mirror tiles do.
template <int T, int DEC>
__global__ void __launch_bounds__(batch_threads<T>(), 1)
k_z_conv_dec(const double *__restrict__ Kt, double2 *__restrict__ W2, const double2 *__restrict__ tw,
             const double2 *__restrict__ E, int zlo, int zhi, int b0, int L, int nd, int ahead = 0)
{
    using C = ZDecCfg<T>;
    constexpr int N = C::N, NN = C::NN, PEN = C::PEN, GX = NN / PEN;   // GX pencil groups per sy row
    constexpr size_t ZS = (size_t)NN * NN;
    using Lay = LayBatch<T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *smem = reinterpret_cast<double2 *>(smem_raw);
    double2 *tw_s = reinterpret_cast<double2 *>(smem_raw + C::OFF_TW), *E_s = reinterpret_cast<double2 *>(smem_raw + C::OFF_E);
    const uint32_t s0 = smem_u32(smem_raw), bar_k = s0 + C::OFF_BAR;
    const int tid = threadIdx.x, px = tid & 7, j = dec_j<T, DEC>((tid >> 3) % T), g = tid / (8 * T), pen = g * 8 + px;
    // CTA -> (fy, group of PEN adjacent sx): fy = 0 .. N (the non-negative y frequencies); the tile at -fy follows
    const int fy = blockIdx.x / GX, gx = blockIdx.x % GX;
    const int sy_a = freq_to_slot(fy, N), sy_b = freq_to_slot((NN - fy) % NN, N);
    const int ntile = (sy_a == sy_b) ? 1 : 2;
    if (tid == 0) {
        mbar_init(bar_k, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(bar_k, PEN * (C::KE + N / 2) * 8);
        const double *ksrc = Kt + ((size_t)sy_a * NN + (size_t)gx * PEN) * C::RSK;
#pragma unroll 1
        for (int q = 0; q < PEN; ++q) {
            const uint32_t dst = s0 + C::OFF_KH + q * (C::RSKH * 8);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                         "l"(ksrc + (size_t)q * C::RSK), "r"(C::KE * 8), "r"(bar_k)
                         : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst + C::KE * 8),
                         "l"(ksrc + (size_t)q * C::RSK + N), "r"((N / 2) * 8), "r"(bar_k)
                         : "memory");
        }
    }
    // One CTA (T = 32) or two per SM and loads straight into registers: nothing hides a tile's load latency (ncu, <32, 4>: fp64
    // pipe 34 % busy, 20 % of the stall samples on the load scoreboard).  Pull into L2 what comes next: the rows of this CTA's
    // mirror tile, and the first tile and the K-hat tile of the CTA `ahead` places later (the next one on this SM).
    if (ahead > 0) {
        auto pull_rows = [&](const double2 *c0) {      // one lane per 128-byte line of the rows this thread will load
            if (px == 0) {
#pragma unroll
                for (int r = 0; r < 16; ++r) {
                    const int z = j + T * r;
                    if (z >= zlo && z < zhi) asm volatile("prefetch.global.L2 [%0];" ::"l"(c0 + (size_t)z * ZS));
                }
            }
        };
        const double2 *lvl = W2 + (size_t)b0 * nd * ZS;
        if (ntile == 2) pull_rows(lvl + ((size_t)sy_b * NN + (size_t)gx * PEN + g * 8));
        const unsigned nb = blockIdx.x + ahead;
        if (nb < gridDim.x) {
            const int sy2 = freq_to_slot((int)(nb / GX), N), gx2 = (int)(nb % GX);
            pull_rows(lvl + ((size_t)sy2 * NN + (size_t)gx2 * PEN + g * 8));
            const char *k2 = reinterpret_cast<const char *>(Kt + ((size_t)sy2 * NN + (size_t)gx2 * PEN) * C::RSK);
            constexpr int LA = (C::KE * 8 + 127) / 128, LB = (N / 2 * 8 + 127) / 128;      // lines of the two stored halves
            for (int i = tid; i < PEN * (LA + LB); i += batch_threads<T>()) {
                const int q = i / (LA + LB), l = i % (LA + LB);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(k2 + (size_t)q * C::RSK * 8 + (l < LA ? l * 128 : N * 8 + (l - LA) * 128)));
            }
        }
    }
    // twiddles and E feed multiplies directly: from global memory their latency was 26 % of the warp time (ncu, T = 32)
    for (int i = tid; i < 32 * T; i += batch_threads<T>()) tw_s[i] = __ldg(&tw[(i % T) * (i / T)]);
    if (DEC > 1)
        for (int i = tid; i < NN; i += batch_threads<T>()) E_s[i] = __ldg(&E[i]);
    __syncthreads();     // tables in place; the barrier is initialised before anyone waits on it
    const double *kh_s = reinterpret_cast<const double *>(smem_raw + C::OFF_KH) + pen * C::RSKH;
    const KhHalf<N> kh0{kh_s, 0}, kh1{kh_s + C::KE, 1};
    double2 *bufA = smem + pen * Lay::PS, *bufB = bufA + PEN * Lay::PS;
    const TwAllShared<T> twg{tw_s + j};

    for (int t = 0; t < ntile * L; ++t) {
        double2 *col = W2 + (size_t)(b0 + t / ntile) * nd * ZS + ((size_t)((t % ntile) ? sy_b : sy_a) * NN + (size_t)gx * PEN + pen);
        double2 a[16], e[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int z = j + T * r;
            a[r] = (z >= zlo && z < zhi) ? col[(size_t)z * ZS] : make_double2(0.0, 0.0);
        }
        {
            double2 v[16];
            fwd_half<T, 0, Lay>(a, v, j, bufA, twg, SyncBlock());
            if (DEC > 1) mul_E<T>(v, E_s, j);
            if (t == 0) mbar_wait(bar_k, 0);
            inv_half<T, 0, Lay, false, true, DEC>(v, e, j, bufB, twg, SyncBlock(), kh0);
        }
        {
            double2 v[16];
            fwd_half<T, 1, Lay>(a, v, j, bufA, twg, SyncBlock());
            if (DEC > 1) mul_E<T>(v, E_s + N, j);
            inv_half<T, 1, Lay, false, true, DEC>(v, e, j, bufB, twg, SyncBlock(), kh1);
        }
        if ((j % DEC) == 0) {
#pragma unroll
            for (int r = 0; r < 16; ++r)
                if ((j + T * r) / DEC < zhi - zlo) col[(size_t)((j + T * r) / DEC) * ZS] = e[r];    // the Nc coarse planes
        }
    }
}

// P4, decimated: plane bz = coarse z; the N / DEC coarse rows a = (j + T r) / DEC of W1 (plane stride as in the plain pass).
template <int T, int DEC>
__global__ void __launch_bounds__(batch_threads<T>()) k_y_inv_dec(const double2 *__restrict__ W2, double2 *__restrict__ W1,
                                                                  const double2 *__restrict__ tw, const double2 *__restrict__ E, int Nc,
                                                                  int ahead = 0)
{
    constexpr int N = 16 * T, NN = 2 * N, PEN = batch_pencils<T>();
    using Lay = LayBatch<T>;
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, px = tid & 7, j = dec_j<T, DEC>((tid >> 3) % T), g = tid / (8 * T);
    const size_t q = (size_t)blockIdx.x * PEN + g * 8 + px;
    const size_t bz = q / NN;
    const int sx = (int)(q % NN);
    const double2 *src = W2 + bz * NN * NN + sx;
    if (ahead > 0 && px == 0 && blockIdx.x + ahead < gridDim.x) {     // the next resident CTA's columns into L2 (see k_y_fwd)
        const size_t q2 = (size_t)(blockIdx.x + ahead) * PEN + g * 8;
        const double2 *s2 = W2 + (q2 / NN) * NN * NN + (q2 % NN);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)vslot<T>(i, j) * NN));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(s2 + (size_t)(N + vslot<T>(i, j)) * NN));
        }
    }
    double2 *dst = W1 + bz * N * NN + sx;
    double2 *bufA = smem + (g * 8 + px) * Lay::PS, *bufB = bufA + PEN * Lay::PS;
    double2 v0[16], v1[16], e[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        v0[i] = src[(size_t)vslot<T>(i, j) * NN];
        v1[i] = src[(size_t)(N + vslot<T>(i, j)) * NN];
    }
    mul_E<T>(v0, E, j);
    mul_E<T>(v1, E + N, j);
    inv_half<T, 0, Lay, false, false, DEC>(v0, e, j, bufA, TwGlobal{tw, j}, SyncBlock());
    inv_half<T, 1, Lay, false, false, DEC>(v1, e, j, bufB, TwGlobal{tw, j}, SyncBlock());
    if ((j % DEC) == 0) {
#pragma unroll
        for (int r = 0; r < 16; ++r)
            if ((j + T * r) / DEC < Nc) dst[(size_t)((j + T * r) / DEC) * NN] = e[r];
    }
}

// P5, decimated: compact row rc = az Nc + ay (Nc coarse cells per axis) of W1 -> the Nc block sums along x, times `scale`;
// real part to out_re, imaginary part (the second field) to out_im if given.  Compact Nc^3 outputs.
template <int T, int DEC>
__global__ void __launch_bounds__(kThreads) k_x_inv_dec(const double2 *__restrict__ W1, double *__restrict__ out_re,
                                                        double *__restrict__ out_im, const double2 *__restrict__ tw,
                                                        const double2 *__restrict__ E, double scale, int Nc)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T;
    using Lay = LayRow<T>;
    extern __shared__ double2 smem[];
    const int tid = threadIdx.x, j = tid % T, rowl = tid / T;
    size_t rc = (size_t)blockIdx.x * ROWS + rowl;
    const bool valid = rc < (size_t)Nc * Nc;
    if (!valid) rc = (size_t)Nc * Nc - 1;
    const size_t az = rc / Nc, ay = rc % Nc;
    const double2 *src = W1 + (az * N + ay) * NN;
    double2 *bufA = smem + rowl * Lay::PS, *bufB = bufA + ROWS * Lay::PS;
    double2 v0[16], v1[16], e[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        v0[i] = src[vslot<T>(i, j)];
        v1[i] = src[N + vslot<T>(i, j)];
    }
    mul_E<T>(v0, E, j);
    mul_E<T>(v1, E + N, j);
    inv_half<T, 0, Lay, false, false, DEC>(v0, e, j, bufA, TwGlobal{tw, j}, SyncWarp());
    inv_half<T, 1, Lay, false, false, DEC>(v1, e, j, bufB, TwGlobal{tw, j}, SyncWarp());
    if (valid && (j % DEC) == 0) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            if ((j + T * r) / DEC >= Nc) continue;
            const size_t o = rc * Nc + (j + T * r) / DEC;
            out_re[o] = scale * e[r].x;
            if (out_im) out_im[o] = scale * e[r].y;
        }
    }
}

}  // namespace cmk
