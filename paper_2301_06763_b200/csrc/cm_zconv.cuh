// cm_zconv.cuh — P3 (step a5): z forward * K-hat * z inverse, TMA-fed persistent kernel.
//
// PAPER.md:L118-L123 (Eq. 11): the convolution is a product in Fourier space.  The z axis
// is the last one transformed, so the forward z transform, the multiplication by the real
// K-hat and the inverse z transform of one pencil happen in registers without the
// (2N)^3 spectrum ever reaching memory.
//
// Why this shape (round 1's first capture): the first k_z_conv was neither
// DRAM- nor fp64-bound; its 8 warps/SM stalled on the tile load, on K-hat loads issued in
// the middle of the dependency chain and on CTA-wide barriers.  Here
//   (the launch covers levels b0 .. b0 + L - 1: all of them in cm_potential, one in cm_potential_host's pipeline)
//   * a CTA is persistent and walks tiles (g, b): g = a group of PEN adjacent (sy,sx)
//     pencils, b = level.  All L levels of a group run back to back so the group's
//     K-hat tile is fetched ONCE (one bulk copy of its pencil-major block) and stays in shared memory;
//   * the next tile's W2 data ([N z-rows][128 B], stride (2N)^2) is fetched by TMA
//     (128B-swizzled box) while the current tile is being transformed; the tile is copied
//     to registers as soon as it lands, which frees the stage for the following load;
//   * the T threads that share a pencil sit in ONE warp (j fastest), so the radix-16 x
//     radix-T exchange needs __syncwarp only; twiddles come from a shared-memory copy.
// Output is staged in shared memory (the idle exchange buffer) and written by a TMA store:
// writing it straight from registers (32-byte sectors per row per warp with this thread
// mapping) cost 6 ms of the 10.6 ms at N = 256 (ablation).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "cm_kernels.cuh"

namespace cmk {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1)
        : "memory");
}

__device__ __forceinline__ void tma_store_2d(const CUtensorMap *map, int c0, int c1, uint32_t src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(map), "r"(src), "r"(c0),
                 "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

template <int T> struct ZConvCfg {
    static_assert(T <= 16, "the TMA-fed kernels cover N <= 256 (k_z_conv_dec<32, 1> above that)");
    static constexpr int N = 16 * T, NN = 2 * N;
    static constexpr int PEN = kThreads / T;          // pencils per tile
    static constexpr int NBOX = PEN / 8;              // 128-byte column groups per tile
    static constexpr int PPW = 32 / T;                // pencils per warp
    static constexpr int RSK = khat_row_stride(N);    // doubles per pencil of the K-hat tile
    static constexpr uint32_t IN_BYTES = 32768, KH_BYTES = PEN * RSK * 8;   // <= 33792, a multiple of 16
    // exchange buffer; at the end of a tile the same bytes stage the output tile for the TMA store
    static constexpr uint32_t EX_BYTES = (T > 1) ? PEN * LayRow<T>::PS * 16 : 32768;
    static_assert(EX_BYTES >= 32768, "the exchange buffer doubles as the 32 KB output stage");
    static constexpr uint32_t TW_BYTES = 32 * T * 16;
    static constexpr int CTAS = 2;                    // per SM (registers and shared memory both)
    static constexpr uint32_t OFF_IN = 0, OFF_KH = IN_BYTES, OFF_EX = OFF_KH + KH_BYTES, OFF_TW = OFF_EX + EX_BYTES,
                              OFF_BAR = OFF_TW + TW_BYTES;
    static constexpr uint32_t SMEM = OFF_BAR + 16 + 1024;   // + slack for the manual 1024-byte alignment
};

template <int T>
__global__ void __launch_bounds__(kThreads, ZConvCfg<T>::CTAS)
k_z_conv_tma(const __grid_constant__ CUtensorMap mapW, const double *__restrict__ Kt,
             double2 *__restrict__ W2, const double2 *__restrict__ tw, int L, int ngroups, int b0, int nd)
{
    // nd <= N: z-rows of data per level (general sizes): the boxes of mapW are nd rows high, the rows
    // nd .. N-1 of the input stage are zeroed once and never written again
    using C = ZConvCfg<T>;
    constexpr int N = C::N, PEN = C::PEN, NBOX = C::NBOX;
    using Lay = LayRow<T>;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t s0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *sbase = smem_raw + (s0 - smem_u32(smem_raw));
    const uint32_t bar_in = s0 + C::OFF_BAR, bar_k = bar_in + 8;
    double2 *ex_s = reinterpret_cast<double2 *>(sbase + C::OFF_EX);
    double2 *tw_s = reinterpret_cast<double2 *>(sbase + C::OFF_TW);

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31, j = lane % T, pxl = lane / T;
    const int pen = w * C::PPW + pxl, bx = pen >> 3, px = pen & 7;
    // Tiles (g, b) in g-major order.  Large grids: CTA c takes groups c, c + gridDim, ... (at any moment the
    // grid works on adjacent 128-byte columns: DRAM page locality).  N <= 64: there are only 1-2 groups per CTA,
    // so the flat tile list is cut into gridDim equal ranges instead (balance; the data is L2-resident anyway).
    constexpr bool FLAT = (T <= 4);
    int t0 = 0, ntiles;
    if (FLAT) {
        const long long total = (long long)ngroups * L;
        t0 = (int)(total * blockIdx.x / gridDim.x);
        ntiles = (int)(total * (blockIdx.x + 1) / gridDim.x) - t0;
        if (ntiles <= 0) return;
    } else {
        if ((int)blockIdx.x >= ngroups) return;
        const int my_groups = (ngroups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
        ntiles = my_groups * L;
    }
    auto tile_of = [&](int t, int &g, int &b) {
        if (FLAT) {
            g = (t0 + t) / L;
            b = (t0 + t) - g * L;
        } else {
            const int gi = t / L;
            b = t - gi * L;
            g = (int)blockIdx.x + gi * (int)gridDim.x;
        }
    };

    auto issue_in = [&](int g, int b) {
        // the stage was last touched through the generic proxy (LDS): order those accesses before
        // the async-proxy write.  Without this fence the refill raced with them (measured: wrong
        // results whenever two CTAs shared an SM).
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(bar_in, (uint32_t)(NBOX * nd * 128));
#pragma unroll
        for (int q = 0; q < NBOX; ++q)
            tma_load_2d(s0 + C::OFF_IN + q * (N * 128), &mapW, 2 * (g * PEN + 8 * q), (b0 + b) * nd, bar_in);
    };
    auto issue_k = [&](int g) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(bar_k, C::KH_BYTES);
        // the PEN pencils of group g are one contiguous block of K-hat (pencil-major layout): one 1-D bulk copy
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s0 + C::OFF_KH),
                     "l"(Kt + (size_t)g * PEN * C::RSK), "r"(C::KH_BYTES), "r"(bar_k)
                     : "memory");
    };

    if (tid == 0) {
        mbar_init(bar_in, 1);
        mbar_init(bar_k, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < 32 * T; i += kThreads) tw_s[i] = __ldg(&tw[(i % T) * (i / T)]);
    if (nd < N) {
        const int tail16 = (N - nd) * 8;       // 16-byte words of the rows nd .. N-1 of one box
        for (int i = tid; i < NBOX * tail16; i += kThreads)
            *reinterpret_cast<double2 *>(sbase + C::OFF_IN + (i / tail16) * (N * 128) + nd * 128 + (i % tail16) * 16) = make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (tid == 0) {
        int g0, b0;
        tile_of(0, g0, b0);
        issue_k(g0);
        issue_in(g0, b0);
    }

    const unsigned char *in_p = sbase + C::OFF_IN + bx * (N * 128);
    const double *kh_p = reinterpret_cast<const double *>(sbase + C::OFF_KH) + pen * C::RSK;
    double2 *ex_p = ex_s + pen * Lay::PS;
    const TwShared<T> tws{tw_s + j, tw_s[2 * T + j]};
    using SyncX = SyncWarp;
    uint32_t ph_in = 0, ph_k = 0;

    for (int t = 0; t < ntiles; ++t) {
        int g, b, gn = 0, bn = 0;
        tile_of(t, g, b);
        if (t + 1 < ntiles) tile_of(t + 1, gn, bn);

        mbar_wait(bar_in, ph_in);
        ph_in ^= 1;
        double2 a[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int z = j + T * r;
            a[r] = *reinterpret_cast<const double2 *>(in_p + z * 128 + ((px ^ (z & 7)) << 4));
        }
        if (tid == 0) tma_store_wait_read();   // the previous tile's output has left the exchange/out buffer
        __syncthreads();   // every thread holds its part of the tile: the stage may be refilled
        if (tid == 0 && t + 1 < ntiles) issue_in(gn, bn);

        double2 e[16];
        if (t == 0 || b == 0) {   // a new group: its K-hat tile was requested during the previous group's last tile
            mbar_wait(bar_k, ph_k);
            ph_k ^= 1;
        }
        {
            double2 v[16];
            fwd_half<T, 0, Lay, true>(a, v, j, ex_p, tws, SyncX());
            inv_half<T, 0, Lay, true, true>(v, e, j, ex_p, tws, SyncX(), kh_p);            // * K-hat, even slots
        }
        {
            double2 v[16];
            fwd_half<T, 1, Lay, true>(a, v, j, ex_p, tws, SyncX());
            inv_half<T, 1, Lay, true, true>(v, e, j, ex_p, tws, SyncX(), kh_p + N);        // * K-hat, odd slots; e += odd half
        }
        // stage the output tile in the (now idle) exchange buffer with the box layout of the
        // input stage, then one thread hands it to the TMA unit: full 128-byte rows to L2.
        __syncthreads();   // every warp is done with its exchanges
        if (tid == 0 && t + 1 < ntiles && gn != g) issue_k(gn);   // last use of this group's K-hat tile is over
        {
            unsigned char *out_p = sbase + C::OFF_EX + bx * (N * 128);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int z = j + T * r;
                *reinterpret_cast<double2 *>(out_p + z * 128 + ((px ^ (z & 7)) << 4)) = e[r];
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
#pragma unroll
            for (int q = 0; q < NBOX; ++q)
                tma_store_2d(&mapW, 2 * (g * PEN + 8 * q), (b0 + b) * nd, s0 + C::OFF_EX + q * (N * 128));
            tma_store_commit();
        }
    }
    if (tid == 0) tma_store_wait_all();
}



template <int T> struct ZWarpCfg {
    using C = ZConvCfg<T>;
    static constexpr int PPW = C::PPW;
    static constexpr uint32_t WIN = C::N * PPW * 16;                                   // a warp's input box
    static constexpr uint32_t EXW = ((PPW * LayRow<T>::PS * 16 + 1023) / 1024) * 1024;   // a warp's exchange region / output box
    static constexpr uint32_t OFF_IN = 0, OFF_KH = 4 * WIN, OFF_EX = ((OFF_KH + C::KH_BYTES + 1023) / 1024) * 1024,
                              OFF_TW = OFF_EX + 4 * EXW, OFF_BAR = OFF_TW + C::TW_BYTES;
    static constexpr uint32_t SMEM = OFF_BAR + 64 + 1024;
};

// ====================== P3, warp-autonomous variant (T = 8, 16) ==========================
// The same tile, but every warp owns its PPW pencils end to end: its own TMA box ([N rows][PPW*16 B], 32B/64B
// swizzle: conflict-free for the j-fastest reads), its own full/empty handshakes, its own output box staged in its
// own exchange region.  No CTA-wide barrier is left in the tile loop (r01d: 9 % of the stall samples sat at the
// three __syncthreads of a tile, 5 % at the TMA waits behind them), and the four warps drift apart, so that one
// warp's exchanges fall under another warp's butterflies.  Only the K-hat tile is shared: a warp reports when it
// is through with a group's tile (bar_kfree, 4 arrivals), warp 0 then fetches the next one.

template <int T>
__global__ void __launch_bounds__(kThreads, 2)
k_z_conv_warp(const __grid_constant__ CUtensorMap mapWw, const double *__restrict__ Kt, const double2 *__restrict__ tw, int L,
              int ngroups, int b0)
{
    using C = ZConvCfg<T>;
    using W = ZWarpCfg<T>;
    constexpr int N = C::N, PEN = C::PEN, PPW = C::PPW, ROWB = PPW * 16;     // bytes of one z row of a warp's box
    constexpr uint32_t WIN = W::WIN, EXW = W::EXW;
    using Lay = LayRow<T>;
    static_assert(T == 8 || T == 16, "one 32- or 64-byte box per warp");
    static_assert(PPW * Lay::PS * 16 >= (int)WIN, "a warp's exchange region doubles as its output stage");
    extern __shared__ unsigned char smem_raw[];
    const uint32_t s0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *sbase = smem_raw + (s0 - smem_u32(smem_raw));
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31, j = lane % T, pxl = lane / T;
    const uint32_t bar_in = s0 + W::OFF_BAR + 8 * w, bar_k = s0 + W::OFF_BAR + 32, bar_kfree = bar_k + 8;
    double2 *tw_s = reinterpret_cast<double2 *>(sbase + W::OFF_TW);
    const int pen = w * PPW + pxl;

    // the flat (group, level) tile list cut into equal ranges (balance: 4096 groups over 296 CTAs would leave 14 against
    // 13.8 groups per CTA; -0.5 % at 8 x 128^3)
    const long long total = (long long)ngroups * L;
    const int t0 = (int)(total * blockIdx.x / gridDim.x);
    const int ntiles = (int)(total * (blockIdx.x + 1) / gridDim.x) - t0;
    if (ntiles <= 0) return;
    auto tile_of = [&](int t, int &g, int &b) {
        g = (t0 + t) / L;
        b = (t0 + t) - g * L;
    };
    const uint32_t in_u = s0 + W::OFF_IN + w * WIN, ex_u = s0 + W::OFF_EX + w * EXW;
    unsigned char *in_p = sbase + W::OFF_IN + w * WIN, *out_p = sbase + W::OFF_EX + w * EXW;
    double2 *ex_p = reinterpret_cast<double2 *>(out_p) + pxl * Lay::PS;
    auto issue_in = [&](int g, int b) {       // lane 0 of the warp
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(bar_in, WIN);
        tma_load_2d(in_u, &mapWw, 2 * (g * PEN + w * PPW), (b0 + b) * N, bar_in);
    };
    auto issue_k = [&](int g) {               // thread 0
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(bar_k, C::KH_BYTES);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s0 + W::OFF_KH),
                     "l"(Kt + (size_t)g * PEN * C::RSK), "r"(C::KH_BYTES), "r"(bar_k)
                     : "memory");
    };
    if (tid == 0) {
        for (int q = 0; q < 4; ++q) mbar_init(s0 + W::OFF_BAR + 8 * q, 1);
        mbar_init(bar_k, 1);
        mbar_init(bar_kfree, 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < 32 * T; i += kThreads) tw_s[i] = __ldg(&tw[(i % T) * (i / T)]);
    __syncthreads();
    {
        int g0, bb0;
        tile_of(0, g0, bb0);
        if (tid == 0) issue_k(g0);
        if (lane == 0) issue_in(g0, bb0);
    }
    const double *kh_p = reinterpret_cast<const double *>(sbase + W::OFF_KH) + pen * C::RSK;
    const TwShared<T, 8> tws{tw_s + j, tw_s[2 * T + j]};
    // swizzled position of (row z, pencil pxl) in a warp's box: 32B rows: chunk bit0 ^= bit 7 of the offset;
    // 64B rows: chunk bits [1:0] ^= bits [8:7]
    auto box_off = [&](int z) -> uint32_t {
        const uint32_t off = (uint32_t)z * ROWB + (uint32_t)pxl * 16;
        return ROWB == 32 ? (off ^ (((off >> 7) & 1u) << 4)) : (off ^ (((off >> 7) & 3u) << 4));
    };
    uint32_t ph_in = 0, ph_k = 0, ph_kfree = 0;

    for (int t = 0; t < ntiles; ++t) {
        int g, b, gn = 0, bn = 0;
        tile_of(t, g, b);
        if (t + 1 < ntiles) tile_of(t + 1, gn, bn);

        mbar_wait(bar_in, ph_in);
        ph_in ^= 1;
        double2 a[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) a[r] = *reinterpret_cast<const double2 *>(in_p + box_off(j + T * r));
        if (lane == 0) tma_store_wait_read();     // this warp's previous output has left its exchange region
        __syncwarp();
        if (lane == 0 && t + 1 < ntiles) issue_in(gn, bn);
        if (t == 0 || b == 0) {
            mbar_wait(bar_k, ph_k);
            ph_k ^= 1;
        }
        double2 e[16];
        {
            double2 v[16];
            fwd_half<T, 0, Lay, true>(a, v, j, ex_p, tws, SyncWarp());
            inv_half<T, 0, Lay, true, true>(v, e, j, ex_p, tws, SyncWarp(), kh_p);         // * K-hat, even slots
        }
        {
            double2 v[16];
            fwd_half<T, 1, Lay, true>(a, v, j, ex_p, tws, SyncWarp());
            // * K-hat (odd slots) rides on the first butterflies of the inverse; the second __syncwarp of inv_half
            // (after the exchange writes) is the point where this warp is through with the group's K-hat tile
            const bool release = t + 1 < ntiles && gn != g;
            int nsync = 0;
            auto sync_release = [&]() {
                __syncwarp();
                if (++nsync == 2 && release) {
                    if (lane == 0) mbar_arrive(bar_kfree);
                    if (tid == 0) {               // warp 0 fetches the next tile once all four warps are through
                        mbar_wait(bar_kfree, ph_kfree);
                        ph_kfree ^= 1;
                        issue_k(gn);
                    }
                }
            };
            inv_half<T, 1, Lay, true, true>(v, e, j, ex_p, tws, sync_release, kh_p + N);     // e += odd half
        }
        __syncwarp();                             // the warp's exchanges are over: its region becomes the output box
#pragma unroll
        for (int r = 0; r < 16; ++r) *reinterpret_cast<double2 *>(out_p + box_off(j + T * r)) = e[r];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
            tma_store_2d(&mapWw, 2 * (g * PEN + w * PPW), (b0 + b) * N, ex_u);
            tma_store_commit();
        }
    }
    if (lane == 0) tma_store_wait_all();
}

}  // namespace cmk
