// cm_fused.cuh — P1+P2 (and P4+P5) as ONE persistent kernel each, so that W1 never leaves L2.
//
// The x pass and the y pass meet in W1 (32 B per level-cell written, 32 B read back): as two
// launches over all levels W1 is 5.4 GB at N = 256 and makes a round trip through HBM.  Here a
// persistent grid pulls work items from a global ticket counter in PLANE order
//     ... A(p+LAG, 0..nA-1), B(p, 0..nB-1), A(p+LAG+1, ...), B(p+1, ...) ...
// (A = x transform of ROWS rows of plane p, B = y transform of PEN columns of plane p), W1 is a
// ring of R planes, and two counters per plane say when a plane has been produced (doneA) and
// when its ring slot may be overwritten (doneB).  The live part of W1 is a few planes (MBs): it
// is written, read once and overwritten while still in the 126 MB L2.
//
// Progress: tickets are handed out in an order in which everything an item waits for has a
// smaller ticket, and a CTA only ever waits while holding a ticket, so the holder of the smallest
// unfinished ticket never waits for ever.  A(p) waits for B(p-R) (ring reuse), whose tickets come
// first because R > LAG; B(p) waits for A(p).  Every wait is bounded (kSpinLimit): on a time-out
// the kernel sets ctl->error and the host reports CM_ECUDA instead of hanging the device.
//
// Memory model: a producer CTA finishes its stores, __syncthreads(), then thread 0 does
// __threadfence() + atomicAdd on the plane counter; a consumer's thread 0 spins on an acquire load
// of the counter, then __syncthreads().  W1 is read with ld.global.cg (L2) — a ring slot is
// re-used, so an L1 line could be stale.
#pragma once

#include "cm_kernels.cuh"

namespace cmk {

struct FusedCtl {
    unsigned ticket;
    unsigned error;
    unsigned pad[30];
    // followed by doneA[P], doneB[P] (unsigned each)
};

constexpr unsigned kSpinLimit = 1u << 22;   // x ~100 ns: seconds, far beyond any legitimate wait

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ---------------------------------------------------------------- the scheduler warp
// A CTA = kThreads compute threads (warps 0-3) + one scheduler warp (lane 0 works).  The scheduler
// runs one item ahead of the compute warps: it takes the ticket of the next item, waits for what the
// item depends on, and publishes it in a two-slot mailbox; it also publishes the completion of the
// items the compute warps finish.  So ticket, dependency and fence latencies sit beside the
// transforms, not between them.
//
// Mailbox protocol (shared memory, CTA scope): slot s = n & 1 for the CTA's n-th item.
//   full[s]  = n + 1 once item n is ready to run (written by the scheduler, read by compute thread 0,
//              which then releases the other compute threads through the compute barrier);
//   done[s]  = n + 1 once every compute thread has issued item n's stores (written by compute
//              thread 0 after the compute barrier).
// The scheduler must publish the completion of item n-1 WHILE it waits for item n's dependency
// (item n may depend on item n-1 of the same CTA), so its wait loop polls done[] as well.
struct FusedItem {
    int kind;   // 0 = A, 1 = B, -1 = no more work, -2 = abort
    int p, w;
};
struct FusedMailbox {
    FusedItem item[2];
    volatile unsigned full[2], done[2];
};

__device__ __forceinline__ void st_release_cta(volatile unsigned *p, unsigned v)
{
    __threadfence_block();
    *p = v;
}
__device__ __forceinline__ unsigned ld_acquire_cta(const volatile unsigned *p)
{
    const unsigned v = *p;
    __threadfence_block();
    return v;
}

// Scheduler (one thread).  next(t, item&, ctr*&, target&) decodes ticket t; done_ctr(item) is the
// global counter an item's completion is published on.
template <class Decode, class DoneCtr>
__device__ __forceinline__ void fused_scheduler(FusedCtl *ctl, FusedMailbox *mb, unsigned total, Decode decode, DoneCtr done_ctr)
{
    unsigned n = 0;            // items handed to the compute warps so far
    unsigned published = 0;    // completions published so far
    auto publish_ready = [&]() {   // publish every completion the compute warps have reported
        while (published < n && ld_acquire_cta(&mb->done[published & 1]) == published + 1) {
            __threadfence();
            atomicAdd(done_ctr(mb->item[published & 1]), 1u);
            ++published;
        }
    };
    bool abort = false;
    for (;;) {
        // the slot of item n was last used by item n-2: it must have been published (=> consumed)
        while (n >= 2 && published < n - 1) publish_ready();
        const unsigned t = atomicAdd(&ctl->ticket, 1u);
        FusedItem it{-1, 0, 0};
        if (t < total) {
            const unsigned *ctr = nullptr;
            unsigned target = 0;
            decode(t, it, ctr, target);
            unsigned spins = 0;
            while (ctr && ld_acquire_u32(ctr) < target) {
                publish_ready();
                __nanosleep(64);
                if (++spins > kSpinLimit || ld_acquire_u32(&ctl->error)) {
                    atomicExch(&ctl->error, 1u);
                    abort = true;
                    break;
                }
            }
        }
        if (abort) it.kind = -2;
        const unsigned s = n & 1;
        mb->item[s] = it;
        st_release_cta(&mb->full[s], n + 1);
        if (it.kind < 0) break;
        ++n;
    }
    if (!abort)
        while (published < n) publish_ready();
}

// Compute side: fetch the n-th item (thread 0 polls the mailbox, the compute barrier spreads it).
__device__ __forceinline__ FusedItem fused_next_item(FusedMailbox *mb, unsigned n)
{
    if (threadIdx.x == 0)
        while (ld_acquire_cta(&mb->full[n & 1]) != n + 1) {}
    SyncCompute()();
    return mb->item[n & 1];
}
__device__ __forceinline__ void fused_item_done(FusedMailbox *mb, unsigned n)
{
    SyncCompute()();            // every compute thread has issued this item's stores and is done with smem
    if (threadIdx.x == 0) st_release_cta(&mb->done[n & 1], n + 1);
}

// ---------------------------------------------------------------- forward: P1 -> P2
template <int T>
__global__ void __launch_bounds__(kThreads + 32, 2) k_xy_fwd(const double *__restrict__ rho, const double *__restrict__ rc,
                                                          double2 *W1ring, double2 *__restrict__ W2,
                                                          const double2 *__restrict__ tw, int L, FusedCtl *ctl, int R, int LAG)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, G = 16 / T, PEN = 8 * G;
    constexpr int nA = N / ROWS, nB = NN / PEN, PER = nA + nB;
    extern __shared__ double2 smem[];
    __shared__ FusedMailbox mb;
    const int P = L * N;
    const unsigned total = (unsigned)(P + LAG) * PER;
    unsigned *doneA = reinterpret_cast<unsigned *>(ctl + 1), *doneB = doneA + P;
    const int tid = threadIdx.x;
    if (tid == 0) mb.full[0] = mb.full[1] = mb.done[0] = mb.done[1] = 0;
    __syncthreads();

    if (tid >= kThreads) {                               // ---- scheduler warp
        if (tid == kThreads) {
            auto decode = [&](unsigned t, FusedItem &it, const unsigned *&ctr, unsigned &target) {
                const int q = (int)(t / PER), w = (int)(t % PER);
                if (w < nA) {                            // A: x transform of ROWS rows of plane q
                    it = FusedItem{q < P ? 0 : 2, q, w};
                    if (q < P && q >= R) { ctr = &doneB[q - R]; target = nB; }   // the ring slot is free
                } else {                                 // B: y transform of PEN columns of plane q - LAG
                    const int p = q - LAG;
                    it = FusedItem{p >= 0 ? 1 : 2, p, w - nA};
                    if (p >= 0) { ctr = &doneA[p]; target = nA; }
                }
            };
            auto done_ctr = [&](const FusedItem &it) { return it.kind == 0 ? &doneA[it.p] : (it.kind == 1 ? &doneB[it.p] : &ctl->pad[0]); };
            fused_scheduler(ctl, &mb, total, decode, done_ctr);
        }
        return;
    }
    for (unsigned n = 0;; ++n) {                         // ---- compute warps
        const FusedItem it = fused_next_item(&mb, n);
        if (it.kind < 0) break;
        if (it.kind == 0) {
            const int rl = it.w * ROWS + tid / T;        // row within the plane
            x_fwd_body<T>(rho, rc, W1ring + ((size_t)(it.p % R) * N + rl) * NN, tw, L, (size_t)it.p * N + rl, smem);
        } else if (it.kind == 1) {
            const int sx = it.w * PEN + (tid / (8 * T)) * 8 + (tid & 7);
            y_fwd_body<T, true, SyncCompute>(W1ring + (size_t)(it.p % R) * N * NN + sx, W2 + (size_t)it.p * NN * NN + sx, tw, smem);
        }                                                // kind 2: an empty ticket (before the first / after the last plane)
        fused_item_done(&mb, n);
    }
}

}  // namespace cmk
