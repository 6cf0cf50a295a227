// cm_plan.h — what the translation units of libcm share: the plan, the error helpers and the shared-memory sizes of the
// passes.  libcm is built from cm_lib.cu (plan, C ABI, the passes of the original method), cm_lib_expand.cu (the pruned /
// decimated passes of the modified method's expanded grids: 9 instantiations of 5 kernels, more than half of the compile
// time) and cm_static.cu, compiled side by side (paper_2301_06763_b200/_build.py).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cm.h"
#include "cm_kernels.cuh"

struct GraphEntry {
    const double *rho;
    double *phi;
    int mode;                      // 0 cm_potential, 1 pairs, 2 triplets (quadrupled grid by FFT), 3 triplets (Eq. B.7)
    cudaGraphExec_t exec;
    unsigned long long last_use;   // for least-recently-used eviction
};
constexpr size_t kGraphCacheSize = 8;

struct cm_plan {
    int N = 0, L = 0, T = 0;       // N: cells per axis of a level; the transforms run at Nf = 16 T = the next power of two >= N
    int Nf = 0;
    bool gen = false;               // N < Nf: the general-size instantiations of the passes
    double dx0 = 0, G = 1.0;
    double2 *W1 = nullptr, *W2 = nullptr, *tw = nullptr;
    double *Khat = nullptr, *rc = nullptr, *hole = nullptr, *pbar = nullptr;
    double *stage_rho = nullptr, *stage_phi = nullptr;
    size_t bytes = 0;
    bool green_ready = false;
    bool split_x = false, split_y = false;   // P1 / P2 split by output parity (256-thread CTAs): N = 256
    cm_plan *dbl = nullptr, *qdp = nullptr;   // single-level plans of the doubled (2N)^3 and quadrupled (4N)^3 fine grid
    double *rho4 = nullptr, *phi4 = nullptr, *tmp3 = nullptr;
    double *rho2 = nullptr, *phi2 = nullptr;   // two doubled grids each: one complex solve serves two pairs
    double2 *decE = nullptr;                    // expanded-grid plans: E(k) of the decimated inverse, slot order (cm_expand.cuh)
    bool use_graph = true;
    cudaStream_t cap_stream = nullptr, copy_stream = nullptr;
    std::vector<cudaEvent_t> ev_level;   // cm_potential_host's pipeline: [0,32) level arrived, [32,64) level's Phi ready, [64] start
    std::vector<GraphEntry> graphs;
    unsigned long long use_counter = 0;
    int launches = 0;
    int num_sms = 148;
    CUtensorMap mapW, mapWw;        // W2 as CTA-wide 128-byte boxes / as per-warp 32- or 64-byte boxes (k_z_conv_warp)
    bool zconv_warp = false;
    int kernels_per_solve = 0;
    char err[512] = {0};
};

inline bool cuda_fail(cm_plan *p, cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return false;
    if (p) std::snprintf(p->err, sizeof(p->err), "%s: %s", what, cudaGetErrorString(e));
    return true;
}
#define CM_CUDA(p, call)                                  \
    do {                                                  \
        if (cuda_fail((p), (call), #call)) return CM_ECUDA; \
    } while (0)

template <int T> size_t smem_row() { return sizeof(double2) * 2 * (cmk::kThreads / T) * cmk::LayRow<T>::PS; }
template <int T> size_t smem_batch() { return sizeof(double2) * 2 * cmk::batch_pencils<T>() * cmk::LayBatch<T>::PS; }

// The five passes of an expanded-grid solve (cm_lib_expand.cu).  attrs_only: set the kernels' attributes and return.
__attribute__((visibility("hidden"))) int cm_dispatch_expanded(cm_plan *pe, int F, const double *src_re, const double *src_im,
                                                               double *out_re, double *out_im, cudaStream_t s, bool attrs_only);
