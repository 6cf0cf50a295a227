// cm_lib.cu — the C ABI of include/cm.h: plan, workspace, CUDA-graph capture (the expanded-grid passes of the modified
// method are in cm_lib_expand.cu, the allocation-free direct sum in cm_static.cu).
#include "cm_plan.h"
#include "cm_zconv.cuh"
#include "cm_expand.cuh"

namespace {

using namespace cmk;

template <int T> int set_attrs(cm_plan *p)
{
    CM_CUDA(p, cudaFuncSetAttribute(k_x_fwd<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
    CM_CUDA(p, cudaFuncSetAttribute(k_x_inv<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
    CM_CUDA(p, cudaFuncSetAttribute(k_y_fwd<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
    CM_CUDA(p, cudaFuncSetAttribute(k_y_inv<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
    CM_CUDA(p, cudaFuncSetAttribute((k_y_fwd<T, false, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
    CM_CUDA(p, cudaFuncSetAttribute((k_y_inv<T, false, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
    if constexpr (T >= 2) {     // general sizes (N < 16 T)
        CM_CUDA(p, cudaFuncSetAttribute(k_x_fwd<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
        CM_CUDA(p, cudaFuncSetAttribute(k_x_inv<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
        CM_CUDA(p, cudaFuncSetAttribute(k_y_fwd<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(p, cudaFuncSetAttribute(k_y_inv<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(p, cudaFuncSetAttribute((k_y_fwd<T, true, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(p, cudaFuncSetAttribute((k_y_inv<T, true, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
    }
    if constexpr (T <= 16) {
        CM_CUDA(p, cudaFuncSetAttribute(k_x_fwd_split<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
        CM_CUDA(p, cudaFuncSetAttribute(k_y_fwd_split<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(p, cudaFuncSetAttribute(k_z_conv_tma<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZConvCfg<T>::SMEM));
        if constexpr (T >= 8)
            CM_CUDA(p, cudaFuncSetAttribute(k_z_conv_warp<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZWarpCfg<T>::SMEM));
    } else {
        CM_CUDA(p, cudaFuncSetAttribute(k_z_conv_dec<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZDecCfg<T>::SMEM));
    }
    return CM_OK;
}

// P3 (step a5) for levels [b0, b0 + L) of W2.
template <int T> void launch_zconv(cm_plan *p, cudaStream_t s, int b0, int L)
{
    constexpr int N = 16 * T, NN = 2 * N;
    if constexpr (T <= 16) {
        const int ngroups = NN * NN / ZConvCfg<T>::PEN;
        // N <= 64: the kernel cuts the flat (group, level) tile list into equal ranges, so up to one CTA per tile
        const long long units = (T <= 4) ? (long long)ngroups * L : ngroups;
        const int grid = units < ZConvCfg<T>::CTAS * p->num_sms ? (int)units : ZConvCfg<T>::CTAS * p->num_sms;
        if constexpr (T >= 8) {
            if (p->zconv_warp) {
                k_z_conv_warp<T><<<grid, kThreads, ZWarpCfg<T>::SMEM, s>>>(p->mapWw, p->Khat, p->tw, L, ngroups, b0);
                return;
            }
        }
        k_z_conv_tma<T><<<grid, kThreads, ZConvCfg<T>::SMEM, s>>>(p->mapW, p->Khat, p->W2, p->tw, L, ngroups, b0, p->N);
    } else {
        // N = 512: the batch-fastest P3 of cm_expand.cuh without decimation (a CTA per (|f_y|, 8 pencils): K-hat tile shared
        // by the two mirror tiles and by the levels)
        k_z_conv_dec<T, 1><<<(unsigned)((size_t)(N + 1) * (NN / batch_pencils<T>())), batch_threads<T>(), ZDecCfg<T>::SMEM, s>>>(
            p->Khat, p->W2, p->tw, nullptr, 0, p->N, b0, L, p->N, /*ahead=*/p->num_sms);
    }
}

// P5 of level b.  chained: programmatic dependent launch on the launch before it in the stream (level b-1's P5), so
// that this level's loads and transforms overlap that level's tail; the kernel waits (griddepcontrol.wait) only
// before it reads what level b-1 wrote.
template <int T>
void launch_x_inv(cm_plan *p, double *phi, cudaStream_t s, int b, unsigned grid, double scale0, bool chained, int hole_all)
{
    const size_t nd = (size_t)p->N;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem_row<T>();
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = chained ? 1 : 0;
    if (p->gen)
        cudaLaunchKernelEx(&cfg, k_x_inv<T, true>, (const double2 *)p->W1, phi, p->hole, (const double *)p->hole, (const double2 *)p->tw,
                           p->L, scale0, (size_t)b * nd * nd, hole_all, p->N);
    else
        cudaLaunchKernelEx(&cfg, k_x_inv<T, false>, (const double2 *)p->W1, phi, p->hole, (const double *)p->hole, (const double2 *)p->tw,
                           p->L, scale0, (size_t)b * nd * nd, hole_all, p->N);
}

// The five FFT passes (steps a3-a7) with the prolongation + Eq. 14 sum (a8) folded into P5:
// P1-P4 take every level in one launch; P5 runs level by level, coarse -> fine, because
// level b adds the prolonged hole potentials of level b-1 (k_x_inv).
template <int T> int launch_passes(cm_plan *p, const double *rho, double *phi, cudaStream_t s, cudaEvent_t *ev, int hole_all)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, PEN = batch_pencils<T>(), BT = batch_threads<T>();
    const int L = p->L, nd = p->N;
    const size_t planes = (size_t)L * nd, rows = planes * nd;
    const double scale0 = -p->G * p->dx0 * p->dx0;
    const unsigned gx = (unsigned)((rows + ROWS - 1) / ROWS), gy = (unsigned)(planes * NN / PEN);
    bool done_x = false, done_y = false;
    // L2 prefetch of the columns of the CTA half a wave (N = 128) or a wave (N = 512: one CTA per SM) ahead in P2 / P4 — measured
    // per size (profiles/r02_pass_variants.md): -10 % / -3 % at N = 128, -16 % / -11 % at N = 512, nothing at N = 256 (P4 is at the
    // copy peak there and P2 is the split kernel with its own prefetch) and at N <= 64 (L2-resident)
    const int ya = (T == 32 || T == 8) ? p->num_sms : 0, ya4 = ya;
    if constexpr (T <= 16) {
        if (p->split_x) {
            k_x_fwd_split<T><<<gx, 2 * kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, L);
            done_x = true;
        }
    }
    if (!done_x) {
        if (p->gen) k_x_fwd<T, true><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, L, 0, nd, rows);
        else k_x_fwd<T, false><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, L, 0);
    }
    if (ev) cudaEventRecord(ev[2], s);
    if constexpr (T <= 16) {
        if (p->split_y) {
            k_y_fwd_split<T><<<gy, 2 * kThreads, smem_batch<T>(), s>>>(p->W1, p->W2, p->tw, /*ahead=*/p->num_sms);
            done_y = true;
        }
    }
    if (!done_y) {
        if (p->gen && ya > 0) k_y_fwd<T, true, true><<<gy, BT, smem_batch<T>(), s>>>(p->W1, p->W2, p->tw, nd, ya);
        else if (p->gen) k_y_fwd<T, true><<<gy, BT, smem_batch<T>(), s>>>(p->W1, p->W2, p->tw, nd);
        else if (ya > 0) k_y_fwd<T, false, true><<<gy, BT, smem_batch<T>(), s>>>(p->W1, p->W2, p->tw, 0, ya);
        else k_y_fwd<T, false><<<gy, BT, smem_batch<T>(), s>>>(p->W1, p->W2, p->tw);
    }
    if (ev) cudaEventRecord(ev[3], s);
    launch_zconv<T>(p, s, 0, L);
    if (ev) cudaEventRecord(ev[4], s);
    if (p->gen && ya4 > 0) k_y_inv<T, true, true><<<gy, BT, smem_batch<T>(), s>>>(p->W2, p->W1, p->tw, nd, ya4);
    else if (p->gen) k_y_inv<T, true><<<gy, BT, smem_batch<T>(), s>>>(p->W2, p->W1, p->tw, nd);
    else if (ya4 > 0) k_y_inv<T, false, true><<<gy, BT, smem_batch<T>(), s>>>(p->W2, p->W1, p->tw, 0, ya4);
    else k_y_inv<T, false><<<gy, BT, smem_batch<T>(), s>>>(p->W2, p->W1, p->tw);
    if (ev) cudaEventRecord(ev[5], s);
    const size_t lrows = (size_t)nd * nd;
    const unsigned gl = (unsigned)((lrows + ROWS - 1) / ROWS);
    for (int b = 0; b < L; ++b) launch_x_inv<T>(p, phi, s, b, gl, scale0, /*chained=*/b > 0, hole_all);
    if (ev) cudaEventRecord(ev[6], s);
    p->launches += 4 + L;
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

// One level's P1..P4 / P5 on their own (cm_potential_host's pipeline): the same kernels on the level's
// slices of W1 / W2; P3 then runs with a one-level range, so K-hat is read once per level (irrelevant there:
// that path is bound by the host link).
template <int T> void level_p1_to_p4(cm_plan *p, const double *rho, cudaStream_t s, int l)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, PEN = batch_pencils<T>(), BT = batch_threads<T>();
    const int nd = p->N;
    const size_t lrows = (size_t)nd * nd;
    double2 *w1 = p->W1 + (size_t)l * lrows * NN, *w2 = p->W2 + (size_t)l * nd * NN * NN;
    const unsigned gx = (unsigned)((lrows + ROWS - 1) / ROWS), gy = (unsigned)((size_t)nd * NN / PEN);
    if (p->gen) {
        k_x_fwd<T, true><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, p->L, (size_t)l * lrows, nd, (size_t)(l + 1) * lrows);
        k_y_fwd<T, true><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw, nd);
        launch_zconv<T>(p, s, l, 1);
        k_y_inv<T, true><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw, nd);
    } else {
        k_x_fwd<T, false><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, p->L, (size_t)l * lrows);
        k_y_fwd<T, false><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw);
        launch_zconv<T>(p, s, l, 1);
        k_y_inv<T, false><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw);
    }
}
template <int T> void level_p5(cm_plan *p, double *phi, cudaStream_t s, int l)
{
    constexpr int ROWS = kThreads / T;
    const size_t lrows = (size_t)p->N * p->N;
    launch_x_inv<T>(p, phi, s, l, (unsigned)((lrows + ROWS - 1) / ROWS), -p->G * p->dx0 * p->dx0, /*chained=*/false, 0);
}
void dispatch_level(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int l, bool p5)
{
    switch (p->T) {
        case 1: p5 ? level_p5<1>(p, phi, s, l) : level_p1_to_p4<1>(p, rho, s, l); break;
        case 2: p5 ? level_p5<2>(p, phi, s, l) : level_p1_to_p4<2>(p, rho, s, l); break;
        case 4: p5 ? level_p5<4>(p, phi, s, l) : level_p1_to_p4<4>(p, rho, s, l); break;
        case 8: p5 ? level_p5<8>(p, phi, s, l) : level_p1_to_p4<8>(p, rho, s, l); break;
        case 16: p5 ? level_p5<16>(p, phi, s, l) : level_p1_to_p4<16>(p, rho, s, l); break;
        case 32: p5 ? level_p5<32>(p, phi, s, l) : level_p1_to_p4<32>(p, rho, s, l); break;
    }
}

// Levels [lo, hi) on their own (the level-sharded solve): the same kernels on those levels' rows of
// W1 / W2, one launch per pass for the whole range (P3 reads K-hat once for the range).
template <int T> void range_p1_to_p4(cm_plan *p, const double *rho, cudaStream_t s, int lo, int hi)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, PEN = batch_pencils<T>(), BT = batch_threads<T>();
    const int nd = p->N, nl = hi - lo;
    const size_t lrows = (size_t)nd * nd;
    double2 *w1 = p->W1 + (size_t)lo * lrows * NN, *w2 = p->W2 + (size_t)lo * nd * NN * NN;
    const unsigned gx = (unsigned)((nl * lrows + ROWS - 1) / ROWS), gy = (unsigned)((size_t)nl * nd * NN / PEN);
    const int ya = (T == 32 || T == 8) ? p->num_sms : 0;      // as in launch_passes
    if (p->gen) {
        k_x_fwd<T, true><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, p->L, (size_t)lo * lrows, nd, (size_t)hi * lrows);
        if (ya > 0) k_y_fwd<T, true, true><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw, nd, ya);
        else k_y_fwd<T, true><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw, nd);
        launch_zconv<T>(p, s, lo, nl);
        if (ya > 0) k_y_inv<T, true, true><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw, nd, ya);
        else k_y_inv<T, true><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw, nd);
    } else {
        k_x_fwd<T, false><<<gx, kThreads, smem_row<T>(), s>>>(rho, p->rc, p->W1, p->tw, p->L, (size_t)lo * lrows);
        if (ya > 0) k_y_fwd<T, false, true><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw, 0, ya);
        else k_y_fwd<T, false><<<gy, BT, smem_batch<T>(), s>>>(w1, w2, p->tw);
        launch_zconv<T>(p, s, lo, nl);
        if (ya > 0) k_y_inv<T, false, true><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw, 0, ya);
        else k_y_inv<T, false><<<gy, BT, smem_batch<T>(), s>>>(w2, w1, p->tw);
    }
}
template <int T> void range_p5(cm_plan *p, double *phi, cudaStream_t s, int lo, int hi)
{
    constexpr int ROWS = kThreads / T;
    const size_t lrows = (size_t)p->N * p->N;
    for (int b = lo; b < hi; ++b)      // the first launch of the range is a normal one: it comes after the unpacked ring
        launch_x_inv<T>(p, phi, s, b, (unsigned)((lrows + ROWS - 1) / ROWS), -p->G * p->dx0 * p->dx0, /*chained=*/b > lo, 0);
}
void dispatch_range(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int lo, int hi, bool p5)
{
    switch (p->T) {
        case 1: p5 ? range_p5<1>(p, phi, s, lo, hi) : range_p1_to_p4<1>(p, rho, s, lo, hi); break;
        case 2: p5 ? range_p5<2>(p, phi, s, lo, hi) : range_p1_to_p4<2>(p, rho, s, lo, hi); break;
        case 4: p5 ? range_p5<4>(p, phi, s, lo, hi) : range_p1_to_p4<4>(p, rho, s, lo, hi); break;
        case 8: p5 ? range_p5<8>(p, phi, s, lo, hi) : range_p1_to_p4<8>(p, rho, s, lo, hi); break;
        case 16: p5 ? range_p5<16>(p, phi, s, lo, hi) : range_p1_to_p4<16>(p, rho, s, lo, hi); break;
        case 32: p5 ? range_p5<32>(p, phi, s, lo, hi) : range_p1_to_p4<32>(p, rho, s, lo, hi); break;
    }
}

// ev (optional): 8 events; ev[0] start, ev[1] after a1, ev[2..6] after P1..P5, ev[7] after a8
// hole_all: P5 keeps H = Phi_hole + ext on every cell, not only on the ring the next level reads (the modified method, Eq. B.1)
int enqueue_solve(cm_plan *p, const double *rho, double *phi, cudaStream_t s, cudaEvent_t *ev = nullptr, int hole_all = 0)
{
    const int N = p->N, L = p->L, H = N / 2;
    const size_t n3 = (size_t)N * N * N, h3 = (size_t)H * H * H;
    p->launches = 0;
    if (ev) cudaEventRecord(ev[0], s);
    // a1: restriction cascade.  Every parent without a child under the next finer grid in one launch for all levels, then
    // fine -> coarse the 1/8 of each level's parents that take already projected values (k_restrict_inner)
    if (L > 1) {
        k_restrict_outer<<<dim3((unsigned)((h3 + 255) / 256), L - 1), 256, 0, s>>>(N, L, rho, p->rc);
        p->launches++;
        const int bx = (3 * (N / 4) + 1) / 2 - (N / 4) / 2;
        for (int lf = L - 2; lf >= 1; --lf) {
            k_restrict_inner<<<(unsigned)(((size_t)bx * bx * bx + 255) / 256), 256, 0, s>>>(N, lf, rho + n3 * lf, p->rc + h3 * lf,
                                                                                             p->rc + h3 * (lf - 1));
            p->launches++;
        }
    }
    CM_CUDA(p, cudaGetLastError());
    if (ev) cudaEventRecord(ev[1], s);
    int rcode = CM_EINVAL;
    switch (p->T) {
        case 1: rcode = launch_passes<1>(p, rho, phi, s, ev, hole_all); break;
        case 2: rcode = launch_passes<2>(p, rho, phi, s, ev, hole_all); break;
        case 4: rcode = launch_passes<4>(p, rho, phi, s, ev, hole_all); break;
        case 8: rcode = launch_passes<8>(p, rho, phi, s, ev, hole_all); break;
        case 16: rcode = launch_passes<16>(p, rho, phi, s, ev, hole_all); break;
        case 32: rcode = launch_passes<32>(p, rho, phi, s, ev, hole_all); break;
    }
    if (rcode != CM_OK) return rcode;
    // a8 (prolongation + Eq. 14 sum) ran inside P5
    if (ev) cudaEventRecord(ev[7], s);
    return CM_OK;
}

void destroy_graphs(cm_plan *p)
{
    for (auto &g : p->graphs)
        if (g.exec) cudaGraphExecDestroy(g.exec);
    p->graphs.clear();
}

template <class Tp> int dev_alloc(cm_plan *p, Tp **ptr, size_t count)
{
    void *q = nullptr;
    cudaError_t e = cudaMalloc(&q, count * sizeof(Tp));
    if (e == cudaErrorMemoryAllocation) {
        cuda_fail(p, e, "cudaMalloc");
        cudaGetLastError();
        return CM_ENOMEM;
    }
    if (cuda_fail(p, e, "cudaMalloc")) return CM_ECUDA;
    *ptr = (Tp *)q;
    p->bytes += count * sizeof(Tp);
    return CM_OK;
}

// TMA descriptors for P3 (cm_zconv.cuh).  cuTensorMapEncodeTiled is a driver entry point;
// it is looked up through the runtime so that libcm does not link libcuda directly.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tensor_maps(cm_plan *p)
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    CM_CUDA(p, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (!fn || q != cudaDriverEntryPointSuccess) {
        std::snprintf(p->err, sizeof(p->err), "cuTensorMapEncodeTiled not available from this driver");
        return CM_ECUDA;
    }
    EncodeTiledFn enc = (EncodeTiledFn)fn;
    const cuuint64_t NN = 2 * (cuuint64_t)p->Nf, N = p->N, L = p->L;     // N rows of data per level, spectra of 2 Nf slots
    const cuuint32_t es[2] = {1, 1};
    {   // W2 as fp64 [L*N rows][2*(2Nf)^2]; box = 16 doubles (8 complex = 128 B) x N rows, 128B swizzle
        const cuuint64_t dims[2] = {2 * NN * NN, L * N};
        const cuuint64_t strides[1] = {NN * NN * 16};
        const cuuint32_t box[2] = {16, (cuuint32_t)N};
        CUresult r = enc(&p->mapW, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, p->W2, dims, strides, box, es,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            std::snprintf(p->err, sizeof(p->err), "cuTensorMapEncodeTiled(W2) failed: %d", (int)r);
            return CM_ECUDA;
        }
    }
    if (p->N >= 128 && !p->gen) {   // per-warp boxes: PPW pencils (32 B at N = 256, 64 B at N = 128) x N rows, swizzle = the row width
        const int ppw = 32 / (p->N / 16);
        const cuuint64_t dims[2] = {2 * NN * NN, L * N};
        const cuuint64_t strides[1] = {NN * NN * 16};
        const cuuint32_t box[2] = {(cuuint32_t)(2 * ppw), (cuuint32_t)N};
        CUresult r = enc(&p->mapWw, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, p->W2, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         ppw == 2 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            std::snprintf(p->err, sizeof(p->err), "cuTensorMapEncodeTiled(W2, per-warp boxes) failed: %d", (int)r);
            return CM_ECUDA;
        }
    }
    return CM_OK;
}

// One call = one CUDA-graph launch.  The sequence of `mode` (0: the original method; 1-3: the modified method, whose
// expanded-grid plans must already exist — nothing may allocate during capture) is captured once per (rho, phi, mode) on the
// plan's own stream and launched on the caller's; the cache keeps the kGraphCacheSize most recently used entries (callers
// that rotate buffers should reuse them).  CM_DEBUG=nograph launches kernel by kernel.
int enqueue_mode(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int mode);

int run_graphed(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int mode)
{
    if (!p->use_graph) return enqueue_mode(p, rho, phi, s, mode);
    for (auto &g : p->graphs)
        if (g.rho == rho && g.phi == phi && g.mode == mode) {
            g.last_use = ++p->use_counter;
            CM_CUDA(p, cudaGraphLaunch(g.exec, s));
            return CM_OK;
        }
    cudaGraph_t graph = nullptr;
    CM_CUDA(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
    const int rc = enqueue_mode(p, rho, phi, p->cap_stream, mode);
    cudaError_t ee = cudaStreamEndCapture(p->cap_stream, &graph);
    if (rc != CM_OK || ee != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        if (rc != CM_OK) return rc;
        CM_CUDA(p, ee);
    }
    GraphEntry ge{rho, phi, mode, nullptr, ++p->use_counter};
    ee = cudaGraphInstantiate(&ge.exec, graph, 0);
    cudaGraphDestroy(graph);   // the executable graph is self-contained
    CM_CUDA(p, ee);
    if (p->graphs.size() >= kGraphCacheSize) {
        size_t lru = 0;
        for (size_t i = 1; i < p->graphs.size(); ++i)
            if (p->graphs[i].last_use < p->graphs[lru].last_use) lru = i;
        cudaGraphExecDestroy(p->graphs[lru].exec);
        p->graphs[lru] = ge;
    } else {
        p->graphs.push_back(ge);
    }
    CM_CUDA(p, cudaGraphLaunch(ge.exec, s));
    return CM_OK;
}

}  // namespace

extern "C" {

int cm_plan_create(cm_plan **out, int N, int levels, double dx0, int refinement)
{
    if (!out) return CM_EINVAL;
    *out = nullptr;
    if (refinement != 2) return CM_EINVAL;
    if (N < 16 || N > 512 || (N % 4) != 0) return CM_EINVAL;
    if (levels < 1 || levels > 32) return CM_EINVAL;
    if (!(dx0 > 0.0) || !std::isfinite(dx0)) return CM_EINVAL;

    cm_plan *p = new (std::nothrow) cm_plan();
    if (!p) return CM_ENOMEM;
    p->N = N;
    p->L = levels;
    p->Nf = 16;
    while (p->Nf < N) p->Nf *= 2;       // the transforms run at the next power of two: 2 Nf >= 2 N - 1 is all a linear
    p->T = p->Nf / 16;                  // convolution needs (L143); the surplus is more zero padding
    p->gen = (p->Nf != N);
    p->dx0 = dx0;
    // the one environment switch (cm.h): CM_DEBUG=nograph launches kernel by kernel instead of through a CUDA graph
    if (const char *dbg = std::getenv("CM_DEBUG")) {
        if (std::strcmp(dbg, "nograph") == 0) p->use_graph = false;
        else if (dbg[0] != '\0') {
            delete p;
            return CM_EINVAL;
        }
    }
    const size_t n = 2 * (size_t)p->Nf, n3 = (size_t)N * N * N, h3 = n3 / 8, L = (size_t)levels;
    int rc = CM_OK;
    if ((rc = dev_alloc(p, &p->W1, L * N * N * n)) == CM_OK &&
        (rc = dev_alloc(p, &p->W2, L * N * n * n)) == CM_OK &&
        (rc = dev_alloc(p, &p->Khat, n * n * (size_t)khat_row_stride(p->Nf))) == CM_OK &&
        (rc = dev_alloc(p, &p->rc, (L > 1 ? L - 1 : 1) * h3)) == CM_OK &&
        (rc = dev_alloc(p, &p->hole, L * n3)) == CM_OK &&
        (rc = dev_alloc(p, &p->pbar, (L > 1 ? L - 1 : 1) * h3)) == CM_OK &&
        (rc = dev_alloc(p, &p->tw, n)) == CM_OK) {
    // twiddles w_2N^m = exp(-2 pi i m / 2N), computed in long double on the host
        std::vector<double2> tw(n);
        const long double tau = 2.0L * acosl(-1.0L);
        for (size_t m = 0; m < n; ++m) {
            const long double a = -tau * (long double)m / (long double)n;
            tw[m] = make_double2((double)cosl(a), (double)sinl(a));
        }
        // exact values on the axes
        tw[0] = make_double2(1.0, 0.0);
        tw[n / 4] = make_double2(0.0, -1.0);
        tw[n / 2] = make_double2(-1.0, 0.0);
        tw[3 * n / 4] = make_double2(0.0, 1.0);
        if (cuda_fail(p, cudaMemcpy(p->tw, tw.data(), n * sizeof(double2), cudaMemcpyHostToDevice), "cudaMemcpy(tw)"))
            rc = CM_ECUDA;
        else if (cuda_fail(p, cudaMemset(p->hole, 0, L * n3 * sizeof(double)), "cudaMemset")) rc = CM_ECUDA;
        else if (cuda_fail(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking), "cudaStreamCreate"))
            rc = CM_ECUDA;
    }
    if (rc == CM_OK) {
        // kernel variants by size, each chosen by measurement
        p->split_y = (N == 256);      // P2 split by output parity: -8 % at N = 256, +4 % at N = 128
        p->split_x = (N == 256);      // P1 split by output parity: -12 % at N = 256, +7 % at N = 128
        p->zconv_warp = (N == 128);   // warp-autonomous P3: -6 % at N = 128; at N = 256 its 32-byte TMA boxes crawl
        int dev = 0;
        if (cuda_fail(p, cudaGetDevice(&dev), "cudaGetDevice") ||
            cuda_fail(p, cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute"))
            rc = CM_ECUDA;
        else if (p->Nf <= 256) rc = make_tensor_maps(p);   // the TMA-fed P3 (Nf = 512 runs k_z_conv_dec<32, 1>)
    }
    if (rc == CM_OK) {
        switch (p->T) {
            case 1: rc = set_attrs<1>(p); break;
            case 2: rc = set_attrs<2>(p); break;
            case 4: rc = set_attrs<4>(p); break;
            case 8: rc = set_attrs<8>(p); break;
            case 16: rc = set_attrs<16>(p); break;
            case 32: rc = set_attrs<32>(p); break;
        }
    }
    if (rc != CM_OK) {
        cm_plan_destroy(p);
        return rc;
    }
    // number of kernels per solve: (L-1) restrictions + P1..P4 + one P5 per level
    p->kernels_per_solve = (levels - 1) + 4 + levels;
    p->launches = p->kernels_per_solve;
    *out = p;
    return CM_OK;
}

int cm_green_precompute(cm_plan *p)
{
    if (!p) return CM_EINVAL;
    if (p->green_ready) return CM_OK;
    const int N = p->Nf, n = 2 * N;          // K-hat of the transform size (a superset of the offsets a level of p->N cells needs)
    const size_t tot = (size_t)n * n * n;
    double2 *Gm = nullptr;
    cudaError_t e = cudaMalloc((void **)&Gm, tot * sizeof(double2));
    if (e != cudaSuccess) {
        cuda_fail(p, e, "cudaMalloc(green scratch)");
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? CM_ENOMEM : CM_ECUDA;
    }
    const double I0 = (double)(3.0L * logl(2.0L + sqrtl(3.0L)) - acosl(-1.0L) / 2.0L);  // Eq. 13, cube
    int log2n = 0;
    while ((1 << log2n) < n) ++log2n;
    cudaStream_t s = p->cap_stream;
    k_green_sample<<<1024, 256, 0, s>>>(Gm, N, I0);
    for (int axis = 0; axis < 3; ++axis)
        k_fft_simple<<<(unsigned)(n * n), n / 2 < 256 ? n / 2 : 256, n * sizeof(double2), s>>>(Gm, n, log2n, axis, p->tw);
    k_green_permute<<<1024, 256, 0, s>>>(Gm, p->Khat, N);
    cudaError_t e1 = cudaGetLastError();
    cudaError_t e2 = cudaStreamSynchronize(s);
    cudaFree(Gm);
    if (cuda_fail(p, e1, "green kernels") || cuda_fail(p, e2, "green sync")) return CM_ECUDA;
    p->green_ready = true;
    return CM_OK;
}

int cm_potential(cm_plan *p, const double *rho, double *phi, void *stream)
{
    if (!p || !rho || !phi) return CM_EINVAL;
    if (((uintptr_t)rho & 15) || ((uintptr_t)phi & 15)) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    const size_t tot = (size_t)p->L * p->N * p->N * p->N;
    if ((rho <= phi && phi < rho + tot) || (phi <= rho && rho < phi + tot)) return CM_EINVAL;
    return run_graphed(p, rho, phi, (cudaStream_t)stream, 0);
}

int cm_potential_profile(cm_plan *p, const double *rho, double *phi, void *stream, float *ms_host, int n_ms)
{
    if (!p || !rho || !phi || !ms_host || n_ms != 7) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    cudaStream_t s = (cudaStream_t)stream;
    cudaEvent_t ev[8];
    for (int i = 0; i < 8; ++i) CM_CUDA(p, cudaEventCreate(&ev[i]));
    int rc = enqueue_solve(p, rho, phi, s, ev);
    if (rc == CM_OK && cuda_fail(p, cudaStreamSynchronize(s), "cudaStreamSynchronize")) rc = CM_ECUDA;
    if (rc == CM_OK)
        for (int i = 0; i < 7; ++i)
            if (cuda_fail(p, cudaEventElapsedTime(&ms_host[i], ev[i], ev[i + 1]), "cudaEventElapsedTime")) rc = CM_ECUDA;
    for (int i = 0; i < 8; ++i) cudaEventDestroy(ev[i]);
    return rc;
}

int cm_potential_host(cm_plan *p, const double *rho_host, double *phi_host, void *stream)
{
    if (!p || !rho_host || !phi_host) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    const size_t n3 = (size_t)p->N * p->N * p->N, tot = (size_t)p->L * n3;
    if (!p->stage_rho) {
        size_t keep = p->bytes;
        int rc = dev_alloc(p, &p->stage_rho, tot);
        if (rc == CM_OK) rc = dev_alloc(p, &p->stage_phi, tot);
        p->bytes = keep;  // staging is reported separately
        if (rc != CM_OK) return rc;
    }
    cudaStream_t s = (cudaStream_t)stream;
    if (p->N < 128) {
        // small grids are launch-bound, not link-bound: one copy in, the graph, one copy out
        CM_CUDA(p, cudaMemcpyAsync(p->stage_rho, rho_host, tot * sizeof(double), cudaMemcpyHostToDevice, s));
        const int rc = cm_potential(p, p->stage_rho, p->stage_phi, stream);
        if (rc != CM_OK) return rc;
        CM_CUDA(p, cudaMemcpyAsync(phi_host, p->stage_phi, tot * sizeof(double), cudaMemcpyDeviceToHost, s));
        CM_CUDA(p, cudaStreamSynchronize(s));
        return CM_OK;
    }
    // Level pipeline (N >= 128: the host link is the bound).  rho arrives finest level first on a copy
    // stream; as soon as level l is there its projection onto level l-1 (a1) and its P1..P4 run, under the
    // copy of the next level.  P5 + a8 must go coarse -> fine, so it starts when level 0 is through, and
    // every level's Phi leaves for the host while the next level's P5 runs.
    const int L = p->L;
    const size_t h3 = n3 / 8;
    if (!p->copy_stream) {
        CM_CUDA(p, cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
        p->ev_level.resize(2 * 32 + 1, nullptr);
        for (auto &e : p->ev_level) CM_CUDA(p, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    cudaEvent_t *ev_in = p->ev_level.data(), *ev_out = ev_in + 32, ev_start = p->ev_level[64];
    CM_CUDA(p, cudaEventRecord(ev_start, s));                       // work already queued on s comes first
    CM_CUDA(p, cudaStreamWaitEvent(p->copy_stream, ev_start, 0));
    for (int l = L - 1; l >= 0; --l) {
        CM_CUDA(p, cudaMemcpyAsync(p->stage_rho + l * n3, rho_host + l * n3, n3 * sizeof(double), cudaMemcpyHostToDevice,
                                   p->copy_stream));
        CM_CUDA(p, cudaEventRecord(ev_in[l], p->copy_stream));
    }
    for (int l = L - 1; l >= 0; --l) {
        CM_CUDA(p, cudaStreamWaitEvent(s, ev_in[l], 0));
        if (l < L - 1) {                                            // rc[l] = projection of level l+1 (a1)
            const double *rc_f = (l + 1 < L - 1) ? p->rc + h3 * (l + 1) : nullptr;
            k_restrict<<<(unsigned)((h3 + 255) / 256), 256, 0, s>>>(p->N, l + 1, L, p->stage_rho + n3 * (l + 1), rc_f, p->rc + h3 * l);
        }
        dispatch_level(p, p->stage_rho, p->stage_phi, s, l, false);
    }
    for (int l = 0; l < L; ++l) {
        dispatch_level(p, p->stage_rho, p->stage_phi, s, l, true);
        CM_CUDA(p, cudaEventRecord(ev_out[l], s));
        CM_CUDA(p, cudaStreamWaitEvent(p->copy_stream, ev_out[l], 0));
        CM_CUDA(p, cudaMemcpyAsync(phi_host + l * n3, p->stage_phi + l * n3, n3 * sizeof(double), cudaMemcpyDeviceToHost,
                                   p->copy_stream));
    }
    CM_CUDA(p, cudaGetLastError());
    CM_CUDA(p, cudaStreamSynchronize(p->copy_stream));
    CM_CUDA(p, cudaStreamSynchronize(s));
    return CM_OK;
}

}  // extern "C"

// ---- level-sharded solve: levels [lo, hi) of the nest on this GPU ----
namespace {
int check_shard(const cm_plan *p, const void *own, int lo, int hi)
{
    if (!p || !own || ((uintptr_t)own & 15)) return CM_EINVAL;
    if (lo < 0 || hi <= lo || hi > p->L) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    return CM_OK;
}
// the caller's arrays hold the levels [lo, hi) only: address of the (virtual) level 0
template <class Tp> Tp *level0(Tp *own, int lo, size_t n3) { return (Tp *)((uintptr_t)own - (uintptr_t)lo * n3 * sizeof(double)); }
}  // namespace

extern "C" {

int cm_shard_restrict(cm_plan *p, const double *rho_own, int lo, int hi, const double *rc_from_finer, double *rc_to_coarser, void *stream)
{
    const int chk = check_shard(p, rho_own, lo, hi);
    if (chk != CM_OK) return chk;
    const int L = p->L;
    if ((hi < L) != (rc_from_finer != nullptr) || (lo > 0) != (rc_to_coarser != nullptr)) return CM_EINVAL;
    const size_t n3 = (size_t)p->N * p->N * p->N, h3 = n3 / 8;
    const double *rho = level0(rho_own, lo, n3);
    cudaStream_t s = (cudaStream_t)stream;
    if (hi < L) CM_CUDA(p, cudaMemcpyAsync(p->rc + h3 * (hi - 1), rc_from_finer, h3 * sizeof(double), cudaMemcpyDeviceToDevice, s));
    // a1 on the own levels, fine -> coarse: level lf projects onto the cavity of level lf - 1; the last one leaves
    for (int lf = hi - 1; lf >= lo && lf >= 1; --lf) {
        const double *rc_f = (lf < L - 1) ? p->rc + h3 * lf : nullptr;
        double *out = (lf - 1 >= lo) ? p->rc + h3 * (lf - 1) : rc_to_coarser;
        k_restrict<<<(unsigned)((h3 + 255) / 256), 256, 0, s>>>(p->N, lf, L, rho + n3 * lf, rc_f, out);
    }
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

int cm_shard_forward(cm_plan *p, const double *rho_own, int lo, int hi, void *stream)
{
    const int chk = check_shard(p, rho_own, lo, hi);
    if (chk != CM_OK) return chk;
    const size_t n3 = (size_t)p->N * p->N * p->N;
    dispatch_range(p, level0(rho_own, lo, n3), nullptr, (cudaStream_t)stream, lo, hi, false);
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

int cm_shard_finish(cm_plan *p, double *phi_own, int lo, int hi, const double *ring_from_coarser, double *ring_to_finer, void *stream)
{
    const int chk = check_shard(p, phi_own, lo, hi);
    if (chk != CM_OK) return chk;
    const int L = p->L, B = p->N / 2 + 2;
    if ((lo > 0) != (ring_from_coarser != nullptr) || (hi < L) != (ring_to_finer != nullptr)) return CM_EINVAL;
    const size_t n3 = (size_t)p->N * p->N * p->N, b3 = (size_t)B * B * B;
    const unsigned gb = (unsigned)((b3 + 255) / 256);
    cudaStream_t s = (cudaStream_t)stream;
    if (lo > 0) k_ring_box<<<gb, 256, 0, s>>>(p->N, p->hole + n3 * (lo - 1), const_cast<double *>(ring_from_coarser), 1);
    dispatch_range(p, nullptr, level0(phi_own, lo, n3), s, lo, hi, true);
    if (hi < L) k_ring_box<<<gb, 256, 0, s>>>(p->N, p->hole + n3 * (hi - 1), ring_to_finer, 0);
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

}  // extern "C" (re-opened below)

namespace {

// one expanded-grid plan (N' = F N, one level, unit G and dx: it supplies K-hat, the twiddles and W1 / W2), the table
// E(k) = sum_{q<F} e^{2 pi i k q / 2N'} in slot order, and compact N^3 buffers for two sources and two results
int ensure_expanded(cm_plan *p, int F, cm_plan **plan, double **src, double **res)
{
    if (*plan && *src && *res) return CM_OK;
    const size_t n3 = (size_t)p->N * p->N * p->N;
    const size_t keep = p->bytes;
    int rc = CM_OK;
    if (!*plan) rc = cm_plan_create(plan, F * p->N, 1, 1.0, 2);
    if (rc == CM_OK) rc = cm_green_precompute(*plan);
    if (rc == CM_OK && !(*plan)->decE) {
        cm_plan *pe = *plan;
        const int n = 2 * pe->Nf;           // the transform length
        rc = dev_alloc(pe, &pe->decE, (size_t)n);
        if (rc == CM_OK) {
            std::vector<double2> E(n);
            const long double tau = 2.0L * acosl(-1.0L);
            for (int sl = 0; sl < n; ++sl) {
                const int k = cmfft::slot_to_freq(sl, pe->Nf);
                long double re = 0, im = 0;
                for (int q = 0; q < F; ++q) {
                    const long double a = tau * (long double)(((long long)k * q) % n) / (long double)n;
                    re += cosl(a);
                    im += sinl(a);
                }
                E[sl] = make_double2((double)re, (double)im);
            }
            if (cuda_fail(p, cudaMemcpy(pe->decE, E.data(), n * sizeof(double2), cudaMemcpyHostToDevice), "cudaMemcpy(E)")) rc = CM_ECUDA;
        }
    }
    if (rc == CM_OK) rc = cm_dispatch_expanded(*plan, F, nullptr, nullptr, nullptr, nullptr, nullptr, /*attrs_only=*/true);
    if (rc == CM_OK && !*src) rc = dev_alloc(p, src, 2 * n3);
    if (rc == CM_OK && !*res) rc = dev_alloc(p, res, 2 * n3);
    if (rc != CM_OK) {
        // all or nothing: a later call must not find a half-built expanded plan
        if (*plan) std::snprintf(p->err, sizeof(p->err), "expanded-grid plan (x%d): %.400s", F, (*plan)->err);
        cm_plan_destroy(*plan);
        *plan = nullptr;
        cudaFree(*src);
        cudaFree(*res);
        *src = *res = nullptr;
        p->bytes = keep;
        return rc;
    }
    p->bytes += (*plan)->bytes;
    return CM_OK;
}

// Expanded grids of levels l1 and (optionally) l1b through ONE complex solve (K-hat real, E Hermitian: the second
// density rides as the imaginary part); res and res + N^3 receive minus the block sums of rho * g over the F^3 cells
// of a coarse cell.
int solve_expanded(cm_plan *p, cm_plan *pe, int F, const double *rho, double *src, double *res, cudaStream_t s, int l1, int hole1,
                   int l1b, int hole1b)
{
    const size_t n3 = (size_t)p->N * p->N * p->N;
    const unsigned g = (unsigned)((n3 + 255) / 256);
    k_level_density<<<g, 256, 0, s>>>(p->N, hole1, l1, p->L, rho, p->rc, src);          // rho-bar of grid l1 (optionally holed)
    if (l1b >= 0) k_level_density<<<g, 256, 0, s>>>(p->N, hole1b, l1b, p->L, rho, p->rc, src + n3);
    return cm_dispatch_expanded(pe, F, src, l1b >= 0 ? src + n3 : nullptr, res, l1b >= 0 ? res + n3 : nullptr, s, /*attrs_only=*/false);
}

int direct_sum_impl(cm_plan *p, const double *rho_src, int src_level, int dst_level, double *phi_dst, cudaStream_t s);

// depth 2: Eq. B.1-B.2 (pairs); depth 3: Eq. B.3-B.6 (triplets), the quadrupled grid by FFT or by Eq. B.7
// everything the modified method allocates (expanded-grid plans with their K-hat, compact buffers): idempotent, all or
// nothing; runs before any capture
int modified_prepare(cm_plan *p, int depth, int qdp_direct)
{
    const size_t n3 = (size_t)p->N * p->N * p->N;
    int rc = CM_OK;
    if (p->L > 1 && (rc = ensure_expanded(p, 2, &p->dbl, &p->rho2, &p->phi2)) != CM_OK) return rc;
    const bool triple = depth == 3 && p->L > 2;
    if (triple && !qdp_direct && (rc = ensure_expanded(p, 4, &p->qdp, &p->rho4, &p->phi4)) != CM_OK) return rc;
    if (triple && qdp_direct && !p->tmp3 && (rc = dev_alloc(p, &p->tmp3, 2 * n3)) != CM_OK) return rc;
    return CM_OK;
}

int modified_impl(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int depth, int qdp_direct)
{
    const int N = p->N, L = p->L;
    const size_t n3 = (size_t)N * N * N;
    const unsigned gn = (unsigned)((n3 + 255) / 256);
    const bool triple = depth == 3 && L > 2;
    // the original solve, keeping H_n = Phi_hole^n + ext_n on every cell; the finest level's Phi is final (B.2 / B.6)
    int rc = enqueue_solve(p, rho, phi, s, nullptr, /*hole_all=*/1);
    if (rc != CM_OK) return rc;
    // doubled grids: Phi(Omega^n) = H_n + reduce(Phi_dbl^{n+1}), two pairs per complex solve; in the triplet scheme the
    // doubled grid has a central hole (grid n+2's mass comes through the quadrupled grid) except for the last pair (B.5)
    for (int n = 0; n + 1 < L; n += 2) {
        const bool two = n + 2 < L;
        const int h0 = triple && n < L - 2, h1 = triple && n + 1 < L - 2;
        rc = solve_expanded(p, p->dbl, 2, rho, p->rho2, p->phi2, s, n + 1, h0, two ? n + 2 : -1, h1);
        if (rc != CM_OK) return rc;
        for (int q = 0; q < (two ? 2 : 1); ++q) {
            const double dxf = p->dx0 * std::exp2(-(double)(n + q + 1));
            k_add_scaled<<<gn, 256, 0, s>>>(n3, p->hole + (n + q) * n3, p->phi2 + q * n3, p->G * dxf * dxf / 8.0, phi + (n + q) * n3);
        }
    }
    // quadrupled grids (B.3): + reduce(Phi_qdp^{n+2}) for n < L-2, by the same convolution or by direct summation (B.7)
    if (triple) {
        for (int n = 0; n + 2 < L; n += (qdp_direct ? 1 : 2)) {
            if (qdp_direct) {
                k_level_density<<<gn, 256, 0, s>>>(N, 0, n + 2, L, rho, p->rc, p->tmp3);           // rho-bar of grid n+2
                rc = direct_sum_impl(p, p->tmp3, n + 2, n, p->tmp3 + n3, s);
                if (rc != CM_OK) return rc;
                k_add_scaled<<<gn, 256, 0, s>>>(n3, phi + n * n3, p->tmp3 + n3, 1.0, phi + n * n3);
            } else {
                const bool two = n + 3 < L;
                rc = solve_expanded(p, p->qdp, 4, rho, p->rho4, p->phi4, s, n + 2, 0, two ? n + 3 : -1, 0);
                if (rc != CM_OK) return rc;
                for (int q = 0; q < (two ? 2 : 1); ++q) {
                    const double dxf = p->dx0 * std::exp2(-(double)(n + q + 2));
                    k_add_scaled<<<gn, 256, 0, s>>>(n3, phi + (n + q) * n3, p->phi4 + q * n3, p->G * dxf * dxf / 64.0, phi + (n + q) * n3);
                }
            }
        }
    }
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

int enqueue_mode(cm_plan *p, const double *rho, double *phi, cudaStream_t s, int mode)
{
    switch (mode) {
        case 0: return enqueue_solve(p, rho, phi, s);
        case 1: return modified_impl(p, rho, phi, s, 2, 0);
        case 2: return modified_impl(p, rho, phi, s, 3, 0);
        case 3: return modified_impl(p, rho, phi, s, 3, 1);
    }
    return CM_EINVAL;
}

int check_modified_args(cm_plan *p, const double *rho, double *phi)
{
    if (!p || !rho || !phi) return CM_EINVAL;
    if (((uintptr_t)rho & 15) || ((uintptr_t)phi & 15)) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    const size_t tot = (size_t)p->L * p->N * p->N * p->N;
    if ((rho <= phi && phi < rho + tot) || (phi <= rho && rho < phi + tot)) return CM_EINVAL;
    return CM_OK;
}

}  // namespace

extern "C" {

int cm_potential_modified(cm_plan *p, const double *rho, double *phi, void *stream)
{
    const int rc = check_modified_args(p, rho, phi);
    if (rc != CM_OK) return rc;
    if (p->N > 256) return CM_EINVAL;                      // the doubled grid must be a supported size (2N <= 512)
    const int rp = modified_prepare(p, 2, 0);
    if (rp != CM_OK) return rp;
    return run_graphed(p, rho, phi, (cudaStream_t)stream, 1);
}

int cm_potential_modified_triplets(cm_plan *p, const double *rho, double *phi, int qdp_direct, void *stream)
{
    const int rc = check_modified_args(p, rho, phi);
    if (rc != CM_OK) return rc;
    if (p->N > 256 || (!qdp_direct && p->N > 128)) return CM_EINVAL;   // 2N (and 4N) must be supported sizes (<= 512)
    const int rp = modified_prepare(p, 3, qdp_direct ? 1 : 0);
    if (rp != CM_OK) return rp;
    return run_graphed(p, rho, phi, (cudaStream_t)stream, qdp_direct ? 3 : 2);
}

int cm_plan_prepare_modified(cm_plan *p, int depth, int qdp_direct)
{
    if (!p || (depth != 2 && depth != 3)) return CM_EINVAL;
    if (!p->green_ready) return CM_ENOTREADY;
    if (p->N > 256 || (depth == 3 && !qdp_direct && p->N > 128)) return CM_EINVAL;
    return modified_prepare(p, depth, qdp_direct ? 1 : 0);
}

int cm_direct_sum(cm_plan *p, const double *rho_levels, int src_level, int dst_level, double *phi_dst, void *stream)
{
    if (!p || !rho_levels || !phi_dst) return CM_EINVAL;
    if (dst_level < 0 || src_level <= dst_level || src_level >= p->L) return CM_EINVAL;
    const size_t n3 = (size_t)p->N * p->N * p->N;
    return direct_sum_impl(p, rho_levels + (size_t)src_level * n3, src_level, dst_level, phi_dst, (cudaStream_t)stream);
}

}  // extern "C"

namespace {
int direct_sum_impl(cm_plan *p, const double *rho_src, int src_level, int dst_level, double *phi_dst, cudaStream_t s)
{
    const size_t n3 = (size_t)p->N * p->N * p->N;
    const double dxs = p->dx0 * std::exp2(-(double)src_level), dxd = p->dx0 * std::exp2(-(double)dst_level);
    // enough source chunks for ~8 CTAs per SM; the partial sums live in W1 (free outside a solve: 4 N^3 doubles per level)
    const unsigned tb = (unsigned)((n3 + 255) / 256);
    int chunks = (8 * p->num_sms + (int)tb - 1) / (int)tb;
    if (chunks < 1) chunks = 1;
    if (chunks > 16) chunks = 16;
    if (chunks > 4 * p->L) chunks = 4 * p->L;          // W1 holds 4 L N^3 doubles
    double *part = reinterpret_cast<double *>(p->W1);
    k_direct_sum<<<dim3(tb, chunks), 256, 0, s>>>(p->N, dxs, dxd, rho_src, part);
    k_direct_reduce<<<tb, 256, 0, s>>>(n3, chunks, p->G, part, phi_dst);
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}
}  // namespace

extern "C" {

int cm_acceleration(cm_plan *p, const double *phi, double *g, void *stream)
{
    if (!p || !phi || !g) return CM_EINVAL;
    if (((uintptr_t)phi & 15) || ((uintptr_t)g & 15)) return CM_EINVAL;
    const size_t n3 = (size_t)p->N * p->N * p->N, tot = (size_t)p->L * n3, h3 = n3 / 8;
    if ((phi <= g && g < phi + tot) || (g <= phi && phi < g + 3 * tot)) return CM_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (p->L > 1) {
        const size_t cnt = (size_t)(p->L - 1) * h3;
        k_child_mean<<<(unsigned)((cnt + 255) / 256), 256, 0, s>>>(p->N, p->L, phi, p->pbar);
    }
    {
        // a CTA is a TX x TY tile of cell pairs marching ZCH planes; all three must divide the grid (any N % 4 == 0)
        auto divisor_le = [](int n, int cap) {
            int d = cap < n ? cap : n;
            while (n % d) --d;
            return d;
        };
        const int N = p->N, TX = divisor_le(N / 2, 32), TY = divisor_le(N, 256 / TX);
        const int ZCH = divisor_le(N, N >= 256 ? 16 : (N >= 128 ? 8 : (N >= 64 ? 4 : 2)));   // planes a thread marches: enough CTAs at small N
        const unsigned grid = (unsigned)((size_t)p->L * (N / ZCH) * (N / TY) * ((N / 2) / TX));
        k_accel<<<grid, TX * TY, 0, s>>>(N, p->L, TX, TY, ZCH, p->dx0, phi, p->pbar, g);
    }
    CM_CUDA(p, cudaGetLastError());
    return CM_OK;
}

int cm_plan_destroy(cm_plan *p)
{
    if (!p) return CM_OK;
    destroy_graphs(p);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (auto e : p->ev_level)
        if (e) cudaEventDestroy(e);
    cudaFree(p->W1);
    cudaFree(p->W2);
    cudaFree(p->Khat);
    cudaFree(p->rc);
    cudaFree(p->hole);
    cudaFree(p->pbar);
    cudaFree(p->rho2);
    cudaFree(p->phi2);
    if (p->dbl) cm_plan_destroy(p->dbl);
    if (p->qdp) cm_plan_destroy(p->qdp);
    cudaFree(p->rho4);
    cudaFree(p->phi4);
    cudaFree(p->tmp3);
    cudaFree(p->tw);
    cudaFree(p->decE);
    cudaFree(p->stage_rho);
    cudaFree(p->stage_phi);
    delete p;
    return CM_OK;
}

int cm_plan_set_G(cm_plan *p, double G)
{
    if (!p || !std::isfinite(G)) return CM_EINVAL;
    if (G != p->G) destroy_graphs(p);  // the scale is baked into the captured kernel arguments
    p->G = G;
    return CM_OK;
}

size_t cm_plan_workspace_bytes(const cm_plan *p) { return p ? p->bytes : 0; }

int cm_plan_kernel_launches(const cm_plan *p) { return p ? p->kernels_per_solve : 0; }

int cm_debug_copy(cm_plan *p, int which, double *dst, size_t n_doubles, void *stream)
{
    if (!p || !dst) return CM_EINVAL;
    const size_t N = p->N, n3 = N * N * N, L = p->L;
    const double *src = nullptr;
    size_t cnt = 0;
    switch (which) {
        case CM_BUF_RESTRICTED: src = p->rc; cnt = (L - 1) * (n3 / 8); break;
        case CM_BUF_HOLE: src = p->hole; cnt = L * n3; break;
        case CM_BUF_KHAT:
            if (n_doubles != 8 * (size_t)p->Nf * p->Nf * p->Nf) return CM_EINVAL;   // K-hat is that of the transform size
            k_khat_export<<<1024, 256, 0, (cudaStream_t)stream>>>(p->Khat, dst, p->Nf);
            CM_CUDA(p, cudaGetLastError());
            return CM_OK;
        default: return CM_EINVAL;
    }
    if (cnt != n_doubles) return CM_EINVAL;
    if (cnt == 0) return CM_OK;
    CM_CUDA(p, cudaMemcpyAsync(dst, src, cnt * sizeof(double), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return CM_OK;
}

int cm_slot_to_freq(int N, int slot)
{
    if (N < 16 || slot < 0 || slot >= 2 * N) return CM_EINVAL;
    return cmfft::slot_to_freq(slot, N);
}

const char *cm_error_string(int code)
{
    switch (code) {
        case CM_OK: return "ok";
        case CM_EINVAL: return "invalid argument";
        case CM_ENOMEM: return "out of memory";
        case CM_ECUDA: return "CUDA error";
        case CM_ENOTREADY: return "cm_green_precompute has not been called";
        default: return "unknown error";
    }
}

const char *cm_last_cuda_error(const cm_plan *p) { return p ? p->err : ""; }

}  // extern "C"
