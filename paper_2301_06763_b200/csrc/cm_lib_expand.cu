// cm_lib_expand.cu — the pruned / decimated passes of the modified method's expanded grids (cm_expand.cuh) as a translation
// unit of their own: 9 (T, F) instantiations of 5 kernels, compiled beside cm_lib.cu.
#include "cm_plan.h"
#include "cm_zconv.cuh"
#include "cm_expand.cuh"

namespace {

using namespace cmk;

// The five passes of an expanded-grid solve (cm_expand.cuh) on the single-level plan pe of size N' = 16 T = F Nc:
// forward passes pruned to the central Nc^3 block, inverse passes decimated by F.  src_re / src_im: compact Nc^3
// densities (src_im optional: the second real field); out_re / out_im: minus the block SUMS of their potentials.
template <int T, int F> int expanded_passes(cm_plan *pe, const double *src_re, const double *src_im, double *out_re, double *out_im,
                                            cudaStream_t s, bool attrs_only)
{
    constexpr int N = 16 * T, NN = 2 * N, ROWS = kThreads / T, PEN = batch_pencils<T>(), BT = batch_threads<T>();
    static bool attrs = false;      // per instantiation; the attribute is per function, not per plan
    if (!attrs) {
        CM_CUDA(pe, cudaFuncSetAttribute(k_x_fwd_blk<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
        CM_CUDA(pe, cudaFuncSetAttribute(k_y_fwd_blk<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(pe, cudaFuncSetAttribute(k_z_conv_dec<T, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZDecCfg<T>::SMEM));
        CM_CUDA(pe, cudaFuncSetAttribute(k_y_inv_dec<T, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_batch<T>()));
        CM_CUDA(pe, cudaFuncSetAttribute(k_x_inv_dec<T, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row<T>()));
        attrs = true;
    }
    if (attrs_only) return CM_OK;
    // the expanded grid has pe->N = F Nc cells per axis (transformed at N = 16 T >= pe->N); the block sits in its middle
    const int Nc = pe->N / F, c0 = (pe->N - Nc) / 2;
    const unsigned gr = (unsigned)(((size_t)Nc * Nc + ROWS - 1) / ROWS);
    const int ya = pe->num_sms;   // y passes: L2 prefetch distance in CTAs (measured 74 ... 148 equal, 296 no gain)
    k_x_fwd_blk<T><<<gr, kThreads, smem_row<T>(), s>>>(src_re, src_im, pe->W1, pe->tw, Nc, c0);
    k_y_fwd_blk<T><<<(unsigned)((size_t)Nc * NN / PEN), BT, smem_batch<T>(), s>>>(pe->W1, pe->W2, pe->tw, Nc, c0, ya);
    k_z_conv_dec<T, F><<<(unsigned)((size_t)(N + 1) * (NN / PEN)), BT, ZDecCfg<T>::SMEM, s>>>(pe->Khat, pe->W2, pe->tw, pe->decE, c0, c0 + Nc, 0, 1, 0,
                                                                                                        /*ahead=*/(T == 32 ? 1 : 2) * pe->num_sms);
    k_y_inv_dec<T, F><<<(unsigned)((size_t)Nc * NN / PEN), BT, smem_batch<T>(), s>>>(pe->W2, pe->W1, pe->tw, pe->decE, Nc, ya);
    k_x_inv_dec<T, F><<<gr, kThreads, smem_row<T>(), s>>>(pe->W1, out_re, out_im, pe->tw, pe->decE, -1.0, Nc);
    CM_CUDA(pe, cudaGetLastError());
    return CM_OK;
}

}  // namespace

int cm_dispatch_expanded(cm_plan *pe, int F, const double *src_re, const double *src_im, double *out_re, double *out_im, cudaStream_t s,
                         bool attrs_only)
{
#define CM_EXP(TT, FF) \
    if (pe->T == TT && F == FF) return expanded_passes<TT, FF>(pe, src_re, src_im, out_re, out_im, s, attrs_only);
    CM_EXP(2, 2) CM_EXP(4, 2) CM_EXP(8, 2) CM_EXP(16, 2) CM_EXP(32, 2)
    CM_EXP(4, 4) CM_EXP(8, 4) CM_EXP(16, 4) CM_EXP(32, 4)
#undef CM_EXP
    return CM_EINVAL;
}
