// cm_static.cu — cm_direct_sum_static: the direct fine -> coarse summation of Eq. B.7 for callers
// that must not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// cm_direct_sum keeps its per-chunk partial sums in the plan's workspace, and a plan is cudaMalloc'ed.  This variant
// needs no plan: the partial sums live in a file-scope __device__ array of fixed size (CM_STATIC_SCRATCH_BYTES, held
// by every GPU that loads libcm until the process exits), so the call is two kernel launches and nothing else — no
// cudaMalloc, cudaFree, or allocating library routine.  Same arithmetic as k_direct_sum / k_direct_reduce
// (cm_kernels.cuh), restated here so that this translation unit stands alone; the existing path is untouched.
//
// The array's name in HOST code is a host-side stand-in, not a device address: its device address is looked up once
// per device with cudaGetSymbolAddress (device current, return code checked) and that pointer is what the kernels get.
//
// Every call on a device shares the one array.  Nothing in it has to start at zero: chunk c of a call writes
// part[c][t] for every target t < N^3 before the reduce kernel of the same call (same stream, after it) reads exactly
// those entries, so what an earlier call left behind is never read.  Two calls that overlap on the GPU (different
// streams, or graphs replayed side by side) race on the array: serialise them.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/cm.h"

namespace {

constexpr int kMaxN = CM_STATIC_MAX_N;          // 32: the size up to which the paper uses Eq. B.7 (L461)
constexpr int kMaxChunks = 16;                  // source chunks (as cm_direct_sum)
constexpr size_t kMaxN3 = (size_t)kMaxN * kMaxN * kMaxN;
static_assert(kMaxChunks * kMaxN3 * sizeof(double) == CM_STATIC_SCRATCH_BYTES, "cm.h states the size of the scratch array");

// [chunk][target] partial sums; 4 MiB per GPU
static __device__ __align__(256) double g_part[kMaxChunks * kMaxN3];

constexpr int kMaxDevices = 64;
struct DeviceSetup {
    double *part = nullptr;   // device address of g_part on this device
    int num_sms = 0;
};
DeviceSetup g_dev[kMaxDevices];
std::mutex g_mu;
thread_local char t_err[256] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

// one thread per target cell, sources through shared memory in tiles of 256 as (x, y, z, M); chunk blockIdx.y sums the
// sources [c, c + 1) n3 / gridDim.y into part[c][t]
__global__ void __launch_bounds__(256) k_direct_sum_static(int N, double dxs, double dxd, const double *__restrict__ rho_src,
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
            src[threadIdx.x] = make_double4(0.0, 0.0, 0.0, 0.0);   // zero mass at the origin: never at a target's centre
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

// chunks added in a fixed order: deterministic
__global__ void k_direct_reduce_static(size_t n3, int chunks, double G, const double *__restrict__ part, double *__restrict__ phi_dst)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n3) return;
    double acc = 0.0;
    for (int c = 0; c < chunks; ++c) acc += part[(size_t)c * n3 + t];
    phi_dst[t] = -G * acc;
}

// once per device, with that device current
int setup_current_device(DeviceSetup **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(CM_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices)
        return fail(CM_EINVAL, "cm_direct_sum_static: device ordinal %d is beyond the %d this entry point keeps set-up for", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_mu);
    DeviceSetup &d = g_dev[dev];
    if (!d.part) {
        double *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_part);
        if (e != cudaSuccess || !ptr) {
            return fail(CM_ECUDA, "cudaGetSymbolAddress(g_part) on device %d: %s", dev, cudaGetErrorString(e));
        }
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || sms <= 0) {
            return fail(CM_ECUDA, "cudaDeviceGetAttribute(SM count) on device %d: %s", dev, cudaGetErrorString(e));
        }
        d.num_sms = sms;
        d.part = ptr;
    }
    *out = &d;
    return CM_OK;
}

}  // namespace

extern "C" {

int cm_direct_sum_static_setup(void)
{
    DeviceSetup *d = nullptr;
    return setup_current_device(&d);
}

int cm_direct_sum_static(int N, double dx_src, double dx_dst, double G, const double *rho_src, double *phi_dst, void *stream)
{
    t_err[0] = 0;
    if (!rho_src || !phi_dst) return fail(CM_EINVAL, "cm_direct_sum_static: rho_src and phi_dst must be device pointers, not NULL");
    if (N < 1) return fail(CM_EINVAL, "cm_direct_sum_static: N = %d must be at least 1", N);
    if (N > kMaxN)
        return fail(CM_EINVAL, "cm_direct_sum_static: N = %d exceeds CM_STATIC_MAX_N = %d (the static scratch array holds %d x %d^3 "
                               "partial sums); use cm_direct_sum with a plan for larger grids", N, kMaxN, kMaxChunks, kMaxN);
    if (!(dx_src > 0.0) || !(dx_dst > 0.0) || !std::isfinite(dx_src) || !std::isfinite(dx_dst))
        return fail(CM_EINVAL, "cm_direct_sum_static: dx_src and dx_dst must be positive and finite");
    DeviceSetup *d = nullptr;
    const int rc = setup_current_device(&d);
    if (rc != CM_OK) return rc;
    const size_t n3 = (size_t)N * N * N;
    const unsigned tb = (unsigned)((n3 + 255) / 256);
    int chunks = (8 * d->num_sms + (int)tb - 1) / (int)tb;      // enough source chunks for ~8 CTAs per SM
    if (chunks < 1) chunks = 1;
    if (chunks > kMaxChunks) chunks = kMaxChunks;
    cudaStream_t s = (cudaStream_t)stream;
    k_direct_sum_static<<<dim3(tb, chunks), 256, 0, s>>>(N, dx_src, dx_dst, rho_src, d->part);
    k_direct_reduce_static<<<tb, 256, 0, s>>>(n3, chunks, G, d->part, phi_dst);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(CM_ECUDA, "cm_direct_sum_static: kernel launch: %s", cudaGetErrorString(e));
    return CM_OK;
}

const char *cm_static_last_error(void) { return t_err; }

}  // extern "C"
