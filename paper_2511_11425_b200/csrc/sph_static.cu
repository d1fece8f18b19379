// sph_static.cu -- sph_timestep_static: the time-step criteria of PAPER.md:263-268 (Eq. 26)
// for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc).  No context, no cudaMalloc / cudaFree, no allocating library call:
// the block minima of the reduction live in a file-scope __device__ array of fixed size that
// every GPU which loads the library holds until exit (SPH_STATIC_SCRATCH_BYTES = 16 KB).
//
// Same arithmetic as k_timestep / k_min_final of sph_misc.cu (FP64 on the FP32 inputs, rounded
// once; a minimum does not depend on the order it is taken in), different blocking: one block
// per SPH_STATIC_BLOCK_N particles and one partial minimum per block, hence the limit
// n <= SPH_STATIC_MAX_N = 4096 x 4096.
//
// The scratch is shared by every call on a device and keeps the last call's contents.  Nothing
// in it has to start at zero: a call writes its nblk partials before its second kernel reads
// exactly those.  Two calls that overlap on one GPU (different streams) race on it.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>
#include "../../include/sph.h"

namespace {

constexpr int      ST_TPB      = 256;
constexpr int      ST_PER_THR  = 16;
constexpr int      ST_BLOCK_N  = ST_TPB * ST_PER_THR;                 // 4096 particles per block
constexpr int      ST_MAX_PART = SPH_STATIC_SCRATCH_BYTES / 4;        // 4096 partial minima
constexpr int      ST_MAX_DEV  = 64;
static_assert((long long)ST_BLOCK_N * ST_MAX_PART == SPH_STATIC_MAX_N, "sph.h states the limit");

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: host
// code takes the address with cudaGetSymbolAddress (static_scratch below); device code could
// name the array directly, the kernels take the pointer so that they read like the others.
static __device__ __align__(256) unsigned char g_static_scratch[SPH_STATIC_SCRATCH_BYTES];

thread_local char g_err[256] = "";
float*            g_addr[ST_MAX_DEV];   // per device: the array's device address (0 = not asked yet)

__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float block_min(float v) {   // result in thread 0
    __shared__ float sh[32];
    v = warp_min(v);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : __int_as_float(0x7f800000);
        v = warp_min(v);
    }
    return v;
}

// dt_a = eta_a sqrt(2h/|a|) (no limit when a = 0), dt_CFL = eta_C h / ((1 + 0.6 alpha) c +
// 0.6 beta |mu_min|), dt_i = min of the two; part[block] = min over the block's particles.
__global__ __launch_bounds__(ST_TPB) void k_timestep_static(
    int64_t n, const float* __restrict__ h, const float* __restrict__ cs,
    const float* __restrict__ ax, const float* __restrict__ ay, const float* __restrict__ az,
    const float* __restrict__ mu_min, float eta_cfl, float eta_acc, float alpha, float beta,
    float* dt_i, float* part) {
    float         best = __int_as_float(0x7f800000);
    const int64_t base = (int64_t)blockIdx.x * ST_BLOCK_N + threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < ST_PER_THR; ++k) {
        const int64_t i = base + (int64_t)k * ST_TPB;
        if (i >= n) break;
        const double hi = h[i], a2 = (double)ax[i] * ax[i] + (double)ay[i] * ay[i] +
                                     (double)az[i] * az[i];
        const double sig = (1.0 + 0.6 * (double)alpha) * (double)cs[i] +
                           0.6 * (double)beta * fabs((double)mu_min[i]);
        double dt = (double)eta_cfl * hi / sig;
        if (a2 > 0.0) dt = fmin(dt, (double)eta_acc * sqrt(2.0 * hi / sqrt(a2)));
        const float f = (float)dt;
        dt_i[i] = f;
        best = fminf(best, f);
    }
    best = block_min(best);
    if (threadIdx.x == 0) part[blockIdx.x] = best;
}

__global__ __launch_bounds__(ST_TPB) void k_min_static(int nparts, const float* __restrict__ part,
                                                      float* out) {
    float v = __int_as_float(0x7f800000);
    for (int i = threadIdx.x; i < nparts; i += blockDim.x) v = fminf(v, part[i]);
    v = block_min(v);
    if (threadIdx.x == 0) *out = v;
}

// Device address of the scratch on the CURRENT device; asked once per device.
int static_scratch(float** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        snprintf(g_err, sizeof(g_err), "sph_timestep_static: cudaGetDevice: %s", cudaGetErrorString(e));
        return SPH_ECUDA;
    }
    if (dev < 0 || dev >= ST_MAX_DEV) {
        snprintf(g_err, sizeof(g_err), "sph_timestep_static: device %d outside [0, %d)", dev, ST_MAX_DEV);
        return SPH_EINVAL;
    }
    float* p = __atomic_load_n(&g_addr[dev], __ATOMIC_ACQUIRE);
    if (p == nullptr) {
        void* q = nullptr;
        e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess || q == nullptr) {
            snprintf(g_err, sizeof(g_err), "sph_timestep_static: cudaGetSymbolAddress: %s",
                     cudaGetErrorString(e));
            return SPH_ECUDA;
        }
        p = (float*)q;   // every thread that gets here is given the same address
        __atomic_store_n(&g_addr[dev], p, __ATOMIC_RELEASE);
    }
    *out = p;
    return SPH_OK;
}

}  // namespace

extern "C" int sph_timestep_static(void* cuda_stream, int64_t n, float eta_cfl, float eta_acc,
                                   float av_alpha, float av_beta, const float* h, const float* c,
                                   const float* ax, const float* ay, const float* az,
                                   const float* mu_min, float* dt_i, float* dt_min_device) {
    if (!h || !c || !ax || !ay || !az || !mu_min || !dt_i || !dt_min_device) {
        snprintf(g_err, sizeof(g_err), "sph_timestep_static: null pointer");
        return SPH_EINVAL;
    }
    if (n <= 0 || n > (int64_t)SPH_STATIC_MAX_N) {
        snprintf(g_err, sizeof(g_err),
                 "sph_timestep_static: n = %lld outside [1, %lld] (the static scratch holds %d block minima "
                 "of %d particles each); use sph_timestep",
                 (long long)n, (long long)SPH_STATIC_MAX_N, ST_MAX_PART, ST_BLOCK_N);
        return SPH_EINVAL;
    }
    if (!(eta_cfl > 0.0f) || !(eta_acc > 0.0f) || !(av_alpha >= 0.0f) || !(av_beta >= 0.0f)) {
        snprintf(g_err, sizeof(g_err), "sph_timestep_static: eta_cfl, eta_acc must be > 0, av_alpha, av_beta >= 0");
        return SPH_EINVAL;
    }
    float* part = nullptr;
    const int rc = static_scratch(&part);
    if (rc != SPH_OK) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int nblk = (int)((n + ST_BLOCK_N - 1) / ST_BLOCK_N);
    k_timestep_static<<<nblk, ST_TPB, 0, s>>>(n, h, c, ax, ay, az, mu_min, eta_cfl, eta_acc, av_alpha,
                                              av_beta, dt_i, part);
    k_min_static<<<1, ST_TPB, 0, s>>>(nblk, part, dt_min_device);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_err, sizeof(g_err), "sph_timestep_static: launch: %s", cudaGetErrorString(e));
        return SPH_ECUDA;
    }
    return SPH_OK;
}

extern "C" const char* sph_static_last_error(void) { return g_err; }
