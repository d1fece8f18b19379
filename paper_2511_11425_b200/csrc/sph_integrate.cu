// sph_integrate.cu -- time integration with a global step, PAPER.md:227-261 (Section 2.3.6),
// Eqs. (19)-(25): the kick-drift-kick leap-frog with predicted v, u for the force pass.
// Element-wise, HBM-bound (one read-modify-write pass per call).  The step length is read
// from device memory (the value sph_timestep wrote), scaled by a host factor, so a whole
// step can be enqueued without a host round trip.
#include <cstdio>
#include "sph_internal.cuh"

namespace {

// out = base + (scale * *dt) * rate  for up to four arrays at once (v_x, v_y, v_z, u)
struct Axpy4 {
    const float* base[4];
    const float* rate[4];
    float*       out[4];
    int          count;
};

__global__ void k_axpy4(int64_t n, Axpy4 a, const float* __restrict__ dt, float scale) {
    const float s = scale * __ldg(dt);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k < a.count) a.out[k][i] = fmaf(s, a.rate[k][i], a.base[k][i]);
    }
}

// Eq. (25): x += dt v, wrapped into [lo, lo + len) on periodic axes
__global__ void k_drift(int64_t n, sph_box box, float* x, float* y, float* z,
                        const float* __restrict__ vx, const float* __restrict__ vy,
                        const float* __restrict__ vz, const float* __restrict__ dt, float scale) {
    const float s = scale * __ldg(dt);
    float* const       xs[3] = {x, y, z};
    const float* const vs[3] = {vx, vy, vz};
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            float xn = fmaf(s, vs[d][i], xs[d][i]);
            if (box.periodic[d]) {
                xn -= box.len[d] * floorf((xn - box.lo[d]) / box.len[d]);
                if (!(xn < box.lo[d] + box.len[d])) xn = box.lo[d];
                if (xn < box.lo[d]) xn = box.lo[d];
            }
            xs[d][i] = xn;
        }
    }
}

// PAPER.md:197 for the ideal gas: u (rho_new / rho_old)^(gamma-1); the ratio is near 1, so
// exp2(gm1 log2(ratio)) in FP32 carries about 1e-7 relative
__global__ void k_isentropic(int64_t n, float gm1, const float* __restrict__ rho_old,
                             const float* __restrict__ rho_new, float* u) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        u[i] *= powf(rho_new[i] / rho_old[i], gm1);
}

int launch_axpy(sph_ctx* c, int64_t n, const Axpy4& a, const float* dt, float scale) {
    int nblk = (int)((n + 255) / 256);
    if (nblk > c->sm_count * 16) nblk = c->sm_count * 16;
    k_axpy4<<<nblk, 256, 0, c->stream>>>(n, a, dt, scale);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace

extern "C" int sph_predict(sph_ctx* c, int64_t n, const float* dt_device, float dt_scale,
                           const float* vx, const float* vy, const float* vz, const float* u,
                           const float* ax, const float* ay, const float* az, const float* dudt,
                           float* vx_pred, float* vy_pred, float* vz_pred, float* u_pred) {
    if (!c || n <= 0 || !dt_device || !vx || !vy || !vz || !u || !ax || !ay || !az || !dudt ||
        !vx_pred || !vy_pred || !vz_pred || !u_pred)
        return SPH_EINVAL;
    Axpy4 a{{vx, vy, vz, u}, {ax, ay, az, dudt}, {vx_pred, vy_pred, vz_pred, u_pred}, 4};
    return launch_axpy(c, n, a, dt_device, 0.5f * dt_scale);   // Eqs. (19), (20)
}

extern "C" int sph_kick(sph_ctx* c, int64_t n, const float* dt_device, float dt_scale, float* vx,
                        float* vy, float* vz, float* u, const float* ax, const float* ay,
                        const float* az, const float* dudt) {
    if (!c || n <= 0 || !dt_device || !vx || !vy || !vz || !u || !ax || !ay || !az || !dudt)
        return SPH_EINVAL;
    Axpy4 a{{vx, vy, vz, u}, {ax, ay, az, dudt}, {vx, vy, vz, u}, 4};
    return launch_axpy(c, n, a, dt_device, 0.5f * dt_scale);   // Eqs. (21)-(24)
}

extern "C" int sph_drift(sph_ctx* c, int64_t n, const float* dt_device, float dt_scale, float* x,
                         float* y, float* z, const float* vx, const float* vy, const float* vz) {
    if (!c || n <= 0 || !dt_device || !x || !y || !z || !vx || !vy || !vz) return SPH_EINVAL;
    int nblk = (int)((n + 255) / 256);
    if (nblk > c->sm_count * 16) nblk = c->sm_count * 16;
    k_drift<<<nblk, 256, 0, c->stream>>>(n, c->box, x, y, z, vx, vy, vz, dt_device, dt_scale);
    SPH_CUDA_CHECK(c, cudaGetLastError());   // Eq. (25)
    return SPH_OK;
}

extern "C" int sph_isentropic_u(sph_ctx* c, int64_t n, const float* rho_old, const float* rho_new,
                                float* u_inout) {
    if (!c || n <= 0 || !rho_old || !rho_new || !u_inout) return SPH_EINVAL;
    int nblk = (int)((n + 255) / 256);
    if (nblk > c->sm_count * 16) nblk = c->sm_count * 16;
    k_isentropic<<<nblk, 256, 0, c->stream>>>(n, c->par.gamma - 1.0f, rho_old, rho_new, u_inout);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
