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

// ---- block time steps (reading R32) ----------------
// Eqs. (19)-(20) for every particle: tau_i = (s - tnext_i) delta + hk_i
__global__ void k_block_predict(int64_t n, Axpy4 a, int32_t s, float delta,
                                const int32_t* __restrict__ tnext, const float* __restrict__ hk) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        const float tau = fmaf((float)(s - tnext[i]), delta, hk[i]);
#pragma unroll
        for (int k = 0; k < 4; ++k) a.out[k][i] = fmaf(tau, a.rate[k][i], a.base[k][i]);
    }
}

__global__ void k_block_active(int64_t n, int32_t s, const int32_t* __restrict__ tnext,
                               uint8_t* active) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        active[i] = tnext[i] == s;
}

// closing kick (Eqs. 21-22), rung change, opening kick (Eqs. 23-24) of the particles whose
// step ends at substep s
__global__ void k_block_kick(int64_t n, Axpy4 a, int32_t s, int32_t R, int32_t floor_rung,
                             float delta, const int32_t* __restrict__ rung_des, int32_t* rung,
                             int32_t* tnext, float* hk, int32_t open) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        if (tnext[i] != s) continue;
        const float   h0 = hk[i];
        if (!open) {   // closing kick alone: v, u at the time of the substep, nothing pending
#pragma unroll
            for (int k = 0; k < 4; ++k) a.out[k][i] = fmaf(h0, a.rate[k][i], a.base[k][i]);
            hk[i] = 0.0f;
            continue;
        }
        const int32_t r  = min(R, max(rung_des[i], floor_rung));
        const int32_t L  = 1 << (R - r);
        const float   h1 = 0.5f * (float)L * delta;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            a.out[k][i] = fmaf(h1, a.rate[k][i], fmaf(h0, a.rate[k][i], a.base[k][i]));
        hk[i]    = h1;
        tnext[i] = s + L;
        rung[i]  = r;
    }
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

namespace {
int block_grid(const sph_ctx* c, int64_t n) {
    int nblk = (int)((n + 255) / 256);
    return nblk > c->sm_count * 16 ? c->sm_count * 16 : nblk;
}
}  // namespace

extern "C" int sph_block_predict(sph_ctx* c, int64_t n, int32_t substep, float delta,
                                 const int32_t* tnext, const float* hk, const float* vx,
                                 const float* vy, const float* vz, const float* u, const float* ax,
                                 const float* ay, const float* az, const float* dudt, float* vx_pred,
                                 float* vy_pred, float* vz_pred, float* u_pred) {
    if (!c || n <= 0 || substep < 0 || !(delta > 0.0f) || !tnext || !hk || !vx || !vy || !vz || !u ||
        !ax || !ay || !az || !dudt || !vx_pred || !vy_pred || !vz_pred || !u_pred)
        return SPH_EINVAL;
    Axpy4 a{{vx, vy, vz, u}, {ax, ay, az, dudt}, {vx_pred, vy_pred, vz_pred, u_pred}, 4};
    k_block_predict<<<block_grid(c, n), 256, 0, c->stream>>>(n, a, substep, delta, tnext, hk);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_block_active(sph_ctx* c, int64_t n, int32_t substep, const int32_t* tnext,
                                uint8_t* active) {
    if (!c || n <= 0 || substep < 0 || !tnext || !active) return SPH_EINVAL;
    k_block_active<<<block_grid(c, n), 256, 0, c->stream>>>(n, substep, tnext, active);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_block_kick(sph_ctx* c, int64_t n, int32_t substep, int32_t max_rung, float delta,
                              const int32_t* rung_desired, int32_t* rung, int32_t* tnext, float* hk,
                              float* vx, float* vy, float* vz, float* u, const float* ax,
                              const float* ay, const float* az, const float* dudt, int32_t open) {
    if (!c || n <= 0 || substep < 0 || max_rung < 0 || max_rung > 24 || !(delta > 0.0f) ||
        !rung_desired || !rung || !tnext || !hk || !vx || !vy || !vz || !u || !ax || !ay || !az || !dudt)
        return SPH_EINVAL;
    // the lowest rung whose steps begin at this substep
    int32_t fl = 0;
    while (fl < max_rung && (substep & ((1 << (max_rung - fl)) - 1)) != 0) ++fl;
    Axpy4 a{{vx, vy, vz, u}, {ax, ay, az, dudt}, {vx, vy, vz, u}, 4};
    k_block_kick<<<block_grid(c, n), 256, 0, c->stream>>>(n, a, substep, max_rung, fl, delta,
                                                          rung_desired, rung, tnext, hk, open);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
