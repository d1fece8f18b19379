// sph_forces.cu -- steps a7-a9 of DESIGN.md: EOS + per-particle precompute, gather-or-
// scatter neighbour search and the hydro force sweep, PAPER.md:186-219 (Section 2.3.5),
// Eqs. (13)-(18), ideal gas of PAPER.md:111.
//
// One warp per target.  Lanes distance-test 32 consecutive candidates of a row, accepted
// pairs (0 < r < 2 max(h_i,h_j)) go through a 64-entry ring in shared memory
// so that the pair arithmetic always runs with 32 busy lanes.
//
// Pair arithmetic (d = x_i - x_j, r = |d|, q_a = r/h_a, g_a = K_a (1-q_a/2)_+^3 with
// K_a = 5 SIGMA / h_a^5, so that dW/dr(r,h_a) = -g_a r):
//   Eq. 13+17:  a_i     = + sum_j m_j (A_i g_i + A_j g_j + Pi_ij gbar) d
//   Eq. 14+18:  du_i/dt = - sum_j m_j (A_i g_i + Pi_ij gbar / 2) (v_ij . d)
//   Eq. 15-16:  mu = hbar (v_ij.d)/(r^2 + eps hbar^2), Pi = mu (beta mu - alpha cbar)/rhobar
//               for v_ij.d < 0, else 0;   gbar = (g_i + g_j)/2;  A = P/(Omega rho^2).
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int F_WARPS   = 8;
constexpr int F_TPB     = F_WARPS * 32;
constexpr int F_TARGETS = 64;
constexpr int RING      = 64;

struct ForcePar {
    float alpha, beta, eps;
};

struct FWarpSmem {
    uint32_t j[RING];
    float    dx[RING], dy[RING], dz[RING], r2[RING], hj[RING];
    RowRec   rows[SPH_RCAP];
};

// a7: EOS and the per-particle factors, written in sorted order (scattered 16-byte stores)
__global__ void k_force_prep(int64_t n, const int32_t* __restrict__ inv_perm,
                             const float* __restrict__ m,
                             const float* __restrict__ vx, const float* __restrict__ vy,
                             const float* __restrict__ vz, const float* __restrict__ u,
                             const float* __restrict__ rho, const float* __restrict__ h,
                             const float* __restrict__ omega, float gamma, float4* pos_h,
                             float4* vel_m, float4* rcak, float* P, float* cs, SphGrid* g) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float   hi = 0.0f;
    if (i < n) {
        const int p = inv_perm[i];
        hi = h[i];
        const float ri = rho[i], ui = u[i], om = omega[i];
        const float Pi = (gamma - 1.0f) * ri * ui;
        const float ci = sqrtf(gamma * Pi / ri);
        P[i]  = Pi;
        cs[i] = ci;
        float4 a = pos_h[p];
        a.w      = hi;
        pos_h[p] = a;
        vel_m[p] = make_float4(vx[i], vy[i], vz[i], m[i]);
        const float h2 = hi * hi;
        rcak[p] = make_float4(ri, ci, Pi / (om * ri * ri), 5.0f * SPH_SIGMA / (h2 * h2 * hi));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) hi = fmaxf(hi, __shfl_xor_sync(SPH_FULL, hi, o));
    if ((threadIdx.x & 31) == 0 && hi > 0.0f) atomicMax(&g->force_hmax_bits, __float_as_uint(hi));
}

__global__ void k_zero_hmax(SphGrid* g) { g->force_hmax_bits = 0u; }

__global__ __launch_bounds__(F_TPB) void k_forces(int n, const SphGrid* __restrict__ gp,
                                                  const uint32_t* __restrict__ cell_start,
                                                  const float4* __restrict__ pos_h,
                                                  const float4* __restrict__ vel_m,
                                                  const float4* __restrict__ rcak,
                                                  const int32_t* __restrict__ perm, ForcePar par,
                                                  float* ax, float* ay, float* az, float* dudt,
                                                  float* mu_min, unsigned long long* stats) {
    __shared__ FWarpSmem sm_all[F_WARPS];
    __shared__ SphGrid   g;
    __shared__ unsigned long long st_sh[3];
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 3) st_sh[threadIdx.x] = 0ull;
    __syncthreads();

    const int      wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned lt  = (1u << lane) - 1u;
    FWarpSmem&     sm  = sm_all[wid];
    const float    hmax_all = __uint_as_float(g.force_hmax_bits);

    unsigned long long c_tested = 0;
    unsigned c_pairs = 0, c_av = 0;

    for (int t = wid; t < F_TARGETS; t += F_WARPS) {
        const int p = blockIdx.x * F_TARGETS + t;
        if (p >= n) break;
        const float4 pi = pos_h[p];
        const float4 vi = vel_m[p];
        const float4 ri = rcak[p];
        const float  hi = pi.w, ihi = 1.0f / hi;
        const float  rho_i = ri.x, c_i = ri.y, A_i = ri.z, K_i = ri.w;
        // scatter neighbours can be as far as 2 h_j: search with the largest h in use
        const float R = 2.0f * fmaxf(hi, hmax_all) * (1.0f + 1e-5f);
        const float hi2x4 = 4.0f * hi * hi;

        float acx = 0.0f, acy = 0.0f, acz = 0.0f, du = 0.0f, mumin = 0.0f;
        int   head = 0, fill = 0;  // ring state (warp-uniform)

        auto process = [&](int k, bool active) {
            // one pair per lane: ring entry k
            if (active) {
                const uint32_t j  = sm.j[k];
                const float    dx = sm.dx[k], dy = sm.dy[k], dz = sm.dz[k], r2 = sm.r2[k];
                const float    hj = sm.hj[k];
                const float4   vj = __ldg(vel_m + j);
                const float4   rj = __ldg(rcak + j);
                const float r  = sqrtf(r2);
                const float ti = fmaxf(1.0f - 0.5f * r * ihi, 0.0f);
                const float tj = fmaxf(1.0f - 0.5f * __fdividef(r, hj), 0.0f);
                const float gi = K_i * ti * ti * ti;
                const float gj = rj.w * tj * tj * tj;
                const float vdx = vi.x - vj.x, vdy = vi.y - vj.y, vdz = vi.z - vj.z;
                const float vr = vdx * dx + vdy * dy + vdz * dz;   // v_ij . r_ij
                float pig = 0.0f;                                   // Pi_ij * gbar
                if (vr < 0.0f) {
                    const float hb  = 0.5f * (hi + hj);
                    const float mu  = hb * vr / (r2 + par.eps * hb * hb);
                    const float cb  = 0.5f * (c_i + rj.y);
                    const float rb  = 0.5f * (rho_i + rj.x);
                    const float Pij = mu * (par.beta * mu - par.alpha * cb) / rb;
                    pig   = Pij * 0.5f * (gi + gj);
                    mumin = fminf(mumin, mu);
                    ++c_av;
                }
                const float Ag = A_i * gi;
                const float ca = vj.w * (Ag + rj.z * gj + pig);
                acx += ca * dx;
                acy += ca * dy;
                acz += ca * dz;
                du -= vj.w * (Ag + 0.5f * pig) * vr;
            }
        };

        sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, R, sm.rows, lane, [&](const RowRec& rr) {
            for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                const uint32_t j = k0 + lane;
                const bool     v = j < rr.end;
                float4 pj = make_float4(3.0e18f, 3.0e18f, 3.0e18f, 0.0f);
                if (v) pj = __ldg(pos_h + j);
                const float dx = rr.sx - pj.x, dy = rr.sy - pj.y, dz = rr.sz - pj.z;
                const float r2 = dx * dx + dy * dy + dz * dz;
                const float Hm = fmaxf(hi2x4, 4.0f * pj.w * pj.w);
                const bool  acc = v && (r2 < Hm) && (r2 > 0.0f);
                const unsigned mk = __ballot_sync(SPH_FULL, acc);
                if (acc) {
                    const int slot = (head + fill + __popc(mk & lt)) & (RING - 1);
                    sm.j[slot]  = j;
                    sm.dx[slot] = dx;
                    sm.dy[slot] = dy;
                    sm.dz[slot] = dz;
                    sm.r2[slot] = r2;
                    sm.hj[slot] = pj.w;
                }
                fill += __popc(mk);
                c_tested += min(32u, rr.end - k0);
                __syncwarp();
                if (fill >= 32) {
                    process((head + lane) & (RING - 1), true);
                    head = (head + 32) & (RING - 1);
                    fill -= 32;
                    c_pairs += 32;
                    __syncwarp();
                }
            }
        });
        __syncwarp();
        if (fill > 0) {
            process((head + lane) & (RING - 1), lane < fill);
            c_pairs += fill;
        }
        acx = sph_warp_sum(acx);
        acy = sph_warp_sum(acy);
        acz = sph_warp_sum(acz);
        du  = sph_warp_sum(du);
        mumin = sph_warp_min(mumin);
        if (lane == 0) {
            const int i = perm[p];
            ax[i] = acx; ay[i] = acy; az[i] = acz;
            dudt[i]   = du;
            mu_min[i] = mumin;
        }
        __syncwarp();
    }

    c_av = __reduce_add_sync(SPH_FULL, c_av);
    if (lane == 0) {
        atomicAdd(&st_sh[0], c_tested);
        atomicAdd(&st_sh[1], (unsigned long long)c_pairs);
        atomicAdd(&st_sh[2], (unsigned long long)c_av);
    }
    __syncthreads();
    if (threadIdx.x < 3 && st_sh[threadIdx.x] != 0ull)
        atomicAdd(stats + ST_FORCE_TESTED + threadIdx.x, st_sh[threadIdx.x]);
}

}  // namespace

int sph_launch_forces(sph_ctx* c, const float* m, const float* vx, const float* vy,
                      const float* vz, const float* u, const float* rho, const float* h,
                      const float* omega, float* ax, float* ay, float* az, float* dudt,
                      float* mu_min, float* P, float* cs) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    k_zero_hmax<<<1, 1, 0, s>>>(c->grid);
    k_force_prep<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->inv_perm, m, vx, vy, vz, u,
                                                        rho, h, omega, c->par.gamma, c->pos_h,
                                                        c->vel_m, c->rcak, P, cs, c->grid);
    ForcePar par{c->par.av_alpha, c->par.av_beta, c->par.av_eps};
    const int nblk = (int)((n + F_TARGETS - 1) / F_TARGETS);
    k_forces<<<nblk, F_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_h, c->vel_m, c->rcak,
                                    c->perm, par, ax, ay, az, dudt, mu_min, c->stats);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
