// sph_forces.cu -- steps a7-a9 of DESIGN.md: EOS + per-particle precompute, gather-or-
// scatter neighbour search and the hydro force sweep, PAPER.md:186-219 (Section 2.3.5),
// Eqs. (13)-(18), ideal gas of PAPER.md:111.
//
// G = 8 lanes per target, four targets per warp.  Phase 1: the lanes of a group distance-
// test the candidates of the rows in reach (0 < r < 2 max(h_i,h_j), gather and scatter,
// PAPER.md:191) and each lane notes the indices it accepted in a private column of a
// shared-memory list.  Phase 2: every lane works through its own column -- the pair
// arithmetic runs without divergence between accepted and rejected candidates.
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

constexpr int F_G      = 8;
constexpr int F_NT     = 32 / F_G;
constexpr int F_WARPS  = 4;
constexpr int F_TPB    = F_WARPS * 32;
constexpr int F_ROUNDS = 2;
constexpr int F_TARGETS = F_WARPS * F_NT * F_ROUNDS;
constexpr int F_SLOTS  = 26;   // list entries per lane

struct ForcePar {
    float alpha, beta, eps;
};

struct FWarpList {
    uint32_t j[F_SLOTS][32];
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

__global__ __launch_bounds__(F_TPB, SPH_MINB) void k_forces(int n, const SphGrid* __restrict__ gp,
                                                     const uint32_t* __restrict__ cell_start,
                                                     const float4* __restrict__ pos_h,
                                                     const float4* __restrict__ vel_m,
                                                     const float4* __restrict__ rcak,
                                                     const int32_t* __restrict__ perm,
                                                     ForcePar par, float* ax, float* ay, float* az,
                                                     float* dudt, float* mu_min,
                                                     unsigned long long* stats) {
    __shared__ FWarpList lists[F_WARPS];
    __shared__ SphGrid   g;
    __shared__ unsigned  st_sh[3];
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 3) st_sh[threadIdx.x] = 0u;
    __syncthreads();

    const int   wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int   gq  = lane / F_G;
    FWarpList&  L   = lists[wid];
    const float hmax_all = __uint_as_float(g.force_hmax_bits);
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;

    unsigned c_tested = 0, c_pairs = 0, c_av = 0;

    for (int round = 0; round < F_ROUNDS; ++round) {
        const int  p      = (blockIdx.x * F_ROUNDS + round) * (F_WARPS * F_NT) + wid * F_NT + gq;
        const bool tvalid = p < n;
        float4 pi = make_float4(0.f, 0.f, 0.f, 1.f), vi = pi, ri = make_float4(1.f, 1.f, 0.f, 0.f);
        if (tvalid) {
            pi = pos_h[p];
            vi = vel_m[p];
            ri = rcak[p];
        }
        const float hi = pi.w, ihi = __fdividef(1.0f, hi);
        const float rho_i = ri.x, c_i = ri.y, A_i = ri.z, K_i = ri.w;
        // scatter neighbours can be as far as 2 h_j: search with the largest h in use
        const float R = 2.0f * fmaxf(hi, hmax_all) * (1.0f + 1e-5f);
        const float hi2x4 = 4.0f * hi * hi;

        float acx = 0.0f, acy = 0.0f, acz = 0.0f, du = 0.0f, mumin = 0.0f;

        // one pair: source j at displacement (dx, dy, dz), smoothing length hj
        auto pair = [&](uint32_t j, float dx, float dy, float dz, float r2, float hj) {
            const float4 vj = __ldg(vel_m + j);
            const float4 rj = __ldg(rcak + j);
            const float r  = r2 * rsqrtf(r2);
            const float ti = fmaxf(1.0f - 0.5f * r * ihi, 0.0f);
            const float tj = fmaxf(1.0f - 0.5f * __fdividef(r, hj), 0.0f);
            const float gi = K_i * ti * ti * ti;
            const float gj = rj.w * tj * tj * tj;
            const float vdx = vi.x - vj.x, vdy = vi.y - vj.y, vdz = vi.z - vj.z;
            const float vr = vdx * dx + vdy * dy + vdz * dz;   // v_ij . r_ij
            float pig = 0.0f;                                   // Pi_ij * gbar
            if (vr < 0.0f) {
                const float hb  = 0.5f * (hi + hj);
                const float mu  = __fdividef(hb * vr, r2 + par.eps * hb * hb);
                const float cb  = 0.5f * (c_i + rj.y);
                const float rb  = 0.5f * (rho_i + rj.x);
                const float Pij = __fdividef(mu * (par.beta * mu - par.alpha * cb), rb);
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
            ++c_pairs;
        };

        // ---- phase 1: lane-private index lists
        int      cnt = 0;
        unsigned rot = 0;
        sph_group_rows<F_G>(g, cell_start, pos_h, pi.x, pi.y, pi.z, R, tvalid, lane, rot, c_tested,
                            [&](uint32_t j, const float4 pj, float sx, float sy, float sz) {
            const float dx = sx - pj.x, dy = sy - pj.y, dz = sz - pj.z;
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float Hm = fmaxf(hi2x4, 4.0f * pj.w * pj.w);
            if (r2 < Hm && r2 > 0.0f) {
                if (cnt < F_SLOTS) L.j[cnt][lane] = j;
                ++cnt;
            }
        });
        const bool ovf = sph_group_any<F_G>(cnt > F_SLOTS, lane);

        // ---- phase 2: the pairs of this lane's column
        const int mycnt  = ovf ? 0 : cnt;
        const int maxcnt = __reduce_max_sync(SPH_FULL, mycnt);
        for (int k = 0; k < maxcnt; ++k) {
            if (k < mycnt) {
                const uint32_t j  = L.j[k][lane];
                const float4   pj = __ldg(pos_h + j);
                float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
                dx -= Lx * rintf(dx * iLx);   // minimum image (no-op on open axes)
                dy -= Ly * rintf(dy * iLy);
                dz -= Lz * rintf(dz * iLz);
                const float r2 = dx * dx + dy * dy + dz * dz;
                pair(j, dx, dy, dz, r2, pj.w);
            }
        }
        // a column overflowed (very crowded neighbourhood): redo the group without lists
        if (__any_sync(SPH_FULL, ovf)) {
            sph_group_rows<F_G>(g, cell_start, pos_h, pi.x, pi.y, pi.z, R, tvalid && ovf, lane, rot,
                                c_tested,
                                [&](uint32_t j, const float4 pj, float sx, float sy, float sz) {
                const float dx = sx - pj.x, dy = sy - pj.y, dz = sz - pj.z;
                const float r2 = dx * dx + dy * dy + dz * dz;
                const float Hm = fmaxf(hi2x4, 4.0f * pj.w * pj.w);
                if (r2 < Hm && r2 > 0.0f) pair(j, dx, dy, dz, r2, pj.w);
            });
        }
        acx = sph_group_sum<F_G>(acx);
        acy = sph_group_sum<F_G>(acy);
        acz = sph_group_sum<F_G>(acz);
        du  = sph_group_sum<F_G>(du);
        mumin = sph_group_min<F_G>(mumin);
        if (tvalid && (lane & (F_G - 1)) == 0) {
            const int i = perm[p];
            ax[i] = acx; ay[i] = acy; az[i] = acz;
            dudt[i]   = du;
            mu_min[i] = mumin;
        }
        __syncwarp();
    }

    unsigned v[3] = {c_tested, c_pairs, c_av};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const unsigned t = __reduce_add_sync(SPH_FULL, v[k]);
        if (lane == 0 && t) atomicAdd(&st_sh[k], t);
    }
    __syncthreads();
    if (threadIdx.x < 3 && st_sh[threadIdx.x] != 0u)
        atomicAdd(stats + ST_FORCE_TESTED + threadIdx.x, (unsigned long long)st_sh[threadIdx.x]);
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
