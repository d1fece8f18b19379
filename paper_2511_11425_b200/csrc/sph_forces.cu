// sph_forces.cu -- steps a7-a9 of DESIGN.md: EOS + per-particle precompute, gather-or-
// scatter neighbour search and the hydro force sweep, PAPER.md:186-219 (Section 2.3.5),
// Eqs. (13)-(18), ideal gas of PAPER.md:111.
//
// G = 8 lanes per target, four targets per warp.  Phase 1: the lanes of a group distance-
// test the candidates of the rows in reach (0 < r < 2 max(h_i,h_j), gather and scatter,
// PAPER.md:191); the accepted ones are numbered by a group ballot into the target's index
// list -- or, when the list the density sweep kept already covers the reach, that list is
// used as it is.  Phase 2: lane l of the group works through entries l, l + 8, ... -- the
// pair arithmetic runs without divergence between accepted and rejected candidates.  A group
// whose column overflows is queued for k_forces_fix (one warp per target, no list).
//
// Pair arithmetic (d = x_i - x_j, r = |d|, q_a = r/h_a, g_a = K_a g(q_a), g = -w'(q)/q, with
// K_a = sigma / h_a^5, so that dW/dr(r,h_a) = -g_a r; Wendland C2: g = 5 (1-q/2)_+^3):
//   Eq. 13+17:  a_i     = + sum_j m_j (A_i g_i + A_j g_j + Pi_ij gbar) d
//   Eq. 14+18:  du_i/dt = - sum_j m_j (A_i g_i + Pi_ij gbar / 2) (v_ij . d)
//   Eq. 15-16:  mu = hbar (v_ij.d)/(r^2 + eps hbar^2), Pi = mu (beta mu - alpha cbar)/rhobar
//               for v_ij.d < 0, else 0;   gbar = (g_i + g_j)/2;  A = P/(Omega rho^2).
#include <cstdio>
#include "sph_internal.cuh"
#include "sph_force_pair.cuh"

namespace {

#ifndef SPH_FMINB
#define SPH_FMINB SPH_MINB
#endif
constexpr int F_G      = SPH_G;
constexpr int F_NT     = 32 / F_G;
constexpr int F_WARPS  = 4;
constexpr int F_TPB    = F_WARPS * 32;
constexpr int F_QUADS  = 16;   // target quads per block, handed out dynamically
constexpr int F_TARGETS = F_NT * F_QUADS;
constexpr int F_SLOTS  = SPH_SLOTS;   // list entries per lane

struct FWarpList {
    uint32_t j[F_SLOTS][32];
};

// a7: EOS and the per-particle factors, written in sorted order (scattered 16-byte stores)
__global__ void k_force_prep(int64_t n, const int32_t* __restrict__ inv_perm,
                             const float* __restrict__ m,
                             const float* __restrict__ vx, const float* __restrict__ vy,
                             const float* __restrict__ vz, const float* __restrict__ u,
                             const float* __restrict__ rho, const float* __restrict__ h,
                             const float* __restrict__ omega, float gamma, float sigma, float4* pos_h,
                             float4* vel_m, float4* rcak, float* P, float* cs, SphGrid* g) {
    int64_t  i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float    hi = 0.0f;
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
        rcak[p] = make_float4(ri, ci, Pi / (om * ri * ri), sigma / (h2 * h2 * hi));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) hi = fmaxf(hi, __shfl_xor_sync(SPH_FULL, hi, o));
    if ((threadIdx.x & 31) == 0 && hi > 0.0f &&
        *(volatile unsigned*)&g->force_hmax_bits < __float_as_uint(hi))
        atomicMax(&g->force_hmax_bits, __float_as_uint(hi));
}

// a6: max h per coarse cell, the bound of the scatter reach.  Runs over the SORTED records, so
// the 32 particles of a warp almost always share one coarse cell: one atomic per warp.
__global__ void k_coarse_hmax(int64_t n, const SphGrid* __restrict__ g,
                              const float4* __restrict__ pos_h, unsigned* coarse) {
    int64_t  p  = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned cc = 0xffffffffu, hb = 0u;
    if (p < n) {
        const float4 a = pos_h[p];
        if (a.w > 0.0f) {
            const int cx = sph_cell_coord(a.x, g->lo[0], g->ics[0], g->cn[0]);
            const int cy = sph_cell_coord(a.y, g->lo[1], g->ics[1], g->cn[1]);
            const int cz = sph_cell_coord(a.z, g->lo[2], g->ics[2], g->cn[2]);
            cc = (unsigned)((cz * g->cn[1] + cy) * g->cn[0] + cx);
            hb = __float_as_uint(a.w);
        }
    }
    const unsigned cc0 = __shfl_sync(SPH_FULL, cc, 0);
    if (__all_sync(SPH_FULL, cc == cc0)) {
        const unsigned mx = __reduce_max_sync(SPH_FULL, hb);
        if ((threadIdx.x & 31) == 0 && cc != 0xffffffffu && __ldcg(coarse + cc) < mx)
            atomicMax(coarse + cc, mx);
    } else if (cc != 0xffffffffu && __ldcg(coarse + cc) < hb) {   // the map only grows
        atomicMax(coarse + cc, hb);
    }
}

// second level of the map: one warp per block of 8 x 8 x 8 coarse cells, written behind the
// first level (the float bits of positive h order like the floats)
__global__ void k_coarse_blocks(const SphGrid* __restrict__ g, unsigned* coarse) {
    const int lane = threadIdx.x & 31, nwarp = (int)((gridDim.x * blockDim.x) >> 5);
    const int nb = g->sn[0] * g->sn[1] * g->sn[2];
    for (int w = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5); w < nb; w += nwarp) {
        const int bx = w % g->sn[0], t = w / g->sn[0], by = t % g->sn[1], bz = t / g->sn[1];
        unsigned  mx = 0u;
        for (int q = lane; q < 512; q += 32) {
            const int cx = bx * 8 + (q & 7), cy = by * 8 + ((q >> 3) & 7), cz = bz * 8 + (q >> 6);
            if (cx < g->cn[0] && cy < g->cn[1] && cz < g->cn[2])
                mx = max(mx, coarse[(cz * g->cn[1] + cy) * g->cn[0] + cx]);
        }
        mx = __reduce_max_sync(SPH_FULL, mx);
        if (lane == 0) coarse[SPH_COARSE_MAX + w] = mx;
    }
}

__global__ void k_zero_hmax(SphGrid* g) { g->force_hmax_bits = 0u; }

template <int KERN, bool ENT>
__global__ __launch_bounds__(F_TPB, SPH_FMINB) void k_forces(
    int n, const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const float4* __restrict__ vel_m,
    const float4* __restrict__ rcak, const int32_t* __restrict__ perm, ForcePar par, float* ax,
    float* ay, float* az, float* dudt, float* mu_min, int32_t* fix_list, unsigned* fix_cnt,
    const unsigned* __restrict__ coarse, const uint32_t* __restrict__ nb_j,
    const uint32_t* __restrict__ nb_cnt, const float* __restrict__ nb_rkeep,
    const uint32_t* __restrict__ act_list_, const unsigned* __restrict__ act_cnt, int all_if_steep,
    unsigned long long* stats) {
    // all_if_steep: the target list is the hand-back list of the tile / list sweeps; under
    // SPH_GRID_STEEP those stand back and this kernel takes every particle
    const uint32_t* __restrict__ act_list = (all_if_steep && (gp->flags & SPH_GRID_STEEP)) ? nullptr : act_list_;
    // targets: all n sorted positions, or the act_cnt entries of act_list (the active set)
    const int nt = act_list ? (int)*act_cnt : n;
    if (blockIdx.x * F_TARGETS >= nt) return;
    __shared__ FWarpList lists[F_WARPS];
    __shared__ SphGrid   g;
    __shared__ unsigned  st_sh[3];
    __shared__ int       next_quad;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 3) st_sh[threadIdx.x] = 0u;
    if (threadIdx.x == 0) next_quad = 0;
    __syncthreads();

    const int   wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int   gq  = lane / F_G;
    uint32_t* const lj = &lists[wid].j[0][lane];   // this lane's column, slot stride 32
    const float hmax_all = __uint_as_float(g.force_hmax_bits);
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;
    const bool  anyper = (g.per[0] | g.per[1] | g.per[2]) != 0;

    unsigned c_tested = 0, c_pairs = 0, c_av = 0;

    for (;;) {
        int quad = 0;
        if (lane == 0) quad = atomicAdd(&next_quad, 1);
        quad = __shfl_sync(SPH_FULL, quad, 0);
        if (quad >= F_QUADS) break;
        const int  idx    = (blockIdx.x * F_QUADS + quad) * F_NT + gq;
        const bool tvalid = idx < nt;
        const int  p      = (act_list && tvalid) ? (int)act_list[idx] : idx;
        Target t;
        t.pi = make_float4(0.f, 0.f, 0.f, 1.f);
        t.vi = t.pi;
        float4 ri = make_float4(1.f, 1.f, 0.f, 0.f);
        if (tvalid) {
            t.pi = pos_h[p];
            t.vi = vel_m[p];
            ri   = rcak[p];
        }
        t.rho = ri.x; t.c = ri.y; t.A = ri.z; t.K = ri.w;
        t.ih  = __fdividef(1.0f, t.pi.w);
        // scatter neighbours can be as far as 2 h_j: the reach is set by the largest h that
        // can get to this target (a6)
        const float R = 2.0f * (1.0f + 1e-5f) *
                        sph_scatter_hmax<F_G>(g, coarse, t.pi.x, t.pi.y, t.pi.z, t.pi.w, hmax_all, lane);
        const float hi2x4 = 4.0f * t.pi.w * t.pi.w;

        // ---- phase 1: the target's index list, entry f handled by lane f % 8 of the group.
        // If the list kept by the density sweep is complete out to R (same positions,
        // DESIGN.md section 7) it is read in place from global memory; else search.
        const int   sl = lane & (F_G - 1), g0 = lane & ~(F_G - 1);
        const float rk      = tvalid ? nb_rkeep[p] : 0.0f;
        const float tau     = 1e-6f + 2.5e-7f * g.xext * t.ih;
        const bool  covered = tvalid && (R * (1.0f + 4.0f * tau) <= rk);
        int cnt = covered ? (int)nb_cnt[p] : 0;
        const bool search = tvalid && !covered;
        if (__any_sync(SPH_FULL, search)) {
            uint32_t* const gl = &lists[wid].j[0][g0];
            sph_group_collect<F_G>(g, cell_start, pos_h, t.pi.x, t.pi.y, t.pi.z, R, search, lane,
                                   c_tested, cnt,
                                   [&](const float4 pj, float r2) {
                                       return r2 < fmaxf(hi2x4, 4.0f * pj.w * pj.w) && r2 > 0.0f;
                                   },
                                   [&](int f, uint32_t j, const float4, float, float, float, float) {
                                       if (f < F_SLOTS * F_G) gl[(f >> 3) * 32 + (f & (F_G - 1))] = j;
                                   });
            __syncwarp();
        }
        const bool ovf = search && cnt > F_SLOTS * F_G;

        // ---- phase 2: entries sl, sl + 8, ... of the list.  The 8 lanes of a group work on 8
        // consecutive entries, i.e. mostly on neighbouring records of the sorted arrays, so the
        // three 16-byte gathers per pair touch a few lines per group instead of one per lane.
        Accum a;
        const uint32_t* const src = covered ? nb_j + ((size_t)p * (F_SLOTS * F_G) + sl) : lj;
        const int stride = covered ? F_G : 32;
        const int mycnt  = ovf ? 0 : (cnt - sl + F_G - 1) >> 3;
        const int maxcnt = __reduce_max_sync(SPH_FULL, mycnt);
        // software-pipelined: the records of entry k+1 are in flight while entry k is worked on.
        // Two record sets used in turn, two entries per trip (no register copies); the loads are
        // unconditional -- past its last entry a lane re-reads that entry (an L1 hit) and a lane
        // without entries reads the target's own record -- so the loop body has no branch
        // around them.
        const uint32_t jself = (uint32_t)(tvalid ? p : 0);
        const int      klast = mycnt - 1;
        auto fetch = [&](int k, float4& pj, float4& vj, float4& rj) {
            uint32_t j = jself;
            if (klast >= 0) j = src[min(k, klast) * stride];
            pj = __ldg(pos_h + j); vj = __ldg(vel_m + j); rj = __ldg(rcak + j);
        };
        auto work = [&](int k, const float4& pj, const float4& vj, const float4& rj) {
            float dx = t.pi.x - pj.x, dy = t.pi.y - pj.y, dz = t.pi.z - pj.z;
            if (anyper) {   // minimum image
                dx -= Lx * rintf(dx * iLx);
                dy -= Ly * rintf(dy * iLy);
                dz -= Lz * rintf(dz * iLz);
            }
            const float r2 = dx * dx + dy * dy + dz * dz;
            // kept lists hold everything inside the kept radius: apply the pair test
            if (k < mycnt && r2 < fmaxf(hi2x4, 4.0f * pj.w * pj.w) && r2 > 0.0f)
                force_pair<KERN, ENT>(t, a, par, vj, rj, dx, dy, dz, r2, pj.w);
        };
        float4 pA, vA, rA, pB, vB, rB;
        fetch(0, pA, vA, rA);
        for (int k = 0; k < maxcnt; k += 2) {
            fetch(k + 1, pB, vB, rB);
            work(k, pA, vA, rA);
            fetch(k + 2, pA, vA, rA);
            work(k + 1, pB, vB, rB);
        }
        a.ax = sph_group_sum<F_G>(a.ax);
        a.ay = sph_group_sum<F_G>(a.ay);
        a.az = sph_group_sum<F_G>(a.az);
        a.du = sph_group_sum<F_G>(a.du);
        a.mumin = sph_group_min<F_G>(a.mumin);
        c_pairs += a.pairs;
        c_av    += a.av;
        if (tvalid && (lane & (F_G - 1)) == 0) {
            if (!ovf) {
                const int i = perm[p];
                ax[i] = a.ax; ay[i] = a.ay; az[i] = a.az;
                dudt[i]   = a.du;
                mu_min[i] = a.mumin;
            } else {
                fix_list[atomicAdd(fix_cnt, 1u)] = p;   // very crowded neighbourhood
            }
        }
        __syncwarp();
    }

    unsigned v[3] = {c_tested, c_pairs, c_av};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const unsigned tt = __reduce_add_sync(SPH_FULL, v[k]);
        if (lane == 0 && tt) atomicAdd(&st_sh[k], tt);
    }
    __syncthreads();
    if (threadIdx.x < 3 && st_sh[threadIdx.x] != 0u)
        atomicAdd(stats + ST_FORCE_TESTED + threadIdx.x, (unsigned long long)st_sh[threadIdx.x]);
}

// The robust path: one warp per queued target, candidates handled as they are met.
template <int KERN, bool ENT>
__global__ __launch_bounds__(256) void k_forces_fix(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const float4* __restrict__ vel_m,
    const float4* __restrict__ rcak, const int32_t* __restrict__ perm, ForcePar par,
    const int32_t* __restrict__ fix_list, const unsigned* __restrict__ fix_cnt, float* ax,
    float* ay, float* az, float* dudt, float* mu_min, unsigned long long* stats) {
    __shared__ RowRec  rows_all[8][SPH_RCAP];
    __shared__ SphGrid g;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    __syncthreads();
    const int      wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned nfix = *fix_cnt;
    const float    hmax_all = __uint_as_float(g.force_hmax_bits);
    unsigned long long c_tested = 0;
    unsigned c_pairs = 0, c_av = 0;
    for (unsigned q = blockIdx.x * 8 + wid; q < nfix; q += gridDim.x * 8) {
        const int p = fix_list[q];
        Target t;
        t.pi = pos_h[p];
        t.vi = vel_m[p];
        const float4 ri = rcak[p];
        t.rho = ri.x; t.c = ri.y; t.A = ri.z; t.K = ri.w;
        t.ih  = 1.0f / t.pi.w;
        const float R = 2.0f * fmaxf(t.pi.w, hmax_all) * (1.0f + 1e-5f);
        const float hi2x4 = 4.0f * t.pi.w * t.pi.w;
        Accum a;
        sph_for_each_row(g, cell_start, t.pi.x, t.pi.y, t.pi.z, R, rows_all[wid], lane,
                         [&](const RowRec& rr) {
            for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                const uint32_t j = k0 + lane;
                if (j < rr.end) {
                    const float4 pj = __ldg(pos_h + j);
                    const float dx = rr.sx - pj.x, dy = rr.sy - pj.y, dz = rr.sz - pj.z;
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 < fmaxf(hi2x4, 4.0f * pj.w * pj.w) && r2 > 0.0f)
                        force_pair<KERN, ENT>(t, a, par, __ldg(vel_m + j), __ldg(rcak + j), dx, dy, dz, r2, pj.w);
                }
                c_tested += min(32u, rr.end - k0);
            }
        });
        a.ax = sph_warp_sum(a.ax);
        a.ay = sph_warp_sum(a.ay);
        a.az = sph_warp_sum(a.az);
        a.du = sph_warp_sum(a.du);
        a.mumin = sph_warp_min(a.mumin);
        c_pairs += a.pairs;
        c_av    += a.av;
        if (lane == 0) {
            const int i = perm[p];
            ax[i] = a.ax; ay[i] = a.ay; az[i] = a.az;
            dudt[i]   = a.du;
            mu_min[i] = a.mumin;
        }
        __syncwarp();
    }
    c_pairs = __reduce_add_sync(SPH_FULL, c_pairs);
    c_av    = __reduce_add_sync(SPH_FULL, c_av);
    if (lane == 0 && (c_tested | c_pairs)) {
        atomicAdd(stats + ST_FORCE_TESTED, c_tested);
        atomicAdd(stats + ST_FORCE_PAIRS, (unsigned long long)c_pairs);
        atomicAdd(stats + ST_FORCE_AV, (unsigned long long)c_av);
    }
}

}  // namespace

// a6 alone: the coarse max-h map of the h held in pos_h.w (used by the marking pass)
int sph_launch_coarse_map(sph_ctx* c) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->coarse_hmax, 0, SPH_COARSE_MAX * sizeof(unsigned), s));
    k_coarse_hmax<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->grid, c->pos_h, c->coarse_hmax);
    k_coarse_blocks<<<c->sm_count, 256, 0, s>>>(c->grid, c->coarse_hmax);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_forces(sph_ctx* c, const float* m, const float* vx, const float* vy,
                      const float* vz, const float* u, const float* rho, const float* h,
                      const float* omega, float* ax, float* ay, float* az, float* dudt,
                      float* mu_min, float* P, float* cs) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    // K = gscale sigma / h^5: dW/dr = -K g_s(q) r
    static const float sigmas[4] = {SphKernel<0>::sigma * SphKernel<0>::gscale,
                                    SphKernel<1>::sigma * SphKernel<1>::gscale,
                                    SphKernel<2>::sigma * SphKernel<2>::gscale,
                                    SphKernel<3>::sigma * SphKernel<3>::gscale};
    const float sigma = sigmas[(c->par.kernel >= 0 && c->par.kernel <= 3) ? c->par.kernel : 1];
    k_zero_hmax<<<1, 1, 0, s>>>(c->grid);
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fix_cnt + 1, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->coarse_hmax, 0, SPH_COARSE_MAX * sizeof(unsigned), s));
    k_force_prep<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->inv_perm, m, vx, vy, vz, u,
                                                        rho, h, omega, c->par.gamma, sigma, c->pos_h,
                                                        c->vel_m, c->rcak, P, cs, c->grid);
    k_coarse_hmax<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->grid, c->pos_h, c->coarse_hmax);
    k_coarse_blocks<<<c->sm_count, 256, 0, s>>>(c->grid, c->coarse_hmax);
    ForcePar par{c->par.av_alpha, c->par.av_beta, c->par.av_eps};
    const int nblk = (int)((n + F_TARGETS - 1) / F_TARGETS);
    // the staged-tile kernel first; what it hands back goes through the 8-lane kernel's target list
    // the buckets of the staged-tile density sweep first: from its kept lists (default) or on
    // staged tiles; what is handed back goes through the 8-lane kernel's target list
    const bool tiled = sph_tile_on(c) && !c->act_on;
    if (tiled) {
        const int rc = c->par.tile_forces == 2 ? sph_launch_forces_tlist(c, ax, ay, az, dudt, mu_min)
                     : c->par.tile_forces > 0 ? sph_launch_forces_tile(c, ax, ay, az, dudt, mu_min)
                                              : sph_launch_forces_list(c, ax, ay, az, dudt, mu_min);
        if (rc != SPH_OK) return rc;
    }
    const uint32_t* tlist = tiled ? c->fb_list : (c->act_on ? c->act_list : nullptr);
    const unsigned* tcnt  = tiled ? c->fb_cnt + 1 : c->act_cnt;
    auto launch2 = [&](auto tag, auto etag) {
        constexpr int  KERN = decltype(tag)::value;
        constexpr bool ENT  = decltype(etag)::value;
        k_forces<KERN, ENT><<<nblk, F_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_h, c->vel_m,
                                              c->rcak, c->perm, par, ax, ay, az, dudt, mu_min,
                                              c->fix_list, c->fix_cnt + 1, c->coarse_hmax, c->nb_j,
                                              c->nb_cnt, c->nb_rkeep, tlist, tcnt, tiled ? 1 : 0, c->stats);
        k_forces_fix<KERN, ENT><<<c->sm_count * 4, 256, 0, s>>>(c->grid, c->cell_start, c->pos_h, c->vel_m,
                                                           c->rcak, c->perm, par, c->fix_list,
                                                           c->fix_cnt + 1, ax, ay, az, dudt, mu_min,
                                                           c->stats);
    };
    auto launch = [&](auto tag) {
        if (c->par.entropy) launch2(tag, std::true_type{});
        else launch2(tag, std::false_type{});
    };
    switch (c->par.kernel) {
    case 0: launch(std::integral_constant<int, 0>{}); break;
    case 2: launch(std::integral_constant<int, 2>{}); break;
    case 3: launch(std::integral_constant<int, 3>{}); break;
    default: launch(std::integral_constant<int, 1>{}); break;
    }
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
