// sph_density.cu -- steps a4-a6 of DESIGN.md: neighbour search, density and smoothing-
// length solve, PAPER.md:137-154 (Section 2.3.3), Eqs. (5)-(7).
//
// G = 8 lanes per target particle, four targets per warp.  The lanes of a group walk the
// candidate rows of the cell grid (coalesced float4 loads); the accepted candidates of a
// target are numbered by a group ballot and dealt out to the 8 lanes' columns of a shared-
// memory list (r, m) -- the paper's "we keep the precomputed interaction list", built for a
// "slightly larger kernel" -- and the root of Eq. (6) is then found on that
// list alone.  The indices j go to a global list that the force sweep reuses.
// Targets the lean kernel cannot finish (a list longer than 192 entries, an entry in the
// FP32-uncertain band around 2h, no convergence) are queued for k_density_fix, which
// re-walks the rows in every sweep with one warp per target and decides borderline
// neighbours in FP64.
//
// With W = sigma h^-3 w(q) (SphKernel<KERN> in sph_internal.cuh) and per target
//   S = sum_j m_j w(q_j),  E = -sum_j m_j q w'(q),  F = -sum_j m_j (q w' + q^2 w''):
//   (Wendland C2: w = (1-q/2)^4 (1+2q), E-term 5 q^2 t^3, F-term q^2 t^2 (10 t - 7.5 q), t = 1-q/2)
//   Eq. (6)  <=>  f(h) = S(h) - T = 0,  T = n_ngb m_i / ((32 pi/3) sigma)       (C2: 14)
//   f' = dS/dh = E/h,   dE/dh = -F/h,   f'' = -(E + F)/h^2
//   Halley step (the paper's Newton-Raphson with the second derivative added):
//       dh = -2 f f' / (2 f'^2 - f f'') = -2 f E h / (2 E^2 + f (E + F))
//   A step with |dh| <= 3e-4 h is accepted; S and E are carried to h + dh by their Taylor
//   series (error O((dh/h)^3) and O((dh/h)^2)), so the accepted sweep is also the last one.
//   Eq. (5)   rho = sigma S / h^3
//   Eq. (7)   Omega = 1 - D/(3S) with D = 3S - E  =>  Omega = E/(3S)
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int   D_G      = SPH_G;         // lanes per target
constexpr int   D_NT     = 32 / D_G;      // targets per warp
constexpr int   D_WARPS  = 4;
constexpr int   D_TPB    = D_WARPS * 32;
constexpr int   D_QUADS  = 16;            // target quads per block, handed out dynamically
constexpr int   D_TARGETS = D_NT * D_QUADS;
constexpr int   D_SLOTS  = SPH_SLOTS;     // list entries per lane
constexpr float D_ACCEPT = 3.0e-4f;

struct DensPar {
    float n_ngb, tol, slack;
    int   max_iter;
};

// A target's list: entry f at float f of its group's segment; the segments of the four groups
// of a warp start 8 banks apart (D_GSTRIDE = 192 + 8), so lane l of every group reading entry
// 8k + l hits 32 different banks.
constexpr int D_GSTRIDE = D_SLOTS * D_G + 8;
struct WarpList {
    float r[D_NT * D_GSTRIDE];
    float m[D_NT * D_GSTRIDE];
};
constexpr int D_MOFF = D_NT * D_GSTRIDE * 4;   // byte offset of m behind r

__global__ void k_pack_pos_m(int64_t n, const float4* __restrict__ pos_h,
                             const int32_t* __restrict__ perm, const float* __restrict__ m,
                             float4* pos_m) {
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    float4 a = pos_h[p];
    a.w      = m[perm[p]];
    pos_m[p] = a;
}

// One safeguarded Halley step from the sums at h.  Returns true if the step is accepted as
// final; hn is the next iterate either way, Sn / En the sums carried to hn.
__device__ __forceinline__ bool halley_step(float s, float e, float f2, float T, float h, float ih,
                                            float hcap, float tol, float& hlo, float& hhi,
                                            float& hn, float& Sn, float& En, bool& conv) {
    const float INF = __int_as_float(0x7f800000);
    const float f = s - T;
    if (f < 0.0f) hlo = h; else hhi = h;
    const float den = 2.0f * e * e + f * (e + f2);
    float dh;
    bool  genuine = true;
    if (e > 0.0f && den > 0.0f)  dh = __fdividef(-2.0f * f * e * h, den);
    else if (e > 0.0f)           dh = __fdividef(-f * h, e);
    else                       { dh = h; genuine = false; }
    hn = h + dh;
    if (!(hn >= 0.5f * h)) { hn = 0.5f * h; genuine = false; }
    if (!(hn <= 2.0f * h)) { hn = 2.0f * h; genuine = false; }
    if (hhi < INF && !(hn >= hlo && hn <= hhi)) { hn = 0.5f * (hlo + hhi); genuine = false; }
    if (hn > hcap) { hn = hcap; genuine = false; }
    dh = hn - h;
    const float x = dh * ih;
    Sn = s + x * (e - 0.5f * x * (e + f2));   // Taylor: S' = E/h, S'' = -(E+F)/h^2
    En = e - x * f2;                          //         E' = -F/h
    const bool small  = fabsf(dh) <= D_ACCEPT * h;
    const bool tight  = (hhi - hlo) <= tol * h;      // bracket closed to the tolerance
    const bool capped = (hn >= hcap && h >= hcap);
    conv = !(capped && f < 0.0f);
    return (genuine && small) || tight || capped;
}

__device__ __forceinline__ float density_hcap(const SphGrid& g) {
    // largest h the search may use: keeps 2 h x 1.25 below half the shortest periodic side
    float hcap = 3.0e37f;
    for (int d = 0; d < 3; ++d)
        if (g.per[d]) hcap = fminf(hcap, g.len[d] / (4.0f * 1.25f) * 0.999f);
        else          hcap = fminf(hcap, 4.0f * fmaxf(g.len[0], fmaxf(g.len[1], g.len[2])));
    return hcap;
}

template <int KERN>
__global__ __launch_bounds__(D_TPB, SPH_MINB) void k_density(
    int n, const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_m, const int32_t* __restrict__ perm, DensPar par, float* h_io,
    float* rho, float* omega, int32_t* nn, int32_t* fix_list, unsigned* fix_cnt, uint32_t* nb_j,
    uint32_t* nb_cnt, float* nb_rkeep, const uint32_t* __restrict__ act_list_,
    const unsigned* __restrict__ act_cnt_, int keep, int all_if_steep, unsigned long long* stats) {
    // keep = 0: no neighbour lists are left behind (the staged-tile sweep owns the list memory,
    // in its own layout; this kernel then only serves the buckets that sweep handed back)
    // all_if_steep: the target list is the tile sweep's hand-back list; under SPH_GRID_STEEP that
    // sweep stands back, this kernel takes every particle and keeps its lists as without tiles
    const bool steep = all_if_steep && (gp->flags & SPH_GRID_STEEP);
    const uint32_t* __restrict__ act_list = steep ? nullptr : act_list_;
    const unsigned* __restrict__ act_cnt  = act_cnt_;
    if (steep) keep = 1;
    // targets: all n sorted positions, or the act_cnt entries of act_list (the active set)
    const int nt = act_list ? (int)*act_cnt : n;
    if (blockIdx.x * D_TARGETS >= nt) return;
    __shared__ WarpList lists[D_WARPS];
    __shared__ SphGrid  g;
    __shared__ unsigned st_sh[5];
    __shared__ int      next_quad;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 5) st_sh[threadIdx.x] = 0u;
    if (threadIdx.x == 0) next_quad = 0;
    // stale list entries are read (with weight 0) by lanes past their count: keep them finite
    for (int k = threadIdx.x; k < (int)(sizeof(lists) / 4); k += D_TPB) ((float*)lists)[k] = 0.0f;
    __syncthreads();

    const int   wid = threadIdx.x >> 5;
    int         lane = threadIdx.x & 31;
    asm volatile("" : "+r"(lane));              // one register instead of SR_TID re-reads
    const int   gq  = lane / D_G;
    const bool  leader = (lane & (D_G - 1)) == 0;
    const int   sl = lane & (D_G - 1);
    // shared addresses (bytes) of the group's segment and of this lane's first entry in it
    const uint32_t gb = sph_smem_addr(&lists[wid].r[gq * D_GSTRIDE]);
    const uint32_t lb = gb + 4u * sl;
    const float hcap   = density_hcap(g);
    const float band_c = 2.5e-7f * g.xext;      // sph_band(h) = 1e-6 + band_c / h

    unsigned c_tested = 0;   // the other counters go to st_sh once per target

    for (;;) {
        int quad = 0;
        if (lane == 0) quad = atomicAdd(&next_quad, 1);
        quad = __shfl_sync(SPH_FULL, quad, 0);
        if (quad >= D_QUADS) break;
        const int  idx    = (blockIdx.x * D_QUADS + quad) * D_NT + gq;
        const bool tvalid = idx < nt;
        const int  p      = (act_list && tvalid) ? (int)act_list[idx] : idx;
        float4 pi = make_float4(0.f, 0.f, 0.f, 1.f);
        int    i  = 0;
        float  h  = g.hmin;
        if (tvalid) {
            pi = pos_m[p];
            i  = perm[p];
            h  = h_io[i];
        }
        if (!(h > 0.0f) || !(h < 3.0e38f)) h = g.hmin;
        h = fminf(h, hcap);
        const float T = par.n_ngb * pi.w * (1.0f / SphKernel<KERN>::self);
        // the target's kept list: entry f at [target][f]
        uint32_t* gj = nb_j + (size_t)(tvalid ? p : 0) * (D_SLOTS * D_G);
        asm volatile("" : "+l"(gj));   // a register pair: entry addresses are one IMAD.WIDE
        float    hlo = 0.0f, hhi = __int_as_float(0x7f800000);
        float    Rc = 0.0f;         // radius the list is complete for
        int      cnt = 0;           // entries in the target's list (uniform in the group)
        bool     first = true, done = !tvalid, fix = false;
        float    S = 0.0f, E = 0.0f;
        int      sweeps = 0;

        while (!__all_sync(SPH_FULL, done)) {
            const float ih  = __fdividef(1.0f, h);
            const float tau = 1e-6f + band_c * ih;
            // ---- (re)build the lists of the groups whose ball outgrew them
            const bool need = !done && (2.0f * h * (1.0f + 2.0f * tau) > Rc);
            if (__any_sync(SPH_FULL, need)) {
                if (need) {
                    Rc = 2.0f * h * (first ? par.slack : fmaxf(par.slack, 1.25f));
                    if (!first && leader) atomicAdd(&st_sh[4], 1u);
                    first = false;
                    cnt   = 0;
                }
                const float Rc2 = Rc * Rc;
                sph_group_collect<D_G>(g, cell_start, pos_m, pi.x, pi.y, pi.z, Rc, need, lane,
                                       c_tested, cnt,
                                       [&](const float4, float r2) { return r2 < Rc2; },
                                       [&](int f, uint32_t j, const float4 pj, float, float, float,
                                           float r2) {
                    if (f < D_SLOTS * D_G) {
                        const uint32_t a = gb + 4u * f;
                        sph_sts<0>(a, sph_sqrt(r2));
                        sph_sts<D_MOFF>(a, pj.w);
                        if (keep) sph_stg(gj + f, j);
                    }
                });
                __syncwarp();
                if (need && cnt > D_SLOTS * D_G) {
                    done = true;     // the list overflowed: leave the target to k_density_fix
                    fix  = true;
                }
            }
            // ---- one sweep over the lists: S(h), E(h), F(h)
            float s = 0.0f, e = 0.0f, f2 = 0.0f;
            const int mycnt  = done ? 0 : (cnt - sl + D_G - 1) >> 3;   // entries sl, sl + 8, ...
            const int maxcnt = __reduce_max_sync(SPH_FULL, mycnt);
            uint32_t la = lb;
            for (int k = 0; k < maxcnt; ++k, la += 4u * D_G) {
                const float mj = (k < mycnt) ? sph_lds<D_MOFF>(la) : 0.0f;
                float wq, eq, fq;
                SphKernel<KERN>::sums_s(sph_lds<0>(la) * ih, wq, eq, fq);
                s  += mj * wq;
                e  += mj * eq;
                f2 += mj * fq;
            }
            s  = sph_group_sum<D_G>(s);
            e  = SphKernel<KERN>::escale * sph_group_sum<D_G>(e);
            f2 = sph_group_sum<D_G>(f2);
            if (done) continue;
            ++sweeps;
            float hn, Sn, En;
            bool  conv;
            const bool acc = halley_step(s, e, f2, T, h, ih, hcap, par.tol, hlo, hhi, hn, Sn, En, conv);
            if (acc && 2.0f * hn * (1.0f + 2.0f * (1e-6f + band_c * __fdividef(1.0f, hn))) <= Rc) {
                S = Sn; E = En; h = hn;   // the list covers the ball of hn (+ band) as well
                done = true;
                fix  = !conv;
                continue;
            }
            h = hn;
            if (sweeps >= par.max_iter) { done = true; fix = true; }
        }

        // ---- n_i = #{j : r_ij < 2h} from the list; an entry inside the FP32-uncertain band
        // around 2h sends the target to the exact recount of k_density_fix.
        // The FP32 distance is uncertain by tau(h) only for sources met through a periodic
        // image (the shifted target coordinate is rounded); when the search ball stays inside
        // the box the displacement x_i - x_j is exact to 2^-24 |d| and 2e-6 covers the rest.
        bool wraps = false;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const float xd = (d == 0 ? pi.x : d == 1 ? pi.y : pi.z) - g.lo[d];
            wraps |= g.per[d] && (xd < Rc || xd + Rc > g.len[d]);
        }
        const float H = 2.0f * h, tauH = (wraps ? 1e-6f + band_c / h : 2e-6f) * H;
        // The whole list is kept for the force sweep: it is complete inside Rc, already in
        // the order of the sorted arrays, and needs no second pass (dropping the entries
        // beyond 2h x 1.05 was measured: the compaction costs the density sweep 9 % and the
        // shorter reach sends most targets of a disordered distribution into a second search).
        int  ni = 0;
        bool edge = false;
        {
            const int mycnt  = (tvalid && !fix) ? (cnt - sl + D_G - 1) >> 3 : 0;
            const int maxcnt = __reduce_max_sync(SPH_FULL, mycnt);
            uint32_t la = lb;
            for (int k = 0; k < maxcnt; ++k, la += 4u * D_G) {
                const float r = (k < mycnt) ? sph_lds<0>(la) : 3.0e38f;
                ni += (r < H) ? 1 : 0;
                edge |= fabsf(r - H) <= tauH;
            }
        }
        const bool recount = sph_group_any<D_G>(edge, lane) && !fix;   // h, rho, Omega stand
        ni = sph_group_sum_int<D_G>(ni);
        if (tvalid && leader) {
            atomicAdd(&st_sh[1], (unsigned)cnt);
            atomicAdd(&st_sh[3], (unsigned)sweeps);
            h_io[i] = h;   // final, or the best iterate for the fix kernel to start from
            nb_rkeep[p] = (fix || !keep) ? 0.0f : Rc;
            nb_cnt[p]   = cnt;
            if (!fix) {
                const float ih = 1.0f / h;
                rho[i]   = SphKernel<KERN>::sigma * S * ih * ih * ih;
                omega[i] = E / (3.0f * S);
                nn[i]    = ni;
            }
            if (fix)          fix_list[atomicAdd(fix_cnt, 1u)] = p;
            else if (recount) fix_list[atomicAdd(fix_cnt, 1u)] = p | (int32_t)0x80000000;
            else              atomicAdd(&st_sh[2], (unsigned)ni);
        }
        __syncwarp();
    }

    // ---- counters: lanes -> warp -> block -> one atomic per block and counter
    {
        const unsigned t = __reduce_add_sync(SPH_FULL, c_tested);
        if (lane == 0 && t) atomicAdd(&st_sh[0], t);
    }
    __syncthreads();
    if (threadIdx.x < 5 && st_sh[threadIdx.x] != 0u)
        atomicAdd(stats + ST_DENS_TESTED + threadIdx.x, (unsigned long long)st_sh[threadIdx.x]);
}

// The robust path: one warp per queued target, no list.  Every sweep re-walks the candidate
// rows (32 lanes over each row), so neither crowding nor a growing h can break it, and the
// final count decides neighbours inside the FP32-uncertain band in FP64.
template <int KERN>
__global__ __launch_bounds__(256) void k_density_fix(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_m, const int32_t* __restrict__ perm, DensPar par,
    const int32_t* __restrict__ fix_list, const unsigned* __restrict__ fix_cnt, float* h_io,
    float* rho, float* omega, int32_t* nn, unsigned long long* stats) {
    __shared__ RowRec  rows_all[8][SPH_RCAP];
    __shared__ SphGrid g;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    __syncthreads();
    const int      wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RowRec*        rows = rows_all[wid];
    const unsigned nfix = *fix_cnt;
    const float    hcap = density_hcap(g);
    unsigned long long c_tested = 0, c_pairs = 0, c_sweeps = 0;
    unsigned c_nonconv = 0, c_recheck = 0, c_targets = 0;

    for (unsigned t = blockIdx.x * 8 + wid; t < nfix; t += gridDim.x * 8) {
        const int    pq = fix_list[t];
        const bool   count_only = pq < 0;   // h, rho, Omega are final: exact n_i only
        const int    p  = pq & 0x7fffffff;
        const float4 pi = pos_m[p];
        const int    i  = perm[p];
        const float  T  = par.n_ngb * pi.w * (1.0f / SphKernel<KERN>::self);
        float h = fminf(h_io[i], hcap);
        float hlo = 0.0f, hhi = __int_as_float(0x7f800000);
        float S = 0.0f, E = 0.0f;
        bool  conv = count_only;
        int   sweeps = 0;
        while (!count_only) {
            const float ih = 1.0f / h, H2 = 4.0f * h * h;
            float s = 0.0f, e = 0.0f, f2 = 0.0f;
            sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, 2.0f * h, rows, lane,
                             [&](const RowRec& rr) {
                for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                    const uint32_t j = k0 + lane;
                    if (j < rr.end) {
                        const float4 pj = __ldg(pos_m + j);
                        const float dx = (rr.sx - pj.x) + rr.lx, dy = (rr.sy - pj.y) + rr.ly, dz = (rr.sz - pj.z) + rr.lz;
                        const float r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 < H2) {
                            float wq, eq, fq;
                            SphKernel<KERN>::sums(sqrtf(r2) * ih, wq, eq, fq);
                            s  += pj.w * wq;
                            e  += pj.w * eq;
                            f2 += pj.w * fq;
                        }
                    }
                    c_tested += min(32u, rr.end - k0);
                }
            });
            s  = sph_warp_sum(s);
            e  = sph_warp_sum(e);
            f2 = sph_warp_sum(f2);
            ++sweeps;
            float hn, Sn, En;
            const bool acc = halley_step(s, e, f2, T, h, ih, hcap, par.tol, hlo, hhi, hn, Sn, En, conv);
            if (acc) { S = Sn; E = En; h = hn; break; }
            if (sweeps >= par.max_iter) { S = s; E = e; conv = false; break; }
            h = hn;
        }
        // ---- exact neighbour count at the final h
        const float  tau = sph_band(g, h), H = 2.0f * h, H2 = H * H;
        const double H2e = 4.0 * (double)h * (double)h;
        int ni = 0;
        sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, H * (1.0f + 2.0f * tau), rows, lane,
                         [&](const RowRec& rr) {
            for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                const uint32_t j = k0 + lane;
                if (j < rr.end) {
                    const float4 pj = __ldg(pos_m + j);
                    const float dx = (rr.sx - pj.x) + rr.lx, dy = (rr.sy - pj.y) + rr.ly, dz = (rr.sz - pj.z) + rr.lz;
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    bool in = r2 < H2;
                    if (fabsf(r2 - H2) <= 2.0f * tau * H2) {
                        in = sph_r2_exact(g, pi.x, pi.y, pi.z, pj.x, pj.y, pj.z) < H2e;
                        ++c_recheck;
                    }
                    ni += in ? 1 : 0;
                }
            }
        });
        ni = sph_warp_sum_int(ni);
        if (lane == 0) {
            nn[i] = ni;
            if (!count_only) {
                const float ih = 1.0f / h;
                h_io[i]  = h;
                rho[i]   = SphKernel<KERN>::sigma * S * ih * ih * ih;
                omega[i] = E / (3.0f * S);
            }
        }
        c_pairs += ni;
        c_sweeps += sweeps;
        c_targets += 1;
        if (!conv) ++c_nonconv;
        __syncwarp();
    }
    c_recheck = __reduce_add_sync(SPH_FULL, c_recheck);
    if (lane == 0 && c_targets) {
        atomicAdd(stats + ST_DENS_TESTED, c_tested);
        atomicAdd(stats + ST_DENS_PAIRS, c_pairs);
        atomicAdd(stats + ST_DENS_SWEEPS, c_sweeps);
        atomicAdd(stats + ST_DENS_OVERFLOW, (unsigned long long)c_targets);
        atomicAdd(stats + ST_DENS_NONCONV, (unsigned long long)c_nonconv);
        atomicAdd(stats + ST_DENS_RECHECK, (unsigned long long)c_recheck);
    }
}

}  // namespace

int sph_launch_density(sph_ctx* c, const float* m, float* h, float* rho, float* omega,
                       int32_t* nn) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    k_pack_pos_m<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->pos_h, c->perm, m, c->pos_m);
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fix_cnt, 0, sizeof(unsigned), s));
    DensPar par{c->par.n_ngb, c->par.h_tol, c->par.search_slack, c->par.h_max_iter};
    const int nblk = (int)((n + D_TARGETS - 1) / D_TARGETS);
    // the staged-tile kernel first (all particles as targets only); what it hands back --
    // buckets its tile cannot hold -- is swept by the 8-lane kernel through a target list
    const bool tiled = sph_tile_on(c) && !c->act_on;
    if (tiled) {
        const int rc = sph_launch_density_tile(c, h, rho, omega, nn);
        if (rc != SPH_OK) return rc;
    }
    const uint32_t* tlist = tiled ? c->fb_list : (c->act_on ? c->act_list : nullptr);
    const unsigned* tcnt  = tiled ? c->fb_cnt : c->act_cnt;
    auto launch = [&](auto tag) {
        constexpr int KERN = decltype(tag)::value;
        k_density<KERN><<<nblk, D_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_m, c->perm, par,
                                               h, rho, omega, nn, c->fix_list, c->fix_cnt, c->nb_j,
                                               c->nb_cnt, c->nb_rkeep, tlist, tcnt,
                                               (tiled && c->par.tile_forces != 1) ? 0 : 1, tiled ? 1 : 0, c->stats);
        k_density_fix<KERN><<<c->sm_count * 4, 256, 0, s>>>(c->grid, c->cell_start, c->pos_m, c->perm,
                                                            par, c->fix_list, c->fix_cnt, h, rho,
                                                            omega, nn, c->stats);
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
