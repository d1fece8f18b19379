// sph_density.cu -- steps a4-a6 of DESIGN.md: neighbour search, density and smoothing-
// length solve, PAPER.md:137-154 (Section 2.3.3), Eqs. (5)-(7).
//
// One warp per target particle.  Lanes sweep the candidate rows of the cell grid in
// parallel (coalesced float4 loads of 32 consecutive sorted particles), the accepted
// candidates are compacted by ballot into a per-warp shared-memory list (r, m, j), and the
// Newton-Raphson iteration for h_i then runs on that list only -- the paper's "we keep the
// precomputed interaction list" with a "slightly larger kernel".
//
// With w(q) = SIGMA wt(q), wt = (1-q/2)^4 (1+2q), and S = sum_j m_j wt(r_ij/h):
//   Eq. (6)  <=>  S(h) = T,  T = n_ngb m_i / 14            ((32 pi/3) SIGMA = 14)
//   dS/dh = E/h,  E = sum_j m_j 5 q^2 (1-q/2)^3            (-q wt'(q) = 5 q^2 (1-q/2)^3)
//   Newton:   h <- h (1 - (S-T)/E)
//   Eq. (5)   rho = SIGMA S / h^3
//   Eq. (7)   Omega = 1 - D/(3S) with D = 3S - E  =>  Omega = E/(3S)
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int D_WARPS   = 8;
constexpr int D_TPB     = D_WARPS * 32;
constexpr int D_TARGETS = 64;   // consecutive sorted targets per block
constexpr int LCAP      = 320;  // list entries per warp

struct DensPar {
    float n_ngb, tol, slack;
    int   max_iter;
};

struct WarpSmem {
    float    r[LCAP];
    float    m[LCAP];
    uint32_t j[LCAP];
    RowRec   rows[SPH_RCAP];
};

__global__ void k_pack_pos_m(int64_t n, const float4* __restrict__ pos_h,
                             const int32_t* __restrict__ perm, const float* __restrict__ m,
                             float4* pos_m) {
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    float4 a = pos_h[p];
    a.w      = m[perm[p]];
    pos_m[p] = a;
}

__global__ __launch_bounds__(D_TPB) void k_density(int n, const SphGrid* __restrict__ gp,
                                                   const uint32_t* __restrict__ cell_start,
                                                   const float4* __restrict__ pos_m,
                                                   const int32_t* __restrict__ perm, DensPar par,
                                                   float* h_io, float* rho, float* omega,
                                                   int32_t* nn, unsigned long long* stats) {
    __shared__ WarpSmem sm_all[D_WARPS];
    __shared__ SphGrid  g;
    __shared__ unsigned long long st_sh[8];
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 8) st_sh[threadIdx.x] = 0ull;
    __syncthreads();

    const int      wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned lt  = (1u << lane) - 1u;
    WarpSmem&      sm  = sm_all[wid];
    const float    INF = __int_as_float(0x7f800000);

    // largest h the search may use: keeps 2 h slack below half the shortest periodic side
    float hcap = 3.0e37f;
    for (int d = 0; d < 3; ++d)
        if (g.per[d]) hcap = fminf(hcap, g.len[d] / (4.0f * 1.25f) * 0.999f);
        else          hcap = fminf(hcap, 4.0f * fmaxf(g.len[0], fmaxf(g.len[1], g.len[2])));

    unsigned long long c_tested = 0, c_listed = 0, c_pairs = 0, c_sweeps = 0;
    unsigned c_recollect = 0, c_overflow = 0, c_nonconv = 0, c_recheck = 0;

    for (int t = wid; t < D_TARGETS; t += D_WARPS) {
        const int p = blockIdx.x * D_TARGETS + t;
        if (p >= n) break;
        const float4 pi = pos_m[p];
        const int    i  = perm[p];
        const float  mi = pi.w;
        const float  T  = par.n_ngb * mi * (1.0f / 14.0f);
        float        h  = h_io[i];
        if (!(h > 0.0f) || !(h < 3.0e38f)) h = g.hmin;
        h = fminf(h, hcap);
        float hlo = 0.0f, hhi = INF;
        float Rc = 0.0f;       // radius the list is complete for
        int   cnt = 0;
        bool  stream = false;  // list overflowed: evaluate by re-enumeration
        bool  first = true;
        float S = 0.0f, E = 0.0f;
        int   sweeps = 0;
        bool  conv = false;

        for (;;) {
            const float tau = sph_band(g, h);
            if (!stream && 2.0f * h * (1.0f + 2.0f * tau) > Rc) {
                // (re)build the list for a ball that over-selects by the slack
                Rc = 2.0f * h * (first ? par.slack : fmaxf(par.slack, 1.25f));
                if (!first) ++c_recollect;
                first = false;
                const float Rc2 = Rc * Rc;
                cnt = 0;
                sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, Rc, sm.rows, lane,
                                 [&](const RowRec& rr) {
                    for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                        const uint32_t j = k0 + lane;
                        const bool     v = j < rr.end;
                        float4 pj = make_float4(3.0e18f, 3.0e18f, 3.0e18f, 0.0f);
                        if (v) pj = __ldg(pos_m + j);
                        const float dx = rr.sx - pj.x, dy = rr.sy - pj.y, dz = rr.sz - pj.z;
                        const float r2 = dx * dx + dy * dy + dz * dz;
                        const bool  acc = v && (r2 < Rc2);
                        const unsigned mk = __ballot_sync(SPH_FULL, acc);
                        if (acc) {
                            const int slot = cnt + __popc(mk & lt);
                            if (slot < LCAP) {
                                sm.r[slot] = sqrtf(r2);
                                sm.m[slot] = pj.w;
                                sm.j[slot] = j;
                            }
                        }
                        cnt += __popc(mk);
                        c_tested += min(32u, rr.end - k0);
                    }
                });
                __syncwarp();
                if (cnt > LCAP) {
                    stream = true;
                    ++c_overflow;
                } else {
                    c_listed += cnt;
                }
            }
            // ---- one sweep: S(h), E(h)
            const float ih = 1.0f / h;
            float s = 0.0f, e = 0.0f;
            if (!stream) {
                for (int k = lane; k < cnt; k += 32) {
                    const float q  = sm.r[k] * ih;
                    const float mj = sm.m[k];
                    const float tt = fmaxf(1.0f - 0.5f * q, 0.0f);
                    const float t3 = tt * tt * tt;
                    s += mj * (t3 * tt * (1.0f + 2.0f * q));
                    e += mj * (5.0f * q * q * t3);
                }
            } else {
                const float H2 = 4.0f * h * h;
                sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, 2.0f * h, sm.rows, lane,
                                 [&](const RowRec& rr) {
                    for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                        const uint32_t j = k0 + lane;
                        if (j < rr.end) {
                            const float4 pj = __ldg(pos_m + j);
                            const float dx = rr.sx - pj.x, dy = rr.sy - pj.y, dz = rr.sz - pj.z;
                            const float r2 = dx * dx + dy * dy + dz * dz;
                            if (r2 < H2) {
                                const float q  = sqrtf(r2) * ih;
                                const float tt = fmaxf(1.0f - 0.5f * q, 0.0f);
                                const float t3 = tt * tt * tt;
                                s += pj.w * (t3 * tt * (1.0f + 2.0f * q));
                                e += pj.w * (5.0f * q * q * t3);
                            }
                        }
                        c_tested += min(32u, rr.end - k0);
                    }
                });
            }
            S = sph_warp_sum(s);
            E = sph_warp_sum(e);
            ++sweeps;
            const float f = S - T;
            if (f < 0.0f) hlo = h; else hhi = h;
            float hn = (E > 0.0f) ? h * (1.0f - f / E) : 2.0f * h;
            hn = fminf(fmaxf(hn, 0.5f * h), 2.0f * h);
            if (hhi < INF && !(hn > hlo && hn < hhi)) hn = 0.5f * (hlo + hhi);
            hn = fminf(hn, hcap);
            if (fabsf(hn - h) <= par.tol * h) {
                conv = (f >= 0.0f) || (h < hcap);
                break;
            }
            if (sweeps >= par.max_iter) break;
            h = hn;
        }
        if (!conv) ++c_nonconv;
        c_sweeps += sweeps;

        // ---- n_i = #{j : r_ij < 2h}; pairs near the edge are decided in FP64
        const float  tau = sph_band(g, h);
        const float  H   = 2.0f * h;
        const double H2e = 4.0 * (double)h * (double)h;
        int ni = 0;
        if (!stream) {
            for (int k = lane; k < cnt; k += 32) {
                const float r = sm.r[k];
                bool in = r < H;
                if (fabsf(r - H) <= tau * H) {
                    const float4 pj = __ldg(pos_m + sm.j[k]);
                    in = sph_r2_exact(g, pi.x, pi.y, pi.z, pj.x, pj.y, pj.z) < H2e;
                    ++c_recheck;
                }
                ni += in ? 1 : 0;
            }
        } else {
            const float H2 = H * H;
            sph_for_each_row(g, cell_start, pi.x, pi.y, pi.z, H * (1.0f + 2.0f * tau), sm.rows,
                             lane, [&](const RowRec& rr) {
                for (uint32_t k0 = rr.start; k0 < rr.end; k0 += 32) {
                    const uint32_t j = k0 + lane;
                    if (j < rr.end) {
                        const float4 pj = __ldg(pos_m + j);
                        const float dx = rr.sx - pj.x, dy = rr.sy - pj.y, dz = rr.sz - pj.z;
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
        }
        ni = sph_warp_sum_int(ni);
        c_pairs += ni;
        if (lane == 0) {
            const float ih = 1.0f / h;
            h_io[i]  = h;
            rho[i]   = SPH_SIGMA * S * ih * ih * ih;
            omega[i] = E / (3.0f * S);
            nn[i]    = ni;
        }
        __syncwarp();
    }

    // ---- counters: warp -> block -> one atomic per block and counter
    c_recheck = __reduce_add_sync(SPH_FULL, c_recheck);
    if (lane == 0) {
        atomicAdd(&st_sh[0], c_tested);
        atomicAdd(&st_sh[1], c_listed);
        atomicAdd(&st_sh[2], c_pairs);
        atomicAdd(&st_sh[3], c_sweeps);
        atomicAdd(&st_sh[4], (unsigned long long)c_recollect);
        atomicAdd(&st_sh[5], (unsigned long long)c_overflow);
        atomicAdd(&st_sh[6], (unsigned long long)c_nonconv);
        atomicAdd(&st_sh[7], (unsigned long long)c_recheck);
    }
    __syncthreads();
    if (threadIdx.x < 8 && st_sh[threadIdx.x] != 0ull)
        atomicAdd(stats + ST_DENS_TESTED + threadIdx.x, st_sh[threadIdx.x]);
}

}  // namespace

int sph_launch_density(sph_ctx* c, const float* m, float* h, float* rho, float* omega,
                       int32_t* nn) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    k_pack_pos_m<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->pos_h, c->perm, m, c->pos_m);
    DensPar par{c->par.n_ngb, c->par.h_tol, c->par.search_slack, c->par.h_max_iter};
    const int nblk = (int)((n + D_TARGETS - 1) / D_TARGETS);
    k_density<<<nblk, D_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_m, c->perm, par, h,
                                     rho, omega, nn, c->stats);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
