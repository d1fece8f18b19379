// sph_density.cu -- steps a4-a6 of DESIGN.md: neighbour search, density and smoothing-
// length solve, PAPER.md:137-154 (Section 2.3.3), Eqs. (5)-(7).
//
// G = 8 lanes per target particle, four targets per warp.  The lanes of a group walk the
// candidate rows of the cell grid (coalesced float4 loads), every lane keeps the candidates
// it accepted in a private column of a shared-memory list (r, m) -- the paper's "we keep the
// precomputed interaction list", built for a "slightly larger kernel" -- and
// the root of Eq. (6) is then found on that list alone.
//
// With w(q) = SIGMA wt(q), wt = (1-q/2)^4 (1+2q), t = 1-q/2, and per target
//   S = sum_j m_j wt(q_j),  E = sum_j m_j 5 q^2 t^3,  F = sum_j m_j q^2 t^2 (10 t - 7.5 q):
//   Eq. (6)  <=>  f(h) = S(h) - T = 0,  T = n_ngb m_i / 14         ((32 pi/3) SIGMA = 14)
//   f' = dS/dh = E/h,   dE/dh = -F/h,   f'' = -(E + F)/h^2
//   Halley step (the paper's Newton-Raphson with the second derivative added):
//       dh = -2 f f' / (2 f'^2 - f f'') = -2 f E h / (2 E^2 + f (E + F))
//   A step with |dh| <= 3e-4 h is accepted; S and E are carried to h + dh by their Taylor
//   series (error O((dh/h)^3) and O((dh/h)^2)), so the accepted sweep is also the last one.
//   Eq. (5)   rho = SIGMA S / h^3
//   Eq. (7)   Omega = 1 - D/(3S) with D = 3S - E  =>  Omega = E/(3S)
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int   D_G      = 8;             // lanes per target
constexpr int   D_NT     = 32 / D_G;      // targets per warp
constexpr int   D_WARPS  = 4;
constexpr int   D_TPB    = D_WARPS * 32;
constexpr int   D_ROUNDS = 2;             // target quads per warp
constexpr int   D_TARGETS = D_WARPS * D_NT * D_ROUNDS;
constexpr int   D_SLOTS  = 28;            // list entries per lane
constexpr float D_ACCEPT = 3.0e-4f;

struct DensPar {
    float n_ngb, tol, slack;
    int   max_iter;
};

struct WarpList {
    float r[D_SLOTS][32];
    float m[D_SLOTS][32];
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

__global__ __launch_bounds__(D_TPB, SPH_MINB) void k_density(int n, const SphGrid* __restrict__ gp,
                                                      const uint32_t* __restrict__ cell_start,
                                                      const float4* __restrict__ pos_m,
                                                      const int32_t* __restrict__ perm,
                                                      DensPar par, float* h_io, float* rho,
                                                      float* omega, int32_t* nn,
                                                      unsigned long long* stats) {
    __shared__ WarpList lists[D_WARPS];
    __shared__ SphGrid g;
    __shared__ unsigned st_sh[8];
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x < 8) st_sh[threadIdx.x] = 0u;
    __syncthreads();

    const int   wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int   gq  = lane / D_G;
    WarpList&   L   = lists[wid];
    const float INF = __int_as_float(0x7f800000);

    // largest h the search may use: keeps 2 h slack below half the shortest periodic side
    float hcap = 3.0e37f;
    for (int d = 0; d < 3; ++d)
        if (g.per[d]) hcap = fminf(hcap, g.len[d] / (4.0f * 1.25f) * 0.999f);
        else          hcap = fminf(hcap, 4.0f * fmaxf(g.len[0], fmaxf(g.len[1], g.len[2])));
    const float band_c = 2.5e-7f * g.xext;   // sph_band(h) = 1e-6 + band_c / h

    unsigned c_tested = 0, c_listed = 0, c_pairs = 0, c_sweeps = 0;
    unsigned c_recollect = 0, c_overflow = 0, c_nonconv = 0, c_recheck = 0;

    for (int round = 0; round < D_ROUNDS; ++round) {
        const int  p      = (blockIdx.x * D_ROUNDS + round) * (D_WARPS * D_NT) + wid * D_NT + gq;
        const bool tvalid = p < n;
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
        const float T = par.n_ngb * pi.w * (1.0f / 14.0f);
        float    hlo = 0.0f, hhi = INF;
        float    Rc = 0.0f;         // radius the list is complete for
        int      cnt = 0;           // entries in this lane's column
        unsigned rot = 0;
        bool     stream = false;    // list overflowed: evaluate by re-enumeration
        bool     first = true, done = !tvalid, conv = false;
        float    S = 0.0f, E = 0.0f;
        int      sweeps = 0;

        while (!__all_sync(SPH_FULL, done)) {
            const float ih  = __fdividef(1.0f, h);
            const float tau = 1e-6f + band_c * ih;
            // ---- (re)build the lists of the groups whose ball outgrew them
            const bool need = !done && !stream && (2.0f * h * (1.0f + 2.0f * tau) > Rc);
            if (__any_sync(SPH_FULL, need)) {
                if (need) {
                    Rc = 2.0f * h * (first ? par.slack : fmaxf(par.slack, 1.25f));
                    if (!first && (lane & (D_G - 1)) == 0) ++c_recollect;
                    first = false;
                    cnt   = 0;
                }
                const float Rc2 = Rc * Rc;
                sph_group_rows<D_G>(g, cell_start, pos_m, pi.x, pi.y, pi.z, Rc, need, lane, rot, c_tested,
                                    [&](uint32_t j, const float4 pj, float sx, float sy, float sz) {
                    const float dx = sx - pj.x, dy = sy - pj.y, dz = sz - pj.z;
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 < Rc2) {
                        if (cnt < D_SLOTS) {
                            L.r[cnt][lane] = r2 * rsqrtf(fmaxf(r2, 1e-35f));
                            L.m[cnt][lane] = pj.w;
                        }
                        ++cnt;
                    }
                });
                const bool ovf = sph_group_any<D_G>(need && cnt > D_SLOTS, lane);
                if (need) {
                    if (ovf) {
                        stream = true;
                        if ((lane & (D_G - 1)) == 0) ++c_overflow;
                    } else {
                        c_listed += cnt;
                    }
                }
            }
            // ---- one sweep: S(h), E(h), F(h)
            float s = 0.0f, e = 0.0f, f2 = 0.0f;
            const bool use_list = !done && !stream;
            const int  mycnt    = use_list ? cnt : 0;
            const int  maxcnt   = __reduce_max_sync(SPH_FULL, mycnt);
            for (int k = 0; k < maxcnt; ++k) {
                if (k < mycnt) {
                    const float q  = L.r[k][lane] * ih;
                    const float mj = L.m[k][lane];
                    const float tt = fmaxf(1.0f - 0.5f * q, 0.0f);
                    const float t2 = tt * tt, q2 = q * q;
                    s  += mj * (t2 * t2 * (1.0f + 2.0f * q));
                    e  += mj * (5.0f * q2 * t2 * tt);
                    f2 += mj * (q2 * t2 * (10.0f * tt - 7.5f * q));
                }
            }
            const bool sgroup = stream && !done;
            if (__any_sync(SPH_FULL, sgroup)) {
                const float H2 = 4.0f * h * h;
                sph_group_rows<D_G>(g, cell_start, pos_m, pi.x, pi.y, pi.z, 2.0f * h, sgroup, lane,
                                    rot, c_tested,
                                    [&](uint32_t j, const float4 pj, float sx, float sy, float sz) {
                    const float dx = sx - pj.x, dy = sy - pj.y, dz = sz - pj.z;
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 < H2) {
                        const float q  = r2 * rsqrtf(fmaxf(r2, 1e-35f)) * ih;
                        const float tt = fmaxf(1.0f - 0.5f * q, 0.0f);
                        const float t2 = tt * tt, q2 = q * q;
                        s  += pj.w * (t2 * t2 * (1.0f + 2.0f * q));
                        e  += pj.w * (5.0f * q2 * t2 * tt);
                        f2 += pj.w * (q2 * t2 * (10.0f * tt - 7.5f * q));
                    }
                });
            }
            s  = sph_group_sum<D_G>(s);
            e  = sph_group_sum<D_G>(e);
            f2 = sph_group_sum<D_G>(f2);
            if (done) continue;
            ++sweeps;
            // ---- safeguarded Halley step
            const float f = s - T;
            if (f < 0.0f) hlo = h; else hhi = h;
            const float den = 2.0f * e * e + f * (e + f2);
            float dh;
            bool  genuine = true;
            if (e > 0.0f && den > 0.0f)  dh = -2.0f * f * e * h / den;
            else if (e > 0.0f)           dh = -f * h / e;
            else                       { dh = h; genuine = false; }
            float hn = h + dh;
            if (!(hn >= 0.5f * h)) { hn = 0.5f * h; genuine = false; }
            if (!(hn <= 2.0f * h)) { hn = 2.0f * h; genuine = false; }
            if (hhi < INF && !(hn >= hlo && hn <= hhi)) { hn = 0.5f * (hlo + hhi); genuine = false; }
            if (hn > hcap) { hn = hcap; genuine = false; }
            dh = hn - h;
            const bool small = fabsf(dh) <= D_ACCEPT * h;
            const bool tight = (hhi - hlo) <= par.tol * h;   // bracket closed to the tolerance
            if ((genuine && small) || tight || (hn >= hcap && h >= hcap)) {
                // carry S and E to hn; the list must cover the ball of hn (+ band) as well
                const float x = dh * ih;
                const float Sn = s + x * (e - 0.5f * x * (e + f2));
                const float En = e - x * f2;
                if (stream || 2.0f * hn * (1.0f + 2.0f * (1e-6f + band_c / hn)) <= Rc) {
                    S = Sn; E = En; h = hn;
                    done = true;
                    conv = !(hn >= hcap && f < 0.0f);
                    continue;
                }
            }
            if (sweeps >= par.max_iter) {
                S = s; E = e;
                done = true;
                continue;
            }
            h = hn;
        }
        if (tvalid && (lane & (D_G - 1)) == 0) {
            if (!conv) ++c_nonconv;
            c_sweeps += sweeps;
        }

        // ---- n_i = #{j : r_ij < 2h}.  From the list; if an entry sits in the FP32-uncertain
        // band around 2h (or there is no list), recount with the FP64 test on the candidates.
        const float  H   = 2.0f * h;
        const float  tau = 1e-6f + band_c / h;
        int  ni = 0;
        bool edge = false;
        if (tvalid && !stream) {
            for (int k = 0; k < cnt; ++k) {
                const float r = L.r[k][lane];
                ni += (r < H) ? 1 : 0;
                edge |= fabsf(r - H) <= tau * H;
            }
        }
        const bool any_edge = sph_group_any<D_G>(edge, lane);
        const bool exact    = tvalid && (stream || any_edge);
        if (__any_sync(SPH_FULL, exact)) {
            if (exact) ni = 0;
            const float  H2  = H * H;
            const double H2e = 4.0 * (double)h * (double)h;
            sph_group_rows<D_G>(g, cell_start, pos_m, pi.x, pi.y, pi.z, H * (1.0f + 2.0f * tau),
                                exact, lane, rot, c_tested,
                                [&](uint32_t j, const float4 pj, float sx, float sy, float sz) {
                const float dx = sx - pj.x, dy = sy - pj.y, dz = sz - pj.z;
                const float r2 = dx * dx + dy * dy + dz * dz;
                bool in = r2 < H2;
                if (fabsf(r2 - H2) <= 2.0f * tau * H2) {
                    in = sph_r2_exact(g, pi.x, pi.y, pi.z, pj.x, pj.y, pj.z) < H2e;
                    ++c_recheck;
                }
                ni += in ? 1 : 0;
            });
        }
        ni = sph_group_sum_int<D_G>(ni);
        if (tvalid && (lane & (D_G - 1)) == 0) {
            const float ih = 1.0f / h;
            h_io[i]  = h;
            rho[i]   = SPH_SIGMA * S * ih * ih * ih;
            omega[i] = E / (3.0f * S);
            nn[i]    = ni;
            c_pairs += ni;
        }
        __syncwarp();
    }

    // ---- counters: lanes -> warp -> block -> one atomic per block and counter
    unsigned v[8] = {c_tested, c_listed, c_pairs, c_sweeps, c_recollect, c_overflow, c_nonconv,
                     c_recheck};
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const unsigned t = __reduce_add_sync(SPH_FULL, v[k]);
        if (lane == 0 && t) atomicAdd(&st_sh[k], t);
    }
    __syncthreads();
    if (threadIdx.x < 8 && st_sh[threadIdx.x] != 0u)
        atomicAdd(stats + ST_DENS_TESTED + threadIdx.x, (unsigned long long)st_sh[threadIdx.x]);
}

}  // namespace

int sph_launch_density(sph_ctx* c, const float* m, float* h, float* rho, float* omega,
                       int32_t* nn) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    k_pack_pos_m<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->pos_h, c->perm, m, c->pos_m);
    DensPar par{c->par.n_ngb, c->par.h_tol, c->par.search_slack, c->par.h_max_iter};
    const int    nblk = (int)((n + D_TARGETS - 1) / D_TARGETS);
    k_density<<<nblk, D_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_m, c->perm, par, h,
                                       rho, omega, nn, c->stats);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
