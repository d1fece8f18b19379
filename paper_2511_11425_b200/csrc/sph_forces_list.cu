// sph_forces_list.cu -- steps a8, a9 of DESIGN.md for the buckets of the staged-tile density
// sweep: the hydro force pass of PAPER.md:186-219 (Section 2.3.5), Eqs. (13)-(18), read from
// the neighbour lists the density sweep kept (one list serves gather and
// scatter as long as it covers the reach 2 max(h_i, h_j)).
//
// One warp per bucket, one lane per pair of targets, NO shared memory: the list of a bucket is
// bucket-major, entry f of target t at [f][t], so the 32 lanes read their f-th entries with one
// coalesced load; the f-th neighbours of adjacent targets are adjacent records of the sorted
// arrays (the lists are in tile order: row by row, ascending inside a row), so the three
// 16-byte gathers per pair -- (x, y, z, h), (v, m), (rho, c, A, K) -- coalesce as well and the
// bucket's ~600 source records stay in L1.  The pair arithmetic is the branch-free form of
// sph_force_pair.cuh, two entries of both targets per trip: four independent dependency chains.
// Targets whose list does not cover their reach (a larger h_j nearby), and buckets without a
// list, go to k_forces (8 lanes per target, own search) through a target list.
#include <cstdio>
#include "sph_tile.cuh"
#include "sph_force_pair.cuh"

namespace {

constexpr int FL_WARPS = 4;
#ifndef FL_MINB
#define FL_MINB 4
#endif

__device__ __forceinline__ float lwarp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}
__device__ __forceinline__ float lwarp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}

template <int KERN, bool ENT>
__global__ __launch_bounds__(FL_WARPS * 32, FL_MINB) void k_forces_list(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const float4* __restrict__ vel_m,
    const float4* __restrict__ rcak, const int32_t* __restrict__ perm,
    const SphBucket* __restrict__ buckets, const unsigned* __restrict__ nbuckets, ForcePar par,
    const unsigned* __restrict__ coarse, const uint32_t* __restrict__ nb_j,
    const uint32_t* __restrict__ bucket_loff, const uint32_t* __restrict__ nb_cnt,
    const float* __restrict__ tl_rkeep, int lcap, unsigned* next, float* ax, float* ay, float* az, float* dudt,
    float* mu_min, uint32_t* fb_list, unsigned* fb_cnt, unsigned long long* stats) {
    __shared__ SphGrid g;
    __shared__ int     rowoff_s[FL_WARPS][32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int k = tid; k < (int)(sizeof(SphGrid) / 4); k += blockDim.x) ((int*)&g)[k] = ((const int*)gp)[k];
    __syncthreads();
    if (g.flags & SPH_GRID_STEEP) return;   // steep h contrast: the 8-lane kernels take every target
    const unsigned nb = *nbuckets;
    const float hmax_all = __uint_as_float(g.force_hmax_bits);
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;
    const bool  anyper = (g.per[0] | g.per[1] | g.per[2]) != 0;
    unsigned c_pairs = 0, c_av = 0;

    for (;;) {   // persistent warps: buckets are handed out by a counter
    unsigned bi = 0;
    if (lane == 0) bi = atomicAdd(next, 1u);
    bi = __shfl_sync(SPH_FULL, bi, 0);
    if (bi >= nb) break;
    const SphBucket bk = buckets[bi];
    __syncwarp();

    // ---- the bucket's targets
    const int nrows = bk.nry * bk.nrz;
    int rs = 0, rc = 0;
    if (lane < nrows) {
        const uint32_t rb = (uint32_t)((bk.rz0 + lane / bk.nry) * g.ny + (bk.ry0 + lane % bk.nry)) * (uint32_t)g.nx;
        const int s0 = (int)__ldg(cell_start + rb + bk.c0) + bk.skip;
        const int s1 = (int)__ldg(cell_start + rb + bk.c1);
        rs = s0;
        rc = min(max(s1 - s0, 0), SPH_TB);
    }
    int inc = rc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(SPH_FULL, inc, o);
        if (lane >= o) inc += t;
    }
    const int ntar = min(__shfl_sync(SPH_FULL, inc, 31), SPH_TB);
    int* const rowoff = rowoff_s[wid];
    rowoff[lane] = inc;
    __syncwarp();
    int    p[2];
    bool   valid[2];
    Target tg[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int k = lane + 32 * t;
        valid[t] = k < ntar;
        int rho_ = 0;
        while (rho_ < 31 && rowoff[rho_] <= k) ++rho_;
        const int before = rho_ ? rowoff[rho_ - 1] : 0;
        const int start  = __shfl_sync(SPH_FULL, rs, rho_);
        p[t] = valid[t] ? start + (k - before) : 0;
        tg[t].pi = make_float4(0.f, 0.f, 0.f, 0.f);
        tg[t].vi = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 ri = make_float4(1.f, 1.f, 0.f, 0.f);
        if (valid[t]) {
            tg[t].pi = pos_h[p[t]];
            tg[t].vi = vel_m[p[t]];
            ri       = rcak[p[t]];
        }
        tg[t].rho = ri.x; tg[t].c = ri.y; tg[t].A = ri.z; tg[t].K = ri.w;
        tg[t].ih  = valid[t] ? __fdividef(1.0f, tg[t].pi.w) : 0.0f;
    }
    float b0[3], b1[3], hown;
    {
        const float INF = __int_as_float(0x7f800000);
        float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF}, hm = 0.0f;
#pragma unroll
        for (int t = 0; t < 2; ++t)
            if (valid[t]) {
                lo[0] = fminf(lo[0], tg[t].pi.x); hi[0] = fmaxf(hi[0], tg[t].pi.x);
                lo[1] = fminf(lo[1], tg[t].pi.y); hi[1] = fmaxf(hi[1], tg[t].pi.y);
                lo[2] = fminf(lo[2], tg[t].pi.z); hi[2] = fmaxf(hi[2], tg[t].pi.z);
                hm = fmaxf(hm, tg[t].pi.w);
            }
#pragma unroll
        for (int d = 0; d < 3; ++d) { b0[d] = lwarp_min(lo[d]); b1[d] = lwarp_max(hi[d]); }
        hown = lwarp_max(hm);
    }
    // a6: the largest h that can reach the bucket sets the reach R = 2 max(h_i, H)
    const float Hs = sph_box_scatter_hmax(g, coarse, b0, b1, hown, hmax_all, lane);

    // ---- which targets the kept lists serve
    const uint32_t reg = bucket_loff[bi];
    const uint32_t* const lb = nb_j + (size_t)(reg == 0xffffffffu ? 0u : reg) * ((size_t)lcap * SPH_TB);
    bool cov[2];
    int  cnt[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const float R   = 2.0f * (1.0f + 1e-5f) * fmaxf(tg[t].pi.w, Hs);
        const float tau = 1e-6f + 2.5e-7f * g.xext * tg[t].ih;
        const float rk  = valid[t] ? tl_rkeep[p[t]] : 0.0f;
        cov[t] = valid[t] && reg != 0xffffffffu && R * (1.0f + 4.0f * tau) <= rk;
        cnt[t] = cov[t] ? (int)nb_cnt[p[t]] : 0;
        // not served: to the 8-lane kernel, which searches (or reads the [target][entry] list its
        // own density kernel left: nb_rkeep, a different array)
        if (valid[t] && !cov[t]) fb_list[atomicAdd(fb_cnt, 1u)] = (uint32_t)p[t];
    }
    const int maxcnt = __reduce_max_sync(SPH_FULL, max(cnt[0], cnt[1]));

    // Does the bucket's reach cross a periodic face?  If not, no pair of it needs the minimum
    // image (warp-uniform, decided once).
    bool wraps = false;
    {
        const float Rb = 2.0f * (1.0f + 1e-4f) * Hs;
#pragma unroll
        for (int d = 0; d < 3; ++d)
            wraps = wraps || (g.per[d] && (b0[d] - Rb < g.lo[d] || b1[d] + Rb > g.lo[d] + g.len[d]));
    }
    Accum acc[2];
    auto entry = [&](int t, int f) -> uint32_t {   // the sorted position of entry f (own record past the end)
        return f < cnt[t] ? __ldg(lb + f * SPH_TB + lane + 32 * t) : (uint32_t)p[t];
    };
    // one pair, in two halves: fetch + geometry (is the pair there, is it approaching), then
    // the arithmetic -- with or without the viscous terms, decided for the four pairs of a trip
    // at once (warp-uniform: a flow at rest, or a receding one, never pays for Eq. 15)
    struct PairIn { float4 vj, rj; float dx, dy, dz, r2, hj; bool ok; };
    auto fetch = [&](int t, int f, uint32_t j, auto wrap_tag, PairIn& q) -> bool {
        constexpr bool WRAP = decltype(wrap_tag)::value;
        const float4 pj = __ldg(pos_h + j);
        q.vj = __ldg(vel_m + j);
        q.rj = __ldg(rcak + j);
        q.dx = tg[t].pi.x - pj.x; q.dy = tg[t].pi.y - pj.y; q.dz = tg[t].pi.z - pj.z;
        if (WRAP) {   // minimum image
            q.dx -= Lx * rintf(q.dx * iLx);
            q.dy -= Ly * rintf(q.dy * iLy);
            q.dz -= Lz * rintf(q.dz * iLz);
        }
        q.r2 = q.dx * q.dx + q.dy * q.dy + q.dz * q.dz;
        q.hj = pj.w;
        const float hm = fmaxf(tg[t].pi.w, pj.w);
        q.ok = f < cnt[t] && q.r2 < 4.0f * hm * hm && q.r2 > 0.0f;
        return q.ok && force_pair_vr(tg[t], q.vj, q.dx, q.dy, q.dz) < 0.0f;
    };
    // two entries of both targets per trip (four independent chains); the list indices of the
    // next trip are loaded before this trip's records are used, so the list stream (HBM) and
    // the record gathers (L1 / L2) are not waited for one after the other
    auto sweep = [&](auto wrap_tag) {
        uint32_t jc[4] = {entry(0, 0), entry(1, 0), entry(0, 1), entry(1, 1)};
        for (int f = 0; f < maxcnt; f += 2) {
            const uint32_t jn[4] = {entry(0, f + 2), entry(1, f + 2), entry(0, f + 3), entry(1, f + 3)};
            PairIn q[4];
            bool   av = false;
#pragma unroll
            for (int k = 0; k < 4; ++k) av = fetch(k & 1, f + (k >> 1), jc[k], wrap_tag, q[k]) || av;
            if (__any_sync(SPH_FULL, av)) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    force_pair_nb<KERN, ENT, true>(tg[k & 1], acc[k & 1], par, q[k].ok, q[k].vj, q[k].rj, q[k].dx,
                                                   q[k].dy, q[k].dz, q[k].r2, q[k].hj);
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    force_pair_nb<KERN, ENT, false>(tg[k & 1], acc[k & 1], par, q[k].ok, q[k].vj, q[k].rj, q[k].dx,
                                                    q[k].dy, q[k].dz, q[k].r2, q[k].hj);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) jc[k] = jn[k];
        }
    };
    if (wraps && anyper) sweep(std::true_type{});
    else                 sweep(std::false_type{});
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        if (!cov[t]) continue;
        const int i = perm[p[t]];
        ax[i] = acc[t].ax; ay[i] = acc[t].ay; az[i] = acc[t].az;
        dudt[i]   = acc[t].du;
        mu_min[i] = acc[t].mumin;
        c_pairs += acc[t].pairs;
        c_av    += acc[t].av;
    }
    }   // bucket loop
    const unsigned tp = __reduce_add_sync(SPH_FULL, c_pairs), ta = __reduce_add_sync(SPH_FULL, c_av);
    if (lane == 0) {
        if (tp) atomicAdd(stats + ST_FORCE_PAIRS, (unsigned long long)tp);
        if (ta) atomicAdd(stats + ST_FORCE_AV, (unsigned long long)ta);
    }
}

}  // namespace

// Sweeps the buckets whose targets have kept lists; the targets it hands back are in
// c->fb_list (c->fb_cnt[1] of them) and are swept by the caller with the 8-lane kernel.
int sph_launch_forces_list(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min) {
    cudaStream_t s = c->stream;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fb_cnt + 1, 0, sizeof(unsigned), s));
    ForcePar par{c->par.av_alpha, c->par.av_beta, c->par.av_eps};
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->tile_next + 2, 0, sizeof(unsigned), s));
    auto launch2 = [&](auto tag, auto etag) {
        constexpr int  KERN = decltype(tag)::value;
        constexpr bool ENT  = decltype(etag)::value;
        int per_sm = 4;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_forces_list<KERN, ENT>, FL_WARPS * 32, 0);
        if (per_sm < 1) per_sm = 1;
        k_forces_list<KERN, ENT><<<c->sm_count * per_sm, FL_WARPS * 32, 0, s>>>(
            c->grid, c->cell_start, c->pos_h, c->vel_m, c->rcak, c->perm, c->buckets, c->bucket_cnt, par,
            c->coarse_hmax, c->nb_j, c->bucket_loff, c->nb_cnt, c->tl_rkeep, c->lcap, c->tile_next + 2, ax, ay, az,
            dudt, mu_min, c->fb_list, c->fb_cnt + 1, c->stats);
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
