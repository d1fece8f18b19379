// sph_forces_tlist.cu -- steps a8, a9 of DESIGN.md for the buckets of the staged-tile density
// sweep, with the SOURCE RECORDS STAGED IN SHARED MEMORY: the hydro force pass of
// PAPER.md:186-219 (Section 2.3.5), Eqs. (13)-(18), read from the neighbour lists the density
// sweep kept.
//
// sph_forces_list.cu gathers the three 16-byte records of every pair from global memory and is
// bound by the L1 data pipe (a warp's 32 records lie in about 12 lines: 12 wavefronts per
// gather).  Here the bucket's tile -- the same rows, cut to the same chords, in the same order
// as in the density sweep, which is why a list entry can be the INDEX of the source in the tile
// (sph_params.tile_forces = 2, TilePar.lmode) -- is brought into shared memory once per bucket
// by bulk copies of the three sorted arrays, and a pair costs three LDS.128 of four wavefronts
// each.  Two warps per bucket, one target per thread, as in the density sweep; the pair
// arithmetic and the order of the sums are those of sph_forces_list.cu.
#include <cstdio>
#include "sph_tile.cuh"
#include "sph_force_pair.cuh"

namespace {

#ifndef TL_NE
#define TL_NE 4
#endif

struct TlPar {
    ForcePar fp;
    int      tcap, lcap;
};

__host__ __device__ inline size_t tl_smem_bytes(int tcap) {
    return (size_t)(tcap + 4) * 48 + (size_t)SPH_TSEGS * 8 + 16;
}

template <int KERN, bool ENT>
__global__ __launch_bounds__(64) void k_forces_tlist(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const float4* __restrict__ vel_m,
    const float4* __restrict__ rcak, const int32_t* __restrict__ perm,
    const SphBucket* __restrict__ buckets, const unsigned* __restrict__ nbuckets,
    const uint32_t* __restrict__ blist, unsigned* big_list, unsigned* big_cnt, unsigned* next,
    TlPar par, const unsigned* __restrict__ coarse, const uint32_t* __restrict__ nb_j,
    const uint32_t* __restrict__ bucket_loff, const float* __restrict__ bucket_rt,
    const uint32_t* __restrict__ nb_cnt, const float* __restrict__ tl_rkeep, float* ax, float* ay,
    float* az, float* dudt, float* mu_min, uint32_t* fb_list, unsigned* fb_cnt,
    unsigned long long* stats) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ SphGrid     g;
    __shared__ SphTileInfo ti;
    __shared__ unsigned    bi_s;
    __shared__ int         rowoff_s[2][32];
    __shared__ float       bb_s[2][8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int k = tid; k < (int)(sizeof(SphGrid) / 4); k += 64) ((int*)&g)[k] = ((const int*)gp)[k];
    // carve: P = (x, y, z, h), V = (v, m), Q = (rho, c, A, K), the segment table, the mbarrier
    SphTileMem sm;
    {
        unsigned char* base = smem_raw;
        sm.tcap  = par.tcap;
        sm.tile  = (float4*)base;   base += (size_t)(par.tcap + 4) * 48;
        sm.ms = nullptr; sm.mask = nullptr; sm.gidx = nullptr; sm.zone = nullptr; sm.rowoff = nullptr;
        sm.seg   = (uint2*)base;    base += (size_t)SPH_TSEGS * 8;
        sm.bar   = (uint32_t)__cvta_generic_to_shared(base);
        sm.tile_sa = (uint32_t)__cvta_generic_to_shared(sm.tile);
        sm.ms_sa = 0u; sm.mask_sa = 0u; sm.zone_sa = 0u; sm.gidx_sa = 0u;
    }
    const uint32_t p_sa = sm.tile_sa;
    const uint32_t v_sa = p_sa + 16u * (uint32_t)(par.tcap + 4);
    const uint32_t q_sa = v_sa + 16u * (uint32_t)(par.tcap + 4);
    if (tid == 0) sph_mbar_init(sm.bar, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t parity = 0;
    if (g.flags & SPH_GRID_STEEP) return;   // steep h contrast: the 8-lane kernels take every target
    const unsigned nb = *nbuckets;
    const float hmax_all = __uint_as_float(g.force_hmax_bits);
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;
    const bool  anyper = (g.per[0] | g.per[1] | g.per[2]) != 0;
    unsigned c_pairs = 0, c_av = 0;
    unsigned nxt = 0;
    if (tid == 0) nxt = atomicAdd(next, 1u);

    for (;;) {
        __syncthreads();                     // the last bucket's tile is free
        if (tid == 0) bi_s = nxt;
        __syncthreads();
        const unsigned bslot = bi_s;
        if (bslot >= nb) break;
        if (tid == 0) nxt = atomicAdd(next, 1u);
        const unsigned  bi = blist ? blist[bslot] : bslot;
        const SphBucket bk = buckets[bi];

        // ---- the bucket's targets: one per thread (column tid)
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
        const bool valid = tid < ntar;
        int p = 0;
        {
            int rho_ = 0;
            while (rho_ < 31 && rowoff[rho_] <= tid) ++rho_;
            const int before = rho_ ? rowoff[rho_ - 1] : 0;
            const int start  = __shfl_sync(SPH_FULL, rs, rho_);
            p = valid ? start + (tid - before) : 0;
        }
        Target tg;
        tg.pi = make_float4(0.f, 0.f, 0.f, 0.f);
        tg.vi = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 ri = make_float4(1.f, 1.f, 0.f, 0.f);
        if (valid) {
            tg.pi = pos_h[p];
            tg.vi = vel_m[p];
            ri    = rcak[p];
        }
        tg.rho = ri.x; tg.c = ri.y; tg.A = ri.z; tg.K = ri.w;
        tg.ih  = valid ? __fdividef(1.0f, tg.pi.w) : 0.0f;
        // bounding box of the block's targets, their largest h
        float b0[3], b1[3], hown;
        {
            const float INF = __int_as_float(0x7f800000);
            float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF}, hm = 0.0f;
            if (valid) {
                lo[0] = hi[0] = tg.pi.x; lo[1] = hi[1] = tg.pi.y; lo[2] = hi[2] = tg.pi.z;
                hm = tg.pi.w;
            }
#pragma unroll
            for (int d = 0; d < 3; ++d) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    lo[d] = fminf(lo[d], __shfl_xor_sync(SPH_FULL, lo[d], o));
                    hi[d] = fmaxf(hi[d], __shfl_xor_sync(SPH_FULL, hi[d], o));
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) hm = fmaxf(hm, __shfl_xor_sync(SPH_FULL, hm, o));
            if (lane == 0) {
#pragma unroll
                for (int d = 0; d < 3; ++d) { bb_s[wid][d] = lo[d]; bb_s[wid][3 + d] = hi[d]; }
                bb_s[wid][6] = hm;
            }
            __syncthreads();
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                b0[d] = fminf(bb_s[0][d], bb_s[1][d]);
                b1[d] = fmaxf(bb_s[0][3 + d], bb_s[1][3 + d]);
            }
            hown = fmaxf(bb_s[0][6], bb_s[1][6]);
        }
        // a6: the largest h that can reach the bucket sets the reach R = 2 max(h_i, H)
        const float Hs = sph_box_scatter_hmax(g, coarse, b0, b1, hown, hmax_all, lane);

        // ---- which targets the kept lists serve
        const uint32_t reg = bucket_loff[bi];
        const float    Rt  = bucket_rt[bi];
        const bool     haslist = reg != 0xffffffffu && Rt > 0.0f;
        const uint32_t* const lb = nb_j + (size_t)(haslist ? reg : 0u) * ((size_t)par.lcap * SPH_TB) + tid;
        bool cov = false;
        {
            const float R   = 2.0f * (1.0f + 1e-5f) * fmaxf(tg.pi.w, Hs);
            const float tau = 1e-6f + 2.5e-7f * g.xext * tg.ih;
            const float rk  = valid ? tl_rkeep[p] : 0.0f;
            cov = valid && haslist && R * (1.0f + 4.0f * tau) <= rk;
        }
        // ---- the bucket's tile, as the density sweep staged it (same box, same radius)
        bool staged = false;
        if (haslist) {
            __syncthreads();
            if (wid == 0) {
                SphTileInfo tl;
                tl.ok = sph_tile_stage(g, cell_start, pos_h, b0, b1, Rt * (1.0f + 1e-5f), sm, lane, tl,
                                       vel_m, v_sa, rcak, q_sa) ? 1 : 0;
                if (lane == 0) ti = tl;
            }
            __syncthreads();
            staged = ti.ok != 0;
        }
        if (haslist && !staged && big_list) {   // to the second pass, which has a larger tile
            if (tid == 0) big_list[atomicAdd(big_cnt, 1u)] = bi;
            continue;
        }
        if (!staged) cov = false;
        // not served: to the 8-lane kernel, which searches
        if (valid && !cov) fb_list[atomicAdd(fb_cnt, 1u)] = (uint32_t)p;
        if (!staged) continue;
        const int cnt    = cov ? (int)nb_cnt[p] : 0;
        const int maxcnt = __reduce_max_sync(SPH_FULL, cnt);
        // Does the bucket's reach cross a periodic face?  If not, no pair of it needs the minimum
        // image (uniform, decided once).
        bool wraps = false;
        {
            const float Rb = 2.0f * (1.0f + 1e-4f) * Hs;
#pragma unroll
            for (int d = 0; d < 3; ++d)
                wraps = wraps || (g.per[d] && (b0[d] - Rb < g.lo[d] || b1[d] + Rb > g.lo[d] + g.len[d]));
        }
        sph_mbar_wait(sm.bar, parity);
        parity ^= 1u;
        Accum acc;
        const uint32_t own = (uint32_t)ti.used;   // past the end of the list: a padding slot (never accepted)
        auto entry = [&](int f) -> uint32_t { return f < cnt ? __ldg(lb + (size_t)f * SPH_TB) : own; };
        struct PairIn { float4 vj, rj; float dx, dy, dz, r2, hj; bool ok; };
        auto fetch = [&](int f, uint32_t j, auto wrap_tag, PairIn& q) -> bool {
            constexpr bool WRAP = decltype(wrap_tag)::value;
            const float4 pj = sph_lds4(p_sa + 16u * j);
            q.vj = sph_lds4(v_sa + 16u * j);
            q.rj = sph_lds4(q_sa + 16u * j);
            q.dx = tg.pi.x - pj.x; q.dy = tg.pi.y - pj.y; q.dz = tg.pi.z - pj.z;
            if (WRAP) {   // minimum image
                q.dx -= Lx * rintf(q.dx * iLx);
                q.dy -= Ly * rintf(q.dy * iLy);
                q.dz -= Lz * rintf(q.dz * iLz);
            }
            q.r2 = q.dx * q.dx + q.dy * q.dy + q.dz * q.dz;
            q.hj = pj.w;
            const float hm = fmaxf(tg.pi.w, pj.w);
            q.ok = f < cnt && q.r2 < 4.0f * hm * hm && q.r2 > 0.0f;
            return q.ok && force_pair_vr(tg, q.vj, q.dx, q.dy, q.dz) < 0.0f;
        };
        auto sweep = [&](auto wrap_tag) {
            constexpr int NE = TL_NE;   // entries per trip: independent chains
            // the list entries (global memory) are loaded two trips ahead
            uint32_t jc[NE], jn[NE];
#pragma unroll
            for (int e = 0; e < NE; ++e) { jc[e] = entry(e); jn[e] = entry(NE + e); }
            for (int f = 0; f < maxcnt; f += NE) {
                uint32_t jf[NE];
#pragma unroll
                for (int e = 0; e < NE; ++e) jf[e] = entry(f + 2 * NE + e);
                PairIn q[NE];
                bool   av = false;
#pragma unroll
                for (int e = 0; e < NE; ++e) av = fetch(f + e, jc[e], wrap_tag, q[e]) || av;
                if (__any_sync(SPH_FULL, av)) {
#pragma unroll
                    for (int e = 0; e < NE; ++e)
                        force_pair_nb<KERN, ENT, true>(tg, acc, par.fp, q[e].ok, q[e].vj, q[e].rj, q[e].dx, q[e].dy,
                                                       q[e].dz, q[e].r2, q[e].hj);
                } else {
#pragma unroll
                    for (int e = 0; e < NE; ++e)
                        force_pair_nb<KERN, ENT, false>(tg, acc, par.fp, q[e].ok, q[e].vj, q[e].rj, q[e].dx, q[e].dy,
                                                        q[e].dz, q[e].r2, q[e].hj);
                }
#pragma unroll
                for (int e = 0; e < NE; ++e) { jc[e] = jn[e]; jn[e] = jf[e]; }
            }
        };
        if (wraps && anyper) sweep(std::true_type{});
        else                 sweep(std::false_type{});
        if (cov) {
            const int i = perm[p];
            ax[i] = acc.ax; ay[i] = acc.ay; az[i] = acc.az;
            dudt[i]   = acc.du;
            mu_min[i] = acc.mumin;
            c_pairs += acc.pairs;
            c_av    += acc.av;
        }
    }
    const unsigned tp = __reduce_add_sync(SPH_FULL, c_pairs), ta = __reduce_add_sync(SPH_FULL, c_av);
    if (lane == 0) {
        if (tp) atomicAdd(stats + ST_FORCE_PAIRS, (unsigned long long)tp);
        if (ta) atomicAdd(stats + ST_FORCE_AV, (unsigned long long)ta);
    }
}

}  // namespace

// Sweeps the buckets whose targets have kept lists of tile indices; the targets it hands back
// are in c->fb_list (c->fb_cnt[1] of them) and are swept by the caller with the 8-lane kernel.
int sph_launch_forces_tlist(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min) {
    cudaStream_t s = c->stream;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fb_cnt + 1, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->tile_next + 2, 0, 2 * sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->big_cnt + 1, 0, sizeof(unsigned), s));
    auto launch2 = [&](auto tag, auto etag) -> cudaError_t {
        constexpr int  KERN = decltype(tag)::value;
        constexpr bool ENT  = decltype(etag)::value;
        for (int pass = 0; pass < 2; ++pass) {
            const int  tcap = pass == 0 ? c->par.tile_cap : c->par.tile_cap2;
            const bool two  = c->par.tile_cap2 >= c->par.tile_cap + 32;
            if (pass == 1 && !two) break;
            TlPar par{ForcePar{c->par.av_alpha, c->par.av_beta, c->par.av_eps}, tcap, c->lcap};
            const size_t smem = tl_smem_bytes(tcap);
            cudaError_t e = cudaFuncSetAttribute(k_forces_tlist<KERN, ENT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            int per_sm = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_forces_tlist<KERN, ENT>, 64, smem);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            const bool last = pass == 1 || !two;
            k_forces_tlist<KERN, ENT><<<c->sm_count * per_sm, 64, smem, s>>>(
                c->grid, c->cell_start, c->pos_h, c->vel_m, c->rcak, c->perm, c->buckets,
                pass == 0 ? c->bucket_cnt : c->big_cnt + 1, pass == 0 ? nullptr : c->big_list,
                last ? nullptr : c->big_list, c->big_cnt + 1, c->tile_next + 2 + pass, par, c->coarse_hmax,
                c->nb_j, c->bucket_loff, c->bucket_rt, c->nb_cnt, c->tl_rkeep, ax, ay, az, dudt, mu_min,
                c->fb_list, c->fb_cnt + 1, c->stats);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    auto launch = [&](auto tag) -> cudaError_t {
        return c->par.entropy ? launch2(tag, std::true_type{}) : launch2(tag, std::false_type{});
    };
    cudaError_t e;
    switch (c->par.kernel) {
    case 0: e = launch(std::integral_constant<int, 0>{}); break;
    case 2: e = launch(std::integral_constant<int, 2>{}); break;
    case 3: e = launch(std::integral_constant<int, 3>{}); break;
    default: e = launch(std::integral_constant<int, 1>{}); break;
    }
    SPH_CUDA_CHECK(c, e);
    return SPH_OK;
}
