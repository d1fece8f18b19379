// sph_tile_forces.cu -- steps a6, a8, a9 of DESIGN.md on the staged-tile path: the hydro force
// pass of PAPER.md:186-219 (Section 2.3.5), Eqs. (13)-(18), pair set 0 < r < 2 max(h_i, h_j)
// (gather and scatter), with one lane per pair of targets over a shared-memory
// tile of source records (sph_tile.cuh).
//
// Per bucket of <= 64 targets: the largest h that can reach the bucket is bounded from the
// coarse max-h map (a6), which fixes the reach R; the three 16-byte records of every source in
// the cell rows within R -- (x, y, z, h), (v, m), (rho, c, A, K) -- are staged by bulk
// asynchronous copies; phase 1 turns the tile into accept masks (a superset: distance below
// R); each lane then walks its two targets' masks and evaluates the pairs that pass the exact
// test with the arithmetic of sph_force_pair.cuh.  No lists in global memory, no reductions
// across lanes.  Buckets the tile cannot hold go to k_forces (8 lanes per target) through a
// target list.
#include <cstdio>
#include "sph_tile.cuh"
#include "sph_force_pair.cuh"

namespace {

struct FTilePar {
    ForcePar fp;
    int      tcap;
};

__host__ __device__ inline size_t ftile_smem_bytes(int tcap, int W) {
    return (size_t)(tcap + 4) * (16 + 4 + 16 + 16) + (size_t)(tcap / 32 + 2 * W) * SPH_TB * 4 +
           sph_tile_xbytes(W, 7) + 16;
}

__device__ __forceinline__ float fwarp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}
__device__ __forceinline__ float fwarp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}

// a6 for a box: the largest h_j of any particle that can reach a point of [b0, b1], bounded
// from the coarse max-h map (the bound of sph_scatter_hmax, for a box instead of a point).
// Starts from the global maximum and tightens: every such j lies within 2 H of the box as long
// as H bounds its h_j.  Warp-collective, all lanes return the same value.
__device__ __forceinline__ float tile_scatter_hmax(const SphGrid& g, const unsigned* __restrict__ coarse,
                                                   const float b0[3], const float b1[3], float hown,
                                                   float hglobal, int lane) {
    float H = fmaxf(hglobal, hown);
#pragma unroll 1
    for (int pass = 0; pass < 3; ++pass) {
        int  u0[3], nn[3];
        bool inside = true;
        const float R = 2.0f * H * (1.0f + 1e-5f);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            float a = floorf((b0[d] - g.lo[d] - R) * g.ics[d] - 1e-3f);
            float b = floorf((b1[d] - g.lo[d] + R) * g.ics[d] + 1e-3f);
            a = fminf(fmaxf(a, -1.0e9f), 1.0e9f);
            b = fminf(fmaxf(b, -1.0e9f), 1.0e9f);
            int lo = (int)a, hi = (int)b;
            if (g.per[d]) {
                inside = inside && lo >= 0 && hi <= g.cn[d] - 1;
                if (hi - lo + 1 >= g.cn[d]) { lo = 0; hi = g.cn[d] - 1; }
            } else {
                lo = min(max(lo, 0), g.cn[d] - 1);
                hi = min(max(hi, 0), g.cn[d] - 1);
            }
            u0[d] = lo;
            nn[d] = hi - lo + 1;
        }
        const bool blocks = inside && nn[0] * nn[1] * nn[2] > 512;   // read the 8^3 blocks instead
        int dx = g.cn[0], dy = g.cn[1], dz = g.cn[2];
        const unsigned* map = coarse;
        if (blocks) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const int q0 = u0[d] >> 3, q1 = (u0[d] + nn[d] - 1) >> 3;
                u0[d] = q0;
                nn[d] = q1 - q0 + 1;
            }
            dx = g.sn[0]; dy = g.sn[1]; dz = g.sn[2];
            map = coarse + SPH_COARSE_MAX;
        }
        const int cnt = nn[0] * nn[1] * nn[2];
        unsigned  best = 0u;
        for (int q = lane; q < cnt; q += 32) {
            const int t  = q / nn[0], ix = q - t * nn[0];
            const int iz = t / nn[1], iy = t - iz * nn[1];
            int cx = u0[0] + ix, cy = u0[1] + iy, cz = u0[2] + iz;
            cx -= (cx >= dx) ? dx : 0; cx += (cx < 0) ? dx : 0;
            cy -= (cy >= dy) ? dy : 0; cy += (cy < 0) ? dy : 0;
            cz -= (cz >= dz) ? dz : 0; cz += (cz < 0) ? dz : 0;
            cx = min(max(cx, 0), dx - 1);
            cy = min(max(cy, 0), dy - 1);
            cz = min(max(cz, 0), dz - 1);
            best = max(best, __ldg(map + (cz * dy + cy) * dx + cx));
        }
        best = __reduce_max_sync(SPH_FULL, best);
        const float Hn = fmaxf(hown, fminf(H, __uint_as_float(best)));
        if (Hn >= H * (1.0f - 1e-6f)) { H = Hn; break; }   // no tighter: done
        H = Hn;
    }
    return H;
}

constexpr int FT_NPART = 7;   // words per target and warp in the exchange area

// Persistent blocks of W warps, one bucket at a time; every warp holds the 64 targets and walks
// its share of the mask words (w = wid, wid + W, ...); the partial sums meet in shared memory.
template <int KERN, bool ENT>
__global__ __launch_bounds__(SPH_TWMAX * 32) void k_forces_tile(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const float4* __restrict__ vel_m,
    const float4* __restrict__ rcak, const int32_t* __restrict__ perm,
    const SphBucket* __restrict__ buckets, const unsigned* __restrict__ nbuckets,
    const uint32_t* __restrict__ blist, unsigned* big_list, unsigned* big_cnt, unsigned* next,
    FTilePar par, const unsigned* __restrict__ coarse, float* ax, float* ay, float* az, float* dudt,
    float* mu_min, uint32_t* fb_list, unsigned* fb_cnt, unsigned long long* stats) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ SphGrid     g;
    __shared__ SphTileInfo ti;
    __shared__ unsigned    bi_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, W = blockDim.x >> 5, nthr = blockDim.x;
    for (int k = tid; k < (int)(sizeof(SphGrid) / 4); k += nthr) ((int*)&g)[k] = ((const int*)gp)[k];
    // carve: tile (x', y', z', |x'|^2), hs = h_j, V = (v, m), Q = (rho, c, A, K), masks, seg / exchange, rowoff, bar
    SphTileMem sm;
    {
        unsigned char* base = smem_raw;
        const int tc = par.tcap;
        sm.tcap = tc;
        sm.tile = (float4*)base;   base += (size_t)(tc + 4) * 16;
        sm.ms   = (float*)base;    base += (size_t)(tc + 4) * 4;      // h_j here
        base += (size_t)(tc + 4) * 32;                                 // V and Q
        sm.mask = (uint32_t*)base; base += (size_t)(tc / 32 + 2 * W) * SPH_TB * 4;
        sm.seg  = (uint2*)base;    base += sph_tile_xbytes(W, FT_NPART);
        sm.zone = nullptr;
        sm.gidx = nullptr;
        sm.gidx_sa = 0u;
        sm.rowoff = (int*)sm.mask;
        sm.bar  = (uint32_t)__cvta_generic_to_shared(base);
        sm.tile_sa = (uint32_t)__cvta_generic_to_shared(sm.tile);
        sm.ms_sa   = (uint32_t)__cvta_generic_to_shared(sm.ms);
        sm.mask_sa = (uint32_t)__cvta_generic_to_shared(sm.mask);
        sm.zone_sa = 0u;
    }
    const uint32_t v_sa = sm.ms_sa + 4u * (uint32_t)(par.tcap + 4);
    const uint32_t q_sa = v_sa + 16u * (uint32_t)(par.tcap + 4);
    float* const xch = (float*)sm.seg;
    if (tid == 0) sph_mbar_init(sm.bar, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t parity = 0;
    if (g.flags & SPH_GRID_STEEP) return;   // steep h contrast: the 8-lane kernels take every target
    const unsigned nb = *nbuckets;
    const float hmax_all = __uint_as_float(g.force_hmax_bits);
    unsigned long long c_tested = 0;
    unsigned c_pairs = 0, c_av = 0;

    for (;;) {
        __syncthreads();                     // the last bucket's tile and tables are free
        if (tid == 0) bi_s = atomicAdd(next, 1u);
        __syncthreads();
        if (bi_s >= nb) break;
        const unsigned  bi = blist ? blist[bi_s] : bi_s;
        const SphBucket bk = buckets[bi];

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
        int* const rowoff = sm.rowoff + 32 * wid;
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
        __syncwarp();
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
            for (int d = 0; d < 3; ++d) { b0[d] = fwarp_min(lo[d]); b1[d] = fwarp_max(hi[d]); }
            hown = fwarp_max(hm);
        }
        // a6: scatter neighbours can be as far as 2 h_j (every warp computes the same bound)
        const float Hs = tile_scatter_hmax(g, coarse, b0, b1, hown, hmax_all, lane);
        const float Rb = 2.0f * Hs * (1.0f + 1e-5f);

        if (wid == 0) {
            SphTileInfo tl;
            tl.ok = sph_tile_stage(g, cell_start, pos_h, b0, b1, Rb * (1.0f + 4e-4f), sm, lane, tl,
                                   vel_m, v_sa, rcak, q_sa) ? 1 : 0;
            if (lane == 0) ti = tl;
        }
        __syncthreads();
        if (!ti.ok) {
            if (wid == 0) {
                if (big_list) {   // to the second pass, which has a larger tile
                    if (lane == 0) big_list[atomicAdd(big_cnt, 1u)] = bi;
                } else {          // whole bucket to the 8-lanes-per-target kernel
#pragma unroll
                    for (int t = 0; t < 2; ++t)
                        if (valid[t]) fb_list[atomicAdd(fb_cnt, 1u)] = (uint32_t)p[t];
                }
            }
            continue;
        }
        // (x, y, z, h) -> (x', y', z', |x'|^2), h -> ms[]; the padding carries h = 1
        sph_tile_finish(g, sm, ti, parity, tid, nthr, 1.0f);
        parity ^= 1u;
        c_tested += (unsigned long long)ti.used * (unsigned)ntar;

        float xt[2], yt[2], zt[2], rr[2];
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            xt[t] = (float)((double)tg[t].pi.x - (double)ti.ox);
            yt[t] = (float)((double)tg[t].pi.y - (double)ti.oy);
            zt[t] = (float)((double)tg[t].pi.z - (double)ti.oz);
            // the mask is a superset: everything within the reach of the target (+ the rounding
            // of the expanded distance); the exact pair test follows in the walk
            rr[t] = valid[t] ? 2.0f * fmaxf(tg[t].pi.w, Hs) * (1.0f + 2e-4f) : 0.0f;
        }
        sph_tile_masks(sm, ti, xt, yt, zt, rr, lane, wid, W);   // this warp's share of the words
        if (W > 1) __syncthreads();                              // every warp walks all of them

        // the pair evaluation dominates the cursor: the warps split the ENTRIES (step wid of
        // every W), each running the cursor over all mask words
        Accum acc[2];
        sph_tile_walk(sm, ti, lane, 0, 1, valid, [&](int t, const SphEntry& en) {
            const float dx = xt[t] - en.c.x, dy = yt[t] - en.c.y, dz = zt[t] - en.c.z;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const float hj = en.m;   // ms[] holds h_j on this path
            const float hm = fmaxf(tg[t].pi.w, hj);
            const bool  ok = en.has && r2 < 4.0f * hm * hm && r2 > 0.0f;
            const float4 vj = sph_lds4(v_sa + 16u * (uint32_t)en.idx);
            const float4 rj = sph_lds4(q_sa + 16u * (uint32_t)en.idx);
            force_pair_nb<KERN, ENT>(tg[t], acc[t], par.fp, ok, vj, rj, dx, dy, dz, r2, hj);
        }, wid, W);
        // ---- the warps' partial sums meet in shared memory; fixed order of addition
        if (W > 1) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                float* x = xch + (wid * FT_NPART) * SPH_TB + lane + 32 * t;
                x[0] = acc[t].ax; x[SPH_TB] = acc[t].ay; x[2 * SPH_TB] = acc[t].az; x[3 * SPH_TB] = acc[t].du;
                x[4 * SPH_TB] = acc[t].mumin;
                x[5 * SPH_TB] = __int_as_float((int)acc[t].pairs);
                x[6 * SPH_TB] = __int_as_float((int)acc[t].av);
            }
            __syncthreads();
            if (wid != 0) continue;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                Accum a;
                for (int w = 0; w < W; ++w) {
                    const float* x = xch + (w * FT_NPART) * SPH_TB + lane + 32 * t;
                    a.ax += x[0]; a.ay += x[SPH_TB]; a.az += x[2 * SPH_TB]; a.du += x[3 * SPH_TB];
                    a.mumin = fminf(a.mumin, x[4 * SPH_TB]);
                    a.pairs += (unsigned)__float_as_int(x[5 * SPH_TB]);
                    a.av    += (unsigned)__float_as_int(x[6 * SPH_TB]);
                }
                acc[t] = a;
            }
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            if (!valid[t]) continue;
            const int i = perm[p[t]];
            ax[i] = acc[t].ax; ay[i] = acc[t].ay; az[i] = acc[t].az;
            dudt[i]   = acc[t].du;
            mu_min[i] = acc[t].mumin;
            c_pairs += acc[t].pairs;
            c_av    += acc[t].av;
        }
    }
    if (wid == 0) {
        const unsigned tp = __reduce_add_sync(SPH_FULL, c_pairs), ta = __reduce_add_sync(SPH_FULL, c_av);
        if (lane == 0) {
            if (c_tested) atomicAdd(stats + ST_FORCE_TESTED, c_tested);
            if (tp) atomicAdd(stats + ST_FORCE_PAIRS, (unsigned long long)tp);
            if (ta) atomicAdd(stats + ST_FORCE_AV, (unsigned long long)ta);
        }
    }
}

}  // namespace

// Runs the tile kernel over all buckets (tile of tile_fcap candidates), then over the buckets
// that did not fit with a larger tile; the targets left after that are in c->fb_list
// (c->fb_cnt[1] of them) and are swept by the caller with the 8-lanes-per-target kernel.
#define SPH_FTCAP_BIG 1536
int sph_launch_forces_tile(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min) {
    cudaStream_t s = c->stream;
    const int    W = c->par.tile_fwarps;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->tile_next + 2, 0, 2 * sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fb_cnt + 1, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->big_cnt + 1, 0, sizeof(unsigned), s));
    auto launch2 = [&](auto tag, auto etag) -> cudaError_t {
        constexpr int  KERN = decltype(tag)::value;
        constexpr bool ENT  = decltype(etag)::value;
        for (int pass = 0; pass < 2; ++pass) {
            const int  tcap = pass == 0 ? c->par.tile_fcap : SPH_FTCAP_BIG;
            const bool two  = c->par.tile_fcap < SPH_FTCAP_BIG && c->par.tile_cap2 >= c->par.tile_cap + 32;
            if (pass == 1 && !two) break;
            FTilePar par{{c->par.av_alpha, c->par.av_beta, c->par.av_eps}, tcap};
            const size_t smem = ftile_smem_bytes(tcap, W);
            cudaError_t e = cudaFuncSetAttribute(k_forces_tile<KERN, ENT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            int per_sm = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_forces_tile<KERN, ENT>, 32 * W, smem);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            const bool last = pass == 1 || !two;
            k_forces_tile<KERN, ENT><<<c->sm_count * per_sm, 32 * W, smem, s>>>(
                c->grid, c->cell_start, c->pos_h, c->vel_m, c->rcak, c->perm, c->buckets,
                pass == 0 ? c->bucket_cnt : c->big_cnt + 1, pass == 0 ? nullptr : c->big_list,
                last ? nullptr : c->big_list, c->big_cnt + 1, c->tile_next + 2 + pass, par, c->coarse_hmax,
                ax, ay, az, dudt, mu_min, c->fb_list, c->fb_cnt + 1, c->stats);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    auto launch = [&](auto tag) -> cudaError_t {
        if (c->par.entropy) return launch2(tag, std::true_type{});
        return launch2(tag, std::false_type{});
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
