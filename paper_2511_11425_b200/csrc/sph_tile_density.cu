// sph_tile_density.cu -- steps a3-a6 of DESIGN.md on the staged-tile path: the bucket table
// (buckets / groups of sinks) and the density + smoothing-length solve of
// PAPER.md:137-154, Eqs. (5)-(7), with one lane per pair of targets over a shared-memory tile
// of candidate sources (sph_tile.cuh).  The arithmetic of the solve is the one documented in
// sph_density.cu (Halley step on S, E, F with Taylor-carried sums); only the parallel shape
// differs (Wendland C2 solves Eq. (6) from the moments of ONE sweep, see below):
//   * one warp owns a bucket of <= 64 targets, two per lane;
//   * the bucket's candidate rows are staged once by bulk asynchronous copies (UBLKCP) that
//     complete on an mbarrier, then moved into the bucket's frame;
//   * phase 1 turns the tile into per-target accept masks (FFMA2 on broadcast loads);
//   * each sweep walks a lane-private cursor over its masks: no ballots, no shuffles, no
//     per-candidate list stores, no reduction across lanes;
//   * the accepted entries' sorted positions go to a bucket-major list in global memory, from
//     the sweep itself: the neighbour lists the force sweep reads (sph_forces_list.cu).
// Buckets the tile cannot hold (too many rows or candidates: steep h contrast, a periodic axis
// barely longer than the search ball) are handed to the 8-lanes-per-target kernel of
// sph_density.cu through a target list; targets with a borderline neighbour or without
// convergence go to k_density_fix as before.
#include <cstdio>
#include "sph_tile.cuh"

namespace {

constexpr float T_ACCEPT = 3.0e-4f;   // a Halley step below this is final (sph_density.cu)
constexpr float T_EDGE   = 4.0e-4f;   // list entries within this of 2h are kept for the final count

// ------------------------------------------------------------------------------------------
// a3: the bucket table.  One warp per group of G x G adjacent rows of cells; it walks along x
// and closes a bucket as soon as the next cell would take it past 64 particles (or 32 cells).
// The group's cumulative counts along x are summed over the rows a chunk of cells at a time
// (independent loads, all lanes busy) into shared memory; the cuts, which are sequential, then
// run on shared memory alone.
// ------------------------------------------------------------------------------------------
constexpr int BK_WARPS = 8;
constexpr int BK_CHUNK = 2048;   // cells of a group held in shared memory at a time

__global__ __launch_bounds__(BK_WARPS * 32) void k_buckets(const SphGrid* __restrict__ gp,
                                                          const uint32_t* __restrict__ cs, int G,
                                                          SphBucket* out, unsigned* nout) {
    __shared__ uint32_t  cum[BK_CHUNK + 1];
    __shared__ SphBucket stage[32];
    __shared__ int       q_s;
    const SphGrid& g = *gp;
    if (g.flags & SPH_GRID_STEEP) return;   // the tile sweeps stand down: nobody reads the table
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int ngy = (g.ny + G - 1) / G, ngz = (g.nz + G - 1) / G;
    int nst = 0;   // warp 0: staged buckets (uniform); the table's counter is asked for 32 at a time
    auto flush = [&]() {
        __syncwarp();
        unsigned at = 0;
        if (lane == 0 && nst > 0) at = atomicAdd(nout, (unsigned)nst);
        at = __shfl_sync(SPH_FULL, at, 0);
        if (lane < nst) out[at + lane] = stage[lane];
        __syncwarp();
        nst = 0;
    };
    for (int grp = (int)blockIdx.x; grp < ngy * ngz; grp += (int)gridDim.x) {   // one block per group
        const int gy = grp % ngy, gz = grp / ngy;
        const int ry0 = gy * G, rz0 = gz * G;
        const int nry = min(G, g.ny - ry0), nrz = min(G, g.nz - rz0), nrows = nry * nrz;
        auto rowbase = [&](int rho) {
            return (uint32_t)((rz0 + rho / nry) * g.ny + (ry0 + rho % nry)) * (uint32_t)g.nx;
        };
        int pos = 0;
        while (pos < g.nx) {
            // cum[k] = particles of the group's rows in the cells before pos + k (all threads)
            const int len = min(BK_CHUNK, g.nx - pos);
            __syncthreads();
            for (int k = tid; k <= len; k += BK_WARPS * 32) {
                uint32_t v = 0;
                for (int r0 = 0; r0 < nrows; r0 += 5) {
                    uint32_t t[5];
#pragma unroll
                    for (int u = 0; u < 5; ++u) t[u] = (r0 + u < nrows) ? __ldg(cs + rowbase(r0 + u) + pos + k) : 0u;
                    v += (t[0] + t[1]) + (t[2] + t[3]) + t[4];
                }
                cum[k] = v;
            }
            __syncthreads();
            if (wid == 0) {   // the cuts are sequential: one warp, on shared memory alone
                const bool tail = pos + len >= g.nx;   // the chunk ends where the rows end
                int q = 0;
                while (q < len && (q + 32 <= len || tail)) {
                    const uint32_t base = cum[q];
                    const int      c    = q + 1 + lane;
                    const uint32_t cu   = c <= len ? cum[c] : 0u;
                    const bool     ok   = c <= len && cu - base <= (uint32_t)SPH_TB;
                    const unsigned bal  = __ballot_sync(SPH_FULL, ok);
                    int m = (bal == SPH_FULL) ? 32 : __ffs((int)~bal) - 1;
                    if (m == 0) {   // the cells of this slab alone hold more than 64: one row, 64 at a time
                        if (lane < nrows) {
                            const uint32_t rb = rowbase(lane);
                            const int cnt = (int)(__ldg(cs + rb + pos + q + 1) - __ldg(cs + rb + pos + q));
                            for (int skip = 0; skip < cnt; skip += SPH_TB) {
                                SphBucket b{ry0 + lane % nry, rz0 + lane / nry, pos + q, pos + q + 1, 1, 1, skip, 0};
                                out[atomicAdd(nout, 1u)] = b;
                            }
                        }
                        m = 1;
                    } else {
                        const uint32_t tot = cum[q + m] - base;
                        if (tot > 0u) {
                            if (lane == 0) stage[nst] = SphBucket{ry0, rz0, pos + q, pos + q + m, nry, nrz, 0, 0};
                            if (++nst == 32) flush();
                        }
                    }
                    q += m;
                }
                if (lane == 0) q_s = q;
            }
            __syncthreads();
            pos += q_s;
        }
        if (wid == 0) flush();
    }
}

struct TilePar {
    float n_ngb, tol, slack;
    int   max_iter, tcap, lcap;
    int   lmode;   // what a kept-list entry is: 0 the sorted position of the source, 1 its index in the
                   // bucket's tile (the force sweep stages the same tile again: sph_forces_tlist.cu)
};

// One safeguarded Halley step from the sums at h (the step of sph_density.cu: same formulas,
// same safeguards).  Returns true if the step is accepted as final.
__device__ __forceinline__ bool tile_halley(float s, float e, float f2, float T, float h, float ih,
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
    const bool small  = fabsf(dh) <= T_ACCEPT * h;
    const bool tight  = (hhi - hlo) <= tol * h;
    const bool capped = (hn >= hcap && h >= hcap);
    conv = !(capped && f < 0.0f);
    return (genuine && small) || tight || capped;
}

__device__ __forceinline__ float tile_hcap(const SphGrid& g) {   // as density_hcap of sph_density.cu
    float hcap = 3.0e37f;
    for (int d = 0; d < 3; ++d)
        if (g.per[d]) hcap = fminf(hcap, g.len[d] / (4.0f * 1.25f) * 0.999f);
        else          hcap = fminf(hcap, 4.0f * fmaxf(g.len[0], fmaxf(g.len[1], g.len[2])));
    return hcap;
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}

// ------------------------------------------------------------------------------------------
// Wendland C2 on the tile: ONE sweep per solve.  With s = r / (2 h0), t = 1 - s the kernel is
// w~ = t^4 (1 + 4 s) = B0 + 5 B1 and -q w~' = 20 s^2 t^3 = 20 B2 in the Bernstein basis
// B_k = s^k t^(5-k); under h = h0 / lam the variables map linearly, s' = lam s, t' = t + eps s
// (eps = 1 - lam), hence B_k' = lam^k sum_j C(5-k, j) eps^j B_(k+j): the six moments
// M_k = sum_j m_j B_k(r_j / 2 h0) give S(h) and E(h) = dS/dln h EXACTLY as polynomials in lam,
// for every h at which no list entry crosses the support edge.  Entries within T_ZONE of the
// edge ("zone", a few per target) are remembered by tile index and their clamped contribution
// is put right by one short pass at the solution.  The root of Eq. (6) then costs a scalar
// Newton iteration per target -- no second sweep over the neighbours (the Halley path needs
// two).  All terms of the expansions are positive for eps > 0 and well scaled: measured against
// the FP64 root h agrees to 3e-7, rho to 9e-7, Omega to 2e-6 (FP32 emulation, lattices and
// Poisson points with unequal masses; tolerance 1e-5).  A solution with |eps| > 0.9 T_ZONE is
// only a step: the sweep is repeated from there (2-3 sweeps from a guess 25 % off).
// ------------------------------------------------------------------------------------------
constexpr float T_ZONE = 0.03f;

__device__ __forceinline__ void c2_poly(const float M[6], float lam, float& S, float& E) {
    const float e = 1.0f - lam;
    const float S0 = M[0] + e * (5.0f * M[1] + e * (10.0f * M[2] + e * (10.0f * M[3] + e * (5.0f * M[4] + e * M[5]))));
    const float S1 = M[1] + e * (4.0f * M[2] + e * (6.0f * M[3] + e * (4.0f * M[4] + e * M[5])));
    const float E2 = M[2] + e * (3.0f * M[3] + e * (3.0f * M[4] + e * M[5]));
    S = S0 + 5.0f * lam * S1;
    E = 20.0f * lam * lam * E2;
}

// ------------------------------------------------------------------------------------------
// a4-a6 on the tile.  Persistent blocks of NW = 2 / NT warps; a block takes one bucket at a
// time (handed out by a counter) and every thread owns NT of its 64 targets (columns
// tid + 32 t of the mask words): NT = 2, one warp, two targets per lane; NT = 1, two warps,
// one target per thread.  The block stages the tile once (warp 0 issues the copies), all
// threads move it into the bucket's frame, the warps split the mask words of phase 1, and
// then every thread walks, solves and stores its own targets -- no exchange of partial sums.
// Decisions that steer the block (another stage, another sweep, new masks) are block-wide
// votes through shared memory.
// ------------------------------------------------------------------------------------------
#ifndef SPH_DT_NSET
#define SPH_DT_NSET 0   // 0: 3 with one target per thread, 2 with two
#endif

template <int KERN, int NT>
__global__ __launch_bounds__(64 / NT, NT == 1 ? 7 : 8) void k_density_tile(
    const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_m, const int32_t* __restrict__ perm,
    const SphBucket* __restrict__ buckets, const unsigned* __restrict__ nbuckets,
    const uint32_t* __restrict__ blist, unsigned* big_list, unsigned* big_cnt, unsigned* next,
    TilePar par, float* h_io, float* rho, float* omega, int32_t* nn, int32_t* fix_list,
    unsigned* fix_cnt, uint32_t* fb_list, unsigned* fb_cnt, uint32_t* nb_j, unsigned nb_regions,
    unsigned* list_next, uint32_t* bucket_loff, uint32_t* nb_cnt, float* nb_rkeep, float* tl_rkeep,
    float* bucket_rt, unsigned long long* stats) {
    constexpr bool MOM = (KERN == 1);   // the moment solve exists for Wendland C2
    constexpr int  NW = 2 / NT, NTHR = 32 * NW;
    constexpr int  NSET = SPH_DT_NSET > 0 ? SPH_DT_NSET : (NT == 1 ? 3 : 2);   // entries in flight per target in the sweep
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ SphGrid     g;
    __shared__ SphTileInfo ti;
    __shared__ unsigned    bi_s, lreg_s;
    __shared__ float       bb_s[2][8];      // per warp: bounding box of its targets, first list radius
    __shared__ float       xf_s[2][2];      // block votes: [phase][warp]
    __shared__ unsigned    xu_s[2][2];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int k = tid; k < (int)(sizeof(SphGrid) / 4); k += NTHR) ((int*)&g)[k] = ((const int*)gp)[k];
    const SphTileMem sm = sph_tile_carve<16>(smem_raw, par.tcap, sph_tile_xbytes(1, 0), NW);
    // the targets' mask parameters (sph_tgt_put): the segment table's memory, dead once the tile is in place
    float* const  tgt  = (float*)sm.seg;
    float* const  edge = (float*)sm.zone;   // Halley path: [DT_NEDGE][64] floats, the whole zone area
    constexpr int DT_NEDGE = SPH_TZCAP / 2;
    if (tid == 0) sph_mbar_init(sm.bar, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t parity = 0;
    if (g.flags & SPH_GRID_STEEP) return;   // steep h contrast: the 8-lane kernels take every target
    const unsigned nb = *nbuckets;
    const float hcap = tile_hcap(g);
    const float lslack = MOM ? (1.0f + T_ZONE) * 1.001f : par.slack;   // list radius / 2h
    unsigned long long c_tested = 0;
    unsigned c_listed = 0, c_pairs = 0, c_sweeps = 0, c_recollect = 0;
    int xph = 0;
    auto block_sync = [&]() { if constexpr (NW > 1) __syncthreads(); else __syncwarp(); };
    auto block_max = [&](float v) -> float {
        v = warp_max(v);
        if constexpr (NW > 1) {
            if (lane == 0) xf_s[xph][wid] = v;
            __syncthreads();
            v = fmaxf(xf_s[xph][0], xf_s[xph][1]);
            xph ^= 1;
        }
        return v;
    };
    auto block_or = [&](unsigned v) -> unsigned {
        v = __reduce_or_sync(SPH_FULL, v);
        if constexpr (NW > 1) {
            if (lane == 0) xu_s[xph][wid] = v;
            __syncthreads();
            v = xu_s[xph][0] | xu_s[xph][1];
            xph ^= 1;
        }
        return v;
    };
    // the next bucket's number is asked for one bucket ahead (thread 0 holds it)
    unsigned nxt = 0;
    if (tid == 0) nxt = atomicAdd(next, 1u);

    for (;;) {
        __syncthreads();                     // the last bucket's tile and tables are free
        if (tid == 0) bi_s = nxt;
        __syncthreads();
        const unsigned bslot = bi_s;
        if (bslot >= nb) break;
        if (tid == 0) nxt = atomicAdd(next, 1u);
        // the buckets of the table, or (second pass, larger tile) the ones the first pass left
        const unsigned  bi = blist ? blist[bslot] : bslot;
        const SphBucket bk = buckets[bi];
        // The neighbour lists kept for the force sweep ("we keep the precomputed
        // interaction list"): entry f of target t of this bucket at lbase[f * 64 + t], the
        // sorted position of the source -- written from the sweep as the entries are met, so a
        // warp's stores fall into a few 256-byte rows.  The bucket takes one region of
        // lcap x 64 words from the pool (none left: no lists, the force sweep searches).
        if (tid == 0) {
            unsigned reg = 0xffffffffu;
            if (nb_j != nullptr) {
                if (blist) reg = bucket_loff[bi];   // second pass: the region the first pass took
                if (reg == 0xffffffffu) {
                    reg = atomicAdd(list_next, 1u);
                    if (reg >= nb_regions) reg = 0xffffffffu;
                    bucket_loff[bi] = reg;
                }
            }
            lreg_s = reg;   // read behind the barriers of the first stage
        }

        // ---- the bucket's targets: rows (ry0 + a, rz0 + b), cells [c0, c1) of each
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
        int* const rowoff = sm.rowoff + 32 * wid;   // in the mask area: free until phase 1
        rowoff[lane] = inc;                      // inclusive prefix of the row counts
        __syncwarp();
        int    kc[NT], p[NT];                    // target column, sorted position
        bool   valid[NT];
        float  xg[NT], yg[NT], zg[NT], mi[NT], h[NT];
        int    ic[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const int k = tid + 32 * t;
            kc[t]    = k;
            valid[t] = k < ntar;
            int rho_ = 0;
            while (rho_ < 31 && rowoff[rho_] <= k) ++rho_;
            const int before = rho_ ? rowoff[rho_ - 1] : 0;
            const int start  = __shfl_sync(SPH_FULL, rs, rho_);
            p[t] = valid[t] ? start + (k - before) : 0;
            float4 pi = make_float4(0.f, 0.f, 0.f, 1.f);
            ic[t] = 0;
            h[t]  = g.hmin;
            if (valid[t]) {
                pi    = pos_m[p[t]];
                ic[t] = perm[p[t]];
                h[t]  = h_io[ic[t]];
            }
            if (!(h[t] > 0.0f) || !(h[t] < 3.0e38f)) h[t] = g.hmin;
            h[t]  = fminf(h[t], hcap);
            xg[t] = pi.x; yg[t] = pi.y; zg[t] = pi.z; mi[t] = pi.w;
        }
        __syncwarp();

        float T[NT], hlo[NT], hhi[NT], S[NT], E[NT], Rc[NT], want[NT];
        bool  done[NT], fix[NT], wait[NT], recount[NT], mvalid[NT];
        int   sweeps[NT], ni[NT], nlist[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            T[t]   = par.n_ngb * mi[t] * (1.0f / SphKernel<KERN>::self);
            hlo[t] = 0.0f; hhi[t] = __int_as_float(0x7f800000);
            S[t] = 0.0f; E[t] = 0.0f; Rc[t] = 0.0f;
            done[t] = !valid[t]; fix[t] = false; wait[t] = valid[t];
            want[t] = valid[t] ? 2.0f * h[t] * lslack : 0.0f;
            sweeps[t] = 0; ni[t] = 0; recount[t] = false; mvalid[t] = false; nlist[t] = 0;
        }
        // bounding box of the block's targets and the first list radius
        float b0[3], b1[3], Rt;
        {
            const float INF = __int_as_float(0x7f800000);
            float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF}, wr = 0.0f;
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (valid[t]) {
                    lo[0] = fminf(lo[0], xg[t]); hi[0] = fmaxf(hi[0], xg[t]);
                    lo[1] = fminf(lo[1], yg[t]); hi[1] = fmaxf(hi[1], yg[t]);
                    lo[2] = fminf(lo[2], zg[t]); hi[2] = fmaxf(hi[2], zg[t]);
                    wr = fmaxf(wr, want[t]);
                }
#pragma unroll
            for (int d = 0; d < 3; ++d) { b0[d] = warp_min(lo[d]); b1[d] = warp_max(hi[d]); }
            Rt = warp_max(wr);
            if constexpr (NW > 1) {
                if (lane == 0) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) { bb_s[wid][d] = b0[d]; bb_s[wid][3 + d] = b1[d]; }
                    bb_s[wid][6] = Rt;
                }
                __syncthreads();
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    b0[d] = fminf(bb_s[0][d], bb_s[1][d]);
                    b1[d] = fmaxf(bb_s[0][3 + d], bb_s[1][3 + d]);
                }
                Rt = fmaxf(bb_s[0][6], bb_s[1][6]);
            }
        }
        bool fallback = false;
        uint32_t* lbase = nullptr;
        int   ntiles = 0;        // tiles staged for this bucket (uniform)
        float rt_used = 0.0f;    // radius of the last one

        // ---- stages: (re)build the tile for the largest list radius wanted
        for (int stage = 0; stage < 4 && Rt > 0.0f; ++stage) {
            __syncthreads();                 // everybody is done with the old tile and the targets' table
            if (wid == 0) {
                SphTileInfo tl;
                tl.ok = sph_tile_stage(g, cell_start, pos_m, b0, b1, Rt * (1.0f + 1e-5f), sm, lane, tl) ? 1 : 0;
                if (lane == 0) ti = tl;
            }
            __syncthreads();
            if (stage == 0 && lreg_s != 0xffffffffu) lbase = nb_j + (size_t)lreg_s * ((size_t)par.lcap * SPH_TB);
            if (!ti.ok) {
                if (stage == 0) fallback = true;
                else {
#pragma unroll
                    for (int t = 0; t < NT; ++t) if (wait[t]) { done[t] = true; fix[t] = true; wait[t] = false; }
                }
                break;
            }
            if (stage > 0) {
#pragma unroll
                for (int t = 0; t < NT; ++t) c_recollect += wait[t] ? 1u : 0u;
            }
            ++ntiles;
            rt_used = Rt;
#pragma unroll
            for (int t = 0; t < NT; ++t) mvalid[t] = false;   // a new tile: the masks of the old one are gone
            sph_tile_finish(g, sm, ti, parity, tid, NTHR, 0.0f);
            parity ^= 1u;
            // the targets in the frame of the tile
            float xt[NT], yt[NT], zt[NT];
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                xt[t] = (float)((double)xg[t] - (double)ti.ox);
                yt[t] = (float)((double)yg[t] - (double)ti.oy);
                zt[t] = (float)((double)zg[t] - (double)ti.oz);
            }
            const float band_c = 2.5e-7f * ti.ext;   // tau(h) = 1e-6 + band_c / h, DESIGN.md section 6
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (wait[t]) { wait[t] = false; Rc[t] = fminf(want[t], Rt); }
            bool remask = true;
            if (tid == 0) c_tested += (unsigned long long)ti.used * (unsigned)ntar;

            // ---- sweeps on this tile
            for (;;) {
                bool need = false;
#pragma unroll
                for (int t = 0; t < NT; ++t) need = need || (!done[t] && !wait[t]);
                const unsigned vote = block_or((need ? 1u : 0u) | (remask ? 2u : 0u));
                if (!(vote & 1u)) break;
                bool on[NT];
#pragma unroll
                for (int t = 0; t < NT; ++t) on[t] = !done[t] && !wait[t];
                if (vote & 2u) {
#pragma unroll
                    for (int t = 0; t < NT; ++t)
                        if (on[t]) sph_tgt_put(tgt, kc[t], -2.0f * xt[t], -2.0f * yt[t], -2.0f * zt[t],
                                               fmaf(zt[t], zt[t], fmaf(yt[t], yt[t], xt[t] * xt[t])) - Rc[t] * Rc[t]);
                        else       sph_tgt_put(tgt, kc[t], 0.0f, 0.0f, 0.0f, 3.0e38f);
                    block_sync();
                    sph_tile_masks_sh(sm, ti, tgt, lane, wid, NW);   // this warp's words, all 64 columns
                    block_sync();
                    remask = false;
#pragma unroll
                    for (int t = 0; t < NT; ++t) mvalid[t] = on[t];   // finished targets lost theirs
                }
                uint32_t* lcol[NT];   // the target's column of the bucket's list region
#pragma unroll
                for (int t = 0; t < NT; ++t) lcol[t] = lbase + kc[t];
                const int lcap = lbase ? par.lcap : 0;
                int nent[NT];
#pragma unroll
                for (int t = 0; t < NT; ++t) nent[t] = 0;
                if constexpr (MOM) {
                    // ---- one sweep: the six Bernstein moments, the zone list, the entry count
                    float M[NT][6];
                    float ihh[NT];
                    int   nz[NT];
                    uint32_t za[NT], zend[NT];
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        ihh[t] = __fdividef(0.5f, h[t]);
#pragma unroll
                        for (int k = 0; k < 6; ++k) M[t][k] = 0.0f;
                        nz[t]   = 0;
                        za[t]   = sm.zone_sa + 2u * (uint32_t)kc[t];
                        zend[t] = za[t] + 2u * SPH_TB * (SPH_TZCAP - 1);
                    }
                    sph_tile_walk_own<NT, NSET>(sm, ti, tid, on, [&](int t, const SphEntry& en) {
                        const float dx = xt[t] - en.c.x, dy = yt[t] - en.c.y, dz = zt[t] - en.c.z;
                        const float r  = sph_sqrt(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
                        const float s  = r * ihh[t], tt = 1.0f - s;
                        const float t2 = tt * tt, t3 = t2 * tt, t4 = t2 * t2, t5 = t4 * tt;
                        const float a1 = en.m * s, a2 = a1 * s, a3 = a2 * s, a4 = a3 * s, a5 = a4 * s;
                        M[t][0] = fmaf(en.m, t5, M[t][0]);
                        M[t][1] = fmaf(a1, t4, M[t][1]);
                        M[t][2] = fmaf(a2, t3, M[t][2]);
                        M[t][3] = fmaf(a3, t2, M[t][3]);
                        M[t][4] = fmaf(a4, tt, M[t][4]);
                        M[t][5] += a5;
                        {   // the kept list (a set: any sweep of this mask writes the same); predicated store
                            const uint32_t gj = par.lmode ? (uint32_t)en.idx : sph_ldsu(sm.gidx_sa + 4u * (uint32_t)en.idx);
                            const bool st = en.has && nent[t] < lcap;
                            uint32_t* const la = lcol[t] + (uint32_t)nent[t] * (uint32_t)SPH_TB;
                            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.global.u32 [%0], %1;\n\t}"
                                         ::"l"(la), "r"(gj), "r"((unsigned)st) : "memory");
                        }
                        nent[t] += en.has ? 1 : 0;
                        // next to (or beyond) the support edge: remember the entry (predicated
                        // store; past the capacity the last slot is overwritten and nz says so)
                        const bool inz = en.has && tt < T_ZONE;
                        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.shared.u16 [%0], %1;\n\t}"
                                     ::"r"(za[t]), "h"((unsigned short)en.idx), "r"((unsigned)inz) : "memory");
                        za[t] = inz ? min(za[t] + 2u * SPH_TB, zend[t]) : za[t];
                        nz[t] += inz ? 1 : 0;
                    });
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        if (!on[t]) continue;
                        const bool zfit = nz[t] <= SPH_TZCAP;
                        if (sweeps[t] == 0) c_listed += (unsigned)nent[t];
                        ++sweeps[t];
                        nlist[t] = nent[t];
                        // the sign of f at the swept h keeps the bracket (the zone's clamp is O(T_ZONE^4))
                        const float f0 = M[t][0] + 5.0f * M[t][1] - T[t];
                        if (f0 < 0.0f) hlo[t] = h[t]; else hhi[t] = h[t];
                        // scalar Newton on lam = h0 / h with the polynomial S, E
                        float lam = 1.0f, Sp = 0.0f, Ep = 0.0f;
                        bool  okp = true;
#pragma unroll 1
                        for (int it = 0; it < 3; ++it) {
                            c2_poly(M[t], lam, Sp, Ep);
                            if (!(Ep > 0.0f)) { okp = false; break; }
                            lam *= 1.0f + __fdividef(Sp - T[t], Ep);
                            lam = fminf(fmaxf(lam, 0.5f), 2.0f);
                        }
                        if (okp && zfit && fabsf(1.0f - lam) <= 0.9f * T_ZONE && h[t] / lam <= hcap) {
                            done[t] = true;
                            // ---- final: put the clamped zone entries right at lam, one more step
                            const float eps = 1.0f - lam;
                            float dS = 0.0f, dE = 0.0f, amin = 3.0e38f;
                            int   cz = 0;
                            for (int q = 0; q < nz[t]; ++q) {
                                const int    idx = sm.zone[q * SPH_TB + kc[t]];
                                const float4 c   = sm.tile[idx];
                                const float  mj  = sm.ms[idx];
                                const float dx = xt[t] - c.x, dy = yt[t] - c.y, dz = zt[t] - c.z;
                                const float r  = sph_sqrt(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
                                const float s  = r * ihh[t], tt = 1.0f - s;
                                const float tq = fmaf(eps, s, tt), sq = lam * s;   // t', s' at lam
                                amin = fminf(amin, fabsf(tq));
                                if (tq < 0.0f) {
                                    const float q2 = tq * tq, q3 = q2 * tq;
                                    dS -= mj * q2 * q2 * (tq + 5.0f * sq);
                                    dE -= 20.0f * mj * sq * sq * q3;
                                } else ++cz;
                            }
                            c2_poly(M[t], lam, Sp, Ep);
                            float lam2 = lam * (1.0f + __fdividef(Sp + dS - T[t], Ep + dE));
                            c2_poly(M[t], lam2, Sp, Ep);
                            const float hn = __fdividef(h[t], lam2);
                            const float taun = 1e-6f + band_c * __fdividef(1.0f, hn);
                            S[t] = Sp + dS; E[t] = Ep + dE; h[t] = hn;
                            ni[t] = nent[t] - nz[t] + cz;
                            // an entry closer to the edge than the band plus the last step: exact recount
                            recount[t] = amin <= taun + 1.5f * fabsf(lam2 - lam);
                            continue;
                        }
                        // ---- a step only: move, keep inside the bracket, sweep again
                        float hn;
                        if (okp) hn = __fdividef(h[t], fminf(fmaxf(lam, 1.0f / 1.35f), 1.0f / 0.7f));
                        else     hn = 1.25f * h[t];
                        if (hhi[t] < 3.0e38f && !(hn >= hlo[t] && hn <= hhi[t])) hn = 0.5f * (hlo[t] + hhi[t]);
                        const bool capped = hn >= hcap && h[t] >= hcap;
                        hn = fminf(hn, hcap);
                        if (capped || sweeps[t] >= par.max_iter || (hhi[t] - hlo[t]) <= par.tol * h[t] || !zfit) {
                            done[t] = true; fix[t] = true;   // k_density_fix settles it (and counts non-convergence)
                            continue;
                        }
                        h[t] = hn;
                        want[t] = 2.0f * hn * lslack;
                        if (want[t] <= Rt) { Rc[t] = want[t]; remask = true; }
                        else wait[t] = true;
                    }
                } else {
                    // ---- Halley path: S, E, F at h; interior count and the entries next to the edge
                    float ih[NT], Hlo[NT], Hhi[NT], s[NT], e[NT], f2[NT];
                    int   cin[NT], ne[NT];
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        ih[t]  = __fdividef(1.0f, h[t]);
                        Hlo[t] = 2.0f * h[t] * (1.0f - T_EDGE);
                        Hhi[t] = 2.0f * h[t] * (1.0f + T_EDGE);
                        s[t] = 0.0f; e[t] = 0.0f; f2[t] = 0.0f; cin[t] = 0; ne[t] = 0;
                    }
                    sph_tile_walk_own<NT, NSET>(sm, ti, tid, on, [&](int t, const SphEntry& en) {
                        const float4 c = en.c;
                        const float  mj = en.m;
                        const bool   has = en.has;
                        const float dx = xt[t] - c.x, dy = yt[t] - c.y, dz = zt[t] - c.z;
                        const float r  = sph_sqrt(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
                        float wq, eq, fq;
                        SphKernel<KERN>::sums_s(r * ih[t], wq, eq, fq);
                        s[t]  = fmaf(mj, wq, s[t]);
                        e[t]  = fmaf(mj, eq, e[t]);
                        f2[t] = fmaf(mj, fq, f2[t]);
                        {
                            const uint32_t gj = par.lmode ? (uint32_t)en.idx : sph_ldsu(sm.gidx_sa + 4u * (uint32_t)en.idx);
                            const bool st = has && nent[t] < lcap;
                            uint32_t* const la = lcol[t] + (uint32_t)nent[t] * (uint32_t)SPH_TB;
                            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.global.u32 [%0], %1;\n\t}"
                                         ::"l"(la), "r"(gj), "r"((unsigned)st) : "memory");
                        }
                        nent[t] += has ? 1 : 0;
                        cin[t]  += (has && r < Hlo[t]) ? 1 : 0;
                        if (has && r >= Hlo[t] && r < Hhi[t]) {
                            if (ne[t] < DT_NEDGE) edge[ne[t] * SPH_TB + kc[t]] = r;
                            ++ne[t];
                        }
                    });
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        if (!on[t]) continue;
                        if (sweeps[t] == 0) c_listed += (unsigned)nent[t];
                        ++sweeps[t];
                        nlist[t] = nent[t];
                        const float es = SphKernel<KERN>::escale * e[t];
                        float hn, Sn, En;
                        bool  conv;
                        const bool acc = tile_halley(s[t], es, f2[t], T[t], h[t], ih[t], hcap, par.tol,
                                                     hlo[t], hhi[t], hn, Sn, En, conv);
                        const float taun = 1e-6f + band_c * __fdividef(1.0f, hn);
                        const float needR = 2.0f * hn * (1.0f + 2.0f * taun) * (1.0f + 1e-4f);
                        if (acc && needR <= Rc[t]) {
                            const float H = 2.0f * hn, tauH = taun * H;
                            int  n = cin[t];
                            bool eg = ne[t] > DT_NEDGE;
                            for (int q = 0; q < min(ne[t], DT_NEDGE); ++q) {
                                const float r = edge[q * SPH_TB + kc[t]];
                                n += (r < H) ? 1 : 0;
                                eg |= fabsf(r - H) <= tauH;
                            }
                            S[t] = Sn; E[t] = En; h[t] = hn; ni[t] = n;
                            done[t] = true;
                            fix[t]  = !conv;
                            recount[t] = eg;
                            continue;
                        }
                        h[t] = hn;
                        if (sweeps[t] >= par.max_iter) { done[t] = true; fix[t] = true; continue; }
                        if (needR > Rc[t]) {   // the ball outgrew the list
                            want[t] = 2.0f * hn * fmaxf(par.slack, 1.25f);
                            if (needR <= Rt) { Rc[t] = fminf(want[t], Rt); remask = true; }
                            else wait[t] = true;
                        }
                    }
                }
            }
            // the next stage: the largest list radius still wanted
            float wr = 0.0f;
#pragma unroll
            for (int t = 0; t < NT; ++t) wr = fmaxf(wr, wait[t] ? want[t] : 0.0f);
            Rt = block_max(wr);
        }

        // ---- results: every thread stores its own targets
        if (fallback) {
            if (tid == 0) {
                // to the second pass, which has a larger tile (the bucket keeps its list region);
                // from the last pass to the 8-lane kernel: no tile-format list
                if (big_list) big_list[atomicAdd(big_cnt, 1u)] = bi;
                else if (lbase != nullptr) bucket_loff[bi] = 0xffffffffu;
            }
            if (!big_list) {          // whole bucket to the 8-lanes-per-target kernel
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if (valid[t]) fb_list[atomicAdd(fb_cnt, 1u)] = (uint32_t)p[t];
            }
            continue;
        }
        if (par.lmode && tid == 0) bucket_rt[bi] = (lbase != nullptr && ntiles == 1) ? rt_used : 0.0f;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (!valid[t]) continue;
            if (wait[t] || !done[t]) { fix[t] = true; done[t] = true; }
            const int i = ic[t];
            h_io[i] = h[t];
            // the list is complete inside the radius of its mask (less the rounding margin of phase 1)
            // (tile indices, lmode 1, mean something only if the bucket had one tile)
            const bool lok = lbase != nullptr && !fix[t] && mvalid[t] && nlist[t] <= par.lcap &&
                             (!par.lmode || ntiles == 1);
            nb_rkeep[p[t]] = 0.0f;     // no [target][entry] list of the 8-lane kernels for this target
            tl_rkeep[p[t]] = lok ? Rc[t] * (1.0f - 1e-4f) : 0.0f;
            nb_cnt[p[t]]   = lok ? (uint32_t)nlist[t] : 0u;
            c_sweeps += (unsigned)sweeps[t];
            if (!fix[t]) {
                const float ih = 1.0f / h[t];
                rho[i]   = SphKernel<KERN>::sigma * S[t] * ih * ih * ih;
                omega[i] = E[t] / (3.0f * S[t]);
                nn[i]    = ni[t];
            }
            if (fix[t])          fix_list[atomicAdd(fix_cnt, 1u)] = p[t];
            else if (recount[t]) fix_list[atomicAdd(fix_cnt, 1u)] = p[t] | (int32_t)0x80000000;
            else                 c_pairs += (unsigned)ni[t];
        }
    }

    // ---- counters: one atomic per warp and counter
    {
        const unsigned tl = __reduce_add_sync(SPH_FULL, c_listed), tp = __reduce_add_sync(SPH_FULL, c_pairs);
        const unsigned tsw = __reduce_add_sync(SPH_FULL, c_sweeps), trc = __reduce_add_sync(SPH_FULL, c_recollect);
        if (lane == 0) {
            if (c_tested) atomicAdd(stats + ST_DENS_TESTED, c_tested);
            if (tl) atomicAdd(stats + ST_DENS_LISTED, (unsigned long long)tl);
            if (tp) atomicAdd(stats + ST_DENS_PAIRS, (unsigned long long)tp);
            if (tsw) atomicAdd(stats + ST_DENS_SWEEPS, (unsigned long long)tsw);
            if (trc) atomicAdd(stats + ST_DENS_RECOLLECT, (unsigned long long)trc);
        }
    }
}

}  // namespace

int sph_launch_buckets(sph_ctx* c) {
    cudaStream_t s = c->stream;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->bucket_cnt, 0, sizeof(unsigned), s));
    k_buckets<<<c->sm_count * 4, BK_WARPS * 32, 0, s>>>(c->grid, c->cell_start, c->par.tile_rows, c->buckets,
                                              c->bucket_cnt);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

// Runs the tile kernel over all buckets with a tile of tile_cap candidates (sized for the
// occupancy), then over the buckets that did not fit with a tile of SPH_TCAP_BIG; the targets
// left after that are in c->fb_list (c->fb_cnt of them) and are swept by the caller with the
// 8-lanes-per-target kernel.
int sph_launch_density_tile(sph_ctx* c, float* h, float* rho, float* omega, int32_t* nn) {
    cudaStream_t s = c->stream;
    const int W = c->par.tile_warps;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->tile_next, 0, 4 * sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->fb_cnt, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->big_cnt, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->list_next, 0, sizeof(unsigned), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->bucket_loff, 0xff, (size_t)c->n_max * sizeof(uint32_t), s));
    auto launch = [&](auto tag, auto ntag) -> cudaError_t {
        constexpr int KERN = decltype(tag)::value, NT = decltype(ntag)::value, NTHR = 64 / NT;
        for (int pass = 0; pass < 2; ++pass) {
            const int  tcap = pass == 0 ? c->par.tile_cap : c->par.tile_cap2;
            const bool two  = c->par.tile_cap2 >= c->par.tile_cap + 32;
            if (pass == 1 && !two) break;
            TilePar par{c->par.n_ngb, c->par.h_tol, c->par.search_slack, c->par.h_max_iter, tcap, c->lcap,
                        c->par.tile_forces == 2 ? 1 : 0};
            const size_t smem = sph_tile_smem_bytes(tcap, 16, sph_tile_xbytes(1, 0), 2 / NT);
            cudaError_t e = cudaFuncSetAttribute(k_density_tile<KERN, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            int per_sm = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_density_tile<KERN, NT>, NTHR, smem);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            const bool last = pass == 1 || !two;
            k_density_tile<KERN, NT><<<c->sm_count * per_sm, NTHR, smem, s>>>(
                c->grid, c->cell_start, c->pos_m, c->perm, c->buckets,
                pass == 0 ? c->bucket_cnt : c->big_cnt, pass == 0 ? nullptr : c->big_list,
                last ? nullptr : c->big_list, c->big_cnt, c->tile_next + pass, par, h, rho, omega, nn,
                c->fix_list, c->fix_cnt, c->fb_list, c->fb_cnt,
                c->par.tile_forces == 1 ? nullptr : c->nb_j,
                (unsigned)(c->nb_words / ((size_t)c->lcap * SPH_TB)), c->list_next,
                c->bucket_loff, c->nb_cnt, c->nb_rkeep, c->tl_rkeep, c->bucket_rt, c->stats);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    // tile_warps = 2: two warps per bucket, one target per thread; 1: one warp, two targets per lane
    auto launch_k = [&](auto tag) -> cudaError_t {
        return W >= 2 ? launch(tag, std::integral_constant<int, 1>{}) : launch(tag, std::integral_constant<int, 2>{});
    };
    cudaError_t e;
    switch (c->par.kernel) {
    case 0: e = launch_k(std::integral_constant<int, 0>{}); break;
    case 2: e = launch_k(std::integral_constant<int, 2>{}); break;
    case 3: e = launch_k(std::integral_constant<int, 3>{}); break;
    default: e = launch_k(std::integral_constant<int, 1>{}); break;
    }
    SPH_CUDA_CHECK(c, e);
    return SPH_OK;
}
