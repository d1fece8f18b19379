// sph_tile.cuh -- the staged-tile sweeps: buckets of up to 64 sorted
// targets, the candidate sources of a bucket staged ONCE in shared memory with 1-D bulk
// asynchronous copies (cp.async.bulk + mbarrier), one lane per target pair.
//
// The paper evaluates groups of sinks against an interaction list that holds "every particle
// that could be a neighbour of any sink in the group", packed in tiles, and selects the actual
// neighbours inside the vectorised evaluation.  This is that
// shape on sm_100a: a bucket is a compact brick of targets (a few adjacent rows of cells over a
// short range of cells along x, "box of balls" = the brick inflated by the search
// radius), its interaction list is the union of the cell rows within reach, each row one
// contiguous range of the sorted arrays and therefore one bulk copy; every lane then tests every
// staged candidate against its own two targets with broadcast shared-memory loads and packed
// FP32 arithmetic (FFMA2), and keeps the accepted set as bit masks over the tile.
// Shares nothing with oracle/.
#pragma once
#include "sph_internal.cuh"

#ifdef __CUDACC__

#define SPH_TB 64        // targets per bucket: two per lane
#define SPH_TROWS 96    // candidate rows of cells per bucket (cap)
#define SPH_TSEGS (2 * SPH_TROWS)   // a row that crosses a periodic face has two segments
#define SPH_TZCAP 28     // per-target slots for list entries next to the support edge (the "zone")
#define SPH_TWMAX 4      // at most this many warps share a bucket

// shared memory of one warp (bytes), tcap = tile capacity in candidates (multiple of 32)
//   tile   float4[tcap]        (x', y', z', |x'|^2) in the bucket's frame
//   ms     float[tcap]         m_j
//   gidx   uint32[tcap]        sorted position of the candidate (density sweep: for the kept lists)
//   mask   uint32[tcap/32][64] accept bits of the 64 targets, word-major
//   seg    uint2[SPH_TSEGS]    (first sorted position, count | tile offset << 12 | image << 24)
//   zone   uint16[SPH_TZCAP][64]  tile indices of the entries next to the support edge
//   rowoff int[32]
//   mbar   uint64
// xbytes: size of the segment table's region, which doubles as the warps' exchange area
__host__ __device__ inline size_t sph_tile_xbytes(int W, int words_per_target) {
    const size_t x = W > 1 ? (size_t)W * words_per_target * SPH_TB * 4 : 0, s = SPH_TSEGS * 8;
    return x > s ? x : s;
}
__host__ __device__ inline size_t sph_tile_smem_bytes(int tcap, int rec_bytes, size_t xbytes, int W) {
    return (size_t)(tcap + 4) * (rec_bytes + 4 + 4) + (size_t)(tcap / 32 + 2 * W) * SPH_TB * 4 +
           xbytes + SPH_TZCAP * SPH_TB * 2 + 16;
}

// ---- mbarrier / bulk-copy primitives (PTX; SASS: SYNCS.*, UBLKCP) -----------------------
__device__ __forceinline__ void sph_mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void sph_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool sph_mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void sph_mbar_wait(uint32_t bar, uint32_t parity) {
    while (!sph_mbar_try_wait(bar, parity)) {}
}
// global -> shared, bytes a multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void sph_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes,
                                             uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}
// generic-proxy accesses of shared memory before this, async-proxy accesses after it
__device__ __forceinline__ void sph_fence_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ---- packed FP32 (two targets of a lane side by side; SASS: FFMA2 / FADD2 / FMUL2) ------
typedef unsigned long long sph_f2;
__device__ __forceinline__ sph_f2 sph_pk(float lo, float hi) {
    sph_f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void sph_upk(sph_f2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ sph_f2 sph_fma2(sph_f2 a, sph_f2 b, sph_f2 c) {
    sph_f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ sph_f2 sph_add2(sph_f2 a, sph_f2 b) {
    sph_f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ sph_f2 sph_mul2(sph_f2 a, sph_f2 b) {
    sph_f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint32_t sph_shl(uint32_t v, uint32_t s) {   // s >= 32 gives 0
    uint32_t r;
    asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(v), "r"(s));
    return r;
}

// The targets of a bucket: rows (ry0 + a, rz0 + b), a < nry, b < nrz, cells [c0, c1) along x
// of each; in single-cell mode (a cell with more than 64 particles) `skip` particles of the
// cell are left to the buckets before this one.
struct SphBucket {
    int32_t ry0, rz0, c0, c1;
    int32_t nry, nrz, skip, pad;
};

// Per-warp view of the dynamic shared memory.
struct SphTileMem {
    float4*   tile;
    float*    ms;
    uint32_t* mask;
    uint32_t* gidx;
    uint2*    seg;
    uint16_t* zone;
    int*      rowoff;   // [W][32]: aliases the head of the mask area (used before the masks exist)
    uint32_t  bar;      // shared-window address of the mbarrier
    uint32_t  tile_sa;  // shared-window addresses of the tile, the masses, the masks, the zone list
    uint32_t  ms_sa, mask_sa, zone_sa, gidx_sa;
    int       tcap;
};

template <int REC>
__device__ __forceinline__ SphTileMem sph_tile_carve(unsigned char* base, int tcap, size_t xbytes, int W) {
    SphTileMem t;
    t.tcap = tcap;
    t.tile = (float4*)base;                 base += (size_t)(tcap + 4) * REC;
 t.ms   = (float*)base;                  base += (size_t)(tcap + 4) * 4;
    t.gidx = (uint32_t*)base;               base += (size_t)(tcap + 4) * 4;
    t.mask = (uint32_t*)base;               base += (size_t)(tcap / 32 + 2 * W) * SPH_TB * 4;
 t.seg  = (uint2*)base;                  base += xbytes;
    t.zone = (uint16_t*)base;               base += SPH_TZCAP * SPH_TB * 2;
    t.rowoff = (int*)t.mask;
    t.bar  = (uint32_t)__cvta_generic_to_shared(base);
    t.tile_sa = (uint32_t)__cvta_generic_to_shared(t.tile);
    t.ms_sa   = (uint32_t)__cvta_generic_to_shared(t.ms);
    t.mask_sa = (uint32_t)__cvta_generic_to_shared(t.mask);
    t.zone_sa = (uint32_t)__cvta_generic_to_shared(t.zone);
    t.gidx_sa = (uint32_t)__cvta_generic_to_shared(t.gidx);
    return t;
}

// What a staged tile is: the frame, the reach it is complete for, its size.
struct SphTileInfo {
    float ox, oy, oz;   // origin of the bucket's frame (centre of the targets' bounding box)
    float R;            // every source within R of any target of the bucket is in the tile
    float ext;          // largest |coordinate| in the frame: bounds the FP32 rounding of r^2
    int   nseg, nrow, used, nwords;
    int   shifted;      // some segment is seen through a periodic image
    int   ok;           // the bucket fits the tile
};

// Squared distance between the slab [u s, (u+1) s) + lo and the interval [b0, b1]; edge cells
// of an open axis extend to infinity.
__device__ __forceinline__ float sph_slab_gap(float b0, float b1, int u, float lo, float s, int n,
                                              int per) {
    const float a = lo + (float)u * s;
    float below = a - b1;           // > 0: the interval lies below the slab
    float above = b0 - (a + s);     // > 0: above
    if (!per) {
        if (u <= 0) below = 0.0f;       // the first cell has no lower face
        if (u >= n - 1) above = 0.0f;   // the last one no upper face
    }
    return fmaxf(fmaxf(below, above) - 1e-3f * s, 0.0f);
}

// Unwrapped cell range along one axis that can hold a particle within R of [b0, b1].
// Returns false if a periodic axis is too short for the images to be unique per bucket.
__device__ __forceinline__ bool sph_axis_span(float b0, float b1, float R, float lo, float len,
                                              float is, int n, int per, int& u0, int& u1) {
    float a = floorf((b0 - lo - R) * is - 1e-3f);
    float b = floorf((b1 - lo + R) * is + 1e-3f);
    a = fminf(fmaxf(a, -1.0e9f), 1.0e9f);
    b = fminf(fmaxf(b, -1.0e9f), 1.0e9f);
    u0 = (int)a;
    u1 = (int)b;
    if (per) {
        if (u1 - u0 + 1 > n || (b1 - b0) + 2.0f * R >= 0.999f * len) return false;
        if (u0 < -n || u1 >= 2 * n) return false;   // targets outside the box
    } else {
        u0 = min(max(u0, 0), n - 1);
        u1 = min(max(u1, 0), n - 1);
    }
    return true;
}

// Warp-collective.  Lists the cell rows within R of the box [b0, b1] (the bucket's targets),
// each cut to its chord, and brings their particle records into the tile with one bulk copy
// per segment.  On return the copies are in flight; sph_tile_wait() completes them.
// Returns false (nothing issued) if the bucket does not fit: too many rows, too many
// candidates, or a periodic axis too short.
__device__ __forceinline__ bool sph_tile_stage(const SphGrid& g, const uint32_t* __restrict__ cell_start,
                                               const float4* __restrict__ rec, const float b0[3],
                                               const float b1[3], float R, const SphTileMem& sm,
                                               int lane, SphTileInfo& ti,
                                               const float4* __restrict__ rec2 = nullptr, uint32_t dst2 = 0u,
                                               const float4* __restrict__ rec3 = nullptr, uint32_t dst3 = 0u) {
    int x0, x1, y0, y1, z0, z1;
    bool ok = sph_axis_span(b0[1], b1[1], R, g.lo[1], g.len[1], g.isy, g.ny, g.per[1], y0, y1);
    ok = sph_axis_span(b0[2], b1[2], R, g.lo[2], g.len[2], g.isz, g.nz, g.per[2], z0, z1) && ok;
    ok = sph_axis_span(b0[0], b1[0], R, g.lo[0], g.len[0], g.isx, g.nx, g.per[0], x0, x1) && ok;
    if (!ok) return false;
    const int nyr = y1 - y0 + 1, nzr = z1 - z0 + 1, nrow = nyr * nzr;
    if (nrow > SPH_TROWS) return false;
    const float R2 = R * R * (1.0f + 1e-5f);
    int  base = 0;
    bool shifted = false;
    for (int rb = 0; rb < nrow; rb += 32) {
        const int r  = rb + lane;
        bool      in = r < nrow;
        const int iz = r / nyr, iy = r - iz * nyr;
        const int uy = y0 + iy, uz = z0 + iz;
        uint32_t  a0 = 0, a1 = 0, c0 = 0, c1 = 0;
        int       ka = 0, kb = 0;
        if (in) {
            const float dy = sph_slab_gap(b0[1], b1[1], uy, g.lo[1], g.sy, g.ny, g.per[1]);
            const float dz = sph_slab_gap(b0[2], b1[2], uz, g.lo[2], g.sz, g.nz, g.per[2]);
            const float d2 = dy * dy + dz * dz;
            in = d2 <= R2;
            if (in) {
                int ky, kz, kx0, u0, u1;
                const int cy = sph_wrap(uy, g.ny, ky), cz = sph_wrap(uz, g.nz, kz);
                sph_axis_span(b0[0], b1[0], sqrtf(R2 - d2), g.lo[0], g.len[0], g.isx, g.nx, g.per[0], u0, u1);
                u0 = max(u0, x0);
                u1 = min(u1, x1);
                const int cx0  = sph_wrap(u0, g.nx, kx0);
                const int span = u1 - u0;
                const uint32_t rq = (uint32_t)(cz * g.ny + cy) * (uint32_t)g.nx;
                a0 = __ldg(cell_start + rq + cx0);
                a1 = __ldg(cell_start + rq + min(cx0 + span, g.nx - 1) + 1);
                const int kyz = ((ky + 1) << 2) | ((kz + 1) << 4);
                ka = (kx0 + 1) | kyz;
                if (cx0 + span > g.nx - 1) {   // the row crosses the periodic face
                    c0 = __ldg(cell_start + rq);
                    c1 = __ldg(cell_start + rq + min(cx0 + span - g.nx, g.nx - 1) + 1);
                    kb = (kx0 + 2) | kyz;
                }
            }
        }
        const int na = (int)(a1 - a0), nb = (int)(c1 - c0);
        shifted = shifted || (na > 0 && ka != 0x15) || nb > 0;
        int inc = na + nb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(SPH_FULL, inc, o);
            if (lane >= o) inc += t;
        }
        const int off = base + inc - (na + nb);
        if (r < nrow) {
            // counts and offsets stay below 4096 (tile_cap), the image code below 64
            const uint32_t oa = (uint32_t)min(off, 4095), ob = (uint32_t)min(off + na, 4095);
            sm.seg[2 * r]     = make_uint2(a0, (uint32_t)min(na, 4095) | (oa << 12) | ((uint32_t)ka << 24));
            sm.seg[2 * r + 1] = make_uint2(c0, (uint32_t)min(nb, 4095) | (ob << 12) | ((uint32_t)kb << 24));
        }
        base += __shfl_sync(SPH_FULL, inc, 31);
    }
    if (base > sm.tcap || base == 0) return false;
    ti.nrow = nrow;
    ti.nseg = 2 * nrow;
    ti.used = base;
    ti.nwords = (base + 31) >> 5;
    ti.R = R;
    ti.ox = 0.5f * (b0[0] + b1[0]);
    ti.oy = 0.5f * (b0[1] + b1[1]);
    ti.oz = 0.5f * (b0[2] + b1[2]);
    ti.ext = R + 0.5f * fmaxf(b1[0] - b0[0], fmaxf(b1[1] - b0[1], b1[2] - b0[2])) +
             fmaxf(g.sx, fmaxf(g.sy, g.sz));
    ti.shifted = __any_sync(SPH_FULL, shifted) ? 1 : 0;
    // the tile's previous contents were read / written through the generic proxy
    sph_fence_async_smem();
    __syncwarp();
    const uint32_t narr = 1u + (rec2 ? 1u : 0u) + (rec3 ? 1u : 0u);
    if (lane == 0) sph_mbar_expect_tx(sm.bar, (uint32_t)base * 16u * narr);
    __syncwarp();
    for (int s = lane; s < ti.nseg; s += 32) {
        const uint2    sg  = sm.seg[s];
        const uint32_t cnt = sg.y & 4095u, off = (sg.y >> 12) & 4095u;
        if (cnt) {
            sph_bulk_g2s(sm.tile_sa + off * 16u, rec + sg.x, cnt * 16u, sm.bar);
            if (rec2) sph_bulk_g2s(dst2 + off * 16u, rec2 + sg.x, cnt * 16u, sm.bar);
            if (rec3) sph_bulk_g2s(dst3 + off * 16u, rec3 + sg.x, cnt * 16u, sm.bar);
        }
    }
    if (sm.gidx) {   // sorted position of every tile entry, written while the copies are in flight
        for (int s = lane; s < ti.nseg; s += 32) {
            const uint2    sg  = sm.seg[s];
            const uint32_t cnt = sg.y & 4095u, off = (sg.y >> 12) & 4095u;
            for (uint32_t k = 0; k < cnt; ++k) sm.gidx[off + k] = sg.x + k;
        }
    }
    return true;
}

// Completes the copies of sph_tile_stage and turns the raw records (x, y, z, w) into the
// bucket's frame: (x', y', z', |x'|^2) with x' = fl((x_j + k L) - origin); the fourth
// component goes to ms[].  Without a periodic image the origin is a float and the FP32
// subtraction is the correctly rounded difference; through an image the shifted origin is not
// representable and the difference is taken in FP64 on the FP32 inputs.  Either way the
// displacement x_i' - x_j' of a pair carries two roundings of 2^-25 |x'|, and |x'| is a few h,
// not the box.  Pads the tile with far-away dummies to a full word and one more entry (the
// record a cursor's bubble reads).
// Called by all nthr threads of the block; ends with a block barrier.
__device__ __forceinline__ void sph_tile_finish(const SphGrid& g, const SphTileMem& sm,
                                                const SphTileInfo& ti, uint32_t parity, int tid,
                                                int nthr, float pad_w) {
    sph_mbar_wait(sm.bar, parity);
    if (!ti.shifted) {
        for (int k = tid; k < ti.used; k += nthr) {
            const float4 p = sm.tile[k];
            const float  x = p.x - ti.ox, y = p.y - ti.oy, z = p.z - ti.oz;
            sm.tile[k] = make_float4(x, y, z, fmaf(z, z, fmaf(y, y, x * x)));
            sm.ms[k]   = p.w;
        }
    } else {
        int    s = -1;
        int    send = 0;
        double ox = 0.0, oy = 0.0, oz = 0.0;
        for (int k = tid; k < ti.used; k += nthr) {
            while (k >= send) {   // the segments are in tile order; each thread only moves forward
                ++s;
                const uint2    sg = sm.seg[s];
                const uint32_t kk = sg.y >> 24;
                send = (int)(((sg.y >> 12) & 4095u) + (sg.y & 4095u));
                const int kx = (int)(kk & 3u) - 1, ky = (int)((kk >> 2) & 3u) - 1, kz = (int)((kk >> 4) & 3u) - 1;
                ox = (double)ti.ox - (double)kx * (double)g.len[0];
                oy = (double)ti.oy - (double)ky * (double)g.len[1];
                oz = (double)ti.oz - (double)kz * (double)g.len[2];
            }
            const float4 p = sm.tile[k];
            const float  x = (float)((double)p.x - ox), y = (float)((double)p.y - oy), z = (float)((double)p.z - oz);
            sm.tile[k] = make_float4(x, y, z, fmaf(z, z, fmaf(y, y, x * x)));
            sm.ms[k]   = p.w;
        }
    }
    for (int k = ti.used + tid; k < ti.nwords * 32 + 1; k += nthr) {
        sm.tile[k] = make_float4(0.0f, 0.0f, 0.0f, 3.0e37f);
        sm.ms[k]   = pad_w;
    }
    __syncthreads();
}

// The first mask word at or behind nwords that belongs to warp wid of W (words w = wid mod W).
__device__ __forceinline__ int sph_first_pad_word(int nwords, int wid, int W) {
    const int r = (wid - nwords % W + W) % W;
    return nwords + r;
}

// Phase 1: the accept masks of the lane's two targets over the whole tile.  Target t of the
// lane (frame coordinates (x, y, z), list radius Rc) accepts candidate j iff
//   |x_j'|^2 - 2 x_t . x_j' + |x_t|^2 - Rc^2 < 0;
// the lane evaluates both targets at once (FADD2 + 3 FFMA2 on a broadcast LDS.128) and shifts
// the two sign bits into the mask words.  Candidate 32 w + b is bit 31 - b of word w.  Only a
// superset of the final neighbour set is needed (kernels vanish outside 2h and the sweeps use
// exact displacements), so the expanded form's rounding (~2^-23 ext^2) is covered by the margin
// the caller leaves between Rc and the ball it relies on.  Rc <= 0 switches a target off.
__device__ __forceinline__ void sph_tile_masks(const SphTileMem& sm, const SphTileInfo& ti,
                                               const float xt[2], const float yt[2],
                                               const float zt[2], const float Rc[2], int lane,
                                               int wid, int W) {
    float ci[2];
#pragma unroll
    for (int t = 0; t < 2; ++t)
        ci[t] = Rc[t] > 0.0f ? fmaf(zt[t], zt[t], fmaf(yt[t], yt[t], xt[t] * xt[t])) - Rc[t] * Rc[t]
                             : 3.0e38f;
    const sph_f2 ax = sph_pk(-2.0f * xt[0], -2.0f * xt[1]);
    const sph_f2 ay = sph_pk(-2.0f * yt[0], -2.0f * yt[1]);
    const sph_f2 az = sph_pk(-2.0f * zt[0], -2.0f * zt[1]);
    const sph_f2 cc = sph_pk(ci[0], ci[1]);
    for (int w = wid; w < ti.nwords; w += W) {
        uint32_t m0 = 0u, m1 = 0u;
        const float4* c = sm.tile + w * 32;
#pragma unroll
        for (int u = 0; u < 32; ++u) {
            const float4 p = c[u];
            sph_f2 t = sph_add2(sph_pk(p.w, p.w), cc);
            t = sph_fma2(ax, sph_pk(p.x, p.x), t);
            t = sph_fma2(ay, sph_pk(p.y, p.y), t);
            t = sph_fma2(az, sph_pk(p.z, p.z), t);
            m0 = __funnelshift_l((uint32_t)t, m0, 1);
            m1 = __funnelshift_l((uint32_t)(t >> 32), m1, 1);
        }
        sm.mask[w * SPH_TB + lane]      = m0;
        sm.mask[w * SPH_TB + 32 + lane] = m1;
    }
    // the cursor reads two words of its own stride ahead: this warp's first two words at or
    // behind nwords are zero
    for (int k = 0, w = sph_first_pad_word(ti.nwords, wid, W); k < 2; ++k, w += W) {
        sm.mask[w * SPH_TB + lane]      = 0u;
        sm.mask[w * SPH_TB + 32 + lane] = 0u;
    }
    __syncwarp();
}

// ---- shared-memory accesses through 32-bit shared-window addresses held in registers --------
__device__ __forceinline__ float4 sph_lds4(uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ float sph_lds1(uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t sph_ldsu(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

// A lane's private cursor over the accept bits of one target, in tile order, over the mask
// words wid, wid + W, wid + 2 W, ... (the W warps that share a bucket split the words).  The
// word after the current one is held in a register (`next`), so a refill never waits.
struct SphCursor {
    uint32_t bits, next;
    uint32_t maddr;    // shared address of the word after `next`
    int      base31;   // 32 w + 31 for the current word w
};
__device__ __forceinline__ void sph_cursor_start(SphCursor& c, const SphTileMem& sm,
                                                 const SphTileInfo& ti, int t, bool on, int wid, int W) {
    const uint32_t a = sm.mask_sa + 4u * (uint32_t)(wid * SPH_TB + t);
    c.base31 = on ? 32 * wid + 31 : ti.nwords * 32 + 31;
    c.bits   = on ? sph_ldsu(a) : 0u;                      // zero words follow the last mask word
    c.next   = on ? sph_ldsu(a + 4u * SPH_TB * (uint32_t)W) : 0u;
    // a cursor that is off must stay empty: it only ever reads the zero word
    const uint32_t zw = sm.mask_sa + 4u * (uint32_t)((sph_first_pad_word(ti.nwords, wid, W) + W) * SPH_TB + t);
    c.maddr  = on ? min(a + 8u * SPH_TB * (uint32_t)W, zw) : zw;
}
__device__ __forceinline__ bool sph_cursor_live(const SphCursor& c, const SphTileInfo& ti) {
    return c.base31 < ti.nwords * 32;
}
// One list entry as the sweeps see it.
struct SphEntry {
    float4 c;      // (x', y', z', |x'|^2) of the source
    float  m;      // its mass; 0 for a bubble
    int    idx;    // tile index
    bool   has;    // false: bubble (an empty mask word was skipped, or the cursor is exhausted)
};
// Takes the next entry of the cursor and starts the loads of its record.  Straight-line code:
// the refill of an exhausted word is predicated, the index of a bubble points at the padding.
__device__ __forceinline__ void sph_cursor_fetch(SphCursor& c, const SphTileMem& sm, int idx_max,
                                                 uint32_t mend, int W, SphEntry& e) {
    uint32_t flo, bit;
    asm("bfind.u32 %0, %1;" : "=r"(flo) : "r"(c.bits));            // 0xffffffff for an empty word
    e.has = c.bits != 0u;
    e.idx = e.has ? c.base31 - (int)flo : idx_max;                   // bubble: the padding entry
    asm("shl.b32 %0, %1, %2;" : "=r"(bit) : "r"(1u), "r"(flo));    // 0 for an empty word
    c.bits ^= bit;
    e.c = sph_lds4(sm.tile_sa + 16u * (uint32_t)e.idx);
    e.m = sph_lds1(sm.ms_sa + 4u * (uint32_t)e.idx);               // padding entries carry m = 0
    if (c.bits == 0u) {
        c.bits   = c.next;
        c.base31 += 32 * W;
        c.next   = sph_ldsu(c.maddr);
        c.maddr  = min(c.maddr + 4u * SPH_TB * (uint32_t)W, mend);
    }
}

// Advances the cursor by one step without touching the records (the steps other warps take).
__device__ __forceinline__ void sph_cursor_skip(SphCursor& c, uint32_t mend, int W) {
    uint32_t flo, bit;
    asm("bfind.u32 %0, %1;" : "=r"(flo) : "r"(c.bits));
    asm("shl.b32 %0, %1, %2;" : "=r"(bit) : "r"(1u), "r"(flo));
    c.bits ^= bit;
    if (c.bits == 0u) {
        c.bits   = c.next;
        c.base31 += 32 * W;
        c.next   = sph_ldsu(c.maddr);
        c.maddr  = min(c.maddr + 4u * SPH_TB * (uint32_t)W, mend);
    }
}

// Walks the accepted entries of the lane's two targets.  Two ways to share a bucket between
// the W warps of a block:
//   by words   (es = 1): this warp's cursor runs over the mask words wid, wid + W, ...;
//   by entries (es = W): every warp's cursor runs over all words, and this warp takes the steps
//                        ep, ep + es, ... of it (bubbles included), which balances the work
//                        of a lane exactly when the per-entry work dominates the cursor's.
// Two entry sets per target are used in turn: the record of an entry is in flight while the
// entry before it is worked on, without register copies.  work(t, entry) sees bubbles too
// (has = false; the padding record, m = pad_w of sph_tile_finish).
template <int NSET = 2, class Work>
__device__ __forceinline__ void sph_tile_walk(const SphTileMem& sm, const SphTileInfo& ti, int lane,
                                              int wid, int W, const bool on[2], Work&& work,
                                              int ep = 0, int es = 1) {
    SphCursor cu[2];
    SphEntry  e[NSET][2];
    const int idx_max = ti.nwords * 32;                               // first padding entry
    // this warp's second zero word behind the masks
    const uint32_t mend = sm.mask_sa + 4u * (uint32_t)((sph_first_pad_word(ti.nwords, wid, W) + W) * SPH_TB);
    auto fetch = [&](int t, SphEntry& en) {
        const uint32_t me = mend + 4u * (uint32_t)(lane + 32 * t);
        for (int s = 0; s < ep; ++s) sph_cursor_skip(cu[t], me, W);
        sph_cursor_fetch(cu[t], sm, idx_max, me, W, en);
        for (int s = ep + 1; s < es; ++s) sph_cursor_skip(cu[t], me, W);
    };
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        sph_cursor_start(cu[t], sm, ti, lane + 32 * t, on[t], wid, W);
#pragma unroll
        for (int q = 0; q < NSET; ++q) fetch(t, e[q][t]);
    }
    for (;;) {
        bool live = sph_cursor_live(cu[0], ti) || sph_cursor_live(cu[1], ti);
#pragma unroll
        for (int q = 0; q < NSET; ++q) live = live || e[q][0].has || e[q][1].has;
        if (!__any_sync(SPH_FULL, live)) break;
#pragma unroll
        for (int q = 0; q < NSET; ++q) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                work(t, e[q][t]);
                fetch(t, e[q][t]);
            }
        }
    }
}

// a6 for a box (the bound of sph_scatter_hmax, for the bucket's bounding box): the largest h_j
// of any particle that can reach a point of [b0, b1].  Warp-collective.
__device__ __forceinline__ float sph_box_scatter_hmax(const SphGrid& g, const unsigned* __restrict__ coarse,
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
        const bool blocks = inside && nn[0] * nn[1] * nn[2] > 512;
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
        if (Hn >= H * (1.0f - 1e-6f)) { H = Hn; break; }
        H = Hn;
    }
    return H;
}

// ---- one thread per target (or two): the forms used when NW = 2 / NT warps share a bucket,
// each thread owning NT targets: columns tid + 32 t, t < NT, of the mask words --------------

// Phase 1 with the targets' parameters in shared memory, as pairs: component c (0..3 =
// -2 x, -2 y, -2 z, |x|^2 - Rc^2 in the tile's frame; (0, 0, 0, 3e38) switches a target off)
// of target columns l and l + 32 side by side at tgt[2 (32 c + l)], so that one 64-bit load
// gives the operand of a packed instruction (sph_tgt_put writes one column).
// Warp wid of NW computes the words w = wid, wid + NW, ... for all 64 columns (lane l: columns
// l and l + 32, as sph_tile_masks) and zeroes its share of the pad words nwords .. nwords +
// 2 NW - 1.  The caller puts a block barrier on both sides.
__device__ __forceinline__ void sph_tgt_put(float* tgt, int col, float x, float y, float z, float c) {
    float* q = tgt + 2 * (col & 31) + (col >> 5);
    q[0] = x; q[64] = y; q[128] = z; q[192] = c;
}
__device__ __forceinline__ void sph_tile_masks_sh(const SphTileMem& sm, const SphTileInfo& ti,
                                                  const float* tgt, int lane, int wid, int NW) {
    const sph_f2* tp = (const sph_f2*)tgt;
    const sph_f2 ax = tp[lane], ay = tp[32 + lane], az = tp[64 + lane], cc = tp[96 + lane];
    for (int w = wid; w < ti.nwords; w += NW) {
        uint32_t m0 = 0u, m1 = 0u;
        const float4* c = sm.tile + w * 32;
#pragma unroll
        for (int u = 0; u < 32; ++u) {
            const float4 p = c[u];
            sph_f2 t = sph_add2(sph_pk(p.w, p.w), cc);
            t = sph_fma2(ax, sph_pk(p.x, p.x), t);
            t = sph_fma2(ay, sph_pk(p.y, p.y), t);
            t = sph_fma2(az, sph_pk(p.z, p.z), t);
            m0 = __funnelshift_l((uint32_t)t, m0, 1);
            m1 = __funnelshift_l((uint32_t)(t >> 32), m1, 1);
        }
        sm.mask[w * SPH_TB + lane]      = m0;
        sm.mask[w * SPH_TB + 32 + lane] = m1;
    }
    for (int k = 0, w = sph_first_pad_word(ti.nwords, wid, NW); k < 2; ++k, w += NW) {
        sm.mask[w * SPH_TB + lane]      = 0u;
        sm.mask[w * SPH_TB + 32 + lane] = 0u;
    }
}

// Walks the accepted entries of the thread's NT targets (columns tid + 32 t) over ALL mask
// words, NSET entries per target in flight.  work(t, entry) sees bubbles too.
template <int NT, int NSET, class Work>
__device__ __forceinline__ void sph_tile_walk_own(const SphTileMem& sm, const SphTileInfo& ti, int tid,
                                                  const bool on[NT], Work&& work) {
    SphCursor cu[NT];
    SphEntry  e[NSET][NT];
    const int idx_max = ti.nwords * 32;                               // first padding entry
    const uint32_t mend = sm.mask_sa + 4u * (uint32_t)((ti.nwords + 1) * SPH_TB);   // second zero word
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        sph_cursor_start(cu[t], sm, ti, tid + 32 * t, on[t], 0, 1);
#pragma unroll
        for (int q = 0; q < NSET; ++q)
            sph_cursor_fetch(cu[t], sm, idx_max, mend + 4u * (uint32_t)(tid + 32 * t), 1, e[q][t]);
    }
    for (;;) {
        bool live = false;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            live = live || sph_cursor_live(cu[t], ti);
#pragma unroll
            for (int q = 0; q < NSET; ++q) live = live || e[q][t].has;
        }
        if (!__any_sync(SPH_FULL, live)) break;
#pragma unroll
        for (int q = 0; q < NSET; ++q) {
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                work(t, e[q][t]);
                sph_cursor_fetch(cu[t], sm, idx_max, mend + 4u * (uint32_t)(tid + 32 * t), 1, e[q][t]);
            }
        }
    }
}

#endif  // __CUDACC__
