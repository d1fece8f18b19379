// sph_internal.cuh -- context, device-resident grid descriptor and the warp-level
// neighbour-row enumeration shared by the sweeps.  Internal to the CUDA library; the public
// boundary is include/sph.h.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>
#include "../../include/sph.h"

// ---------------------------------------------------------------------------------------
// Spatial index.  Uniform grid, cell = (cz*ny + cy)*nx + cx, so that
// a run of cells along x is ONE contiguous range of the sorted particle arrays
// (the paper's "particles of a cell are contiguous", applied to rows).
// The descriptor lives in device memory and is written by a kernel from min(h): no host
// round trip between sph_build_cells and the sweeps.
// ---------------------------------------------------------------------------------------
struct SphGrid {
    int   nx, ny, nz, ncells;
    float sx, sy, sz;          // cell sides
    float isx, isy, isz;       // inverse cell sides
    float lo[3], len[3];
    int   per[3];
    float hmin, hmax;          // of the h given to sph_build_cells
    float xext;                // largest |coordinate| that enters a displacement
    int   flags;               // bit0: periodic side too short; bit1: cell table clipped; bit2: no valid h;
                               // bit3: steep h contrast (max h > 1.6 min h): the staged-tile sweeps stand
                               // back and every target takes the 8-lane kernels (set only in automatic mode)
    unsigned force_hmax_bits;  // max h given to sph_forces (float bits, atomicMax)
    int   cn[3];               // coarse grid (max-h map for the scatter reach of the force search)
    float ics[3];              // inverse coarse cell sides
    int   sn[3];               // second level of the map: blocks of 8 x 8 x 8 coarse cells
};
#define SPH_COARSE_MAX (1 << 18)   // entries of the coarse max-h map (the second level, of
                                   // at most as many, follows it in the same allocation)
#define SPH_POS_PAD 64             // records of padding behind the sorted float4 arrays
#define SPH_G 8                    // lanes per target in the sweeps
#define SPH_SLOTS 24               // list entries per lane (24 x 8 = 192 per target)
#define SPH_LCAP_MIN 128           // entries per target of a bucket-major list region: at least this (sph_ctx.lcap)

enum {  // indices into the device counter block (uint64 each), mirrors sph_stats_t
    ST_DENS_TESTED = 0, ST_DENS_LISTED, ST_DENS_PAIRS, ST_DENS_SWEEPS, ST_DENS_RECOLLECT,
    ST_DENS_OVERFLOW, ST_DENS_NONCONV, ST_DENS_RECHECK, ST_FORCE_TESTED, ST_FORCE_PAIRS,
    ST_FORCE_AV, ST_NCOUNTERS
};

struct sph_ctx {
    sph_params   par;
    sph_box      box;
    int64_t      n_max, n;
    int64_t      n_build;      // n of the sph_build_cells call in progress / last
    int64_t      cap_cells;
    cudaStream_t stream;
    bool         built;
    bool         forces_ready; // sph_forces ran since the last build: pos_h.w, coarse map valid
    int          sm_count;
    // device memory
    SphGrid*     grid;
    unsigned*    red;          // [8] uint: hmin bits, hmax bits, max|x| bits ...
    uint32_t*    cell_cnt;     // cap_cells + 1
    uint32_t*    cell_start;   // cap_cells + 1
    uint32_t*    key;          // n_max
    uint32_t*    rank;         // n_max
    int32_t*     perm;         // n_max: sorted position -> caller index
    int32_t*     inv_perm;     // n_max: caller index -> sorted position
    uint32_t*    scan_part;    // SCAN_BLOCKS + 1
    float4*      pos_h;        // sorted (x, y, z, h)
    float4*      pos_m;        // sorted (x, y, z, m)
    float4*      vel_m;        // sorted (vx, vy, vz, m)
    float4*      rcak;         // sorted (rho, c, A = P/(Omega rho^2), K = gscale sigma / h^5)
    unsigned*    coarse_hmax;  // SPH_COARSE_MAX: max h (float bits) per coarse cell, step a6
    unsigned long long* stats; // ST_NCOUNTERS
    uint32_t*    nb_j;         // n_max x SPH_SLOTS x SPH_G: the density sweep's neighbour indices,
                               // [target][entry]; reused by the force sweep
    uint32_t*    nb_cnt;       // n_max: entries of the kept list
    float*       nb_rkeep;     // n_max: radius inside which the kept list is complete (0: none)
    int32_t*     fix_list;     // n_max: sorted positions queued for the robust (fix) kernels
    unsigned*    fix_cnt;      // [2]: queue lengths (density, forces)
    uint32_t*    act_list;     // n_max: sorted positions of the active set, ascending
    unsigned*    act_cnt;      // [2]: its length; [1]: length of the marking pass's source list
    bool         act_on;       // sph_set_active gave a mask since the last build
    struct SphBucket* buckets; // n_max: the bucket table of the staged-tile sweeps (sph_tile.cuh)
    unsigned*    bucket_cnt;   // [1]
    unsigned*    tile_next;    // [4]: work counters of the persistent tile kernels (density, forces; two passes)
    unsigned*    big_list;     // n_max: buckets the first pass of a tile sweep left to the second (larger tile)
    unsigned*    big_cnt;      // [2]: their number (density, forces)
    unsigned*    list_next;    // [1]: next free region of nb_j (bucket-major lists of the tile sweep)
    float*       bucket_rt;    // n_max: radius of the tile a bucket's lists index (tile_forces = 2), 0: none
    int          lcap;         // entries per target of a bucket-major list region (from n_ngb, sph_create)
    size_t       nb_words;     // words in nb_j
    uint32_t*    bucket_loff;  // n_max: list region of a bucket (0xffffffff: none)
    float*       tl_rkeep;     // n_max: radius inside which a target's bucket-major list is complete (0: none);
                               // nb_rkeep stays the radius of the 8-lane kernels' [target][entry] lists
    uint32_t*    fb_list;      // n_max: targets the tile kernels hand to the 8-lane kernels
    unsigned*    fb_cnt;       // [2]: their number (density, forces)
    float*       dt_part;      // per-block minima of the time-step reduction
    int64_t*     nb_total;     // neighbour-list total (device) + pinned mirror
    char         err[256];
};

#define SPH_SCAN_BLOCKS 1024
#define SPH_GRID_STEEP 8           // SphGrid.flags bit 3
#define SPH_TILE_MIN_N (1 << 17)   // automatic mode: fewer particles than this cannot fill the GPU with
                                   // one block per bucket of 64 (148 SMs x 7 blocks x a few buckets each);
                                   // measured: the tile sweeps win from about 10^5 particles up
#define SPH_STEEP_RATIO 1.6f       // automatic mode: max h beyond this x min h stands the tile sweeps down

// The staged-tile sweeps are in use for this index: forced (tile > 0), or automatic (tile = 0) with
// enough particles.  (In automatic mode the device may still stand them down: SPH_GRID_STEEP.)
static inline bool sph_tile_on(const sph_ctx* c) {
    return c->par.tile > 0 || (c->par.tile == 0 && c->n_build >= SPH_TILE_MIN_N);
}

#define SPH_CUDA_CHECK(ctx, call)                                                          \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__,   \
                     #call, cudaGetErrorString(e_));                                       \
            return SPH_ECUDA;                                                              \
        }                                                                                  \
    } while (0)

#ifdef __CUDACC__

#define SPH_FULL 0xffffffffu
#ifndef SPH_UNROLL
#define SPH_UNROLL 3   // candidate windows loaded ahead per lane
#endif
#ifndef SPH_MINB
#define SPH_MINB 8     // resident blocks per SM the sweeps are compiled for
#endif

// SPH kernels with support radius 2h (PAPER.md:105 offers the cubic spline and the Wendland
// C2, C4, C6 functions; forms of Dehnen & Aly 2012 rescaled to 2h, reading R3):
// W(r,h) = sigma h^-3 w(q), q = r/h, x = q/2, y = (1-x)_+.  Every kernel provides
//   sums(q, w, e, f):  w(q),  e = -q w'(q),  f = -(q w'(q) + q^2 w''(q))
//                      (S = sum m w, dS/dh = E/h, dE/dh = -F/h with E = sum m e, F = sum m f)
//   g(q) = -w'(q)/q    (dW/dr = -sigma h^-5 g(q) r: no division by r in the force sweep)
//   self = (32 pi/3) sigma w(0): the neighbour "count" of a particle alone in its kernel.
template <int KERN> struct SphKernel;
// sums_s / escale: the same sums with a constant factor of e left out of the loop,
// E = escale * sum m e_s (only Wendland C2 has a cheaper form; the others pass through)
// g_s / gscale: g(q) = gscale * g_s(q); the force sweep folds gscale into K = gscale sigma / h^5.
template <class K> struct SphKernelPlain {
    static constexpr float escale = 1.0f;
    static constexpr float gscale = 1.0f;
    static __device__ __forceinline__ float g_s(float q) { return K::g(q); }
    static __device__ __forceinline__ void sums_s(float q, float& w, float& e, float& f) {
        K::sums(q, w, e, f);
    }
};
template <> struct SphKernel<0> : SphKernelPlain<SphKernel<0>> {   // cubic spline (Monaghan 1992)
    static constexpr float sigma = 0.31830988618379067f, self = 32.0f / 3.0f;
    static __device__ __forceinline__ void sums(float q, float& w, float& e, float& f) {
        const float u = fmaxf(2.0f - q, 0.0f), q2 = q * q;
        const bool  in = q < 1.0f;
        w = in ? 1.0f - q2 * (1.5f - 0.75f * q) : 0.25f * u * u * u;
        e = in ? q2 * (3.0f - 2.25f * q) : 0.75f * q * u * u;
        f = in ? q2 * (6.0f - 6.75f * q) : 0.75f * q * u * (u - 2.0f * q);
    }
    static __device__ __forceinline__ float g(float q) {
        const float u = fmaxf(2.0f - q, 0.0f);
        return q < 1.0f ? 3.0f - 2.25f * q : __fdividef(0.75f * u * u, q);
    }
    static __device__ __forceinline__ float w(float q) {
        const float u = fmaxf(2.0f - q, 0.0f);
        return q < 1.0f ? 1.0f - q * q * (1.5f - 0.75f * q) : 0.25f * u * u * u;
    }
};
template <> struct SphKernel<1> {   // Wendland C2: w = y^4 (1 + 4x)
    static constexpr float sigma = 0.41778172561566733f, self = 14.0f;
    static __device__ __forceinline__ void sums(float q, float& w, float& e, float& f) {
        const float t = fmaxf(1.0f - 0.5f * q, 0.0f), t2 = t * t, q2 = q * q;
        w = t2 * t2 * (1.0f + 2.0f * q);
        e = 5.0f * q2 * t2 * t;
        f = q2 * t2 * (10.0f * t - 7.5f * q);
    }
    // 15 instead of 18 FP instructions per entry: a = q^2 t^2 shared, e_s = a t (factor 5
    // outside), and 10 t - 7.5 q = 10 - 12.5 q wherever t > 0 (a = 0 elsewhere)
    static constexpr float gscale = 5.0f;
    static __device__ __forceinline__ float g_s(float q) {
        const float t = fmaxf(1.0f - 0.5f * q, 0.0f);
        return t * t * t;
    }
    static constexpr float escale = 5.0f;
    static __device__ __forceinline__ void sums_s(float q, float& w, float& e, float& f) {
        const float t = fmaxf(1.0f - 0.5f * q, 0.0f), t2 = t * t, a = (q * q) * t2;
        w = (t2 * t2) * (1.0f + 2.0f * q);
        e = a * t;
        f = a * (10.0f - 12.5f * q);
    }
    static __device__ __forceinline__ float g(float q) {
        const float t = fmaxf(1.0f - 0.5f * q, 0.0f);
        return 5.0f * t * t * t;
    }
    static __device__ __forceinline__ float w(float q) {
        const float t = fmaxf(1.0f - 0.5f * q, 0.0f), t2 = t * t;
        return t2 * t2 * (1.0f + 2.0f * q);
    }
};
template <> struct SphKernel<2> : SphKernelPlain<SphKernel<2>> {   // Wendland C4: w = y^6 (1 + 6x + 35/3 x^2)
    static constexpr float sigma = 0.61548200648818910f, self = 20.625f;
    static __device__ __forceinline__ void sums(float q, float& w, float& e, float& f) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y, y4 = y2 * y2, x2 = x * x;
        w = y4 * y2 * (1.0f + x * (6.0f + (35.0f / 3.0f) * x));
        e = (56.0f / 3.0f) * x2 * y4 * y * (1.0f + 5.0f * x);
        f = (56.0f / 3.0f) * x2 * y4 * (2.0f + x * (8.0f - 40.0f * x));
    }
    static __device__ __forceinline__ float g(float q) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y;
        return (14.0f / 3.0f) * y2 * y2 * y * (1.0f + 5.0f * x);
    }
    static __device__ __forceinline__ float w(float q) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y;
        return y2 * y2 * y2 * (1.0f + x * (6.0f + (35.0f / 3.0f) * x));
    }
};
template <> struct SphKernel<3> : SphKernelPlain<SphKernel<3>> {   // Wendland C6: w = y^8 (1 + 8x + 25x^2 + 32x^3)
    static constexpr float sigma = 0.84861913015795750f, self = 28.4375f;
    static __device__ __forceinline__ void sums(float q, float& w, float& e, float& f) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y, y6 = y2 * y2 * y2, x2 = x * x;
        w = y6 * y2 * (1.0f + x * (8.0f + x * (25.0f + 32.0f * x)));
        e = 22.0f * x2 * y6 * y * (1.0f + x * (7.0f + 16.0f * x));
        f = 22.0f * x2 * y6 * (2.0f + x * (12.0f - x * (6.0f + 176.0f * x)));
    }
    static __device__ __forceinline__ float g(float q) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y;
        return 5.5f * y2 * y2 * y2 * y * (1.0f + x * (7.0f + 16.0f * x));
    }
    static __device__ __forceinline__ float w(float q) {
        const float x = 0.5f * q, y = fmaxf(1.0f - x, 0.0f), y2 = y * y, y4 = y2 * y2;
        return y4 * y4 * (1.0f + x * (8.0f + x * (25.0f + 32.0f * x)));
    }
};

// Shared-memory accesses through a 32-bit shared-window address that lives in a register
// (base + immediate): the hot list stores/loads cost one address add each instead of the
// re-derivation from SR_TID / the CTA's shared base that the compiler otherwise emits.
__device__ __forceinline__ uint32_t sph_smem_addr(const void* p) {
    uint32_t a = (uint32_t)__cvta_generic_to_shared(p);
    asm volatile("" : "+r"(a));
    return a;
}
// sqrt.approx: one MUFU.SQRT, relative error 2^-23, sqrt(0) = 0
__device__ __forceinline__ float sph_sqrt(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
template <int OFF> __device__ __forceinline__ void sph_sts(uint32_t a, float v) {
    asm volatile("st.shared.f32 [%0+%2], %1;" ::"r"(a), "f"(v), "n"(OFF));
}
// global store through a pointer that was pinned to a register pair (the pin hides the
// address space from the compiler, which would otherwise emit a generic store)
__device__ __forceinline__ void sph_stg(uint32_t* p, uint32_t v) {
    asm volatile("st.global.u32 [%0], %1;" ::"l"(p), "r"(v));
}
template <int OFF> __device__ __forceinline__ float sph_lds(uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF));
    return v;
}

__device__ __forceinline__ int sph_fdiv(int u, int n) {   // floor(u / n), n > 0
    return (u >= 0) ? (u / n) : -((-u + n - 1) / n);
}

__device__ __forceinline__ int sph_cell_coord(float x, float lo, float is, int n) {
    float c = floorf((x - lo) * is);
    c = fminf(fmaxf(c, 0.0f), (float)(n - 1));
    return (int)c;   // NaN -> 0 through fmaxf
}

// Range of (unwrapped) cell coordinates that can hold a particle within R of x.
__device__ __forceinline__ void sph_axis_range(float x, float R, float lo, float is, int n,
                                               int per, int& u0, int& u1) {
    float a = floorf((x - lo - R) * is - 1e-3f);
    float b = floorf((x - lo + R) * is + 1e-3f);
    a = fminf(fmaxf(a, -1.0e9f), 1.0e9f);
    b = fminf(fmaxf(b, -1.0e9f), 1.0e9f);
    u0 = (int)a;
    u1 = (int)b;
    if (per) {
        if (u1 - u0 + 1 > n) {   // whole axis: every cell once, image nearest to the target
            int c = (int)fminf(fmaxf(floorf((x - lo) * is), -1.0e9f), 1.0e9f);
            u0 = c - (n - 1) / 2;
            u1 = u0 + n - 1;
        }
    } else {
        u0 = min(max(u0, 0), n - 1);
        u1 = min(max(u1, 0), n - 1);
    }
}

// The target coordinate seen from periodic image k: s + l = x - k L exactly (FP64 on the FP32
// inputs), s the nearest float.  d = (s - x_j) + l then has the relative error of one FP32
// subtraction, as for a pair that does not wrap.
__device__ __forceinline__ void sph_image_shift(float x, int k, float L, float& s, float& l) {
    if (abs(k) <= 1) {   // k L is a float: the sum and its rounding error in six additions
        const float b = -(float)k * L;
        s = x + b;
        const float bb = s - x;
        l = (x - (s - bb)) + (b - bb);
    } else {             // grids of fewer than 8 cells along an axis
        const double t = (double)x - (double)k * (double)L;
        s = (float)t;
        l = (float)(t - (double)s);
    }
}

// One contiguous run of candidate sources: sorted positions [start, end), and the target's
// coordinates shifted by the periodic image of the run, so that d = s - x_j (+ l: what the
// rounding of the shift dropped, for the callers that want the displacement to 2^-24 |d|).
struct RowRec {
    uint32_t start, end;
    float    sx, sy, sz;
    float    lx, ly, lz;
};
#define SPH_RCAP 64   // two x segments for each of 32 rows built per batch

// Squared distance from coordinate y to the slab [u*s, (u+1)*s) + lo; edge cells of a
// non-periodic axis extend to infinity (particles outside the box are binned there).
__device__ __forceinline__ float sph_slab_dist(float y, int u, float lo, float s, int n, int per) {
    float a = lo + (float)u * s;
    float below = a - y;           // > 0: y is below the slab
    float above = y - (a + s);     // > 0: y is above the slab
    if (!per) {
        if (u <= 0) below = 0.0f;
        if (u >= n - 1) above = 0.0f;
    }
    float d = fmaxf(fmaxf(below, above) - 1e-3f * s, 0.0f);
    return d;
}

// Warp-collective.  Calls body(const RowRec&) for every non-empty row segment whose cells
// can hold a particle within R of (xi, yi, zi).  `rows` is SPH_RCAP records of this warp's
// shared memory.  All 32 lanes must call with identical arguments.
template <class Body>
__device__ __forceinline__ void sph_for_each_row(const SphGrid& g,
                                                 const uint32_t* __restrict__ cell_start,
                                                 float xi, float yi, float zi, float R,
                                                 RowRec* rows, int lane, Body&& body) {
    int x0, x1, y0, y1, z0, z1;
    sph_axis_range(xi, R, g.lo[0], g.isx, g.nx, g.per[0], x0, x1);
    sph_axis_range(yi, R, g.lo[1], g.isy, g.ny, g.per[1], y0, y1);
    sph_axis_range(zi, R, g.lo[2], g.isz, g.nz, g.per[2], z0, z1);
    const int   kx0  = sph_fdiv(x0, g.nx);
    const int   c0   = x0 - kx0 * g.nx;
    const int   span = x1 - x0;
    const int   a_c1 = min(c0 + span, g.nx - 1);
    const bool  two  = (c0 + span > g.nx - 1);
    const int   b_c1 = c0 + span - g.nx;
    float sxA = xi, sxB = xi, lxA = 0.0f, lxB = 0.0f;
    if (kx0) sph_image_shift(xi, kx0, g.len[0], sxA, lxA);
    if (kx0 + 1) sph_image_shift(xi, kx0 + 1, g.len[0], sxB, lxB);
    const int   nyr  = y1 - y0 + 1, nzr = z1 - z0 + 1, nrow = nyr * nzr;
    const float R2   = R * R * (1.0f + 1e-5f);
    const unsigned lt = (1u << lane) - 1u;

    for (int base = 0; base < nrow; base += 32) {
        const int r  = base + lane;
        bool      ok = r < nrow;
        const int iz = r / nyr, iy = r - iz * nyr;
        const int uy = y0 + iy, uz = z0 + iz;
        uint32_t  a0 = 0, a1 = 0, b0 = 0, b1 = 0;
        float     sy = yi, sz = zi, ly = 0.0f, lz = 0.0f;
        if (ok) {
            float dy = sph_slab_dist(yi, uy, g.lo[1], g.sy, g.ny, g.per[1]);
            float dz = sph_slab_dist(zi, uz, g.lo[2], g.sz, g.nz, g.per[2]);
            ok = (dy * dy + dz * dz <= R2);
        }
        if (ok) {
            const int ky = sph_fdiv(uy, g.ny), cy = uy - ky * g.ny;
            const int kz = sph_fdiv(uz, g.nz), cz = uz - kz * g.nz;
            if (ky) sph_image_shift(yi, ky, g.len[1], sy, ly);
            if (kz) sph_image_shift(zi, kz, g.len[2], sz, lz);
            const uint32_t rb = (uint32_t)(cz * g.ny + cy) * (uint32_t)g.nx;
            a0 = __ldg(cell_start + rb + c0);
            a1 = __ldg(cell_start + rb + a_c1 + 1);
            if (two) {
                b0 = __ldg(cell_start + rb);
                b1 = __ldg(cell_start + rb + b_c1 + 1);
            }
        }
        const bool     va = ok && (a1 > a0), vb = ok && (b1 > b0);
        const unsigned ma = __ballot_sync(SPH_FULL, va), mb = __ballot_sync(SPH_FULL, vb);
        const int      na = __popc(ma);
        if (va) {
            RowRec rr{a0, a1, sxA, sy, sz, lxA, ly, lz};
            rows[__popc(ma & lt)] = rr;
        }
        if (vb) {
            RowRec rr{b0, b1, sxB, sy, sz, lxB, ly, lz};
            rows[na + __popc(mb & lt)] = rr;
        }
        __syncwarp();
        const int cnt = na + __popc(mb);
        for (int q = 0; q < cnt; ++q) {
            const RowRec rr = rows[q];
            body(rr);
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------
// Sub-warp enumeration: the warp holds 32/G targets, G consecutive lanes each.  All loops
// have warp-uniform trip counts (maxima over the groups), groups that have nothing to do
// are predicated off, so the warp never splits.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ int sph_wrap(int u, int n, int& k) {   // u = c + k n, 0 <= c < n
    if (n >= 8) k = (u < 0) ? -1 : ((u >= n) ? 1 : 0);
    else        k = sph_fdiv(u, n);
    int c = u - k * n;
    return min(max(c, 0), n - 1);   // memory-safe even for coordinates outside a periodic box
}

// The image k that a rounded shift s = fl(x - k L) belongs to (0 on a non-periodic axis).
__device__ __forceinline__ int sph_image_of(float x, float s, float L, int per) {
    return per ? __float2int_rn(__fdividef(x - s, L)) : 0;
}

// Walks the candidate sources of every group's target and compacts the accepted ones.
// For candidate j (pj = pos[j], d = displacement to the right periodic image, r2 = |d|^2)
// `accept(pj, r2)` decides; the accepted candidates of a target are numbered 0, 1, 2, ... in
// the order of the sorted arrays (group ballot), and `store(f, j, pj, dx, dy, dz, r2)` is
// called on the lane that tested number f.  Keeping entry f in slot f / G of lane f % G
// gives every lane of the group an equally long column AND makes the G lanes work on G
// consecutive -- mostly memory-adjacent -- sources later.  `total` (uniform in a group) is
// advanced by the number accepted, `tested` by the number of candidates (summed over the lanes).
// `active` (uniform in a group) switches a group off.
template <int G, class Accept, class Store>
__device__ __forceinline__ void sph_group_collect(const SphGrid& g,
                                                  const uint32_t* __restrict__ cell_start,
                                                  const float4* __restrict__ pos, float xi,
                                                  float yi, float zi, float R, bool active,
                                                  int lane, unsigned& tested, int& total,
                                                  Accept&& accept, Store&& store) {
    constexpr unsigned GM = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    int      sl = lane & (G - 1);
    int      g0 = lane & ~(G - 1);
    unsigned lt = (1u << sl) - 1u;   // the lanes of the group below this one
    // kept in registers: without this the compiler re-derives them from SR_TID in every trip
    asm volatile("" : "+r"(sl), "+r"(g0), "+r"(lt));
    int y0, y1, z0, z1;
    sph_axis_range(yi, R, g.lo[1], g.isy, g.ny, g.per[1], y0, y1);
    sph_axis_range(zi, R, g.lo[2], g.isz, g.nz, g.per[2], z0, z1);
    const int   nyr  = y1 - y0 + 1, nzr = z1 - z0 + 1;
    const int   nrow = active ? nyr * nzr : 0;
    const float inv_nyr = __fdividef(1.0f, (float)nyr);
    const float R2   = R * R * (1.0f + 1e-5f);
    const int   nrow_max = __reduce_max_sync(SPH_FULL, nrow);

    for (int rb = 0; rb < nrow_max; rb += G) {
        const int r  = rb + sl;
        bool      ok = r < nrow;
        const int iz = (int)(((float)r + 0.5f) * inv_nyr), iy = r - iz * nyr;
        const int uy = y0 + iy, uz = z0 + iz;
        uint32_t  a0 = 0, a1 = 0, b0 = 0, b1 = 0;
        float     sy = yi, sz = zi, sxa = xi;
        bool      shifted = false;
        float     d2 = 0.0f;
        if (ok) {
            const float dy = sph_slab_dist(yi, uy, g.lo[1], g.sy, g.ny, g.per[1]);
            const float dz = sph_slab_dist(zi, uz, g.lo[2], g.sz, g.nz, g.per[2]);
            d2 = dy * dy + dz * dz;
            ok = (d2 <= R2);
        }
        if (ok) {
            int ky, kz, kx0;
            const int cy = sph_wrap(uy, g.ny, ky), cz = sph_wrap(uz, g.nz, kz);
            sy = yi - (float)ky * g.len[1];
            sz = zi - (float)kz * g.len[2];
            // the row only matters over the chord of the search ball at its distance
            int x0, x1;
            sph_axis_range(xi, sqrtf(R2 - d2), g.lo[0], g.isx, g.nx, g.per[0], x0, x1);
            const int c0   = sph_wrap(x0, g.nx, kx0);
            const int span = x1 - x0;
            sxa = xi - (float)kx0 * g.len[0];
            const uint32_t rq = (uint32_t)(cz * g.ny + cy) * (uint32_t)g.nx;
            a0 = __ldg(cell_start + rq + c0);
            a1 = __ldg(cell_start + rq + min(c0 + span, g.nx - 1) + 1);
            if (c0 + span > g.nx - 1) {   // the row crosses the periodic face: second segment
                b0 = __ldg(cell_start + rq);
                b1 = __ldg(cell_start + rq + min(c0 + span - g.nx, g.nx - 1) + 1);
            }
            shifted = (ky | kz | kx0) != 0 || b1 > b0;
        }
        // Warp-uniform: some row of this batch is met through a periodic image.  The rounded
        // shift x_i - k L is off by up to 2^-24 |x|, which relative to a displacement of a few
        // h is far more than one FP32 subtraction's 2^-24 |d|.  Such a batch takes the second
        // copy of the candidate loop, which carries what the rounding dropped (three more
        // additions per candidate); batches inside the box run the plain loop unchanged.
        const bool wrapany = __any_sync(SPH_FULL, shifted);
        const int  nseg = __any_sync(SPH_FULL, b1 > b0) ? 2 : 1;
        auto segments = [&](auto wrap_tag) {
            constexpr bool WRAP = decltype(wrap_tag)::value;
            float ly = 0.0f, lz = 0.0f;
            if (WRAP) {   // exact shifts of this lane's row, redone from the image it was given
                sph_image_shift(yi, sph_image_of(yi, sy, g.len[1], g.per[1]), g.len[1], sy, ly);
                sph_image_shift(zi, sph_image_of(zi, sz, g.len[2], g.per[2]), g.len[2], sz, lz);
            }
            for (int seg = 0; seg < nseg; ++seg) {
                const uint32_t s0 = seg ? b0 : a0, s1 = seg ? b1 : a1;
                float          sxs = seg ? sxa - g.len[0] : sxa, lxs = 0.0f;
                if (WRAP)
                    sph_image_shift(xi, sph_image_of(xi, sxa, g.len[0], g.per[0]) + seg, g.len[0], sxs, lxs);
                unsigned gm = (__ballot_sync(SPH_FULL, s1 > s0) >> g0) & GM;
                const int nk = __reduce_max_sync(SPH_FULL, __popc(gm));
                if (s1 > s0) tested += s1 - s0;   // every candidate of this lane's row gets tested
                for (int k = 0; k < nk; ++k) {
                    const bool have = gm != 0u;
                    const int  src  = g0 + (have ? (__ffs(gm) - 1) : 0);
                    gm &= gm - 1u;
                    uint32_t       rs  = __shfl_sync(SPH_FULL, s0, src);
                    uint32_t       re  = __shfl_sync(SPH_FULL, s1, src);
                    const float    sxx = __shfl_sync(SPH_FULL, sxs, src);
                    const float    rsy = __shfl_sync(SPH_FULL, sy, src);
                    const float    rsz = __shfl_sync(SPH_FULL, sz, src);
                    float          rlx = 0.0f, rly = 0.0f, rlz = 0.0f;
                    if (WRAP) {
                        rlx = __shfl_sync(SPH_FULL, lxs, src);
                        rly = __shfl_sync(SPH_FULL, ly, src);
                        rlz = __shfl_sync(SPH_FULL, lz, src);
                    }
                    if (!have) re = rs;
                    uint32_t c = rs + sl;
                    // NW windows of G candidates per trip, loaded unconditionally (the sorted arrays
                    // are padded by SPH_POS_PAD records, so reading past a row's end is harmless)
                    auto trip = [&](auto nw_tag) {
                        constexpr int NW = decltype(nw_tag)::value;
                        float4 pp[NW];
#pragma unroll
                        // (a group whose own row is short walks as many windows as the longest
                        // row of the warp: the index is clamped to the row's padded end)
                        for (int u = 0; u < NW; ++u) pp[u] = __ldg(pos + min(c + u * G, re + (uint32_t)(G - 1)));
#pragma unroll
                        for (int u = 0; u < NW; ++u) {
                            float dx = sxx - pp[u].x, dy = rsy - pp[u].y, dz = rsz - pp[u].z;
                            if (WRAP) { dx += rlx; dy += rly; dz += rlz; }
                            const float r2 = dx * dx + dy * dy + dz * dz;
                            const bool  acc = (c + u * G < re) && accept(pp[u], r2);
                            const unsigned gm = (__ballot_sync(SPH_FULL, acc) >> g0) & GM;
                            if (acc)
                                store(total + __popc(gm & lt), c + u * G, pp[u], dx, dy, dz, r2);
                            total += __popc(gm);
                        }
                        c += NW * G;
                    };
                    // the longest row among the four groups decides how many windows are issued
                    const int nwin = (__reduce_max_sync(SPH_FULL, re - rs) + (G - 1)) / G;
                    if (nwin == 1) {
                        trip(std::integral_constant<int, 1>{});
                    } else if (nwin == 2) {
                        trip(std::integral_constant<int, 2>{});
                    } else {
                        for (int w = 0; w < nwin; w += SPH_UNROLL) trip(std::integral_constant<int, SPH_UNROLL>{});
                    }
                }
            }
        };
        if (wrapany) segments(std::true_type{});
        else         segments(std::false_type{});
    }
}

// Step a6: the largest h_j of any particle that can reach (x, y, z), i.e. with
// |x - x_j| < 2 h_j, bounded from the coarse max-h map.  Starts from the
// global maximum and tightens two or three times: every such j lies within 2 H of the target as long
// as H bounds its h_j, so the maximum over the coarse cells meeting that ball is again a bound.
// The map has two levels (coarse cells, and blocks of 8^3 of them behind SPH_COARSE_MAX): a
// pass whose ball meets more than SPH_HMAP_CELLS coarse cells reads the blocks instead, so a
// target with a very large h -- or the first pass, from the global maximum, under a deep h
// contrast -- costs tens of loads, not tens of thousands.  (A ball that crosses a periodic
// face always reads the first level.)
#define SPH_HMAP_CELLS 64
template <int G>
__device__ __forceinline__ float sph_scatter_hmax(const SphGrid& g,
                                                  const unsigned* __restrict__ coarse, float xi,
                                                  float yi, float zi, float hi, float hglobal,
                                                  int lane) {
    const int sl = lane & (G - 1);
    float H = fmaxf(hglobal, hi);
    const float xs[3] = {xi, yi, zi};
    int npass = 2;        // one more if the first one had to read the blocks (warp-uniform)
#pragma unroll 1
    for (int pass = 0; pass < npass; ++pass) {
        int  u0[3], nn[3];
        bool inside = true;   // the ball stays clear of the periodic faces
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const float R = 2.0f * H * (1.0f + 1e-5f);
            float a = floorf((xs[d] - g.lo[d] - R) * g.ics[d] - 1e-3f);
            float b = floorf((xs[d] - g.lo[d] + R) * g.ics[d] + 1e-3f);
            a = fminf(fmaxf(a, -1.0e9f), 1.0e9f);
            b = fminf(fmaxf(b, -1.0e9f), 1.0e9f);
            int lo = (int)a, hi_ = (int)b;
            if (g.per[d]) {
                inside = inside && lo >= 0 && hi_ <= g.cn[d] - 1;
                if (hi_ - lo + 1 >= g.cn[d]) { lo = 0; hi_ = g.cn[d] - 1; }
            } else {
                lo  = min(max(lo, 0), g.cn[d] - 1);
                hi_ = min(max(hi_, 0), g.cn[d] - 1);
            }
            u0[d] = lo;
            nn[d] = hi_ - lo + 1;
        }
        // second level: the blocks that hold the cells [u0, u0 + nn)
        const bool blocks = inside && nn[0] * nn[1] * nn[2] > SPH_HMAP_CELLS;
        const bool anyblk = __any_sync(SPH_FULL, blocks);
        if (pass == 0 && anyblk) npass = 3;
        unsigned best = 0u;
        auto sweep = [&](const unsigned* __restrict__ map, int dx, int dy, int dz) {
            const int   cnt  = nn[0] * nn[1] * nn[2];
            const int   cmax = __reduce_max_sync(SPH_FULL, cnt);
            const float i0 = __fdividef(1.0f, (float)nn[0]), i1 = __fdividef(1.0f, (float)nn[1]);
            for (int q = sl; q < cmax; q += G) {
                if (q < cnt) {
                    const int t  = (int)(((float)q + 0.5f) * i0);          // q / nn[0]
                    const int ix = q - t * nn[0];
                    const int iz = (int)(((float)t + 0.5f) * i1);          // t / nn[1]
                    const int iy = t - iz * nn[1];
                    int cx = u0[0] + ix, cy = u0[1] + iy, cz = u0[2] + iz;
                    cx -= (cx >= dx) ? dx : 0; cx += (cx < 0) ? dx : 0;    // periodic images
                    cy -= (cy >= dy) ? dy : 0; cy += (cy < 0) ? dy : 0;    // (first level only)
                    cz -= (cz >= dz) ? dz : 0; cz += (cz < 0) ? dz : 0;
                    cx = min(max(cx, 0), dx - 1);
                    cy = min(max(cy, 0), dy - 1);
                    cz = min(max(cz, 0), dz - 1);
                    best = max(best, __ldg(map + (cz * dy + cy) * dx + cx));
                }
            }
        };
        if (!anyblk) {   // the common case: every ball of the warp meets a few coarse cells
            sweep(coarse, g.cn[0], g.cn[1], g.cn[2]);
        } else {
            if (blocks) {
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const int b0 = u0[d] >> 3, b1 = (u0[d] + nn[d] - 1) >> 3;
                    u0[d] = b0;
                    nn[d] = b1 - b0 + 1;
                }
            }
            sweep(blocks ? coarse + SPH_COARSE_MAX : coarse, blocks ? g.sn[0] : g.cn[0],
                  blocks ? g.sn[1] : g.cn[1], blocks ? g.sn[2] : g.cn[2]);
        }
#pragma unroll
        for (int o = G / 2; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(SPH_FULL, best, o));
        H = fmaxf(hi, fminf(H, __uint_as_float(best)));
    }
    return H;
}

template <int G>
__device__ __forceinline__ float sph_group_sum(float v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL, v, o);
    return v;
}
template <int G>
__device__ __forceinline__ float sph_group_min(float v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}
template <int G>
__device__ __forceinline__ int sph_group_sum_int(int v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL, v, o);
    return v;
}
template <int G>
__device__ __forceinline__ bool sph_group_any(bool p, int lane) {
    constexpr unsigned GM = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    return ((__ballot_sync(SPH_FULL, p) >> (lane & ~(G - 1))) & GM) != 0u;
}

// Exact (FP64) squared distance of two particles under the minimum-image convention,
// evaluated on the FP32 inputs -- the definition the neighbour sets are tested against
// (reading R7).  Rare: only pairs within a relative band tau of the support edge.
__device__ __forceinline__ double sph_r2_exact(const SphGrid& g, float ax, float ay, float az,
                                               float bx, float by, float bz) {
    double dx = (double)ax - (double)bx, dy = (double)ay - (double)by, dz = (double)az - (double)bz;
    if (g.per[0]) { double L = (double)g.len[0]; dx -= L * rint(dx / L); }
    if (g.per[1]) { double L = (double)g.len[1]; dy -= L * rint(dy / L); }
    if (g.per[2]) { double L = (double)g.len[2]; dz -= L * rint(dz / L); }
    return dx * dx + dy * dy + dz * dz;
}

// Relative half-width of the band around r^2 = 4h^2 inside which the FP32 distance cannot
// be trusted: |delta r^2| / r^2 <= 2 sqrt(3) 2^-24 xext / r + O(2^-22).
__device__ __forceinline__ float sph_band(const SphGrid& g, float h) {
    return 1e-6f + 2.5e-7f * g.xext / h;
}

__device__ __forceinline__ float sph_warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL, v, o);
    return v;
}
__device__ __forceinline__ float sph_warp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(SPH_FULL, v, o));
    return v;
}
__device__ __forceinline__ int sph_warp_sum_int(int v) {
    return __reduce_add_sync(SPH_FULL, v);
}

#endif  // __CUDACC__

// host-side launch helpers implemented across the .cu files
int sph_launch_build(sph_ctx* c, int64_t n, const float* x, const float* y, const float* z,
                     const float* h);
int sph_launch_density(sph_ctx* c, const float* m, float* h, float* rho, float* omega,
                       int32_t* nn);
int sph_launch_forces(sph_ctx* c, const float* m, const float* vx, const float* vy,
                      const float* vz, const float* u, const float* rho, const float* h,
                      const float* omega, float* ax, float* ay, float* az, float* dudt,
                      float* mu_min, float* P, float* cs);
int sph_launch_timestep(sph_ctx* c, const float* h, const float* cs, const float* ax,
                        const float* ay, const float* az, const float* mu_min, float* dt_i,
                        float* dt_min);
int sph_launch_neighbors(sph_ctx* c, const float* h, int32_t mode, int64_t* offsets,
                         int32_t* indices, int64_t capacity, int64_t* needed);
int sph_launch_fp32_peak(cudaStream_t s, float seconds, double* tflops);
int sph_launch_rungs(sph_ctx* c, const float* dt_i, float dt0, int32_t max_rung, int32_t* rung);
int sph_launch_coarse_map(sph_ctx* c);
int sph_launch_buckets(sph_ctx* c);
int sph_launch_density_tile(sph_ctx* c, float* h, float* rho, float* omega, int32_t* nn);
int sph_launch_forces_tile(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min);
int sph_launch_forces_tlist(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min);
int sph_launch_forces_list(sph_ctx* c, float* ax, float* ay, float* az, float* dudt, float* mu_min);
int sph_launch_mark(sph_ctx* c, const uint8_t* src, uint8_t* mark);
int sph_launch_set_active(sph_ctx* c, const uint8_t* active);
int sph_launch_compact(sph_ctx* c, const uint8_t* mask, uint32_t* list, unsigned* cnt);
int sph_launch_interface(sph_ctx* c, const float* m, const float* u, const float* rho, const float* h,
                         const int32_t* mat, float alpha, float* imbalance, float* rho_corr,
                         float* P_corr);
