// sph_build.cu -- steps a1-a3 of DESIGN.md: cell keys, counting sort, cell table.
// Stands in for the tree build of PAPER.md:66-68 ("particles of a cell are contiguous").
// Everything, including the choice of the cell size from min(h), runs on the device.
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int TPB = 256;

__global__ void k_init_red(unsigned* red) {
    red[0] = 0x7f800000u;  // min h  (+inf)
    red[1] = 0u;           // max h
    red[2] = 0u;           // max |coordinate|
}

// min / max of h (positive finite values only) and the largest |coordinate|
__global__ void k_reduce_h(int64_t n, const float* __restrict__ x, const float* __restrict__ y,
                           const float* __restrict__ z, const float* __restrict__ h,
                           unsigned* red) {
    float hmin = __int_as_float(0x7f800000), hmax = 0.0f, xm = 0.0f;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    // four particles per trip: sixteen independent loads in flight per thread
    for (int64_t i0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i0 < n; i0 += 4 * stride) {
        float hv[4], av[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int64_t i = i0 + k * stride;
            const bool in = i < n;
            hv[k] = in ? h[i] : 0.0f;
            av[k] = in ? fmaxf(fabsf(x[i]), fmaxf(fabsf(y[i]), fabsf(z[i]))) : 0.0f;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (hv[k] > 0.0f && hv[k] < 3.0e38f) {
                hmin = fminf(hmin, hv[k]);
                hmax = fmaxf(hmax, hv[k]);
            }
            if (av[k] < 3.0e38f) xm = fmaxf(xm, av[k]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        hmin = fminf(hmin, __shfl_xor_sync(SPH_FULL, hmin, o));
        hmax = fmaxf(hmax, __shfl_xor_sync(SPH_FULL, hmax, o));
        xm   = fmaxf(xm, __shfl_xor_sync(SPH_FULL, xm, o));
    }
    // one set of atomics per block (they all hit the same three words)
    __shared__ float sh[3][TPB / 32];
    if ((threadIdx.x & 31) == 0) {
        sh[0][threadIdx.x >> 5] = hmin; sh[1][threadIdx.x >> 5] = hmax; sh[2][threadIdx.x >> 5] = xm;
    }
    __syncthreads();
    if (threadIdx.x == 0) {  // positive floats order like their bit patterns
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) {
            hmin = fminf(hmin, sh[0][w]); hmax = fmaxf(hmax, sh[1][w]); xm = fmaxf(xm, sh[2][w]);
        }
        atomicMin(red + 0, __float_as_uint(hmin));
        atomicMax(red + 1, __float_as_uint(hmax));
        atomicMax(red + 2, __float_as_uint(xm));
    }
}

// One thread: derive the grid from min(h).  Cell sides: the smallest density search radius
// R_min = 2 h_min slack, divided by cell_div_x along x (rows are contiguous, so fine cells
// along x cost nothing and trim the row ends) and by cell_div_yz along y and z.
// steep_check: automatic tile mode -- a contrast of h above 3 sets SPH_GRID_STEEP and takes the
// cell sides of the 8-lane kernels (divx_s, divyz_s) instead of the tile sweeps' (divx, divyz).
__global__ void k_grid_setup(SphGrid* g, const unsigned* red, sph_box box, float slack, float divx,
                             float divyz, float divx_s, float divyz_m, float divyz_s, int steep_check,
                             long long cap_cells) {
    float hmin = __uint_as_float(red[0]), hmax = __uint_as_float(red[1]);
    float xm = __uint_as_float(red[2]);
    int   flags = 0;
    if (steep_check && hmax > SPH_STEEP_RATIO * hmin) {
        flags |= SPH_GRID_STEEP;
        divx = divx_s;
        // the 8-lane kernels' cells; coarser rows only where h really spreads (measured on C5)
        divyz = hmax > 3.0f * hmin ? divyz_s : divyz_m;
    }
    float lmax = fmaxf(box.len[0], fmaxf(box.len[1], box.len[2]));
    if (!(hmin < 3.0e38f) || !(hmin > 0.0f)) {  // no valid h at all: one coarse grid
        hmin = hmax = lmax * 0.05f;
        flags |= 4;
    }
    float Rmin = 2.0f * hmin * slack;
    float want[3] = {Rmin / divx, Rmin / divyz, Rmin / divyz};
    int   n[3];
    float scale = 1.0f;
    for (int it = 0; it < 64; ++it) {
        double prod = 1.0;
        for (int d = 0; d < 3; ++d) {
            float s  = want[d] * scale;
            float fn = box.len[d] / s;
            fn = fminf(fmaxf(fn, 1.0f), 2.0e9f);
            int nd = box.periodic[d] ? (int)floorf(fn) : (int)ceilf(fn);
            n[d] = max(nd, 1);
            prod *= (double)n[d];
        }
        if (prod <= (double)cap_cells && n[0] < (1 << 20) && n[1] < (1 << 20) && n[2] < (1 << 20))
            break;
        flags |= 2;  // clipped: coarser cells than asked for (slower, still correct)
        double f = cbrt(prod / (double)cap_cells);
        scale *= (float)fmax(f * 1.02, 1.05);
    }
    g->nx = n[0]; g->ny = n[1]; g->nz = n[2];
    g->ncells = n[0] * n[1] * n[2];
    g->sx = box.len[0] / n[0]; g->sy = box.len[1] / n[1]; g->sz = box.len[2] / n[2];
    g->isx = n[0] / box.len[0]; g->isy = n[1] / box.len[1]; g->isz = n[2] / box.len[2];
    float ext = xm;
    for (int d = 0; d < 3; ++d) {
        g->lo[d]  = box.lo[d];
        g->len[d] = box.len[d];
        g->per[d] = box.periodic[d] ? 1 : 0;
        float e = fmaxf(fabsf(box.lo[d]), fabsf(box.lo[d] + box.len[d]));
        if (box.periodic[d]) {
            e += box.len[d];
            // minimum image must be unique for the largest search ball
            if (box.len[d] < 4.0f * hmax * slack) flags |= 1;
        }
        ext = fmaxf(ext, e);
    }
    g->hmin = hmin; g->hmax = hmax; g->xext = ext; g->flags = flags;
    g->force_hmax_bits = 0u;
    // coarse max-h map: cells of about 8 h_min, at most SPH_COARSE_MAX of them
    float cs = 8.0f * hmin * slack;
    for (int it = 0; it < 64; ++it) {
        double prod = 1.0;
        for (int d = 0; d < 3; ++d) {
            float fn = fminf(fmaxf(box.len[d] / cs, 1.0f), 1.0e6f);
            g->cn[d] = max((int)floorf(fn), 1);
            prod *= (double)g->cn[d];
        }
        if (prod <= (double)SPH_COARSE_MAX) break;
        cs *= (float)fmax(cbrt(prod / (double)SPH_COARSE_MAX) * 1.02, 1.05);
    }
    for (int d = 0; d < 3; ++d) g->ics[d] = (float)g->cn[d] / box.len[d];
    for (int d = 0; d < 3; ++d) g->sn[d] = (g->cn[d] + 7) >> 3;
}

__global__ void k_zero_cells(const SphGrid* __restrict__ g, uint32_t* cnt) {
    const int64_t nc = g->ncells;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i <= nc;
         i += (int64_t)gridDim.x * blockDim.x)
        cnt[i] = 0u;
}

// a1: cell key of every particle, and its arrival rank within the cell
__global__ void k_bin(int64_t n, const SphGrid* __restrict__ gp, const float* __restrict__ x,
                      const float* __restrict__ y, const float* __restrict__ z, uint32_t* cnt,
                      uint32_t* key, uint32_t* rank) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const SphGrid& g = *gp;
    int cx = sph_cell_coord(x[i], g.lo[0], g.isx, g.nx);
    int cy = sph_cell_coord(y[i], g.lo[1], g.isy, g.ny);
    int cz = sph_cell_coord(z[i], g.lo[2], g.isz, g.nz);
    uint32_t k = (uint32_t)(cz * g.ny + cy) * (uint32_t)g.nx + (uint32_t)cx;
    key[i]  = k;
    rank[i] = atomicAdd(cnt + k, 1u);
}

// a3: exclusive scan cnt[0..ncells) -> start[0..ncells], three phases over fixed segments
__global__ void k_scan_sum(const SphGrid* __restrict__ g, const uint32_t* __restrict__ cnt,
                           uint32_t* part) {
    const int64_t nc  = g->ncells;
    const int64_t seg = (nc + gridDim.x - 1) / gridDim.x;
    const int64_t a = blockIdx.x * seg, b = min(a + seg, nc);
    uint32_t s = 0;
    for (int64_t i = a + threadIdx.x; i < b; i += blockDim.x) s += cnt[i];
    __shared__ uint32_t sh[TPB / 32];
    s = __reduce_add_sync(SPH_FULL, s);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < TPB / 32; ++w) t += sh[w];
        part[blockIdx.x] = t;
    }
}

__global__ void k_scan_part(uint32_t* part, int nparts) {  // one block of nparts threads
    __shared__ uint32_t sh[SPH_SCAN_BLOCKS];
    int t = threadIdx.x;
    sh[t] = part[t];
    __syncthreads();
    for (int o = 1; o < nparts; o <<= 1) {
        uint32_t v = (t >= o) ? sh[t - o] : 0u;
        __syncthreads();
        sh[t] += v;
        __syncthreads();
    }
    part[t] = (t == 0) ? 0u : sh[t - 1];
    if (t == nparts - 1) part[nparts] = sh[t];
}

__global__ void k_scan_write(const SphGrid* __restrict__ g, const uint32_t* __restrict__ cnt,
                             const uint32_t* __restrict__ part, uint32_t* start) {
    const int64_t nc  = g->ncells;
    const int64_t seg = (nc + gridDim.x - 1) / gridDim.x;
    const int64_t a = blockIdx.x * seg, b = min(a + seg, nc);
    __shared__ uint32_t wsum[TPB / 32];
    __shared__ uint32_t carry_sh;
    if (threadIdx.x == 0) carry_sh = part[blockIdx.x];
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int64_t base = a; base < b; base += TPB) {
        int64_t  i = base + threadIdx.x;
        uint32_t v = (i < b) ? cnt[i] : 0u;
        uint32_t inc = v;  // inclusive warp scan
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(SPH_FULL, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[wid] = inc;
        __syncthreads();
        uint32_t woff = 0, tot = 0;
#pragma unroll
        for (int w = 0; w < TPB / 32; ++w) {
            uint32_t s = wsum[w];
            if (w < wid) woff += s;
            tot += s;
        }
        const uint32_t carry = carry_sh;
        if (i < b) start[i] = carry + woff + inc - v;
        __syncthreads();
        if (threadIdx.x == 0) carry_sh = carry + tot;
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) start[nc] = part[gridDim.x];
}

// a2: place every particle; the order inside a cell is the atomic arrival order for now
__global__ void k_scatter(int64_t n, const uint32_t* __restrict__ key,
                          const uint32_t* __restrict__ rank, const uint32_t* __restrict__ start,
                          int32_t* perm) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    perm[start[key[i]] + rank[i]] = (int32_t)i;
}

// Make the order inside each cell the caller's index order, so that the whole sort (and
// with it every floating-point sum of the sweeps) is deterministic.  One thread per cell
// leader; cells hold a handful of particles.  Cells above the cap keep arrival order.
__global__ void k_cell_sort(int64_t n, const uint32_t* __restrict__ key,
                            const uint32_t* __restrict__ start, int32_t* perm) {
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    const uint32_t k = key[perm[p]];
    const uint32_t a = start[k];
    if (a != (uint32_t)p) return;
    const uint32_t b = start[k + 1];
    if (b - a > 512u) return;
    for (uint32_t i = a + 1; i < b; ++i) {
        int32_t  v = perm[i];
        uint32_t j = i;
        while (j > a && perm[j - 1] > v) {
            perm[j] = perm[j - 1];
            --j;
        }
        perm[j] = v;
    }
}

__global__ void k_gather(int64_t n, const int32_t* __restrict__ perm, const float* __restrict__ x,
                         const float* __restrict__ y, const float* __restrict__ z,
                         const float* __restrict__ h, float4* pos_h, int32_t* inv_perm) {
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int32_t i = perm[p];
    pos_h[p]    = make_float4(x[i], y[i], z[i], h[i]);
    inv_perm[i] = (int32_t)p;
}

}  // namespace

int sph_launch_build(sph_ctx* c, int64_t n, const float* x, const float* y, const float* z,
                     const float* h) {
    cudaStream_t s  = c->stream;
    const int    nb = (int)((n + TPB - 1) / TPB);
    const int    gs = c->sm_count * 8;
    // new positions: the neighbour lists kept from the last density sweep are void
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->nb_rkeep, 0, (size_t)n * sizeof(float), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->bucket_loff, 0xff, (size_t)n * sizeof(uint32_t), s));
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->tl_rkeep, 0, (size_t)n * sizeof(float), s));
    k_init_red<<<1, 1, 0, s>>>(c->red);
    k_reduce_h<<<min(nb, gs), TPB, 0, s>>>(n, x, y, z, h, c->red);
    c->n_build = n;
    const bool  tl = sph_tile_on(c);
    const float ux = c->par.cell_div_x, uyz = c->par.cell_div_yz;   // > 0: the caller's choice
    k_grid_setup<<<1, 1, 0, s>>>(c->grid, c->red, c->box, c->par.search_slack,
                                 ux > 0.0f ? ux : (tl ? 8.0f : 4.0f),
                                 // several hundred neighbours: finer rows keep a bucket of 64 compact
                                 uyz > 0.0f ? uyz : (tl ? (c->par.n_ngb > 100.0f ? 3.0f : 2.0f) : 1.5f),
                                 // steep h contrast: coarser rows (fewer near-empty rows around large-h targets)
                                 ux > 0.0f ? ux : 4.0f, uyz > 0.0f ? uyz : 1.5f, uyz > 0.0f ? uyz : 1.0f,
                                 (tl && c->par.tile == 0) ? 1 : 0, (long long)c->cap_cells);
    k_zero_cells<<<gs, TPB, 0, s>>>(c->grid, c->cell_cnt);
    k_bin<<<nb, TPB, 0, s>>>(n, c->grid, x, y, z, c->cell_cnt, c->key, c->rank);
    k_scan_sum<<<SPH_SCAN_BLOCKS, TPB, 0, s>>>(c->grid, c->cell_cnt, c->scan_part);
    k_scan_part<<<1, SPH_SCAN_BLOCKS, 0, s>>>(c->scan_part, SPH_SCAN_BLOCKS);
    k_scan_write<<<SPH_SCAN_BLOCKS, TPB, 0, s>>>(c->grid, c->cell_cnt, c->scan_part,
                                                 c->cell_start);
    k_scatter<<<nb, TPB, 0, s>>>(n, c->key, c->rank, c->cell_start, c->perm);
    k_cell_sort<<<nb, TPB, 0, s>>>(n, c->key, c->cell_start, c->perm);
    k_gather<<<nb, TPB, 0, s>>>(n, c->perm, x, y, z, h, c->pos_h, c->inv_perm);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    if (sph_tile_on(c)) return sph_launch_buckets(c);   // a3: the bucket table
    return SPH_OK;
}
