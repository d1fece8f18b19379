// sph_api.cu -- the extern "C" boundary of include/sph.h: context life cycle, argument
// checks, error text, counters.  All compute is in the sph_*.cu kernels it dispatches to.
#include <cstdio>
#include <cstring>
#include <new>
#include "sph_internal.cuh"
#include "sph_tile.cuh"

static void fill_defaults(sph_params& p) {
    if (!(p.n_ngb > 0.0f)) p.n_ngb = 64.0f;
    if (!(p.gamma > 1.0f)) p.gamma = 5.0f / 3.0f;
    if (!(p.av_eps > 0.0f)) p.av_eps = 0.01f;
    if (!(p.eta_cfl > 0.0f)) p.eta_cfl = 0.3f;
    if (!(p.eta_acc > 0.0f)) p.eta_acc = 0.2f;
    if (!(p.h_tol > 0.0f)) p.h_tol = 1e-6f;
    if (p.h_max_iter <= 0) p.h_max_iter = 40;
    if (!(p.search_slack > 1.0f)) p.search_slack = 1.1f;
    // cell_div_x / cell_div_yz <= 0 stay "automatic": sph_build_cells picks 8 x 2 for the staged-
    // tile sweeps and 4 x 1.5 for the 8-lane kernels (4 x 1 under the grid's steep-h flag)
    if (p.tile_rows <= 0) p.tile_rows = p.n_ngb > 100.0f ? 2 : 3;
    if (p.tile_rows > 5) p.tile_rows = 5;
    // tile capacities follow the neighbour number: ~12 x n_ngb candidates reach a bucket of 64 targets
    if (p.tile_cap <= 0) p.tile_cap = (int)fminf(fmaxf(12.0f * p.n_ngb, 768.0f), 3072.0f);
    p.tile_cap = (p.tile_cap + 31) & ~31;
    if (p.tile_cap > 4096) p.tile_cap = 4096;
    if (p.tile_cap2 <= 0) p.tile_cap2 = p.n_ngb > 64.0f ? 4064 : 2560;
    p.tile_cap2 = (p.tile_cap2 + 31) & ~31;
    if (p.tile_cap2 > 4064) p.tile_cap2 = 4064;
    if (p.tile_warps <= 0) p.tile_warps = 2;
    if (p.tile_warps > 2) p.tile_warps = 2;
    if (p.tile_fcap <= 0) p.tile_fcap = 576;
    p.tile_fcap = (p.tile_fcap + 31) & ~31;
    if (p.tile_fcap > 4096) p.tile_fcap = 4096;
    if (p.tile_fwarps <= 0) p.tile_fwarps = 1;
    if (p.tile_fwarps > SPH_TWMAX) p.tile_fwarps = SPH_TWMAX;
}

template <class T>
static cudaError_t dalloc(T** p, size_t count) {
    return cudaMalloc((void**)p, count * sizeof(T));
}

extern "C" int sph_create(sph_ctx** out, const sph_params* params, const sph_box* box,
                          int64_t n_max, void* cuda_stream) {
    if (!out || !params || !box || n_max <= 0 || n_max > (int64_t)0x7fffff00) return SPH_EINVAL;
    if (params->kernel < 0 || params->kernel > 3) return SPH_EINVAL;
    {   // Eq. (6) has a root only if the target exceeds the self contribution (32 pi/3) W(0) h^3
        static const float self[4] = {32.0f / 3.0f, 14.0f, 20.625f, 28.4375f};
        if (params->n_ngb > 0.0f && params->n_ngb <= self[params->kernel]) return SPH_EINVAL;
    }
    for (int d = 0; d < 3; ++d)
        if (!(box->len[d] > 0.0f)) return SPH_EINVAL;
    sph_ctx* c = new (std::nothrow) sph_ctx;
    if (!c) return SPH_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->par = *params;
    fill_defaults(c->par);
    c->box    = *box;
    c->n_max  = n_max;
    c->stream = (cudaStream_t)cuda_stream;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete c;
        return SPH_ECUDA;
    }
    // cell table: a few cells per particle is the working point; vacuum around free
    // surfaces needs more, hence the generous cap (4 B per cell)
    c->cap_cells = 8 * n_max + (1 << 20);
    if (c->cap_cells > ((int64_t)1 << 30)) c->cap_cells = (int64_t)1 << 30;
    bool ok = true;
    ok = ok && dalloc(&c->grid, 1) == cudaSuccess;
    ok = ok && dalloc(&c->red, 8) == cudaSuccess;
    ok = ok && dalloc(&c->cell_cnt, (size_t)c->cap_cells + 1) == cudaSuccess;
    ok = ok && dalloc(&c->cell_start, (size_t)c->cap_cells + 1) == cudaSuccess;
    ok = ok && dalloc(&c->key, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->rank, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->perm, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->inv_perm, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->scan_part, (size_t)SPH_SCAN_BLOCKS + 1) == cudaSuccess;
    ok = ok && dalloc(&c->pos_h, (size_t)n_max + SPH_POS_PAD) == cudaSuccess;
    ok = ok && dalloc(&c->pos_m, (size_t)n_max + SPH_POS_PAD) == cudaSuccess;
    // every array handed to sph_group_collect carries the padding its window loads rely on
    ok = ok && dalloc(&c->vel_m, (size_t)n_max + SPH_POS_PAD) == cudaSuccess;
    ok = ok && dalloc(&c->rcak, (size_t)n_max + SPH_POS_PAD) == cudaSuccess;
    ok = ok && dalloc(&c->stats, (size_t)ST_NCOUNTERS) == cudaSuccess;
    ok = ok && dalloc(&c->coarse_hmax, (size_t)2 * SPH_COARSE_MAX) == cudaSuccess;
    // bucket-major lists of the tile sweep: lcap entries per target hold the list ball (2h x 1.03 for
    // the moment solve of Wendland C2, 2h x search_slack for the Halley sweeps) with a margin of 30 %;
    // the pool holds a region of lcap x 64 words for every bucket at an average fill of 43 targets,
    // and never less than the [target][192] lists of the 8-lane kernels need
    {
        const float sl = c->par.kernel == 1 ? 1.031f : c->par.search_slack;
        int lc = (int)(c->par.n_ngb * sl * sl * sl * 1.3f) + 32;
        lc = (lc + 31) & ~31;
        c->lcap = lc < SPH_LCAP_MIN ? SPH_LCAP_MIN : lc;
        size_t per = (size_t)c->lcap * 3 / 2;
        if (per < (size_t)SPH_SLOTS * SPH_G) per = (size_t)SPH_SLOTS * SPH_G;
        c->nb_words = (size_t)n_max * per;
    }
    ok = ok && dalloc(&c->nb_j, c->nb_words) == cudaSuccess;
    ok = ok && dalloc(&c->nb_cnt, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->nb_rkeep, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->fix_list, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->fix_cnt, (size_t)2) == cudaSuccess;
    ok = ok && dalloc(&c->act_list, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->act_cnt, (size_t)2) == cudaSuccess;
    ok = ok && dalloc(&c->buckets, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->bucket_cnt, (size_t)1) == cudaSuccess;
    ok = ok && dalloc(&c->tile_next, (size_t)4) == cudaSuccess;
    ok = ok && dalloc(&c->big_list, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->big_cnt, (size_t)2) == cudaSuccess;
    ok = ok && dalloc(&c->list_next, (size_t)1) == cudaSuccess;
    ok = ok && dalloc(&c->bucket_rt, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->bucket_loff, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->tl_rkeep, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->fb_list, (size_t)n_max) == cudaSuccess;
    ok = ok && dalloc(&c->fb_cnt, (size_t)2) == cudaSuccess;
    ok = ok && dalloc(&c->dt_part, (size_t)1024) == cudaSuccess;
    ok = ok && dalloc(&c->nb_total, (size_t)2) == cudaSuccess;
    if (ok) ok = cudaMemsetAsync(c->stats, 0, ST_NCOUNTERS * sizeof(unsigned long long),
                                 c->stream) == cudaSuccess;
    if (ok) ok = cudaMemsetAsync(c->grid, 0, sizeof(SphGrid), c->stream) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        sph_destroy(c);
        return SPH_ENOMEM;
    }
    *out = c;
    return SPH_OK;
}

extern "C" void sph_destroy(sph_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    cudaFree(c->grid);      cudaFree(c->red);       cudaFree(c->cell_cnt);
    cudaFree(c->cell_start); cudaFree(c->key);      cudaFree(c->rank);
    cudaFree(c->perm);      cudaFree(c->inv_perm);  cudaFree(c->scan_part);
    cudaFree(c->pos_h);     cudaFree(c->pos_m);     cudaFree(c->vel_m);
    cudaFree(c->rcak);      cudaFree(c->stats);     cudaFree(c->dt_part);
    cudaFree(c->nb_total);  cudaFree(c->fix_list);  cudaFree(c->fix_cnt);
    cudaFree(c->coarse_hmax);
    cudaFree(c->act_list);  cudaFree(c->act_cnt);
    cudaFree(c->nb_j);      cudaFree(c->nb_cnt);   cudaFree(c->nb_rkeep);
    cudaFree(c->buckets);   cudaFree(c->bucket_cnt); cudaFree(c->tile_next);
    cudaFree(c->fb_list);   cudaFree(c->fb_cnt);
    cudaFree(c->big_list);  cudaFree(c->big_cnt);
    cudaFree(c->list_next); cudaFree(c->bucket_loff); cudaFree(c->tl_rkeep); cudaFree(c->bucket_rt);
    delete c;
}

static int fail(sph_ctx* c, int code, const char* what) {
    if (c) snprintf(c->err, sizeof(c->err), "%s: %s", sph_strerror(code), what);
    return code;
}

extern "C" int sph_build_cells(sph_ctx* c, int64_t n, const float* x, const float* y,
                               const float* z, const float* h) {
    if (!c) return SPH_EINVAL;
    if (!x || !y || !z || !h) return fail(c, SPH_EINVAL, "sph_build_cells: null array");
    if (n <= 0 || n > c->n_max) return fail(c, SPH_EINVAL, "sph_build_cells: n out of range");
    c->built = false;
    c->forces_ready = false;
    c->act_on = false;   // the active set is a list of sorted positions of the old index
    int rc = sph_launch_build(c, n, x, y, z, h);
    if (rc == SPH_OK) {
        c->n     = n;
        c->built = true;
    }
    return rc;
}

extern "C" int sph_density_h(sph_ctx* c, const float* m, float* h, float* rho, float* omega,
                             int32_t* nn) {
    if (!c) return SPH_EINVAL;
    if (!m || !h || !rho || !omega || !nn) return fail(c, SPH_EINVAL, "sph_density_h: null array");
    if (!c->built) return fail(c, SPH_ESTALE, "sph_density_h before sph_build_cells");
    return sph_launch_density(c, m, h, rho, omega, nn);
}

extern "C" int sph_forces(sph_ctx* c, const float* m, const float* vx, const float* vy,
                          const float* vz, const float* u, const float* rho, const float* h,
                          const float* omega, float* ax, float* ay, float* az, float* dudt,
                          float* mu_min, float* P, float* cs) {
    if (!c) return SPH_EINVAL;
    if (!m || !vx || !vy || !vz || !u || !rho || !h || !omega || !ax || !ay || !az || !dudt ||
        !mu_min || !P || !cs)
        return fail(c, SPH_EINVAL, "sph_forces: null array");
    if (!c->built) return fail(c, SPH_ESTALE, "sph_forces before sph_build_cells");
    const int rc = sph_launch_forces(c, m, vx, vy, vz, u, rho, h, omega, ax, ay, az, dudt, mu_min, P, cs);
    c->forces_ready = (rc == SPH_OK);
    return rc;
}

extern "C" int sph_interface_correction(sph_ctx* c, const float* m, const float* u,
                                        const float* rho, const float* h, const int32_t* mat,
                                        float alpha, float* imbalance, float* rho_corr,
                                        float* P_corr) {
    if (!c) return SPH_EINVAL;
    if (!m || !u || !rho || !h || !imbalance || !rho_corr || !(alpha >= 0.0f))
        return fail(c, SPH_EINVAL, "sph_interface_correction: bad argument");
    if (!c->built) return fail(c, SPH_ESTALE, "sph_interface_correction before sph_build_cells");
    return sph_launch_interface(c, m, u, rho, h, mat, alpha, imbalance, rho_corr, P_corr);
}

// sweeps over the active set of a rung, and the FastGas marking pass
extern "C" int sph_set_active(sph_ctx* c, const uint8_t* active) {
    if (!c) return SPH_EINVAL;
    if (!c->built) return fail(c, SPH_ESTALE, "sph_set_active before sph_build_cells");
    if (!active) {
        c->act_on = false;
        return SPH_OK;
    }
    const int rc = sph_launch_set_active(c, active);
    c->act_on = (rc == SPH_OK);
    return rc;
}

extern "C" int sph_mark_neighbors(sph_ctx* c, const uint8_t* src, uint8_t* mark) {
    if (!c) return SPH_EINVAL;
    if (!src || !mark) return fail(c, SPH_EINVAL, "sph_mark_neighbors: null array");
    if (!c->built) return fail(c, SPH_ESTALE, "sph_mark_neighbors before sph_build_cells");
    return sph_launch_mark(c, src, mark);
}

extern "C" int sph_rungs(sph_ctx* c, const float* dt_i, float dt0, int32_t max_rung, int32_t* rung) {
    if (!c) return SPH_EINVAL;
    if (!dt_i || !rung || !(dt0 > 0.0f) || max_rung < 0 || max_rung > 62)
        return fail(c, SPH_EINVAL, "sph_rungs: bad argument");
    if (!c->built || !c->forces_ready)
        return fail(c, SPH_ESTALE, "sph_rungs needs sph_forces on the current positions");
    return sph_launch_rungs(c, dt_i, dt0, max_rung, rung);
}

extern "C" int sph_timestep(sph_ctx* c, const float* h, const float* cs, const float* ax,
                            const float* ay, const float* az, const float* mu_min, float* dt_i,
                            float* dt_min) {
    if (!c) return SPH_EINVAL;
    if (!h || !cs || !ax || !ay || !az || !mu_min || !dt_i || !dt_min)
        return fail(c, SPH_EINVAL, "sph_timestep: null array");
    if (c->n <= 0) return fail(c, SPH_ESTALE, "sph_timestep before sph_build_cells");
    return sph_launch_timestep(c, h, cs, ax, ay, az, mu_min, dt_i, dt_min);
}

extern "C" int sph_neighbors(sph_ctx* c, const float* h, int32_t mode, int64_t* offsets,
                             int32_t* indices, int64_t capacity, int64_t* needed) {
    if (!c) return SPH_EINVAL;
    if (!h || !offsets || !needed || (mode != 0 && mode != 1) || capacity < 0 ||
        (capacity > 0 && !indices))
        return fail(c, SPH_EINVAL, "sph_neighbors: bad argument");
    if (!c->built) return fail(c, SPH_ESTALE, "sph_neighbors before sph_build_cells");
    return sph_launch_neighbors(c, h, mode, offsets, indices, capacity, needed);
}

extern "C" int sph_stats(sph_ctx* c, sph_stats_t* out) {
    if (!c || !out) return SPH_EINVAL;
    unsigned long long v[ST_NCOUNTERS];
    SphGrid g;
    SPH_CUDA_CHECK(c, cudaMemcpyAsync(v, c->stats, sizeof(v), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_CHECK(c, cudaMemcpyAsync(&g, c->grid, sizeof(g), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    memset(out, 0, sizeof(*out));
    out->dens_tested    = (int64_t)v[ST_DENS_TESTED];
    out->dens_listed    = (int64_t)v[ST_DENS_LISTED];
    out->dens_pairs     = (int64_t)v[ST_DENS_PAIRS];
    out->dens_sweeps    = (int64_t)v[ST_DENS_SWEEPS];
    out->dens_recollect = (int64_t)v[ST_DENS_RECOLLECT];
    out->dens_overflow  = (int64_t)v[ST_DENS_OVERFLOW];
    out->dens_nonconv   = (int64_t)v[ST_DENS_NONCONV];
    out->dens_recheck   = (int64_t)v[ST_DENS_RECHECK];
    out->force_tested   = (int64_t)v[ST_FORCE_TESTED];
    out->force_pairs    = (int64_t)v[ST_FORCE_PAIRS];
    out->force_av_pairs = (int64_t)v[ST_FORCE_AV];
    out->n_cells        = g.ncells;
    out->grid_flags     = g.flags;
    out->reserved[0]    = g.nx;
    out->reserved[1]    = g.ny;
    out->reserved[2]    = g.nz;
    return SPH_OK;
}

extern "C" int sph_stats_reset(sph_ctx* c) {
    if (!c) return SPH_EINVAL;
    SPH_CUDA_CHECK(c, cudaMemsetAsync(c->stats, 0, ST_NCOUNTERS * sizeof(unsigned long long),
                                      c->stream));
    return SPH_OK;
}

extern "C" int sph_permutation(sph_ctx* c, int32_t* perm_out) {
    if (!c || !perm_out) return SPH_EINVAL;
    if (!c->built) return fail(c, SPH_ESTALE, "sph_permutation before sph_build_cells");
    SPH_CUDA_CHECK(c, cudaMemcpyAsync(perm_out, c->perm, (size_t)c->n * sizeof(int32_t),
                                      cudaMemcpyDeviceToDevice, c->stream));
    return SPH_OK;
}

extern "C" int sph_fp32_peak(void* cuda_stream, float seconds, double* tflops) {
    if (!tflops || !(seconds > 0.0f)) return SPH_EINVAL;
    return sph_launch_fp32_peak((cudaStream_t)cuda_stream, seconds, tflops);
}

extern "C" const char* sph_strerror(int code) {
    switch (code) {
    case SPH_OK:     return "ok";
    case SPH_EINVAL: return "invalid argument";
    case SPH_EBOX:   return "periodic box too small for the kernel support";
    case SPH_ENOMEM: return "out of device memory";
    case SPH_ECUDA:  return "CUDA error";
    case SPH_ESTALE: return "index not built";
    case SPH_ENOSPC: return "output capacity too small";
    }
    return "unknown error";
}

extern "C" const char* sph_last_error(const sph_ctx* c) { return c ? c->err : ""; }
