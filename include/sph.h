/*
 * sph.h -- C-ABI of the B200-native SPH interaction sweep (arxiv/paper_2511_11425,
 * "SPH in pkdgrav3 for Shock Physics Simulations. I. Hydrodynamics").
 *
 * The library computes, on ONE GPU (sm_100a), the data-parallel hot path of the paper's
 * SPH method: neighbour search within the kernel support 2h (Section
 * 2.3.2), the density / smoothing-length solve (Eqs. 5-7), the hydro
 * force pass with Monaghan artificial viscosity and the ideal-gas EOS (PAPER.md:186-219,
 * Eqs. 13-18) and the time-step criteria (Eq. 26).
 *
 * Conventions for every call
 *   - All array pointers are DEVICE pointers to FP32 (or int32 / int64 where stated)
 *     arrays of length n in the CALLER'S particle order, both for inputs and outputs.
 *     The spatial sort is internal.  The caller owns every array it passes; the context
 *     owns its sorted copies, cell table and scratch, all allocated in sph_create.
 *   - Work is enqueued on the CUDA stream given to sph_create; calls do not synchronise
 *     unless stated (sph_stats, sph_neighbors, sph_fp32_peak do).
 *   - Return value: SPH_OK (0) or a negative error code.  No exceptions, no exit, no
 *     printing.  sph_last_error gives a text for the last failure of a context.
 *   - Positions on a periodic axis must lie in [lo, lo + len) (sph_drift wraps them); a
 *     coordinate outside is binned into the edge cell and its neighbours across the face
 *     are missed.  On an open axis any coordinate is fine (edge cells extend to infinity).
 *   - Device memory of a context: about 1 KB per particle of n_max (768 B of it the neighbour
 *     lists kept between sph_density_h and sph_forces; for n_ngb > 64 that part grows to about
 *     8 n_ngb s^3 bytes, s = search_slack: 4.4 KB per particle at Wendland C6 / 400) plus 4 B per
 *     cell of the index.
 *   - Call order: sph_build_cells -> sph_density_h -> sph_forces -> sph_timestep.
 *     sph_forces / sph_neighbors may be fed rho, h, Omega from elsewhere as long as
 *     sph_build_cells ran on the same positions (else SPH_ESTALE).
 *   - Kernels have support radius 2h (readings R2, R3), e.g. Wendland C2
 *       W(r,h) = h^-3 (21/(16 pi)) (1-q/2)^4 (1+2q),  q = r/h < 2.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SPH_OK      = 0,
    SPH_EINVAL  = -1, /* null pointer, n <= 0, n > n_max, bad parameter                  */
    SPH_EBOX    = -2, /* a periodic side is shorter than 2 x the search diameter, so the  */
                      /* minimum image is not unique; reported by sph_stats */
    SPH_ENOMEM  = -3, /* device allocation failed                                         */
    SPH_ECUDA   = -4, /* CUDA runtime error (text in sph_last_error)                      */
    SPH_ESTALE  = -5, /* sph_build_cells has not run for this n                           */
    SPH_ENOSPC  = -6  /* sph_neighbors: `capacity` too small; *needed holds the size      */
};

typedef struct {
    float   lo[3];        /* lower corner                                                  */
    float   len[3];       /* side lengths (> 0)                                            */
    int32_t periodic[3];  /* 1: periodic in that dimension (minimum image)    */
} sph_box;

typedef struct {
    int32_t kernel;       /* 0 cubic spline, 1 Wendland C2, 2 Wendland C4, 3 Wendland C6, all  */
                          /* with support radius 2h                           */
    float   n_ngb;        /* kernel mass in units of m_i, Eq. (6) with R_kernel = 2h       */
    float   gamma;        /* ideal gas P = (gamma-1) rho u                  */
    float   av_alpha;     /* Eq. (15) alpha                                                */
    float   av_beta;      /* Eq. (15) beta                                                 */
    float   av_eps;       /* Eq. (16) epsilon (0.01, Monaghan 1992)                        */
    float   eta_cfl;      /* Eq. (26) Courant parameter eta_C                              */
    float   eta_acc;      /* eta_a = 0.2                                    */
    float   h_tol;        /* relative width at which a bisection bracket of h counts as     */
                          /* converged (<= 0: default 1e-6); regular steps stop earlier:    */
                          /* a Halley step below 3e-4 h is final      */
    int32_t h_max_iter;   /* sweep cap per particle (<= 0: default 40)                      */
    float   search_slack; /* density search radius = 2 h_guess x this (<= 1: default 1.1);  */
                          /* PAPER.md:152 "slightly larger kernel"; results do not depend   */
                          /* on it                                                         */
    float   cell_div_x;   /* cells per minimum search radius along x (<= 0: automatic: 8     */
                          /* when the staged-tile sweeps run, 4 otherwise)                   */
    float   cell_div_yz;  /* ... along y and z (<= 0: automatic: 2 with tiles (3 for n_ngb >  */
                          /* 100), else 1.5, or 1 where max h > 3 min h)                      */
    int32_t entropy;      /* 1: entropy-conserving variant: sph_forces drops */
                          /* the Eq. (14) term, dudt is the viscous heating of Eq. (18)     */
                          /* alone; the caller advances u with sph_isentropic_u             */
    int32_t tile;         /* staged-tile sweeps (buckets of 64 targets over a shared-memory   */
                          /* tile of sources).  0 (default) = automatic: */
                          /* on for n >= 2^17 particles unless max h > 1.6 min h at build time */
                          /* (decided on the device); 1 = on whatever the size or h contrast; */
                          /* -1 = off: every target takes the 8-lanes-per-target kernels.     */
                          /* Results do not depend on it beyond rounding                      */
    int32_t tile_rows;    /* a bucket spans tile_rows x tile_rows rows of cells (<= 0:        */
                          /* default 3, or 2 for n_ngb > 100; at most 5)                      */
    int32_t tile_cap;     /* candidates a tile holds (<= 0: default 12 n_ngb, between 768 and */
                          /* 3072); buckets that need more go to the second pass              */
    int32_t tile_cap2;    /* tile of the second pass (<= 0: default 2560 for n_ngb <= 64,     */
                          /* else 4064, the largest; below tile_cap + 32: no second pass);    */
                          /* buckets it cannot hold either fall back to the 8-lane kernels    */
    int32_t tile_warps;   /* warps per bucket of the density sweep: 2 (default, <= 0) = one   */
                          /* target per thread; 1 = one warp, two targets per lane            */
    int32_t tile_forces;  /* 0 (default): the force sweep reads the bucket-major neighbour    */
                          /* lists the tile density sweep kept and gathers the source records */
                          /* from global memory (one warp per bucket); 2: the same lists as   */
                          /* tile indices, the bucket's records staged in shared memory; 1:   */
                          /* no lists, the force sweep runs on staged tiles with its own      */
                          /* accept masks (1 and 2 measured slower)      */
    int32_t tile_fcap;    /* tile_cap and tile_warps of the force sweep (<= 0: defaults 576   */
    int32_t tile_fwarps;  /* and 1); its tile holds 52 B per candidate, the density tile 20   */
} sph_params;

/* 64-bit counters accumulated on the device since the last sph_stats_reset.             */
typedef struct {
    int64_t dens_tested;      /* candidate pairs distance-tested by sph_density_h          */
    int64_t dens_listed;      /* pairs put on the per-target lists (within the slack ball)  */
    int64_t dens_pairs;       /* sum_i n_i at the final h (self included)                  */
    int64_t dens_sweeps;      /* sweeps over the neighbour lists, summed over particles    */
    int64_t dens_recollect;   /* targets whose search ball had to be rebuilt larger        */
    int64_t dens_overflow;    /* targets finished by the robust list-free kernel (a list   */
                              /* column overflowed, or an entry sat in the FP64 band)      */
    int64_t dens_nonconv;     /* particles not converged within h_max_iter                 */
    int64_t dens_recheck;     /* borderline pairs re-evaluated in FP64                     */
    int64_t force_tested;     /* candidate pairs distance-tested by sph_forces             */
    int64_t force_pairs;      /* pairs with 0 < r < 2 max(h_i,h_j) (FP32 test)             */
    int64_t force_av_pairs;   /* of those, approaching pairs (v_ij . r_ij < 0)             */
    int64_t n_cells;          /* cells in the index of the last sph_build_cells            */
    int64_t grid_flags;       /* bit 0: SPH_EBOX condition met; bit 1: cell table clipped   */
    int64_t reserved[3];
} sph_stats_t;

typedef struct sph_ctx sph_ctx;

/* Create a context for up to n_max particles on the current CUDA device.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Allocates all scratch.    */
int  sph_create(sph_ctx** out, const sph_params* params, const sph_box* box, int64_t n_max,
                void* cuda_stream);
void sph_destroy(sph_ctx* ctx);

/* Steps a1-a3: spatial index standing in for the tree of PAPER.md:66-68,
 * 121-127.  Bins the n particles into a uniform grid whose cell sides derive from
 * min(h) (device-side, no host round trip), counting-sorts them so that every x-row of
 * cells is one contiguous particle range, and keeps the permutation.  h is the caller's
 * current guess of the smoothing lengths (> 0); it only sizes the cells.                 */
int  sph_build_cells(sph_ctx* ctx, int64_t n, const float* x, const float* y, const float* z,
                     const float* h);

/* Steps a4-a6: Eqs. (5)-(7).  For every particle finds h_i with
 * (32 pi/3) sum_j m_j w(r_ij/h_i) = n_ngb m_i (gather, self included) by a safeguarded
 * Newton-type (Halley) iteration on a per-target neighbour list, then writes
 *   h_inout (in: guess, out: solution), rho = sum_j m_j W_ij(h_i), omega (Eq. 7),
 *   n_ngb_out = #{j : r_ij < 2 h_i} (borderline pairs decided in FP64).
 * Along a periodic axis of side L, h_i is capped at L/5: the search ball 2 h x 1.25 then
 * stays below L/2, where the minimum image is unique (PAPER.md:297 asks for the same).  A
 * particle whose root lies above the cap, or that runs out of h_max_iter sweeps, keeps its
 * last iterate and is counted in sph_stats_t.dens_nonconv (no host synchronisation here). */
int  sph_density_h(sph_ctx* ctx, const float* m, float* h_inout, float* rho, float* omega,
                   int32_t* n_ngb_out);

/* Steps a7-a9: Eqs. (13)-(18), with P = (gamma-1) rho u, c = sqrt(gamma
 * P/rho).  Pair set: 0 < r_ij < 2 max(h_i,h_j) (gather and scatter).
 * Outputs: acceleration a, du/dt = Eq. (14) + Eq. (18), mu_min_i = min(0, min_j mu_ij),
 * and the EOS values P, c.  v and u are whatever the caller wants used (the "predicted"
 * values of PAPER.md:232-240).                                                           */
int  sph_forces(sph_ctx* ctx, const float* m, const float* vx, const float* vy, const float* vz,
                const float* u, const float* rho, const float* h, const float* omega,
                float* ax, float* ay, float* az, float* dudt, float* mu_min, float* P,
                float* c);

/* Steps a10-a11: PAPER.md:263-268.  dt_a = eta_a sqrt(2h/|a|) (no limit if a = 0),
 * dt_CFL = eta_C h/((1+0.6 alpha) c + 0.6 beta |mu_min|), dt_i = min of the two,
 * *dt_min_device = min_i dt_i (one float in device memory).                              */
int  sph_timestep(sph_ctx* ctx, const float* h, const float* c, const float* ax, const float* ay,
                  const float* az, const float* mu_min, float* dt_i, float* dt_min_device);

/* Time-step rungs.  rung_i = the smallest r >= 0 with 2^-r dt0 <= dt_i
 * (Eq. 27, capped at max_rung <= 62), then the limiter of Saitoh & Makino (2009): rung_i >=
 * rung_j - 2 for every particle j of the force pair set of i, one pass over the Eq. (27)
 * values.  Uses the neighbour data of the last sph_forces (same positions, same h), else
 * SPH_ESTALE.  rung: n int32, caller order.                                                  */
int  sph_rungs(sph_ctx* ctx, const float* dt_i, float dt0, int32_t max_rung, int32_t* rung);

/* The active set of a rung, PAPER.md:229, 274 ("only the particles on the active rungs are
 * updated").  active: n bytes in device memory, caller order, non-zero = active; NULL = all
 * particles again.  Until the next sph_build_cells (which clears the set: it is held as a
 * list of positions in the index) sph_density_h and sph_forces take their TARGETS from the
 * set only -- the entries of their output arrays that belong to inactive particles are not
 * touched -- while the sources remain all particles, whose input arrays (m, h, rho, ...)
 * must therefore be valid for every particle.  The results for an active particle are the
 * ones of the full sweep.  sph_timestep, sph_rungs and the other calls ignore the set.
 * SPH_ESTALE before sph_build_cells.                                                       */
int  sph_set_active(sph_ctx* ctx, const uint8_t* active);

/* The FastGas marking pass: "mark all particles that would end up on
 * interaction lists of active particles".  mark_i = 1 if src_i != 0 or if some particle j
 * with src_j != 0 interacts with i (the force pair set 0 < r_ij < 2 max(h_i, h_j), with the
 * h given to sph_build_cells or, once sph_forces has run on this index, the h given to it);
 * else 0.  Borderline pairs are decided in FP64, so the marks are exact.  A second call with
 * src = the first marks gives the paper's second marking pass.  src, mark: n bytes, device
 * memory, caller order; they may not alias.  Only the particles of src walk their
 * neighbourhood (the pair set is symmetric), so the cost follows the size of the set.
 * SPH_ESTALE before sph_build_cells.                                                       */
int  sph_mark_neighbors(sph_ctx* ctx, const uint8_t* src, uint8_t* mark);

/* Interface correction for the ideal gas, PAPER.md:158-182 (Section 2.3.4), Eqs. (8)-(12);
 * call between sph_density_h and sph_forces and hand rho_corr to sph_forces.  Gather sums over
 * r_ij < 2 h_i, self included.
 *   imbalance  I_i = alpha |sum_j kappa_ij (r_j - r_i) m_j W_ij(h_i)| / (h_i sum_j m_j W_ij(h_i)),
 *              kappa_ij = +1 for equal material ids, -1 otherwise (mat may be NULL: one material)
 *   rho_corr   Eq. (12) with T = u / c_v: P~ / ((gamma-1) u~), where P~, u~ are P_i, u_i mixed
 *              with their e^{-I_j^2} W_ij(h_i)-weighted kernel averages by e^{-I_i^2} (Eqs. 9-11)
 *   P_corr     P~ (may be NULL)
 * alpha: the "normalization parameter" of Eq. (8); the paper gives no value (1.5 in the
 * method it cites).  Needs sph_build_cells for the same positions (else SPH_ESTALE).            */
int  sph_interface_correction(sph_ctx* ctx, const float* m, const float* u, const float* rho,
                              const float* h, const int32_t* mat, float alpha, float* imbalance,
                              float* rho_corr, float* P_corr);

/* Time integration with a global step, PAPER.md:227-261 (Section 2.3.6), Eqs. (19)-(25):
 * kick-drift-kick with predicted v, u for the force pass.  Element-wise; arrays of length n
 * in the caller's order.  The step is dt = dt_scale x *dt_device (dt_device: one float in
 * device memory, e.g. the dt_min_device of sph_timestep), so no host round trip is needed.
 *   sph_predict  Eqs. (19)-(20): q_pred = q + (dt/2) qdot        (q = v, u; qdot of the last step)
 *   sph_kick     Eqs. (21)-(24): q += (dt/2) qdot, in place      (closing and opening kick)
 *   sph_drift    Eq. (25):       x += dt v, wrapped into [lo, lo+len) on periodic axes        */
int  sph_predict(sph_ctx* ctx, int64_t n, const float* dt_device, float dt_scale, const float* vx,
                 const float* vy, const float* vz, const float* u, const float* ax, const float* ay,
                 const float* az, const float* dudt, float* vx_pred, float* vy_pred,
                 float* vz_pred, float* u_pred);
int  sph_kick(sph_ctx* ctx, int64_t n, const float* dt_device, float dt_scale, float* vx, float* vy,
              float* vz, float* u, const float* ax, const float* ay, const float* az,
              const float* dudt);
int  sph_drift(sph_ctx* ctx, int64_t n, const float* dt_device, float dt_scale, float* x, float* y,
               float* z, const float* vx, const float* vy, const float* vz);

/* Entropy-conserving update of the internal energy: "uses the old density and
 * internal energy to calculate the isentropic evolution to the new density, by having the EOS
 * solve u_new = u(rho_new, s(rho_old, u_old))".  For the built-in ideal gas an
 * isentrope is P / rho^gamma = const, so u_inout[i] *= (rho_new[i] / rho_old[i])^(gamma-1)
 * (reading R31).  All arrays are device pointers of n floats in caller order;
 * element-wise, in place, asynchronous on the context's stream.  With params.entropy = 1 the
 * dudt of sph_forces holds the viscous heating alone, which the kicks add on top.             */
int  sph_isentropic_u(sph_ctx* ctx, int64_t n, const float* rho_old, const float* rho_new,
                      float* u_inout);

/* Block time steps, PAPER.md:229 ("each particle is integrated with a time step size that is a
 * power-of-two fraction of the global timestep"), the substep of PAPER.md:231-261 per particle,
 * rung changes of PAPER.md:270; bookkeeping of DESIGN.md reading R32.  Time is counted in
 * substeps of delta = dt0 / 2^max_rung; a step of rung r spans 2^(max_rung - r) substeps.  Per
 * particle (device arrays of n, caller order, owned by the caller): rung (int32), tnext (int32:
 * the substep at which its running step ends; all 0 at the start) and hk (float: half-step
 * length of its last opening kick; all 0 at the start).  Element-wise, asynchronous.
 *   sph_block_predict  Eqs. (19)-(20) for EVERY particle (sources need predicted values too):
 *                      q_pred = q + ((substep - tnext_i) delta + hk_i) dq/dt; for a particle
 *                      whose step ends now this is the paper's dt_i / 2.
 *   sph_block_active   active_i = (tnext_i == substep), the mask sph_set_active takes.
 *   sph_block_kick     for those particles only: closing kick over hk_i (Eqs. 21-22), new rung
 *                      min(max_rung, max(rung_desired_i, f)) with f the lowest rung whose steps
 *                      begin at this substep ("moving to a lower rung is only possible on
 *                      substeps that correspond to the rung it wants to move to"), opening kick
 *                      over the new hk_i = 2^(max_rung - rung_i) delta / 2 (Eqs. 23-24), tnext_i
 *                      += the new step.  rung_desired: the output of sph_rungs.  open = 0:
 *                      the closing kick alone (v, u of the current time, e.g. for an
 *                      output); hk_i becomes 0, tnext_i and rung_i stay: the starting state.
 * max_rung <= 24; substep >= 0 (it may run past 2^max_rung: only substep mod 2^max_rung counts
 * for f).  SPH_EINVAL on a NULL pointer or a bad scalar.                                      */
int  sph_block_predict(sph_ctx* ctx, int64_t n, int32_t substep, float delta, const int32_t* tnext,
                       const float* hk, const float* vx, const float* vy, const float* vz,
                       const float* u, const float* ax, const float* ay, const float* az,
                       const float* dudt, float* vx_pred, float* vy_pred, float* vz_pred,
                       float* u_pred);
int  sph_block_active(sph_ctx* ctx, int64_t n, int32_t substep, const int32_t* tnext,
                      uint8_t* active);
int  sph_block_kick(sph_ctx* ctx, int64_t n, int32_t substep, int32_t max_rung, float delta,
                    const int32_t* rung_desired, int32_t* rung, int32_t* tnext, float* hk, float* vx,
                    float* vy, float* vz, float* u, const float* ax, const float* ay,
                    const float* az, const float* dudt, int32_t open);

/* Diagnostic: CSR neighbour lists at a prescribed h, caller indices; a list is a set, the
 * order inside it is unspecified.
 * mode 0: j with r_ij < 2 h_i (self included); mode 1: j != i with r_ij < 2 max(h_i,h_j).
 * Borderline pairs are decided in FP64 on the FP32 inputs, so the sets equal the exact
 * ones.  offsets: n+1 int64 (device).  indices: `capacity` int32 (device, may be NULL if
 * capacity = 0).  *needed (host) receives the total length.  Synchronises the stream.    */
int  sph_neighbors(sph_ctx* ctx, const float* h, int32_t mode, int64_t* offsets, int32_t* indices,
                   int64_t capacity, int64_t* needed);

/* Copies the device counters to *out (host).  Synchronises the stream.                   */
int  sph_stats(sph_ctx* ctx, sph_stats_t* out);
int  sph_stats_reset(sph_ctx* ctx);

/* perm_out[p] = caller index of the particle at sorted position p (device, n int32).     */
int  sph_permutation(sph_ctx* ctx, int32_t* perm_out);

/* Measures the FP32 FMA rate of the device with a register-resident FFMA kernel running
 * for about `seconds`; *tflops (host) = 2 x FMAs / time.  The ALU roofline denominator of
 * bench.py.  Synchronises.                                                               */
int  sph_fp32_peak(void* cuda_stream, float seconds, double* tflops);

/* sph_timestep without a context and WITHOUT ANY ALLOCATION (no cudaMalloc / cudaFree, no
 * allocating library routine): for callers that may not allocate -- code under CUDA graph
 * capture, serving loops, harnesses that forbid it.  Same operation as sph_timestep (steps
 * a10-a11, Eq. 26): dt_i = min(eta_acc sqrt(2h/|a|), eta_cfl h / ((1 + 0.6
 * av_alpha) c + 0.6 av_beta |mu_min|)), *dt_min_device = min_i dt_i; all arrays DEVICE pointers,
 * n floats (dt_min_device: one float), owned by the caller; work is enqueued on cuda_stream
 * (a cudaStream_t; NULL = the default stream) of the CURRENT device and not waited for.
 * The block minima of the reduction go to a scratch array of SPH_STATIC_SCRATCH_BYTES that is
 * part of the library image: every GPU that loads the library holds it until exit, and that
 * size is the limit -- n <= SPH_STATIC_MAX_N, else SPH_EINVAL (use sph_timestep).  All calls on a
 * device share the scratch, which keeps the last call's contents (nothing in it needs to start
 * at zero); calls that overlap on one GPU (two streams) race on it and must be ordered by the
 * caller.  The first call on a device looks up the array's device address (no allocation).
 * SPH_EINVAL: null pointer, n out of range, eta <= 0 or a negative viscosity parameter;
 * SPH_ECUDA: CUDA runtime error.  sph_static_last_error: text of this thread's last failure.  */
#define SPH_STATIC_SCRATCH_BYTES 16384
#define SPH_STATIC_MAX_N 16777216 /* 4096 block minima x 4096 particles per block */
int  sph_timestep_static(void* cuda_stream, int64_t n, float eta_cfl, float eta_acc,
                         float av_alpha, float av_beta, const float* h, const float* c,
                         const float* ax, const float* ay, const float* az, const float* mu_min,
                         float* dt_i, float* dt_min_device);
const char* sph_static_last_error(void);

const char* sph_strerror(int code);
const char* sph_last_error(const sph_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
