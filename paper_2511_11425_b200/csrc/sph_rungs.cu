// sph_rungs.cu -- time-step rungs: Eq. (27) and the limiter of Saitoh &
// Makino (2009), r_i >= r_j - 2 for every particle j that i interacts with (the force pair set
// 0 < r_ij < 2 max(h_i, h_j)), one pass over the rungs of Eq. (27) (reading R28).
// The neighbour walk is the force sweep's: the kept list where it covers the scatter reach,
// the cell rows otherwise.  Rungs are integers, so pairs inside the FP32-uncertain band of the
// support edge are decided in FP64.
//
// The same walk is the FastGas marking pass: mark every particle that is on
// the interaction list of a particle of the source set (the set itself included; DESIGN.md
// reading R29).  Only the particles of the source set walk -- the pair set is symmetric -- and
// store a 1 for each partner, so the cost follows the size of the set.
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int R_G = SPH_G, R_NT = 32 / R_G, R_WARPS = 4, R_TPB = R_WARPS * 32, R_QUADS = 16;
constexpr int R_TARGETS = R_NT * R_QUADS;

// Eq. (27): the smallest r >= 0 with 2^-r dt0 <= dt_i (halving is exact), capped at max_rung;
// written in sorted order for the limiter's gathers
__global__ void k_rung_eq27(int64_t n, const int32_t* __restrict__ inv_perm,
                            const float* __restrict__ dt_i, float dt0, int max_rung,
                            int32_t* rung_sorted) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float d = dt_i[i];
    int   r = 0;
    float t = dt0;
    while (r < max_rung && t > d) { t *= 0.5f; ++r; }
    rung_sorted[inv_perm[i]] = r;
}

// marks start as the source set itself
__global__ void k_mark_init(int64_t n, const uint8_t* __restrict__ src, uint8_t* mark) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) mark[i] = src[i] ? 1 : 0;
}

// MODE 0: rung limiter over all particles, out_i = max(r_i, max_j r_j - 2) as int32.
// MODE 1: marking pass; the targets are the tcnt sorted positions in tlist (the source set),
//         out[j] = 1 (uint8, caller order) for every partner j of a target.
template <int MODE>
__global__ __launch_bounds__(R_TPB, SPH_MINB) void k_rung_limiter(
    int n, const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ pos_h, const int32_t* __restrict__ rung_sorted,
    const int32_t* __restrict__ perm, const unsigned* __restrict__ coarse,
    const uint32_t* __restrict__ nb_j, const uint32_t* __restrict__ nb_cnt,
    const float* __restrict__ nb_rkeep, const uint32_t* __restrict__ tlist,
    const unsigned* __restrict__ tcnt, void* out) {
    const int nt = (MODE == 1) ? (int)*tcnt : n;
    if (blockIdx.x * R_TARGETS >= nt) return;
    __shared__ SphGrid g;
    __shared__ int     next_quad;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x == 0) next_quad = 0;
    __syncthreads();
    const int   lane = threadIdx.x & 31, gq = lane / R_G, sl = lane & (R_G - 1);
    // pos_h.w holds the h of the build (<= g.hmax) or, after sph_forces, the solved h
    const float hmax_all = fmaxf(g.hmax, __uint_as_float(g.force_hmax_bits));
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;
    unsigned tested = 0;

    for (;;) {
        int quad = 0;
        if (lane == 0) quad = atomicAdd(&next_quad, 1);
        quad = __shfl_sync(SPH_FULL, quad, 0);
        if (quad >= R_QUADS) break;
        const int  idx    = (blockIdx.x * R_QUADS + quad) * R_NT + gq;
        const bool tvalid = idx < nt;
        const int  p      = (MODE == 1 && tvalid) ? (int)tlist[idx] : idx;
        const float4 pi = tvalid ? pos_h[p] : make_float4(0.f, 0.f, 0.f, 1.f);
        const float  hi = pi.w;
        int best = (MODE == 0 && tvalid) ? rung_sorted[p] : 0;
        const float Hs  = sph_scatter_hmax<R_G>(g, coarse, pi.x, pi.y, pi.z, hi, hmax_all, lane);
        const float tau = 1e-6f + 2.5e-7f * g.xext / hi;
        const float R   = 2.0f * Hs * (1.0f + 4.0f * tau) * (1.0f + 1e-5f);
        const bool  covered = tvalid && (R * (1.0f + 4.0f * tau) <= nb_rkeep[tvalid ? p : 0]);

        auto pair = [&](uint32_t j, const float4 pj, float r2) {
            if (j == (uint32_t)p || !(r2 > 0.0f)) return;
            const float hm = fmaxf(hi, pj.w), H2 = 4.0f * hm * hm;
            bool in = r2 < H2;
            if (fabsf(r2 - H2) <= 2.0f * (1e-6f + 2.5e-7f * g.xext / hm) * H2)
                in = sph_r2_exact(g, pi.x, pi.y, pi.z, pj.x, pj.y, pj.z) <
                     4.0 * (double)hm * (double)hm;
            if (in) {
                if (MODE == 0) best = max(best, __ldg(rung_sorted + j) - 2);
                else           ((uint8_t*)out)[perm[j]] = 1;
            }
        };
        if (covered) {
            const uint32_t* src = nb_j + ((size_t)p * (SPH_SLOTS * R_G) + sl);
            const int mycnt = ((int)nb_cnt[p] - sl + R_G - 1) >> 3;
            for (int k = 0; k < mycnt; ++k) {
                const uint32_t j  = src[k * R_G];
                const float4   pj = __ldg(pos_h + j);
                float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
                dx -= Lx * rintf(dx * iLx);
                dy -= Ly * rintf(dy * iLy);
                dz -= Lz * rintf(dz * iLz);
                pair(j, pj, dx * dx + dy * dy + dz * dz);
            }
        }
        const bool search = tvalid && !covered;
        if (__any_sync(SPH_FULL, search)) {
            int dummy = 0;
            const float R2 = R * R;
            sph_group_collect<R_G>(g, cell_start, pos_h, pi.x, pi.y, pi.z, R, search, lane, tested,
                                   dummy, [&](const float4, float r2) { return r2 < R2; },
                                   [&](int, uint32_t j, const float4 pj, float, float, float,
                                       float r2) { pair(j, pj, r2); });
        }
#pragma unroll
        for (int o = R_G / 2; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(SPH_FULL, best, o));
        if (MODE == 0 && tvalid && sl == 0) ((int32_t*)out)[perm[p]] = best;
        __syncwarp();
    }
}

}  // namespace

int sph_launch_rungs(sph_ctx* c, const float* dt_i, float dt0, int32_t max_rung, int32_t* rung) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    int32_t* rs = (int32_t*)c->key;   // build-time scratch, free once the index exists
    k_rung_eq27<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->inv_perm, dt_i, dt0, max_rung, rs);
    const int nblk = (int)((n + R_TARGETS - 1) / R_TARGETS);
    k_rung_limiter<0><<<nblk, R_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_h, rs, c->perm,
                                             c->coarse_hmax, c->nb_j, c->nb_cnt, c->nb_rkeep, nullptr,
                                             nullptr, rung);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_mark(sph_ctx* c, const uint8_t* src, uint8_t* mark) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    uint32_t* list = (uint32_t*)c->fix_list;   // the sweeps' queue, free between their calls
    int rc = sph_launch_coarse_map(c);         // of the h now in pos_h.w
    if (rc != SPH_OK) return rc;
    rc = sph_launch_compact(c, src, list, c->act_cnt + 1);
    if (rc != SPH_OK) return rc;
    k_mark_init<<<(int)((n + 255) / 256), 256, 0, s>>>(n, src, mark);
    const int nblk = (int)((n + R_TARGETS - 1) / R_TARGETS);
    k_rung_limiter<1><<<nblk, R_TPB, 0, s>>>((int)n, c->grid, c->cell_start, c->pos_h, nullptr,
                                             c->perm, c->coarse_hmax, c->nb_j, c->nb_cnt,
                                             c->nb_rkeep, list, c->act_cnt + 1, mark);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}
