// sph_interface.cu -- interface correction for the ideal gas, PAPER.md:158-182 (Section 2.3.4),
// Eqs. (8)-(12): the kernel imbalance I_i (pass 1) and the imbalance-weighted kernel averages of
// pressure and temperature that replace P_i, T_i where I_i is large (pass 2); the corrected
// density follows from the EOS.  Both passes are gather sums over r_ij < 2 h_i.
//
// Same machinery as the force sweep: 8 lanes per target; where the neighbour list kept by the
// density sweep covers the support it is read in place, otherwise the group walks the cell
// rows and accumulates as it goes.  Ideal gas: T = u / c_v, so u stands in for T and
// Eq. (12) reads rho~ = P~ / ((gamma - 1) u~)  (readings R24-R27).
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int I_G     = SPH_G;
constexpr int I_NT    = 32 / I_G;
constexpr int I_WARPS = 4;
constexpr int I_TPB   = I_WARPS * 32;
constexpr int I_QUADS = 16;
constexpr int I_TARGETS = I_NT * I_QUADS;

// sorted records: ica = (x, y, z, m), icb = (P, u, h, material bits)
__global__ void k_ic_prep(int64_t n, const int32_t* __restrict__ inv_perm,
                          const float4* __restrict__ pos_h, const float* __restrict__ m,
                          const float* __restrict__ u, const float* __restrict__ rho,
                          const float* __restrict__ h, const int32_t* __restrict__ mat, float gamma,
                          float4* ica, float4* icb) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int    p = inv_perm[i];
    const float4 a = pos_h[p];
    ica[p] = make_float4(a.x, a.y, a.z, m[i]);
    icb[p] = make_float4((gamma - 1.0f) * rho[i] * u[i], u[i], h[i],
                         __int_as_float(mat ? mat[i] : 0));
}

// PASS 1: Eq. (8) -> imbalance (caller order) and e^{-I^2} (sorted order)
// PASS 2: Eqs. (9)-(12) -> rho_corr, P_corr (caller order)
template <int KERN, int PASS>
__global__ __launch_bounds__(I_TPB, SPH_MINB) void k_interface(
    int n, const SphGrid* __restrict__ gp, const uint32_t* __restrict__ cell_start,
    const float4* __restrict__ ica, const float4* __restrict__ icb, const float* expI,
    const int32_t* __restrict__ perm, const uint32_t* __restrict__ nb_j,
    const uint32_t* __restrict__ nb_cnt, const float* __restrict__ nb_rkeep, float alpha,
    float gamma, float* imbalance, float* expI_out, float* rho_corr, float* P_corr) {
    __shared__ SphGrid g;
    __shared__ int     next_quad;
    if (threadIdx.x < sizeof(SphGrid) / 4)
        ((int*)&g)[threadIdx.x] = ((const int*)gp)[threadIdx.x];
    if (threadIdx.x == 0) next_quad = 0;
    __syncthreads();
    const int   lane = threadIdx.x & 31, gq = lane / I_G, sl = lane & (I_G - 1);
    const float iLx = g.per[0] ? 1.0f / g.len[0] : 0.0f, Lx = g.per[0] ? g.len[0] : 0.0f;
    const float iLy = g.per[1] ? 1.0f / g.len[1] : 0.0f, Ly = g.per[1] ? g.len[1] : 0.0f;
    const float iLz = g.per[2] ? 1.0f / g.len[2] : 0.0f, Lz = g.per[2] ? g.len[2] : 0.0f;
    unsigned tested = 0;

    for (;;) {
        int quad = 0;
        if (lane == 0) quad = atomicAdd(&next_quad, 1);
        quad = __shfl_sync(SPH_FULL, quad, 0);
        if (quad >= I_QUADS) break;
        const int  p      = (blockIdx.x * I_QUADS + quad) * I_NT + gq;
        const bool tvalid = p < n;
        float4 ai = make_float4(0.f, 0.f, 0.f, 1.f), bi = make_float4(1.f, 1.f, 1.f, 0.f);
        if (tvalid) {
            ai = ica[p];
            bi = icb[p];
        }
        const float hi = bi.z, ih = __fdividef(1.0f, hi), H2 = 4.0f * hi * hi;
        const int   mat_i = __float_as_int(bi.w);
        const float R   = 2.0f * hi * (1.0f + 1e-5f);
        const float tau = 1e-6f + 2.5e-7f * g.xext * ih;
        const bool  covered = tvalid && (R * (1.0f + 4.0f * tau) <= nb_rkeep[tvalid ? p : 0]);
        float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;   // pass 1: sum kappa d m w (3), sum m w
                                                            // pass 2: sum u e w, sum P e w, sum e w
        auto pair = [&](uint32_t j, const float4 aj, float dx, float dy, float dz, float r2) {
            const float w = SphKernel<KERN>::w(r2 * rsqrtf(fmaxf(r2, 1e-35f)) * ih);
            if (PASS == 1) {
                const int   mat_j = __float_as_int(__ldg(&icb[j].w));
                const float mw = aj.w * w, k = (mat_j != mat_i) ? mw : -mw;   // kappa (r_j - r_i) = -kappa d
                s0 += k * dx; s1 += k * dy; s2 += k * dz;
                s3 += mw;
            } else {
                const float4 bj = __ldg(icb + j);
                const float  ew = __ldg(expI + j) * w;
                s0 += bj.y * ew; s1 += bj.x * ew; s2 += ew;
            }
        };
        if (covered) {
            const uint32_t* src = nb_j + ((size_t)p * (SPH_SLOTS * I_G) + sl);
            const int mycnt = ((int)nb_cnt[p] - sl + I_G - 1) >> 3;
            for (int k = 0; k < mycnt; ++k) {
                const uint32_t j  = src[k * I_G];
                const float4   aj = __ldg(ica + j);
                float dx = ai.x - aj.x, dy = ai.y - aj.y, dz = ai.z - aj.z;
                dx -= Lx * rintf(dx * iLx);
                dy -= Ly * rintf(dy * iLy);
                dz -= Lz * rintf(dz * iLz);
                const float r2 = dx * dx + dy * dy + dz * dz;
                if (r2 < H2) pair(j, aj, dx, dy, dz, r2);
            }
        }
        const bool search = tvalid && !covered;
        if (__any_sync(SPH_FULL, search)) {
            int dummy = 0;
            sph_group_collect<I_G>(g, cell_start, ica, ai.x, ai.y, ai.z, R, search, lane, tested,
                                   dummy, [&](const float4, float r2) { return r2 < H2; },
                                   [&](int, uint32_t j, const float4 aj, float dx, float dy, float dz,
                                       float r2) { pair(j, aj, dx, dy, dz, r2); });
        }
        s0 = sph_group_sum<I_G>(s0);
        s1 = sph_group_sum<I_G>(s1);
        s2 = sph_group_sum<I_G>(s2);
        s3 = sph_group_sum<I_G>(s3);
        if (tvalid && sl == 0) {
            const int i = perm[p];
            if (PASS == 1) {
                const float I = alpha * sqrtf(s0 * s0 + s1 * s1 + s2 * s2) / (hi * s3);   // Eq. (8)
                imbalance[i] = I;
                expI_out[p]  = expf(-I * I);
            } else {
                const float e  = expI[p];
                const float Pt = e * bi.x + (1.0f - e) * (s1 / s2);    // Eq. (10)
                const float ut = e * bi.y + (1.0f - e) * (s0 / s2);    // Eq. (11), T = u / c_v
                rho_corr[i] = Pt / ((gamma - 1.0f) * ut);              // Eq. (12), ideal gas
                if (P_corr) P_corr[i] = Pt;
            }
        }
        __syncwarp();
    }
}

}  // namespace

int sph_launch_interface(sph_ctx* c, const float* m, const float* u, const float* rho, const float* h,
                         const int32_t* mat, float alpha, float* imbalance, float* rho_corr,
                         float* P_corr) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    float4* ica  = c->vel_m;          // scratch shared with the force sweep (rebuilt by its prep)
    float4* icb  = c->rcak;
    float*  expI = (float*)c->rank;   // build-time scratch, free once the index exists
    k_ic_prep<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->inv_perm, c->pos_h, m, u, rho, h, mat,
                                                     c->par.gamma, ica, icb);
    const int nblk = (int)((n + I_TARGETS - 1) / I_TARGETS);
    auto launch = [&](auto tag) {
        constexpr int KERN = decltype(tag)::value;
        k_interface<KERN, 1><<<nblk, I_TPB, 0, s>>>((int)n, c->grid, c->cell_start, ica, icb, expI,
                                                    c->perm, c->nb_j, c->nb_cnt, c->nb_rkeep, alpha,
                                                    c->par.gamma, imbalance, expI, rho_corr, P_corr);
        k_interface<KERN, 2><<<nblk, I_TPB, 0, s>>>((int)n, c->grid, c->cell_start, ica, icb, expI,
                                                    c->perm, c->nb_j, c->nb_cnt, c->nb_rkeep, alpha,
                                                    c->par.gamma, imbalance, expI, rho_corr, P_corr);
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
