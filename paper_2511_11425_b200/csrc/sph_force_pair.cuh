// sph_force_pair.cuh -- the pair arithmetic of the hydro force pass
// (Section 2.3.5), Eqs. (13)-(18), shared by the force kernels (sph_forces.cu: 8 lanes per
// target; sph_tile_forces.cu: staged tiles).  Shares nothing with oracle/.
//
// d = x_i - x_j, r = |d|, q_a = r/h_a, g_a = K_a g(q_a), g = -w'(q)/q, K_a = sigma / h_a^5, so
// that dW/dr(r,h_a) = -g_a r:
//   Eq. 13+17:  a_i     = + sum_j m_j (A_i g_i + A_j g_j + Pi_ij gbar) d
//   Eq. 14+18:  du_i/dt = - sum_j m_j (A_i g_i + Pi_ij gbar / 2) (v_ij . d)
//   Eq. 15-16:  mu = hbar (v_ij.d)/(r^2 + eps hbar^2), Pi = mu (beta mu - alpha cbar)/rhobar
//               for v_ij.d < 0, else 0;   gbar = (g_i + g_j)/2;  A = P/(Omega rho^2).
#pragma once
#include "sph_internal.cuh"

#ifdef __CUDACC__
struct ForcePar {
    float alpha, beta, eps;
};


// Per-target constants and accumulators of the pair sum.
struct Target {
    float4 pi, vi;                       // (x, y, z, h), (vx, vy, vz, m)
    float  rho, c, A, K, ih;
};
struct Accum {
    float    ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, mumin = 0.f;
    unsigned pairs = 0, av = 0;
};

// One pair of Eqs. (13)-(18): source j at displacement d = x_i - x_j (minimum image).
// ENT: the entropy-conserving variant drops the Eq. (14) term of du/dt.
template <int KERN, bool ENT>
__device__ __forceinline__ void force_pair(const Target& t, Accum& a, const ForcePar& par,
                                           const float4 vj, const float4 rj, float dx,
                                           float dy, float dz, float r2, float hj) {
    const float r  = sph_sqrt(r2);
    const float gi = t.K * SphKernel<KERN>::g_s(r * t.ih);   // K carries gscale
    const float gj = rj.w * SphKernel<KERN>::g_s(__fdividef(r, hj));
    const float vdx = t.vi.x - vj.x, vdy = t.vi.y - vj.y, vdz = t.vi.z - vj.z;
    const float vr = vdx * dx + vdy * dy + vdz * dz;   // v_ij . r_ij
    float pig = 0.0f;                                   // Pi_ij * gbar
    if (vr < 0.0f) {
        const float hb  = 0.5f * (t.pi.w + hj);
        const float mu  = __fdividef(hb * vr, r2 + par.eps * hb * hb);
        const float cb  = 0.5f * (t.c + rj.y);
        const float rb  = 0.5f * (t.rho + rj.x);
        const float Pij = __fdividef(mu * (par.beta * mu - par.alpha * cb), rb);
        pig     = Pij * 0.5f * (gi + gj);
        a.mumin = fminf(a.mumin, mu);
        ++a.av;
    }
    const float Ag = t.A * gi;
    const float ca = vj.w * (Ag + rj.z * gj + pig);
    a.ax += ca * dx;
    a.ay += ca * dy;
    a.az += ca * dz;
    a.du -= vj.w * (ENT ? 0.5f * pig : Ag + 0.5f * pig) * vr;   // Eq. (18) [+ Eq. (14)]
    ++a.pairs;
}

// The same pair without a branch: everything is evaluated, `ok` (the pair test) selects what
// is added.  Eq. (15)'s case distinction becomes mu^- = min(mu, 0): for a receding pair
// mu^- = 0 and Pi_ij = 0 exactly, for an approaching one mu^- = mu.  Straight-line code lets
// the compiler interleave the dependency chains of several pairs (the staged-tile sweep
// evaluates four per trip); a source whose records are not meaningful (ok = false: a cursor
// bubble, the self pair) may produce anything, the selects drop it.
// v_ij . r_ij of a pair (the sign decides Eq. 15)
__device__ __forceinline__ float force_pair_vr(const Target& t, const float4 vj, float dx, float dy, float dz) {
    return (t.vi.x - vj.x) * dx + (t.vi.y - vj.y) * dy + (t.vi.z - vj.z) * dz;
}
// AV = false: the caller knows that no pair it evaluates together is approaching (a warp-uniform
// decision); the viscous terms are then exactly zero and are left out.
template <int KERN, bool ENT, bool AV = true>
__device__ __forceinline__ void force_pair_nb(const Target& t, Accum& a, const ForcePar& par, bool ok,
                                              const float4 vj, const float4 rj, float dx, float dy,
                                              float dz, float r2, float hj) {
    const float r  = sph_sqrt(r2);
    const float gi = t.K * SphKernel<KERN>::g_s(r * t.ih);   // K carries gscale
    const float gj = rj.w * SphKernel<KERN>::g_s(__fdividef(r, hj));
    const float vr = force_pair_vr(t, vj, dx, dy, dz);   // v_ij . r_ij
    float mu = 0.0f, pig = 0.0f;
    if (AV) {
        const float hb  = 0.5f * (t.pi.w + hj);
        mu = fminf(__fdividef(hb * vr, r2 + par.eps * hb * hb), 0.0f);
        const float cb  = 0.5f * (t.c + rj.y);
        const float rb  = 0.5f * (t.rho + rj.x);
        const float Pij = __fdividef(mu * (par.beta * mu - par.alpha * cb), rb);
        pig = Pij * 0.5f * (gi + gj);           // Pi_ij * gbar
    }
    const float Ag  = t.A * gi;
    const float ca  = ok ? vj.w * (Ag + rj.z * gj + pig) : 0.0f;
    const float du  = ok ? vj.w * (ENT ? 0.5f * pig : Ag + 0.5f * pig) * vr : 0.0f;   // Eq. (18) [+ Eq. (14)]
    a.ax += ca * dx;
    a.ay += ca * dy;
    a.az += ca * dz;
    a.du -= du;
    a.mumin = fminf(a.mumin, ok ? mu : 0.0f);
    a.pairs += ok ? 1u : 0u;
    a.av    += (ok && vr < 0.0f) ? 1u : 0u;
}

#endif  // __CUDACC__
