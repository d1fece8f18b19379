"""Seeded synthetic workloads shaped like the paper's tests.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: it only lays particles out and assigns initial fields.  The paper's own
initial conditions (BCC lattices relaxed for Wendland C6 / 400 neighbours, `ballic` planet
models, ANEOS tables -- PAPER.md:282, 297, 424) are not available; these stand in for them:

  C1 uniform   PAPER.md:297 (lattice ICs)         16^3 jittered cubic lattice, random v
  C2 sod       PAPER.md:307-309 (Section 3.2)     1 x 1/8 x 1/8 tube, 8:1 density jump
  C3 sedov     PAPER.md:311-325 (Section 3.3)     128^3 lattice, energy 1 at the centre
  C4 kh        PAPER.md:381-388 (Section 3.8)     shear layer, ~2:1 density, Eq. (31) seed
  C5 impact    PAPER.md:424, 462-467              two n=1 polytropes, free surfaces

All arrays are FP32 (BASELINE.json configs).  Seeds: 114250 + config number.
"""
from __future__ import annotations

import numpy as np

H_OVER_DELTA = 1.2347      # h / (m/rho)^(1/3) that holds ~64 m in the 2h ball on a cubic lattice


def _lattice(nx, ny, nz, dx, origin=(0.0, 0.0, 0.0)):
    i, j, k = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    x = origin[0] + (i.ravel() + 0.5) * dx
    y = origin[1] + (j.ravel() + 0.5) * dx
    z = origin[2] + (k.ravel() + 0.5) * dx
    return x, y, z


def _finish(w, rng, rho_nominal, h_start):
    """Cast to FP32 and attach the starting guess for h ('warm' = +-2 %, 'cold' = 0.8..1.25)."""
    n = len(w["x"])
    m = np.broadcast_to(np.asarray(w["m"], np.float64), (n,))
    h0 = H_OVER_DELTA * np.cbrt(m / rho_nominal)
    if h_start == "warm":
        h0 = h0 * rng.uniform(0.98, 1.02, n)
    elif h_start == "cold":
        h0 = h0 * rng.uniform(0.8, 1.25, n)
    elif h_start != "exact":
        raise ValueError(h_start)
    w["h"] = h0
    for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h"):
        w[k] = np.ascontiguousarray(np.broadcast_to(np.asarray(w[k], np.float64), (n,)), np.float32)
    # wrap after the cast so that FP32 positions stay inside [lo, lo+len)
    for d, k in enumerate(("x", "y", "z")):
        if w["periodic"][d]:
            L = np.float32(w["box_len"][d])
            a = w[k]
            a[a >= L] -= L
            a[a < 0] += L
            a[a >= L] = np.float32(0.0)
    w["n"] = n
    return w


def uniform_cube(nside=16, jitter=0.05, seed=114251, h_start="cold", v_sigma=0.01):
    """C1: unit periodic cube, rho = 1, u = 1, gamma = 5/3, alpha = 1, beta = 2."""
    rng = np.random.default_rng(seed)
    dx = 1.0 / nside
    x, y, z = _lattice(nside, nside, nside, dx)
    n = len(x)
    x = x + rng.uniform(-jitter, jitter, n) * dx
    y = y + rng.uniform(-jitter, jitter, n) * dx
    z = z + rng.uniform(-jitter, jitter, n) * dx
    w = dict(name="uniform_cube", x=x % 1.0, y=y % 1.0, z=z % 1.0, m=1.0 / n,
             vx=rng.normal(0, v_sigma, n), vy=rng.normal(0, v_sigma, n),
             vz=rng.normal(0, v_sigma, n), u=1.0,
             box_lo=(0.0, 0.0, 0.0), box_len=(1.0, 1.0, 1.0), periodic=(1, 1, 1),
             gamma=5.0 / 3.0, av_alpha=1.0, av_beta=2.0)
    return _finish(w, rng, 1.0, h_start)


def sod_tube(ncross=38, seed=114252, h_start="warm", jitter=0.0):
    """C2: periodic 1 x 1/8 x 1/8 box; left half rho=1,P=1; right half rho=1/8,P=0.1; gamma=1.4.
    jitter > 0 (in units of the local spacing) breaks the symmetry of the perfect lattice, which
    otherwise cannot rearrange when the flow stretches it along x only (evolution tests)."""
    rng = np.random.default_rng(seed)
    dl = 0.125 / ncross
    dr = 2.0 * dl
    xl, yl, zl = _lattice(4 * ncross, ncross, ncross, dl)
    xr, yr, zr = _lattice(2 * ncross, ncross // 2, ncross // 2, dr, origin=(0.5, 0.0, 0.0))
    x = np.concatenate([xl, xr]); y = np.concatenate([yl, yr]); z = np.concatenate([zl, zr])
    m = dl ** 3
    left = np.arange(len(x)) < len(xl)
    if jitter > 0:
        sp = np.where(left, dl, dr)
        x = (x + rng.uniform(-jitter, jitter, len(x)) * sp) % 1.0
        y = (y + rng.uniform(-jitter, jitter, len(x)) * sp) % 0.125
        z = (z + rng.uniform(-jitter, jitter, len(x)) * sp) % 0.125
    rho = np.where(left, 1.0, 0.125)
    P = np.where(left, 1.0, 0.1)
    gamma = 1.4
    w = dict(name="sod_tube", x=x, y=y, z=z, m=m, vx=0.0, vy=0.0, vz=0.0,
             u=P / ((gamma - 1.0) * rho),
             box_lo=(0.0, 0.0, 0.0), box_len=(1.0, 0.125, 0.125), periodic=(1, 1, 1),
             gamma=gamma, av_alpha=1.5, av_beta=3.0)
    return _finish(w, rng, rho, h_start)


def sedov(nside=128, jitter=0.01, seed=114253, h_start="warm", v_sigma=0.0):
    """C3: unit periodic cube, rho=1, u_bg=1e-5, E=1 spread smoothly over the particles within
    2.5 lattice spacings of the centre (PAPER.md:311 uses a top-hat of radius 0.02).
    v_sigma > 0 gives the throughput variant C3v with random velocities."""
    rng = np.random.default_rng(seed)
    dx = 1.0 / nside
    x, y, z = _lattice(nside, nside, nside, dx)
    n = len(x)
    x = (x + rng.uniform(-jitter, jitter, n) * dx) % 1.0
    y = (y + rng.uniform(-jitter, jitter, n) * dx) % 1.0
    z = (z + rng.uniform(-jitter, jitter, n) * dx) % 1.0
    m = 1.0 / n
    # initial-condition profile of the deposited energy: a smooth bump (1 - s^2)^2 of radius
    # 2.5 lattice spacings -- a recipe of this generator, not a formula of the method
    R = 2.5 * dx
    s2 = ((x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2) / R ** 2
    bump = np.where(s2 < 1.0, (1.0 - s2) ** 2, 0.0)
    u = 1e-5 + 1.0 * bump / (m * bump.sum())
    vel = (lambda: rng.normal(0, v_sigma, n)) if v_sigma > 0 else (lambda: 0.0)
    w = dict(name="sedov" if v_sigma == 0 else "sedov_v", x=x, y=y, z=z, m=m,
             vx=vel(), vy=vel(), vz=vel(), u=u,
             box_lo=(0.0, 0.0, 0.0), box_len=(1.0, 1.0, 1.0), periodic=(1, 1, 1),
             gamma=5.0 / 3.0, av_alpha=1.0, av_beta=2.0)
    return _finish(w, rng, 1.0, h_start)


def kelvin_helmholtz(nout=280, nin=352, jitter=0.01, seed=114254, h_start="warm"):
    """C4: periodic 1 x 1 x 1/8 box; slab |y-1/2|<1/4 with spacing 1/nin and vx=+0.5, outside
    spacing 1/nout and vx=-0.5; equal masses => rho_in = (nin/nout)^3; P=2.5; gamma=5/3."""
    rng = np.random.default_rng(seed)
    do, di = 1.0 / nout, 1.0 / nin
    xo, yo, zo = _lattice(nout, nout // 2, nout // 8, do)
    yo = np.where(yo < 0.25, yo, yo + 0.5)            # two outer quarter-slabs
    xi, yi, zi = _lattice(nin, nin // 2, nin // 8, di, origin=(0.0, 0.25, 0.0))
    no = len(xo)
    x = np.concatenate([xo, xi]); y = np.concatenate([yo, yi]); z = np.concatenate([zo, zi])
    n = len(x)
    sp = np.where(np.arange(n) < no, do, di)
    x = (x + rng.uniform(-jitter, jitter, n) * sp) % 1.0
    y = (y + rng.uniform(-jitter, jitter, n) * sp) % 1.0
    z = (z + rng.uniform(-jitter, jitter, n) * sp) % 0.125
    m = do ** 3
    inner = np.arange(n) >= no
    rho = np.where(inner, (nin / nout) ** 3, 1.0)
    gamma = 5.0 / 3.0
    lam = 0.5
    vy = 0.025 * (np.sin(2 * np.pi * (x + lam / 2) / lam) * np.exp(-(10 * (y - 0.25)) ** 2)
                  + np.sin(2 * np.pi * x / lam) * np.exp(-(10 * (y - 0.75)) ** 2))
    w = dict(name="kelvin_helmholtz", x=x, y=y, z=z, m=m, vx=np.where(inner, 0.5, -0.5), vy=vy,
             vz=0.0, u=2.5 / ((gamma - 1.0) * rho),
             box_lo=(0.0, 0.0, 0.0), box_len=(1.0, 1.0, 0.125), periodic=(1, 1, 1),
             gamma=gamma, av_alpha=1.0, av_beta=2.0)
    return _finish(w, rng, rho, h_start)


def _polytrope(n_target, R, rho_c, rng, jitter):
    """Equal-mass particles following rho = rho_c sin(xi)/xi, xi = pi r/R: a jittered cubic
    lattice in the unit ball whose radii are remapped so the enclosed-mass fraction matches
    (sin xi - xi cos xi)/pi (the radial-stretch idea of PAPER.md:341)."""
    nside = int(np.ceil(np.cbrt(n_target * 6.0 / np.pi)))
    d = 2.0 / nside
    x, y, z = _lattice(nside, nside, nside, d, origin=(-1.0, -1.0, -1.0))
    k = len(x)
    x = x + rng.uniform(-jitter, jitter, k) * d
    y = y + rng.uniform(-jitter, jitter, k) * d
    z = z + rng.uniform(-jitter, jitter, k) * d
    s = np.sqrt(x * x + y * y + z * z)
    keep = (s < 1.0) & (s > 0)
    x, y, z, s = x[keep], y[keep], z[keep], s[keep]
    xi_tab = np.linspace(0.0, np.pi, 20001)
    frac_tab = (np.sin(xi_tab) - xi_tab * np.cos(xi_tab)) / np.pi
    xi = np.interp(s ** 3, frac_tab, xi_tab)
    dens = rho_c * np.where(xi > 0, np.sin(xi) / np.maximum(xi, 1e-30), 1.0)
    ok = dens / rho_c >= 1e-3
    scale = (xi * R / np.pi) / s
    M = 4.0 * rho_c * R ** 3 / np.pi
    m = M / len(s)                                   # mass per lattice point before truncation
    return x[ok] * scale[ok], y[ok] * scale[ok], z[ok] * scale[ok], dens[ok], m


def impact(n_target=12_000_000, n_impactor=1_500_000, jitter=0.05, seed=114255, h_start="warm"):
    """C5: two n=1 polytropes (gamma=2, u = K rho, K = 2 R^2/pi with G=1) in vacuum; impactor
    arriving at 45 degrees with 1.5 x the mutual escape speed; non-periodic box."""
    rng = np.random.default_rng(seed)
    rho_c = np.pi / 4.0
    Rt, Ri = 1.0, 0.5
    xt, yt, zt, dt_, mt = _polytrope(n_target, Rt, rho_c, rng, jitter)
    xq, yq, zq, dq, mq = _polytrope(n_impactor, Ri, rho_c, rng, jitter)
    Mt, Mi = 4.0 * rho_c * Rt ** 3 / np.pi, 4.0 * rho_c * Ri ** 3 / np.pi
    sep = Rt + Ri
    c45 = np.sqrt(0.5)
    off = np.array([sep * c45, sep * c45, 0.0])
    vesc = np.sqrt(2.0 * (Mt + Mi) / sep)
    vrel = 1.5 * vesc
    v_t = +vrel * Mi / (Mt + Mi)
    v_i = -vrel * Mt / (Mt + Mi)
    x = np.concatenate([xt, xq + off[0]]); y = np.concatenate([yt, yq + off[1]])
    z = np.concatenate([zt, zq + off[2]])
    nt = len(xt)
    n = len(x)
    isT = np.arange(n) < nt
    rho = np.concatenate([dt_, dq])
    K = np.where(isT, 2.0 * Rt ** 2 / np.pi, 2.0 * Ri ** 2 / np.pi)
    lo = np.array([x.min(), y.min(), z.min()]) - 0.05
    hi = np.array([x.max(), y.max(), z.max()]) + 0.05
    w = dict(name="impact", x=x, y=y, z=z, m=np.where(isT, mt, mq), vx=np.where(isT, v_t, v_i),
             vy=0.0, vz=0.0, u=K * rho,
             box_lo=tuple(float(np.float32(v)) for v in lo),
             box_len=tuple(float(np.float32(v)) for v in (hi - lo)), periodic=(0, 0, 0),
             gamma=2.0, av_alpha=1.5, av_beta=3.0)
    return _finish(w, rng, rho, h_start)


CONFIGS = {
    "uniform_cube": uniform_cube,
    "sod_tube": sod_tube,
    "sedov": sedov,
    "kelvin_helmholtz": kelvin_helmholtz,
    "impact": impact,
}


def make(name: str, **kw):
    return CONFIGS[name](**kw)
