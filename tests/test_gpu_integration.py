"""GPU tests of the time integration (Eqs. 19-25): element-wise parity of
predict / kick / drift with the oracle, a few chained steps against the oracle-driven
evolution, conservation over many steps, and the Sod shock tube against the exact Riemann
solution (Fig. 4)."""
import numpy as np
import pytest
import torch

from oracle import sph_oracle as orc
from paper_2511_11425_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gu():
    import gpu_util
    return gpu_util


def _wrapdiff(a, b, L, periodic):
    d = a - b
    return d - L * np.rint(d / L) if periodic else d


def test_predict_kick_drift_elementwise(gu):
    from paper_2511_11425_b200 import sph
    rng = np.random.default_rng(3)
    n = 100_003
    box = sph.Box((-0.5, 0.0, 1.0), (1.0, 2.0, 0.5), (1, 0, 1))
    ctx = sph.Sph(sph.Params(), box, n)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()
    q = {k: rng.normal(0, 1, n).astype(np.float32) for k in ("vx", "vy", "vz", "u")}
    r = {k: rng.normal(0, 3, n).astype(np.float32) for k in ("ax", "ay", "az", "dudt")}
    x = {"x": rng.uniform(-0.5, 0.5, n), "y": rng.uniform(0, 2, n), "z": rng.uniform(1, 1.5, n)}
    x = {k: v.astype(np.float32) for k, v in x.items()}
    dt, scale = np.float32(0.0371), 0.75
    tdt = f(np.array([dt]))
    dq, dr = {k: f(v) for k, v in q.items()}, {k: f(v) for k, v in r.items()}
    pred = [torch.empty(n, device="cuda") for _ in range(4)]
    ctx.predict(tdt, scale, dq["vx"], dq["vy"], dq["vz"], dq["u"], dr["ax"], dr["ay"], dr["az"],
                dr["dudt"], *pred)
    step = float(dt) * scale
    for p, kq, kr in zip(pred, ("vx", "vy", "vz", "u"), ("ax", "ay", "az", "dudt")):
        ref = orc.axpy(0.5 * step, r[kr], q[kq])
        assert np.abs(gu.np64(p) - ref).max() <= 2e-7 * (np.abs(ref).max() + 1)
    ctx.kick(tdt, scale, dq["vx"], dq["vy"], dq["vz"], dq["u"], dr["ax"], dr["ay"], dr["az"],
             dr["dudt"])
    for kq, kr in zip(("vx", "vy", "vz", "u"), ("ax", "ay", "az", "dudt")):
        ref = orc.axpy(0.5 * step, r[kr], q[kq])
        assert np.abs(gu.np64(dq[kq]) - ref).max() <= 2e-7 * (np.abs(ref).max() + 1)
    dx = {k: f(v) for k, v in x.items()}
    vq = {k: f(q[k]) for k in ("vx", "vy", "vz")}
    ctx.drift(tdt, scale, dx["x"], dx["y"], dx["z"], vq["vx"], vq["vy"], vq["vz"])
    for d, (k, kv) in enumerate(zip("xyz", ("vx", "vy", "vz"))):
        ref = orc.drift(x[k], q[kv], step, box.lo[d], box.len[d], box.periodic[d])
        g = gu.np64(dx[k])
        assert np.abs(_wrapdiff(g, ref, box.len[d], box.periodic[d])).max() <= 3e-7
        if box.periodic[d]:
            assert (g >= box.lo[d]).all() and (g < box.lo[d] + box.len[d]).all()


def test_three_steps_against_the_oracle_driven_evolution(gu):
    """The same kick-drift-kick sequence driven through the FP64 oracle (cell-list variant)."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.uniform_cube(h_start="warm", v_sigma=0.05)
    _, op = gu.make_params(w)
    _, ob = gu.make_boxes(w)
    sim = Simulation(w)
    # oracle state in FP64, started from the same FP32 inputs
    s = {k: w[k].astype(np.float64) for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h")}
    a = {k: np.zeros(w["n"]) for k in ("ax", "ay", "az", "dudt")}
    dt_prev, t_or = 0.0, 0.0
    for _ in range(3):
        sim.step()
        h, rho, om, _ = orc.density(s["x"], s["y"], s["z"], s["m"], s["h"], ob, op, cells=True)
        vp = [orc.axpy(0.5 * dt_prev, a[ka], s[kv]) for kv, ka in
              (("vx", "ax"), ("vy", "ay"), ("vz", "az"), ("u", "dudt"))]
        o = orc.forces(s["x"], s["y"], s["z"], s["m"], vp[0], vp[1], vp[2], vp[3], rho, h, om, ob,
                       op, cells=True)
        P, c = orc.eos(rho, vp[3], op.gamma)
        _, dt = orc.timestep(h, c, o["ax"], o["ay"], o["az"], o["mu_min"], op)
        a = {k: o[k] for k in ("ax", "ay", "az", "dudt")}
        for kv, ka in (("vx", "ax"), ("vy", "ay"), ("vz", "az"), ("u", "dudt")):
            s[kv] = orc.axpy(0.5 * dt_prev, a[ka], s[kv])     # closing kick
            s[kv] = orc.axpy(0.5 * dt, a[ka], s[kv])          # opening kick
        for d, (k, kv) in enumerate(zip("xyz", ("vx", "vy", "vz"))):
            s[k] = orc.drift(s[k], s[kv], dt, ob.lo[d], ob.len[d], ob.periodic[d])
        s["h"] = h
        dt_prev = dt
        t_or += dt
    assert abs(float(sim.t.item()) / t_or - 1) <= 1e-5
    for d, k in enumerate("xyz"):
        assert np.abs(_wrapdiff(gu.np64(sim.d[k]), s[k], 1.0, 1)).max() <= 5e-7
    vscale = max(np.abs(s[k]).max() for k in ("vx", "vy", "vz"))
    for k in ("vx", "vy", "vz"):
        assert np.abs(gu.np64(sim.d[k]) - s[k]).max() <= 2e-5 * vscale
    assert np.abs(gu.np64(sim.d["u"]) / s["u"] - 1).max() <= 2e-5
    assert np.abs(gu.np64(sim.d["h"]) / s["h"] - 1).max() <= 1e-5


def test_energy_and_momentum_conservation_over_many_steps(gu):
    """PAPER.md:325 quotes < 0.2 % energy error for the Sedov run with a global step; here a
    small periodic cube with random velocities (all pairs approaching or receding)."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.uniform_cube(nside=24, h_start="warm", v_sigma=0.3)
    sim = Simulation(w)
    sim.synchronise()
    ek0, eu0 = sim.energies()
    p0 = sim.momentum()
    for _ in range(40):
        sim.step()
    sim.synchronise()
    ek1, eu1 = sim.energies()
    p1 = sim.momentum()
    e0, e1 = ek0 + eu0, ek1 + eu1
    assert abs(e1 - e0) <= 1e-3 * e0, (e0, e1)        # 0.1 %; PAPER.md:325 quotes < 0.2 %
    assert ek1 < ek0                                   # viscosity turns kinetic into internal energy
    pscale = float((w["m"].astype(np.float64) * np.abs(w["vx"]).astype(np.float64)).sum())
    assert max(abs(b - a_) for a_, b in zip(p0, p1)) <= 1e-5 * pscale
    assert sim.ctx.stats()["dens_nonconv"] == 0


def _sod_exact(x, t, gamma=1.4, left=(1.0, 0.0, 1.0), right=(0.125, 0.0, 0.1), x0=0.5):
    """Exact solution of the Riemann problem for an ideal gas (textbook: Toro, ch. 4):
    Newton iteration for the star pressure, then sampling.  Returns density at x."""
    rl, ul, pl = left
    rr, ur, pr = right
    cl, cr = np.sqrt(gamma * pl / rl), np.sqrt(gamma * pr / rr)
    g1, g2 = (gamma - 1) / (2 * gamma), (gamma + 1) / (2 * gamma)

    def fk(p, rk, pk, ck):
        if p > pk:   # shock
            A, B = 2 / ((gamma + 1) * rk), (gamma - 1) / (gamma + 1) * pk
            return (p - pk) * np.sqrt(A / (p + B)), np.sqrt(A / (p + B)) * (1 - (p - pk) / (2 * (B + p)))
        return 2 * ck / (gamma - 1) * ((p / pk) ** g1 - 1), 1 / (rk * ck) * (p / pk) ** (-g2)

    p = 0.5 * (pl + pr)
    for _ in range(50):
        f1, d1 = fk(p, rl, pl, cl)
        f2, d2 = fk(p, rr, pr, cr)
        dp = (f1 + f2 + ur - ul) / (d1 + d2)
        p = max(p - dp, 1e-8)
        if abs(dp) < 1e-14:
            break
    us = 0.5 * (ul + ur) + 0.5 * (fk(p, rr, pr, cr)[0] - fk(p, rl, pl, cl)[0])
    rho = np.empty_like(x)
    xi = (x - x0) / t
    # left rarefaction (p < pl), right shock (p > pr): the Sod configuration
    rsl = rl * (p / pl) ** (1 / gamma)
    csl = cl * (p / pl) ** g1
    rsr = rr * ((p / pr + (gamma - 1) / (gamma + 1)) / ((gamma - 1) / (gamma + 1) * p / pr + 1))
    S = ur + cr * np.sqrt(g2 * p / pr + g1)
    for i, s in enumerate(xi):
        if s <= ul - cl:
            rho[i] = rl
        elif s <= us - csl:
            rho[i] = rl * (2 / (gamma + 1) + (gamma - 1) / ((gamma + 1) * cl) * (ul - s)) ** (2 / (gamma - 1))
        elif s <= us:
            rho[i] = rsl
        elif s <= S:
            rho[i] = rsr
        else:
            rho[i] = rr
    return rho, p, us


def test_sod_shock_tube_against_the_exact_solution(gu):
    """Config 2 (lattice jittered by 0.2 spacings) evolved to t = 0.1: the binned SPH density follows the exact Riemann solution
    around the x = 0.5 diaphragm (plateaus to 2 %, L1 error of the profile below 3 %)."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.sod_tube(h_start="warm", jitter=0.2)   # a perfect lattice cannot rearrange
    sim = Simulation(w)
    sim.synchronise()
    e0 = sum(sim.energies())
    sim.run_until(0.1)
    e1 = sum(sim.energies())
    assert abs(e1 - e0) <= 2e-3 * e0                     # PAPER.md:325 quotes 0.2 %
    assert sim.ctx.stats()["dens_nonconv"] == 0
    x = gu.np64(sim.d["x"])
    rho = gu.np64(sim.out["rho"])
    edges = np.linspace(0.25, 0.75, 126)
    idx = np.digitize(x, edges) - 1
    ok = (idx >= 0) & (idx < 125)
    mean = np.bincount(idx[ok], rho[ok], 125) / np.maximum(np.bincount(idx[ok], None, 125), 1)
    xc = 0.5 * (edges[1:] + edges[:-1])
    exact, pstar, ustar = _sod_exact(xc, 0.1)
    assert abs(pstar - 0.30313) < 1e-4 and abs(ustar - 0.92745) < 1e-4   # textbook star values
    l1 = np.abs(mean - exact).mean() / exact.mean()
    assert l1 <= 0.03, l1
    # plateaus between the waves: rho*_L = 0.4263 (x in [0.50, 0.58]), rho*_R = 0.2656 ([0.61, 0.66])
    pl = mean[(xc > 0.51) & (xc < 0.57)].mean()
    prr = mean[(xc > 0.615) & (xc < 0.655)].mean()
    assert abs(pl / 0.42632 - 1) <= 0.02, pl
    assert abs(prr / 0.26557 - 1) <= 0.03, prr


def test_sedov_taylor_blast_shock_radius_and_energy(gu):
    """Config 3's shape at 64^3 evolved with the dynamic global step: the
    shock sits at the Sedov-Taylor radius R = 1.152 (E t^2 / rho)^(1/5) (gamma = 5/3), the
    compression behind it is strong (4 in the continuum limit, smeared over ~2h here) and the
    total energy is conserved to the paper's 0.2 % class."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.sedov(nside=64, h_start="warm")
    sim = Simulation(w)
    sim.synchronise()
    e0 = sum(sim.energies())
    R = 0.3
    sim.run_until((R / 1.152) ** 2.5)
    e1 = sum(sim.energies())
    assert abs(e1 / e0 - 1) <= 3e-3, e1 / e0 - 1
    assert sim.ctx.stats()["dens_nonconv"] == 0
    x, y, z = (gu.np64(sim.d[k]) - 0.5 for k in "xyz")
    r = np.sqrt(x * x + y * y + z * z)
    rho = gu.np64(sim.out["rho"])
    edges = np.linspace(0.0, 0.5, 101)
    idx = np.digitize(r, edges) - 1
    ok = idx < 100
    mean = np.bincount(idx[ok], rho[ok], 100) / np.maximum(np.bincount(idx[ok], None, 100), 1)
    k = int(np.argmax(mean))
    r_peak = 0.5 * (edges[k] + edges[k + 1])
    assert abs(r_peak / R - 1) <= 0.04, r_peak           # shock position
    assert mean[k] >= 2.3, mean[k]                       # compression behind the shock
    assert abs(mean[edges[:-1] > 0.4].mean() / 1.0146 - 1) <= 2e-3   # undisturbed gas ahead
    assert mean[:20].max() < 0.2                         # evacuated interior


def test_entropy_variant_conserves_the_entropic_function_without_viscosity(gu):
    """with the viscosity off, the entropy-conserving scheme keeps
    A_i = u_i rho_i^(1-gamma) of every particle over many steps (u follows the isentrope to
    each new density; the kicks add nothing), while the flow compresses and expands; with
    the viscosity on, A_i never decreases and total energy stays close (the scheme trades the
    exact energy budget for the entropy one)."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.uniform_cube(nside=24, h_start="warm", v_sigma=0.3)
    gamma = float(np.float32(w["gamma"]))
    w0 = dict(w, av_alpha=0.0, av_beta=0.0)

    def entropic(sim):
        return gu.np64(sim.d["u"]) * gu.np64(sim.out["rho"]) ** (1.0 - gamma)

    sim = Simulation(w0, entropy=1)
    sim.synchronise()
    A0, rho0 = entropic(sim), gu.np64(sim.out["rho"]).copy()
    ek0, eu0 = sim.energies()
    for _ in range(20):
        sim.step()
    sim.synchronise()
    A1, rho1 = entropic(sim), gu.np64(sim.out["rho"])
    assert np.abs(rho1 / rho0 - 1).max() > 0.02          # the gas did compress / expand
    assert (np.abs(A1 - A0) / A0).max() <= 2e-5, (np.abs(A1 - A0) / A0).max()
    assert np.abs(gu.np64(sim.out["dudt"])).max() == 0.0
    ek1, eu1 = sim.energies()
    assert abs((ek1 + eu1) - (ek0 + eu0)) <= 1e-2 * (ek0 + eu0), (ek0, eu0, ek1, eu1)

    simv = Simulation(w, entropy=1)
    simv.synchronise()
    B0 = entropic(simv)
    e0 = sum(simv.energies())
    for _ in range(20):
        simv.step()
    simv.synchronise()
    B1 = entropic(simv)
    assert ((B1 - B0) / B0).min() >= -2e-5               # viscous heating only raises entropy
    assert ((B1 - B0) / B0).max() > 1e-4
    assert abs(sum(simv.energies()) - e0) <= 1e-2 * e0, (sum(simv.energies()), e0)


# ------------------------------------------- block time steps (reading R32)
def test_block_predict_active_kick_elementwise(gu):
    """sph_block_predict / sph_block_active / sph_block_kick against the oracle on a seeded
    state with every rung populated, some steps ending at the substep, desired rungs below
    the floor of the substep and above the cap; closing-only mode as well."""
    from paper_2511_11425_b200 import sph
    rng = np.random.default_rng(17)
    n, R, s = 50_003, 5, 40                      # floor rung of substep 40 with R = 5: 2
    delta = float(np.float32(0.0123))
    ctx = sph.Sph(sph.Params(), sph.Box(), n)
    rung = rng.integers(0, R + 1, n).astype(np.int32)
    L = 2 ** (R - rung)
    ends = rng.random(n) < 0.4
    tnext = np.where(ends, s, s + rng.integers(1, 32, n)).astype(np.int32)
    hk = np.float32(0.5 * L * delta)
    hk[rng.random(n) < 0.05] = 0.0               # particles that have not been kicked yet
    des = rng.integers(0, R + 3, n).astype(np.int32)
    q = [rng.normal(0, 1, n).astype(np.float32) for _ in range(4)]
    r = [rng.normal(0, 3, n).astype(np.float32) for _ in range(4)]
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dq, dr = [f(a) for a in q], [f(a) for a in r]
    pred = [torch.empty(n, device="cuda") for _ in range(4)]
    ctx.block_predict(s, delta, f(tnext), f(hk), *dq, *dr, *pred)
    for k in range(4):
        ref = orc.block_predict(s, delta, tnext, hk, q[k], r[k])
        assert np.abs(gu.np64(pred[k]) - ref).max() <= 3e-7 * (np.abs(ref).max() + 1)
    act = torch.empty(n, dtype=torch.uint8, device="cuda")
    ctx.block_active(s, f(tnext), act)
    assert np.array_equal(act.cpu().numpy().astype(bool), tnext == s)
    assert orc.block_floor_rung(s, R) == 2
    for open_ in (1, 0):
        drung, dtn, dhk, dqq = f(rung), f(tnext), f(hk), [f(a) for a in q]
        ctx.block_kick(s, R, delta, f(des), drung, dtn, dhk, *dqq, *dr, open=open_)
        torch.cuda.synchronize()
        org, otn, ohk, oq = orc.block_kick(s, R, delta, des, rung, tnext, hk, q, r, open=open_)
        assert np.array_equal(drung.cpu().numpy(), org)
        assert np.array_equal(dtn.cpu().numpy(), otn)
        assert np.abs(gu.np64(dhk) - ohk).max() <= 1e-7 * ohk.max() + 0.0
        for k in range(4):
            assert np.abs(gu.np64(dqq[k]) - oq[k]).max() <= 3e-7 * (np.abs(oq[k]).max() + 1)
            assert np.array_equal(dqq[k].cpu().numpy()[~ends], q[k][~ends])   # others untouched
        if open_:
            assert (org[ends] >= 2).all() and (org[ends] <= R).all() and set(org[ends]) == {2, 3, 4, 5}


def test_block_driver_on_one_rung_is_the_global_step_driver(gu):
    """max_rung = 0: every particle steps with dt0, and the block driver must reproduce the
    global-step driver run with that fixed step bit for bit (same kernels for density and
    forces, the same fused multiply-adds in the kicks and the drift).  The block driver's
    active sets are swept by the 8-lanes-per-target kernels, so the global-step driver runs on
    those as well here (tile = -1); on the staged-tile sweeps it agrees to rounding."""
    from paper_2511_11425_b200.integrate import BlockSimulation, Simulation
    w = workloads.uniform_cube(h_start="warm", v_sigma=0.05)
    dt0 = 2.0e-3                                  # below the CFL step of this state (~7e-3)
    a, b = Simulation(w, tile=-1), BlockSimulation(w, dt0=dt0, max_rung=0, tile=-1)
    t = Simulation(w)
    for _ in range(5):
        a.step(dt_cap=dt0)
        b.step()
        t.step(dt_cap=dt0)
    assert float(a.out["dt_min"].item()) == float(np.float32(dt0))   # the cap was the step
    for k in ("x", "y", "z", "vx", "vy", "vz", "u", "h"):
        assert (t.d[k] - a.d[k]).abs().max() <= 2e-5 * a.d[k].abs().max(), k
    for k in ("x", "y", "z", "vx", "vy", "vz", "u", "h"):
        assert torch.equal(a.d[k], b.d[k]), k
    a.synchronise()
    b.synchronise()
    for k in ("vx", "vy", "vz", "u"):
        assert torch.equal(a.d[k], b.d[k]), k
    assert not b.hk.any() and (b.tnext == 5).all()


@pytest.mark.parametrize("fastgas", [False, True])
def test_block_steps_on_the_sod_tube(gu, fastgas):
    """Config 2 with block time steps (dt0 = 3.2e-3, rungs 0..3): the dense left half steps
    with dt0/8, the dilute right half with dt0/4 or dt0/2; after 32 big steps (t = 0.1024)
    the density profile follows the exact Riemann solution as with the global step (L1 < 3 %),
    energy is conserved to 0.5 %, and FastGas (marking pass + density of the marked only on
    the substeps between the full ones) gives the same flow."""
    from paper_2511_11425_b200.integrate import BlockSimulation
    w = workloads.sod_tube(h_start="warm", jitter=0.2)
    sim = BlockSimulation(w, dt0=3.2e-3, max_rung=3, fastgas=fastgas)
    sim.synchronise()
    e0 = sum(sim.energies())
    for _ in range(31):
        sim.big_step()
    pop = np.bincount(sim.rung.cpu().numpy(), minlength=4)
    sim.run_until(0.1)                       # one more big step (to 32 dt0), then synchronise
    assert sim.s == 32 * 8
    t = float(sim.t.item())
    assert abs(t - 0.1024) <= 1e-6
    e1 = sum(sim.energies())
    assert abs(e1 - e0) <= 5e-3 * e0, (e0, e1)
    assert (pop > 0.02 * pop.sum()).sum() >= 2, pop          # at least two rungs carry particles
    assert sim.ctx.stats()["dens_nonconv"] == 0
    x = gu.np64(sim.d["x"])
    rho = gu.np64(sim.out["rho"])
    edges = np.linspace(0.25, 0.75, 126)
    idx = np.digitize(x, edges) - 1
    ok = (idx >= 0) & (idx < 125)
    mean = np.bincount(idx[ok], rho[ok], 125) / np.maximum(np.bincount(idx[ok], None, 125), 1)
    xc = 0.5 * (edges[1:] + edges[:-1])
    exact, _, _ = _sod_exact(xc, t)
    l1 = np.abs(mean - exact).mean() / exact.mean()
    assert l1 <= 0.03, l1


@pytest.mark.parametrize("fastgas", [0.0, 0.5, 1.0])
def test_block_steps_with_the_entropy_variant_keep_the_entropic_function(gu, fastgas):
    """Block time steps + PAPER.md:197 without viscosity: u rho^(1-gamma) of every particle is
    kept over two big steps of 8 substeps, on whatever rung it moves and whether its density
    is refreshed on every substep or (FastGas) only when a neighbour is active."""
    from paper_2511_11425_b200.integrate import BlockSimulation
    w = dict(workloads.uniform_cube(nside=24, h_start="warm", v_sigma=0.3), av_alpha=0.0, av_beta=0.0)
    gamma = float(np.float32(w["gamma"]))
    sim = BlockSimulation(w, dt0=0.03, max_rung=3, fastgas=fastgas, entropy=1)
    sim.synchronise()
    A0 = gu.np64(sim.d["u"]) * gu.np64(sim.out["rho"]) ** (1.0 - gamma)
    rho0 = gu.np64(sim.out["rho"]).copy()
    for _ in range(2):
        sim.big_step()
    pop = np.bincount(sim.rung.cpu().numpy(), minlength=4)
    sim.synchronise()
    rho1 = gu.np64(sim.out["rho"])
    A1 = gu.np64(sim.d["u"]) * rho1 ** (1.0 - gamma)
    assert (pop > 0).sum() >= 2, pop
    assert np.abs(rho1 / rho0 - 1).max() > 0.02
    assert (np.abs(A1 - A0) / A0).max() <= 2e-5, (np.abs(A1 - A0) / A0).max()


def test_block_substeps_against_the_oracle_driven_evolution(gu):
    """One big step of four substeps on mixed rungs (config 1 with fast random velocities), the
    same sequence driven through the FP64 oracle: density of all, prediction of all, forces of
    the particles whose step ends (brute force over those targets), Eq. (26), Eq. (27) +
    limiter, closing kick / rung change / opening kick, drift.  Rungs and step ends must agree
    exactly, the state within the tolerances of the global-step test."""
    from paper_2511_11425_b200.integrate import BlockSimulation
    w = workloads.uniform_cube(h_start="warm", v_sigma=0.3)
    _, op = gu.make_params(w)
    _, ob = gu.make_boxes(w)
    R, dt0 = 2, float(np.float32(0.016))     # dt_i from 0.0058 to 0.0114: rungs 1 and 2
    sim = BlockSimulation(w, dt0=dt0, max_rung=R)
    delta = sim.delta
    n = int(w["n"])
    s = {k: w[k].astype(np.float64) for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h")}
    a = {k: np.zeros(n) for k in ("ax", "ay", "az", "dudt")}
    mu_min = np.zeros(n)
    rung, tnext, hk = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n)
    kv, ka = ("vx", "vy", "vz", "u"), ("ax", "ay", "az", "dudt")
    seen, partial = set(), 0
    for sub in range(6):                              # one big step and two more substeps
        sim.step()
        act = np.flatnonzero(tnext == sub)
        partial += 0 < len(act) < n
        h, rho, om, _ = orc.density(s["x"], s["y"], s["z"], s["m"], s["h"], ob, op, cells=True)
        vp = [orc.block_predict(sub, delta, tnext, hk, s[q], a[r]) for q, r in zip(kv, ka)]
        o = orc.forces(s["x"], s["y"], s["z"], s["m"], vp[0], vp[1], vp[2], vp[3], rho, h, om, ob,
                       op, targets=act)
        for k in ka:
            a[k][act] = o[k]
        mu_min[act] = o["mu_min"]
        _, c = orc.eos(rho, vp[3], op.gamma)
        dt_i, _ = orc.timestep(h, c, a["ax"], a["ay"], a["az"], mu_min, op)
        des = orc.rung_limiter(s["x"], s["y"], s["z"], h, orc.rungs(dt_i, dt0, R), ob)
        rung, tnext, hk, q = orc.block_kick(sub, R, delta, des, rung, tnext, hk,
                                            [s[k] for k in kv], [a[k] for k in ka])
        for k, v in zip(kv, q):
            s[k] = v
        for d, (k, v) in enumerate(zip("xyz", ("vx", "vy", "vz"))):
            s[k] = orc.drift(s[k], s[v], delta, ob.lo[d], ob.len[d], ob.periodic[d])
        s["h"] = h
        seen |= set(rung.tolist())
        assert np.array_equal(sim.rung.cpu().numpy(), rung), (sub, int((sim.rung.cpu().numpy() != rung).sum()))
        assert np.array_equal(sim.tnext.cpu().numpy(), tnext), sub
    assert len(seen) >= 2, seen                       # more than one rung in use
    assert partial >= 2                               # substeps with a partial active set
    for d, k in enumerate("xyz"):
        assert np.abs(_wrapdiff(gu.np64(sim.d[k]), s[k], 1.0, 1)).max() <= 5e-7
    vscale = max(np.abs(s[k]).max() for k in ("vx", "vy", "vz"))
    for k in ("vx", "vy", "vz"):
        assert np.abs(gu.np64(sim.d[k]) - s[k]).max() <= 2e-5 * vscale
    assert np.abs(gu.np64(sim.d["u"]) / s["u"] - 1).max() <= 2e-5
    assert np.abs(gu.np64(sim.d["h"]) / s["h"] - 1).max() <= 1e-5
    assert np.abs(gu.np64(sim.hk) - hk).max() <= 1e-7 * hk.max()


def test_driver_with_the_interface_correction_pass(gu):
    """Step 3 of PAPER.md:241 in the global-step driver, two materials split at x = 0.5 (and at
    the periodic face).  One step = one force pass: the imbalance is non-zero within 2h of the
    boundary and at the level of the lattice noise elsewhere, so the corrected density and
    the velocities differ from the uncorrected run's near the boundary and hardly beyond 4h of
    it.  With one uniform state the correction only smooths the lattice noise (below 5 % at the
    boundary); with a 4:1 jump of u across it (P and T jump alike, so rho(P~, T~) moves little)
    it acts somewhat more strongly, in the same place."""
    from paper_2511_11425_b200.integrate import Simulation
    w = workloads.uniform_cube(nside=32, h_start="warm", v_sigma=0.01)
    w["mat"] = (w["x"] >= 0.5).astype(np.int32)
    dist = np.minimum(np.abs(w["x"] - 0.5), np.minimum(w["x"], 1 - w["x"]))
    far, near = dist > 0.2, dist < 0.03            # h = 0.04 here: 4h = 0.16

    def run(ww, alpha):
        sim = Simulation(ww, interface_alpha=alpha)
        sim.step(dt_cap=2e-3)
        return sim

    def check(a, b):
        ratio = gu.np64(b.rho_corr) / gu.np64(b.out["rho"]) - 1
        imb = gu.np64(b.imbalance)
        dv = np.abs(gu.np64(a.d["vx"]) - gu.np64(b.d["vx"]))
        assert imb[near].mean() > 0.1 and imb[near].mean() > 5 * imb[far].max()
        assert np.abs(ratio[far]).max() <= 1e-4          # e^(-I^2) of the lattice noise
        assert dv[near].max() > 50 * dv[far].max(), (dv[near].max(), dv[far].max())
        return np.abs(ratio[near]).max(), dv[near].max()

    r1, dv1 = check(run(w, None), run(w, 1.5))
    assert r1 <= 0.05
    w2 = dict(w)
    w2["u"] = np.where(w["x"] < 0.5, 4.0, 1.0).astype(np.float32)
    r2, dv2 = check(run(w2, None), run(w2, 1.5))
    assert r2 > r1 and dv2 > dv1, (r1, r2, dv1, dv2)


def _two_material_cube(v_sigma):
    """Config 1 on 24^3 particles, two materials split at x = 0.5 (and at the periodic face), a
    4:1 jump of u across it: the imbalance and the density correction are not small there."""
    w = workloads.uniform_cube(nside=24, h_start="warm", v_sigma=v_sigma)
    w["mat"] = (w["x"] >= 0.5).astype(np.int32)
    w["u"] = np.where(w["x"] < 0.5, 4.0, 1.0).astype(np.float32)
    return w


def test_block_driver_with_the_interface_correction_on_one_rung_is_the_global_step_driver(gu):
    """Step 3 inside the block-step driver: with max_rung = 0 it must reproduce the
    global-step driver with the correction bit for bit (same passes in the same order), and the
    correction must matter (the run without it differs near the material boundary)."""
    from paper_2511_11425_b200.integrate import BlockSimulation, Simulation
    w = _two_material_cube(0.05)
    dt0 = 1.0e-3
    a = Simulation(w, interface_alpha=1.5, tile=-1)
    b = BlockSimulation(w, dt0=dt0, max_rung=0, interface_alpha=1.5, tile=-1)
    plain = BlockSimulation(w, dt0=dt0, max_rung=0, tile=-1)
    for _ in range(4):
        a.step(dt_cap=dt0)
        b.step()
        plain.step()
    assert float(a.out["dt_min"].item()) == float(np.float32(dt0))   # the cap was the step
    for k in ("x", "y", "z", "vx", "vy", "vz", "u", "h"):
        assert torch.equal(a.d[k], b.d[k]), k
    assert torch.equal(a.rho_corr, b.rho_corr) and torch.equal(a.imbalance, b.imbalance)
    near = torch.from_numpy(np.abs(w["x"] - 0.5) < 0.03).cuda()
    dv = (b.d["vx"] - plain.d["vx"]).abs()
    assert float(dv[near].max()) > 1e-4 * float(b.d["vx"].abs().max())
    assert float((b.rho_corr / b.out["rho"] - 1).abs()[near].max()) > 1e-3


def test_block_steps_with_the_interface_correction_do_not_depend_on_fastgas(gu):
    """Mixed rungs with the interface correction: FastGas (first marking pass from the active
    particles, second from the marked ones, density for either mark) must give the
    flow of the run that updates every density on every substep -- the same rungs and step ends,
    the state to rounding (the sweeps of a subset sum in the same order; a density that is not
    refreshed belongs to a particle no active particle interacts with)."""
    from paper_2511_11425_b200.integrate import BlockSimulation
    w = _two_material_cube(0.3)
    R, dt0 = 2, float(np.float32(0.008))
    a = BlockSimulation(w, dt0=dt0, max_rung=R, interface_alpha=1.5)
    b = BlockSimulation(w, dt0=dt0, max_rung=R, interface_alpha=1.5, fastgas=1.0)
    seen = set()
    for _ in range(2 * (1 << R)):
        a.step()
        b.step()
        seen |= set(a.rung.cpu().numpy().tolist())
        assert torch.equal(a.rung, b.rung) and torch.equal(a.tnext, b.tnext)
    assert len(seen) >= 2, seen
    a.synchronise()
    b.synchronise()
    for k in ("x", "y", "z"):
        assert np.abs(_wrapdiff(gu.np64(a.d[k]), gu.np64(b.d[k]), 1.0, 1)).max() <= 1e-6
    vscale = max(float(a.d[k].abs().max()) for k in ("vx", "vy", "vz"))
    for k in ("vx", "vy", "vz"):
        assert float((a.d[k] - b.d[k]).abs().max()) <= 2e-5 * vscale, k
    assert float((a.d["u"] / b.d["u"] - 1).abs().max()) <= 2e-5


def test_block_substep_with_the_interface_correction_against_the_oracle(gu):
    """The first substep of the block driver with the correction, driven through the FP64 oracle:
    density, prediction (no kick pending), imbalance (Eq. 8) and corrected density (Eqs. 9-12) from
    the predicted u, forces with the corrected density, Eq. (26), Eq. (27) + limiter."""
    from paper_2511_11425_b200.integrate import BlockSimulation
    w = _two_material_cube(0.3)
    _, op = gu.make_params(w)
    _, ob = gu.make_boxes(w)
    R, dt0, alpha = 2, float(np.float32(0.008)), 1.5
    sim = BlockSimulation(w, dt0=dt0, max_rung=R, interface_alpha=alpha)
    sim.step()
    s = {k: w[k].astype(np.float64) for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h")}
    h, rho, om, _ = orc.density(s["x"], s["y"], s["z"], s["m"], s["h"], ob, op, cells=True)
    imb = orc.imbalance(s["x"], s["y"], s["z"], s["m"], h, w["mat"], ob, op, alpha)
    rho_c = orc.interface_correction(s["x"], s["y"], s["z"], h, s["u"], rho, imb, ob, op)
    rho_c = rho_c[0] if isinstance(rho_c, tuple) else rho_c
    assert np.abs(gu.np64(sim.imbalance) - imb).max() <= 1e-4 * max(imb.max(), 1.0)
    assert np.abs(gu.np64(sim.rho_corr) / rho_c - 1).max() <= 2e-5
    o = orc.forces(s["x"], s["y"], s["z"], s["m"], s["vx"], s["vy"], s["vz"], s["u"], rho_c, h, om, ob, op)
    ea, eu = gu.force_errors(sim.out.t, o)
    assert ea.max() <= 1e-4 and eu.max() <= 1e-4, (ea.max(), eu.max())
    _, c = orc.eos(rho_c, s["u"], op.gamma)
    dt_i, _ = orc.timestep(h, c, o["ax"], o["ay"], o["az"], o["mu_min"], op)
    des = orc.rung_limiter(s["x"], s["y"], s["z"], h, orc.rungs(dt_i, dt0, R), ob)
    got = sim.rung.cpu().numpy()
    # a dt_i within rounding of a rung boundary may fall either way; the rest must agree
    edge = np.abs(np.log2(dt0 / dt_i) - np.round(np.log2(dt0 / dt_i))) < 1e-4
    assert np.array_equal(got[~edge], des[~edge]) and edge.mean() < 0.01
    assert len(set(des.tolist())) >= 2


def test_step_graph_replays_the_same_step(gu):
    """sph.StepGraph: the hot path captured in a CUDA graph (no allocation, no host
    synchronisation and no host-dependent branch inside a step, so the capture is legal) and
    replayed gives bit for bit what the same calls give when launched one by one -- on the
    8-lane path (config 1, where the launches set the time) and on the tile path."""
    from paper_2511_11425_b200 import sph
    for w, kw in ((workloads.uniform_cube(h_start="warm", v_sigma=0.05), dict(tile=-1)),
                  (workloads.sedov(nside=48, h_start="warm", v_sigma=0.05), dict(tile=1))):
        n = int(w["n"])
        d = gu.to_device(w)
        gp, _ = gu.make_params(w, **kw)
        gb, _ = gu.make_boxes(w)
        a = sph.Sph(gp, gb, n)
        oa, ha = sph.StepBuffers(n), d["h"].clone()
        sph.step(a, d, oa, ha)
        s = torch.cuda.Stream()
        b = sph.Sph(gp, gb, n, stream=s)
        ob, hb = sph.StepBuffers(n), d["h"].clone()
        g = sph.StepGraph(b, d, ob, hb)
        assert torch.equal(hb, d["h"])                 # capturing ran nothing on the caller's arrays
        for _ in range(2):                             # twice: a replay leaves no state behind
            hb.copy_(d["h"])
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(ha, hb)
            for k in ("rho", "omega", "n_ngb", "ax", "ay", "az", "dudt", "mu_min", "P", "c", "dt_i", "dt_min"):
                assert torch.equal(oa[k], ob[k]), k
        with pytest.raises(sph.SphError):
            sph.StepGraph(a, d, oa, ha)                # a context on the default stream cannot be captured
        a.close()
        b.close()
