"""Global-time-step kick-drift-kick driver over the C-ABI calls (Section 2.3.6,
Eqs. 19-25; the dynamic global step of PAPER.md:325).  Plumbing only: every update runs in the
library's kernels, the step length never leaves the device.

One step, in the paper's order:
  1. density pass at time i                                   sph_build_cells, sph_density_h
  2. predict v, u to time i with the derivatives of i-1       sph_predict          (Eqs. 19-20)
  4. force pass with the predicted values, new global dt      sph_forces, sph_timestep
     closing kick of the previous step (its dt)               sph_kick             (Eqs. 21-22)
     opening kick of the new step (new dt)                    sph_kick             (Eqs. 23-24)
  5. drift                                                    sph_drift            (Eq. 25)
Step 3, the interface correction (Eqs. 8-12), runs between 2 and 4 when `interface_alpha` is given
(material ids from w["mat"], one material without it): sph_interface_correction on the predicted
u, and the corrected density goes into the force pass.  Between steps v and u live at the half step.

With `entropy=1` the force pass returns the viscous heating of Eq. (18) alone and,
right after each density pass, u follows the isentrope from the previous pass's density to the new
one (sph_isentropic_u); the kicks then add the viscous heating.
"""
from __future__ import annotations

import numpy as np
import torch

from . import sph

_KEYS = ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h")


class Simulation:
    def __init__(self, w: dict, interface_alpha: float | None = None, **params):
        n = int(w["n"])
        self.interface_alpha = interface_alpha
        self.n = n
        self.d = {k: torch.from_numpy(np.ascontiguousarray(w[k], np.float32)).cuda() for k in _KEYS}
        self.ctx = sph.Sph(sph.Params(gamma=float(w["gamma"]), av_alpha=float(w["av_alpha"]),
                                      av_beta=float(w["av_beta"]), **params),
                           sph.Box(w["box_lo"], w["box_len"], w["periodic"]), n)
        self.out = sph.StepBuffers(n)
        f = dict(dtype=torch.float32, device="cuda")
        self.pred = {k: torch.empty(n, **f) for k in ("vx", "vy", "vz", "u")}
        for k in ("ax", "ay", "az", "dudt"):
            self.out[k].zero_()
        self.dt_prev = torch.zeros(1, **f)     # no half kick is pending before the first step
        self.dt_new = self.out["dt_min"]
        self.t = torch.zeros(1, dtype=torch.float64, device="cuda")
        self.steps = 0
        if interface_alpha is not None:
            self.mat = (torch.from_numpy(np.ascontiguousarray(w["mat"], np.int32)).cuda()
                        if "mat" in w else None)
            self.imbalance = torch.empty(n, **f)
            self.rho_corr = torch.empty(n, **f)
        self.entropy = bool(params.get("entropy", 0))
        self.rho_prev = None                   # density of the previous pass (entropy variant)

    def _derivatives(self):
        """Steps 1, 2, 4a: density, prediction, forces and the new global dt."""
        d, o, c = self.d, self.out, self.ctx
        c.build_cells(d["x"], d["y"], d["z"], d["h"])
        c.density_h(d["m"], d["h"], o["rho"], o["omega"], o["n_ngb"])
        if self.entropy:
            if self.rho_prev is None:
                self.rho_prev = torch.empty_like(o["rho"])
            else:
                c.isentropic_u(self.rho_prev, o["rho"], d["u"])
            self.rho_prev.copy_(o["rho"])
        p = self.pred
        c.predict(self.dt_prev, 1.0, d["vx"], d["vy"], d["vz"], d["u"], o["ax"], o["ay"], o["az"],
                  o["dudt"], p["vx"], p["vy"], p["vz"], p["u"])
        rho = o["rho"]
        if self.interface_alpha is not None:      # step 3
            c.interface_correction(d["m"], p["u"], o["rho"], d["h"], self.mat, self.interface_alpha,
                                   self.imbalance, self.rho_corr)
            rho = self.rho_corr
        c.forces(d["m"], p["vx"], p["vy"], p["vz"], p["u"], rho, d["h"], o["omega"], o["ax"],
                 o["ay"], o["az"], o["dudt"], o["mu_min"], o["P"], o["c"])
        c.timestep(d["h"], o["c"], o["ax"], o["ay"], o["az"], o["mu_min"], o["dt_i"], self.dt_new)
        # closing kick of the step that ends here (Eqs. 21-22); a no-op before the first step
        c.kick(self.dt_prev, 1.0, d["vx"], d["vy"], d["vz"], d["u"], o["ax"], o["ay"], o["az"],
               o["dudt"])

    def step(self, dt_cap: float | None = None):
        """Advance by one global step dt = min_i dt_i (optionally capped)."""
        d, o, c = self.d, self.out, self.ctx
        self._derivatives()
        if dt_cap is not None:
            self.dt_new.clamp_(max=float(dt_cap))
        c.kick(self.dt_new, 1.0, d["vx"], d["vy"], d["vz"], d["u"], o["ax"], o["ay"], o["az"],
               o["dudt"])                                             # opening kick, Eqs. 23-24
        c.drift(self.dt_new, 1.0, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"])   # Eq. 25
        self.t += self.dt_new.double()
        self.dt_prev.copy_(self.dt_new)
        self.steps += 1

    def synchronise(self):
        """Bring v, u from the half step to the current time (density, forces, closing kick),
        e.g. before measuring energies.  The next step() then starts without a pending kick."""
        self._derivatives()
        self.dt_prev.zero_()

    def run_until(self, t_end: float, max_steps: int = 100000):
        while self.steps < max_steps:
            t = float(self.t.item())
            if t >= t_end * (1.0 - 1e-12):
                break
            self.step(dt_cap=t_end - t)
        self.synchronise()

    def energies(self):
        """Total kinetic and internal energy (FP64 sums on the device)."""
        d = self.d
        m = d["m"].double()
        ek = 0.5 * (m * (d["vx"].double() ** 2 + d["vy"].double() ** 2 + d["vz"].double() ** 2)).sum()
        eu = (m * d["u"].double()).sum()
        return float(ek.item()), float(eu.item())

    def momentum(self):
        d = self.d
        m = d["m"].double()
        return [float((m * d[k].double()).sum().item()) for k in ("vx", "vy", "vz")]


def floor_rung(substep: int, max_rung: int) -> int:
    """Lowest rung whose steps begin at this substep: max_rung minus the number of
    trailing zero bits of substep mod 2^max_rung; 0 at the start of a big step."""
    sub = substep % (1 << max_rung)
    return 0 if sub == 0 else max_rung - ((sub & -sub).bit_length() - 1)


class BlockSimulation(Simulation):
    """Block-time-step driver (reading R32): every particle
    advances with dt0 / 2^rung, rung <= max_rung; time runs in substeps of delta = dt0 / 2^max_rung.

    One substep s, in the paper's order (Figure 2):
      1. density pass for all particles (with `fastgas`, on the substeps that do not start a
         step of rung 0: marking pass, then the density of the marked particles only,
         PAPER.md:276; with the interface correction a second marking pass from the marked
         particles, and the density of the particles with either mark)
                                                            sph_build_cells, sph_mark_neighbors,
                                                            sph_density_h
      2. prediction of v, u of every particle to the time of the substep   sph_block_predict
      3. interface correction (`interface_alpha`; Eqs. 8-12) from the predicted u:
         the corrected density replaces rho in the force pass.  The pass runs over all particles
         (the paper restricts it to the first mark; the values it needs -- of the active
         particles' neighbours -- are the same)             sph_interface_correction
      4. forces of the particles whose step ends now        sph_block_active, sph_set_active,
                                                            sph_forces
         their new desired rungs (Eq. 27 + limiter)         sph_timestep, sph_rungs
         closing kick, rung change, opening kick            sph_block_kick
      5. drift of all particles by delta                    sph_drift
    Plumbing only; nothing is read back to the host inside a substep."""

    def __init__(self, w: dict, dt0: float, max_rung: int, fastgas: float = 0.0, **params):
        """fastgas: 0 / False = off; a fraction in (0, 1] = use the marking pass on a substep when
        the share of particles on its active rungs (rung histogram read once per big step, a
        performance heuristic only: the results do not depend on it) is below it; True = 1."""
        super().__init__(w, **params)
        if not 0 <= int(max_rung) <= 24:
            raise ValueError("max_rung must be in 0..24")
        n = self.n
        self.dt0, self.max_rung = float(np.float32(dt0)), int(max_rung)
        self.delta = float(np.float32(self.dt0 / 2 ** self.max_rung))
        self.delta_dev = torch.full((1,), self.delta, dtype=torch.float32, device="cuda")
        i32 = dict(dtype=torch.int32, device="cuda")
        self.rung = torch.zeros(n, **i32)
        self.rung_des = torch.zeros(n, **i32)
        self.tnext = torch.zeros(n, **i32)
        self.hk = torch.zeros(n, dtype=torch.float32, device="cuda")
        self.active = torch.empty(n, dtype=torch.uint8, device="cuda")
        self.mark = torch.empty(n, dtype=torch.uint8, device="cuda")
        self.mark2 = torch.empty(n, dtype=torch.uint8, device="cuda") if self.interface_alpha is not None else None
        self.fastgas = float(fastgas)
        self.rung_share = None                  # share of particles on rungs >= r, per r
        self.s = 0                              # substep counter (host integer, plumbing)
        self.have_density = False

    def _substep_derivatives(self):
        d, o, c, s = self.d, self.out, self.ctx, self.s
        c.block_active(s, self.tnext, self.active)
        c.build_cells(d["x"], d["y"], d["z"], d["h"])
        sub = s % (1 << self.max_rung)
        full = sub == 0
        use_fastgas = False
        if self.fastgas > 0.0 and self.have_density:
            if full:
                if self.fastgas < 1.0:    # one host read per big step
                    pop = torch.bincount(self.rung, minlength=self.max_rung + 1).double().cpu().numpy()
                    self.rung_share = np.cumsum(pop[::-1])[::-1] / max(pop.sum(), 1.0)
            elif self.fastgas >= 1.0:
                use_fastgas = True
            elif self.rung_share is not None:
                fl = floor_rung(s, self.max_rung)
                use_fastgas = bool(self.rung_share[fl] < self.fastgas)
        if use_fastgas:
            c.mark_neighbors(self.active, self.mark)          # index holds the last pass's h
            if self.interface_alpha is not None:
                # the corrected density of a marked particle needs the densities of ITS
                # neighbours: second marking pass, density for either mark
                c.mark_neighbors(self.mark, self.mark2)
                torch.maximum(self.mark, self.mark2, out=self.mark2)
                c.set_active(self.mark2)
            else:
                c.set_active(self.mark)
        c.density_h(d["m"], d["h"], o["rho"], o["omega"], o["n_ngb"])
        self.have_density = True
        if self.entropy:
            # PAPER.md:197; entries the pass did not update (FastGas) hold the same density in
            # both arrays, so their u stays as it is
            if self.rho_prev is None:
                self.rho_prev = torch.empty_like(o["rho"])
            else:
                c.isentropic_u(self.rho_prev, o["rho"], d["u"])
            self.rho_prev.copy_(o["rho"])
        p = self.pred
        c.block_predict(s, self.delta, self.tnext, self.hk, d["vx"], d["vy"], d["vz"], d["u"],
                        o["ax"], o["ay"], o["az"], o["dudt"], p["vx"], p["vy"], p["vz"], p["u"])
        rho = o["rho"]
        if self.interface_alpha is not None:      # step 3
            c.interface_correction(d["m"], p["u"], o["rho"], d["h"], self.mat, self.interface_alpha,
                                   self.imbalance, self.rho_corr)
            rho = self.rho_corr
        c.set_active(self.active)
        c.forces(d["m"], p["vx"], p["vy"], p["vz"], p["u"], rho, d["h"], o["omega"], o["ax"],
                 o["ay"], o["az"], o["dudt"], o["mu_min"], o["P"], o["c"])
        c.timestep(d["h"], o["c"], o["ax"], o["ay"], o["az"], o["mu_min"], o["dt_i"], self.dt_new)
        c.rungs(o["dt_i"], self.dt0, self.max_rung, self.rung_des)

    def step(self, dt_cap=None):
        """One substep of length delta (dt_cap is ignored: the substep length is fixed)."""
        d, o, c = self.d, self.out, self.ctx
        self._substep_derivatives()
        c.block_kick(self.s, self.max_rung, self.delta, self.rung_des, self.rung, self.tnext,
                     self.hk, d["vx"], d["vy"], d["vz"], d["u"], o["ax"], o["ay"], o["az"],
                     o["dudt"])
        c.drift(self.delta_dev, 1.0, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"])
        self.s += 1
        self.t += self.delta
        self.steps += 1

    def big_step(self):
        """All substeps of one dt0; ends where every particle's step ends."""
        for _ in range(1 << self.max_rung):
            self.step()

    def run_until(self, t_end: float, max_steps: int = 100000):
        """Whole big steps until t >= t_end (the end time is a multiple of dt0), then the
        closing kicks."""
        if self.s % (1 << self.max_rung) != 0:
            raise ValueError("run_until() starts at the end of a big step")
        while self.steps < max_steps and self.s * self.delta < t_end * (1.0 - 1e-12):
            self.big_step()
        self.synchronise()

    def synchronise(self):
        """At the end of a big step (every particle active): density, forces and the closing
        kicks; v, u are then those of the current time and no kick is pending."""
        if self.s % (1 << self.max_rung) != 0:
            raise ValueError("synchronise() needs the end of a big step")
        d, o, c = self.d, self.out, self.ctx
        self._substep_derivatives()
        c.block_kick(self.s, self.max_rung, self.delta, self.rung_des, self.rung, self.tnext,
                     self.hk, d["vx"], d["vy"], d["vz"], d["u"], o["ax"], o["ay"], o["az"],
                     o["dudt"], open=0)
