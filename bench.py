#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

A "step" is one pass of the whole hot path over one batch of synthetic input:
    sph_build_cells -> sph_density_h -> sph_forces -> sph_timestep
on the 128^3 Sedov-Taylor workload (BASELINE.json configs[2], the one north_star's target is
quoted on).  `value` = particle-neighbour interactions per second (density pairs at the final
h, counted once, plus force pairs), whole job; `particles_per_s` beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives), so each rank
runs an independent replica and the values add up ("replicas only", weak scaling).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-neighbour interactions/sec per density+force step"
UNIT = "interactions/s"
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x FP32 lanes x 2 (FMA) x max clock
KERNELS_PER_STEP = 11 + 3 + 6 + 2   # build_cells, density_h, forces, timestep kernel launches
# algorithmic FLOPs: per accepted density pair and Newton
# sweep 27; per force pair 50 (AV branch not taken) or 70 (taken)
FLOP_DENS, FLOP_FORCE, FLOP_FORCE_AV = 27.0, 50.0, 70.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch on sedov_128^3, from the ncu --set full
# capture summarised in profiles/r1h_density_forces.md (k_density / k_forces)
NCU_DRAM_BYTES = {"density_h": 158.0e6 + 783.7e6, "forces": 941.9e6 + 43.6e6}
# executed FP32 lane-operations per cycle (fadd + fmul + 2 ffma, predicated-on threads) over the
# 148 x 128 x 2 the chip can retire, same capture: what the kernel executes, rejected candidates,
# culling and Taylor/Halley bookkeeping included -- printed beside the useful (reject-free) fraction
NCU_EXECUTED_FP32_FRAC = {"density_h": (1013.1 + 1190.0 + 2 * 1101.9) / (148 * 128 * 2),
                          "forces": (783.6 + 1742.4 + 2 * 1495.4) / (148 * 128 * 2)}

KERNEL_IDS = {"cubic_spline": 0, "wendland_c2": 1, "wendland_c4": 2, "wendland_c6": 3}


def workloads_names():
    from paper_2511_11425_b200 import workloads
    return workloads.CONFIGS.keys()


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--nside", type=int, default=int(os.environ.get("BENCH_NSIDE", "128")))
    ap.add_argument("--ref-nside", type=int, default=96,
                    help="lattice side of the bounded sample the CPU oracle is timed on")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="sedov", choices=sorted(workloads_names()),
                    help="sedov (BASELINE.json's metric configuration, the default) or another of "
                         "the five configurations at its full size, for the per-configuration table")
    ap.add_argument("--slack", type=float, default=0.0, help="sph_params.search_slack (0: default)")
    ap.add_argument("--cell-div-x", type=float, default=0.0, help="sph_params.cell_div_x (0: default)")
    ap.add_argument("--cell-div-yz", type=float, default=0.0, help="sph_params.cell_div_yz (0: default)")
    ap.add_argument("--tile", type=int, default=0, help="sph_params.tile (-1: 8-lane kernels only)")
    ap.add_argument("--tile-rows", type=int, default=0, help="sph_params.tile_rows (0: default)")
    ap.add_argument("--tile-cap", type=int, default=0, help="sph_params.tile_cap (0: default)")
    ap.add_argument("--tile-warps", type=int, default=0, help="sph_params.tile_warps (0: default)")
    ap.add_argument("--tile-forces", type=int, default=0, help="sph_params.tile_forces (1: force sweep on staged tiles)")
    ap.add_argument("--tile-fcap", type=int, default=0, help="sph_params.tile_fcap (0: default)")
    ap.add_argument("--tile-fwarps", type=int, default=0, help="sph_params.tile_fwarps (0: default)")
    ap.add_argument("--kernel", default="wendland_c2", choices=list(KERNEL_IDS),
                    help="SPH kernel (sph_params.kernel); the metric configuration is wendland_c2")
    ap.add_argument("--n-ngb", type=float, default=64.0,
                    help="neighbour number of Eq. (6); the metric configuration is 64 "
                         "(PAPER.md:297 uses wendland_c6 with 400)")
    ap.add_argument("--v-sigma", type=float, default=0.0,
                    help="> 0: Sedov variant with random velocities (AV branch exercised)")
    return ap.parse_args()


def oracle_sample(nside, v_sigma=0.0):
    """Times the FP64 cell-list oracle, as it stands, on a Sedov lattice of side `nside`."""
    from oracle import sph_oracle as orc
    from paper_2511_11425_b200 import workloads
    orc.build()
    w = workloads.sedov(nside=nside, v_sigma=v_sigma)
    op = orc.Params(gamma=float(np.float32(w["gamma"])), av_alpha=w["av_alpha"], av_beta=w["av_beta"])
    ob = orc.Box(w["box_lo"], w["box_len"], w["periodic"])
    t0 = time.perf_counter()
    h, rho, om, nn = orc.density(w["x"], w["y"], w["z"], w["m"], w["h"], ob, op, cells=True)
    o = orc.forces(w["x"], w["y"], w["z"], w["m"], w["vx"], w["vy"], w["vz"], w["u"], rho, h, om,
                   ob, op, cells=True)
    P, c = orc.eos(rho, w["u"], op.gamma)
    orc.timestep(h, c, o["ax"], o["ay"], o["az"], o["mu_min"], op)
    dt = time.perf_counter() - t0
    inter = int(nn.sum()) + int(o["n_pairs"].sum())
    return dict(value=inter / dt, unit=UNIT, cores=orc.num_threads(), kind="oracle",
                sample=f"sedov {nside}^3 = {w['n']} particles, one density+force+dt pass, "
                       f"FP64 cell-list oracle (oracle/sph_oracle.c), {dt:.2f} s",
                particles_per_s=w["n"] / dt, seconds=dt, n=int(w["n"]))


def run_reference(a):
    """--impl reference: the oracle on the host cores, same metric, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    res = []
    for _ in range(max(a.warmup, 0)):
        oracle_sample(min(a.ref_nside, 32), a.v_sigma)
    for _ in range(max(a.steps, 1)):
        res.append(oracle_sample(a.ref_nside, a.v_sigma))
    tot_t = sum(r["seconds"] for r in res)
    val = sum(r["value"] * r["seconds"] for r in res) / tot_t
    cb = dict(res[-1])
    cb["value"] = val
    for k in ("seconds", "n", "particles_per_s"):
        cb.pop(k, None)
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=a.gpus,
                steps=len(res), warmup=a.warmup, ms_per_step=1e3 * tot_t / len(res),
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic",
                config=dict(workload=f"sedov_{a.nside}^3 (bounded sample: sedov {a.ref_nside}^3 "
                                     f"per step)", kernel="wendland_c2", n_ngb=64),
                particles_per_s=res[-1]["n"] * len(res) / tot_t, cpu_baseline=cb,
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line), flush=True)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            c = [s.strip() for s in ln.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)),
                       power_w_max=float(max(pw)), reasons=sorted(reasons), samples=len(sm))
        return out


def run_gpu(a):
    import torch
    import torch.distributed as dist
    from paper_2511_11425_b200 import build as sph_build, sph, workloads

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the SPH path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        sph_build.build()          # no-op when libsph_b200.so is up to date
    if world > 1:
        dist.barrier()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- synthetic input (seeded; every rank its own replica of the same workload) --------
    if a.workload == "sedov":
        w = workloads.sedov(nside=a.nside, v_sigma=a.v_sigma, h_start="warm")
        wname = f"sedov_{a.nside}^3" + ("_v" if a.v_sigma > 0 else "")
    else:
        w = workloads.make(a.workload, h_start="warm")
        wname = a.workload
    n = int(w["n"])
    keys = ("x", "y", "z", "m", "vx", "vy", "vz", "u", "h")
    host = {k: torch.from_numpy(w[k]).pin_memory() for k in keys}
    d = {k: host[k].cuda() for k in keys}
    custom = a.kernel != "wendland_c2" or a.n_ngb != 64.0
    ctx = sph.Sph(sph.Params(kernel=KERNEL_IDS[a.kernel], n_ngb=a.n_ngb, gamma=w["gamma"],
                             av_alpha=w["av_alpha"], av_beta=w["av_beta"], search_slack=a.slack, cell_div_x=a.cell_div_x,
                             cell_div_yz=a.cell_div_yz, tile=a.tile, tile_rows=a.tile_rows,
                             tile_cap=a.tile_cap, tile_warps=a.tile_warps,
                             tile_forces=a.tile_forces,
                             tile_fcap=a.tile_fcap, tile_fwarps=a.tile_fwarps),
                  sph.Box(w["box_lo"], w["box_len"], w["periodic"]), n)
    out = sph.StepBuffers(n)
    h = torch.empty_like(d["h"])
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB of L2
    if custom:
        # the generators' guess is for wendland_c2 / 64: converge once from the rescaled guess
        # (untimed) and start every step from that solution
        d["h"] *= (a.n_ngb / 64.0) ** (1.0 / 3.0)
        ctx.build_cells(d["x"], d["y"], d["z"], d["h"])
        ctx.density_h(d["m"], d["h"], out["rho"], out["omega"], out["n_ngb"])
        torch.cuda.synchronize()
        host["h"].copy_(d["h"])

    def one_step(ev=None):
        h.copy_(d["h"])                      # every step starts from the same warm guess
        if ev: ev[0].record()
        ctx.build_cells(d["x"], d["y"], d["z"], h)
        if ev: ev[1].record()
        ctx.density_h(d["m"], h, out["rho"], out["omega"], out["n_ngb"])
        if ev: ev[2].record()
        ctx.forces(d["m"], d["vx"], d["vy"], d["vz"], d["u"], out["rho"], h, out["omega"],
                   out["ax"], out["ay"], out["az"], out["dudt"], out["mu_min"], out["P"], out["c"])
        if ev: ev[3].record()
        ctx.timestep(h, out["c"], out["ax"], out["ay"], out["az"], out["mu_min"], out["dt_i"],
                     out["dt_min"])
        if ev: ev[4].record()

    for _ in range(max(a.warmup, 3)):
        one_step()
        flush.fill_(1)
    barrier()
    ctx.stats_reset()
    sampler = ClockSampler(local) if rank == 0 else None
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(a.steps)]
    barrier()
    for k in range(a.steps):
        one_step(evs[k])
        flush.fill_(k & 0xff)                # L2 flush between timed steps, outside the events
    barrier()
    st = ctx.stats()
    per = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in evs])  # ms
    step_ms = per.sum(axis=1)
    total_ms = torch.tensor([float(step_ms.sum())], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_s = float(total_ms.item()) * 1e-3

    # ---- end to end: host (pinned) inputs in, all outputs back, every step ----------------
    outs_host = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.t.items()}
    h_host = torch.empty(n, dtype=torch.float32).pin_memory()
    h2d = sum(host[k].numel() * 4 for k in keys)
    d2h = sum(v.numel() * v.element_size() for v in outs_host.values()) + n * 4
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # The copies of step k+1 (host -> device) and of step k-1 (device -> host) overlap the
    # kernels of step k: two sets of device buffers, one copy stream per direction, events
    # between them.  Every step still moves all of its inputs in and all of its results out.
    main = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    din = [d, {k: torch.empty_like(d[k]) for k in keys}]
    dout = [out, sph.StepBuffers(n)]
    dh = [h, torch.empty_like(h)]
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_comp = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def e2e_step(k):
        b = k & 1
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_comp[b])          # step k-2 no longer reads this input set
            for key in keys:
                din[b][key].copy_(host[key], non_blocking=True)
            ev_in[b].record(s_in)
        main.wait_event(ev_in[b])
        main.wait_event(ev_out[b])               # step k-2's results have left this output set
        dh[b].copy_(din[b]["h"])
        sph.step(ctx, din[b], dout[b], dh[b])
        ev_comp[b].record(main)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_comp[b])
            for key, v in dout[b].t.items():
                outs_host[key].copy_(v, non_blocking=True)
            h_host.copy_(dh[b], non_blocking=True)
            ev_out[b].record(s_out)

    e2e_step(0)
    e2e_step(1)
    barrier()
    e0.record(main)
    s_in.wait_event(e0)
    for k in range(a.steps):
        e2e_step(k)
    main.wait_stream(s_out)
    main.wait_stream(s_in)
    e1.record(main)
    barrier()
    e2e_ms = torch.tensor([e0.elapsed_time(e1)], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    clocks = sampler.stop() if sampler else None
    assert abs(float(outs_host["dt_min"][0]) - float(dout[(a.steps - 1) & 1]["dt_min"].item())) == 0.0

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    K = a.steps
    i_dens, i_force = st["dens_pairs"] / K, st["force_pairs"] / K
    inter = i_dens + i_force
    value = world * inter * K / total_s
    e2e_val = world * inter * K / (float(e2e_ms.item()) * 1e-3)
    sweeps = st["dens_sweeps"] / K / n
    f_dens = FLOP_DENS * i_dens * sweeps
    av = st["force_av_pairs"] / K
    f_force = FLOP_FORCE * (i_force - av) + FLOP_FORCE_AV * av
    call_ms = per.mean(axis=0)
    names = ["build_cells", "density_h", "forces", "timestep"]
    dom = int(np.argmax(call_ms))
    dom_flops = {1: f_dens, 2: f_force}.get(dom, 0.0)
    ach = dom_flops / (call_ms[dom] * 1e-3) / 1e12
    fma_peak = sph.fp32_peak(1.0)
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=max(a.warmup, 3),
        ms_per_step=float(step_ms.mean()), higher_is_better=True, scaling="weak",
        vs_baseline=None, dtype="f32", data="synthetic",
        config=dict(workload=wname,
                    n_particles=n, kernel=a.kernel, n_ngb=a.n_ngb if custom else 64,
                    h_start="converged h of an untimed pass; FLOP model of the roofline is "
                            "wendland_c2's" if custom else "warm +-2%",
                    l2_flush="256 MiB device write between timed steps, outside the events; "
                             "working set ~320 MB > L2",
                    parallelism="replicas only" if world > 1 else "single GPU"),
        particles_per_s=world * n * K / total_s,
        interactions_per_step=dict(density=i_dens, force=i_force),
        ms_per_call={nm: float(v) for nm, v in zip(names, call_ms)},
        ms_per_step_best=float(step_ms.min()),
        stats_per_step={k: v / K for k, v in st.items() if isinstance(v, int) and
                        k not in ("n_cells", "grid_flags")},
        newton_sweeps_per_particle=sweeps, grid_dims=st["grid_dims"],
        roofline=dict(bound="alu", kernel=names[dom], achieved=ach, peak=NOMINAL_FP32_TFLOPS,
                      unit="TFLOP/s", frac=ach / NOMINAL_FP32_TFLOPS,
                      traffic=(NCU_DRAM_BYTES.get(names[dom]) if wname == "sedov_128^3" else None),
                      traffic_source="profiles/r1h_density_forces.md (ncu --set full, bytes per launch)",
                      peak_source="derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz",
                      measured_fma_peak=fma_peak, frac_of_measured_fma=ach / fma_peak,
                      useful_frac=ach / NOMINAL_FP32_TFLOPS,
                      executed_fp32_frac=(NCU_EXECUTED_FP32_FRAC.get(names[dom])
                                          if wname == "sedov_128^3" else None),
                      algorithmic_flops_per_launch=dom_flops,
                      step_frac=(f_dens + f_force) / (float(step_ms.mean()) * 1e-3) / 1e12 /
                                NOMINAL_FP32_TFLOPS),
        e2e=dict(value=e2e_val, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                 ms_per_step=float(e2e_ms.item()) / K,
                 overlap="copies of steps k+1 / k-1 overlap the kernels of step k (two device "
                         "buffer sets, one copy stream per direction)"),
        gpu_launches=KERNELS_PER_STEP * K, clocks=clocks)
    if world == 1 and not a.no_cpu_baseline and not custom:   # the oracle sample is wendland_c2 / 64
        cb = oracle_sample(a.ref_nside, a.v_sigma)
        for k in ("seconds", "n"):
            cb.pop(k, None)
        line["cpu_baseline"] = cb
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)
