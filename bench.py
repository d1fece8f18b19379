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
KERNELS_PER_STEP = 12 + 5 + 7 + 2   # build_cells, density_h, forces, timestep kernel launches
# algorithmic FLOPs: per accepted density pair and Newton
# sweep 27; per force pair 50 (AV branch not taken) or 70 (taken)
FLOP_DENS, FLOP_FORCE, FLOP_FORCE_AV = 27.0, 50.0, 70.0
# What ncu measured on the dominant kernels (DRAM bytes per launch, executed FP32 lane-operations)
# lives in profiles/ncu_current.json together with a hash of the CUDA sources it was taken at;
# the numbers are printed only while that hash matches the sources that run (else null + stale).
NCU_JSON = os.path.join(ROOT, "profiles", "ncu_current.json")
NCU_KERNEL_OF_CALL = {"density_h": "k_density_tile", "forces": "k_forces_list"}


def csrc_hash():
    """sha256 over the CUDA sources and the C header, in name order."""
    import hashlib
    d = os.path.join(ROOT, "paper_2511_11425_b200", "csrc")
    hh = hashlib.sha256()
    for f in sorted(os.listdir(d)) + ["../../include/sph.h"]:
        with open(os.path.join(d, f), "rb") as fh:
            hh.update(f.encode() + b"\0" + fh.read())
    return hh.hexdigest()[:16]


def ncu_numbers(call):
    """(traffic bytes per launch, executed FP32 fraction, stale) of the kernel behind a call."""
    try:
        with open(NCU_JSON) as fh:
            j = json.load(fh)
    except Exception:
        return None, None, None
    k = j.get("kernels", {}).get(NCU_KERNEL_OF_CALL.get(call, ""), None)
    if k is None:
        return None, None, None
    if j.get("csrc_hash") != csrc_hash():
        return None, None, True
    return k.get("dram_bytes"), k.get("executed_fp32_frac"), False


def write_ncu_json(paths):
    """--ncu-raw-csv: turns `ncu -i rep --page raw --csv` dumps (one launch each) into
    profiles/ncu_current.json, stamped with the hash of the sources as they are now."""
    import csv
    out = dict(csrc_hash=csrc_hash(), workload="sedov_128^3", kernels={},
               note="per launch; executed_fp32_frac = (fadd + fmul + 2 ffma predicated-on thread "
                    "instructions per elapsed cycle, as ncu counts them) / (148 x 128 x 2)")
    for path in paths:
        rows = list(csv.reader(open(path)))
        hdr, val = rows[0], rows[2]
        g = lambda k: float(val[hdr.index(k)].replace(",", "")) if k in hdr else 0.0
        name = val[hdr.index("Kernel Name")]
        short = [k for k in NCU_KERNEL_OF_CALL.values() if k in name]
        if not short:
            continue
        cyc = 1.0   # the --set full page gives the counters per elapsed cycle, summed over the chip
        fl = (g("smsp__sass_thread_inst_executed_op_fadd_pred_on.sum.per_cycle_elapsed") +
              g("smsp__sass_thread_inst_executed_op_fmul_pred_on.sum.per_cycle_elapsed") +
              2.0 * g("smsp__sass_thread_inst_executed_op_ffma_pred_on.sum.per_cycle_elapsed"))
        unit = {"Mbyte": 1e6, "Gbyte": 1e9, "Kbyte": 1e3, "byte": 1.0}
        u = lambda k: unit.get(rows[1][hdr.index(k)], 1.0)
        out["kernels"][short[0]] = dict(
            dram_bytes=g("dram__bytes_read.sum") * u("dram__bytes_read.sum") +
                       g("dram__bytes_write.sum") * u("dram__bytes_write.sum"),
            executed_fp32_frac=fl / (cyc * 148 * 128 * 2) if cyc else None,
            duration_ms=g("gpu__time_duration.sum") * {"ms": 1.0, "us": 1e-3, "ns": 1e-6}.get(
                rows[1][hdr.index("gpu__time_duration.sum")], 1.0),
            issue_active_pct=g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
            warp_inst=g("smsp__inst_executed.sum"),
            registers=g("launch__registers_per_thread"))
    with open(NCU_JSON, "w") as fh:
        json.dump(out, fh, indent=1)
    print(json.dumps(out))


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
    ap.add_argument("--no-cpu-legs", dest="cpu_legs", action="store_false",
                    help="skip the oracle legs of BASELINE.md section 3 (brute force on C1 with 1 "
                         "and all threads, cell list with 1 thread: 15 s)")
    ap.add_argument("--ncu-raw-csv", nargs="+", default=None,
                    help="write profiles/ncu_current.json from `ncu --page raw --csv` dumps and exit")
    ap.add_argument("--workload", default="sedov", choices=sorted(workloads_names()),
                    help="sedov (BASELINE.json's metric configuration, the default) or another of "
                         "the five configurations at its full size, for the per-configuration table")
    ap.add_argument("--slack", type=float, default=0.0, help="sph_params.search_slack (0: default)")
    ap.add_argument("--cell-div-x", type=float, default=0.0, help="sph_params.cell_div_x (0: default)")
    ap.add_argument("--cell-div-yz", type=float, default=0.0, help="sph_params.cell_div_yz (0: default)")
    ap.add_argument("--tile", type=int, default=0, help="sph_params.tile (-1: 8-lane kernels only)")
    ap.add_argument("--tile-rows", type=int, default=0, help="sph_params.tile_rows (0: default)")
    ap.add_argument("--tile-cap", type=int, default=0, help="sph_params.tile_cap (0: default)")
    ap.add_argument("--tile-cap2", type=int, default=0, help="sph_params.tile_cap2 (0: default; 1: no second pass)")
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


def oracle_legs():
    """The other oracle timings BASELINE.md section 3 lists, each in a subprocess so that the
    thread count (OMP_NUM_THREADS) can differ: brute force O(N^2) on C1 (4096 particles) with one
    and with all threads, the cell-list oracle on a 40^3 Sedov lattice with one thread."""
    code = (
        "import sys, json, time, numpy as np\n"
        "sys.path.insert(0, %r)\n"
        "from oracle import sph_oracle as orc\n"
        "from paper_2511_11425_b200 import workloads\n"
        "orc.build()\n"
        "kind = sys.argv[1]\n"
        "w = workloads.uniform_cube() if kind == 'brute' else workloads.sedov(nside=40)\n"
        "op = orc.Params(gamma=float(np.float32(w['gamma'])), av_alpha=w['av_alpha'], av_beta=w['av_beta'])\n"
        "ob = orc.Box(w['box_lo'], w['box_len'], w['periodic'])\n"
        "c = kind != 'brute'\n"
        "t0 = time.perf_counter()\n"
        "h, rho, om, nn = orc.density(w['x'], w['y'], w['z'], w['m'], w['h'], ob, op, cells=c)\n"
        "o = orc.forces(w['x'], w['y'], w['z'], w['m'], w['vx'], w['vy'], w['vz'], w['u'], rho, h, om, ob, op, cells=c)\n"
        "dt = time.perf_counter() - t0\n"
        "print(json.dumps(dict(value=(int(nn.sum()) + int(o['n_pairs'].sum())) / dt, unit='interactions/s',\n"
        "      cores=orc.num_threads(), seconds=dt, n=int(w['n']))))\n") % ROOT
    legs = {}
    for name, kind, threads in (("brute_force_c1_1_thread", "brute", "1"), ("brute_force_c1_all_threads", "brute", None),
                                ("cell_list_sedov40_1_thread", "fast", "1")):
        env = dict(os.environ)
        if threads:
            env["OMP_NUM_THREADS"] = threads
        else:
            env.pop("OMP_NUM_THREADS", None)
        try:
            r = subprocess.run([sys.executable, "-c", code, kind], env=env, capture_output=True, text=True,
                               timeout=300)
            legs[name] = json.loads(r.stdout.strip().splitlines()[-1])
        except Exception as e:   # a leg that cannot run is reported, not fatal
            legs[name] = dict(error=str(e)[:200])
    return legs


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
                             tile_cap=a.tile_cap, tile_cap2=a.tile_cap2, tile_warps=a.tile_warps,
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
        # ... perturbed by +-2 % like the generators' warm guess
        gen = torch.Generator(device="cuda").manual_seed(20251111)
        d["h"] *= 0.98 + 0.04 * torch.rand(n, device="cuda", generator=gen)
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

    # ---- the same steps with random velocities (Sedov variant C3v of SURVEY.md 8(d)): half of the
    # pairs are approaching and take the viscosity of Eqs. (15)-(18); reported beside the headline
    av_line = None
    if a.workload == "sedov" and a.v_sigma == 0.0 and not custom:
        gsd = torch.Generator(device="cuda").manual_seed(114253)
        keep = {k: d[k].clone() for k in ("vx", "vy", "vz")}
        for k in keep:
            d[k].normal_(0.0, 0.01, generator=gsd)
        one_step(); one_step()
        ctx.stats_reset()
        ev2 = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(a.steps)]
        for k in range(a.steps):
            one_step(ev2[k])
            flush.fill_(k & 0xff)
        torch.cuda.synchronize()
        st2 = ctx.stats()
        per2 = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in ev2]).mean(axis=0)
        av_line = dict(workload=wname + "_v (v ~ N(0, 0.01))", ms_per_step=float(per2.sum()),
                       ms_forces=float(per2[2]), force_av_pairs=st2["force_av_pairs"] / a.steps,
                       force_pairs=st2["force_pairs"] / a.steps,
                       value=(st2["dens_pairs"] + st2["force_pairs"]) / a.steps / (float(per2.sum()) * 1e-3))
        for k in keep:
            d[k].copy_(keep[k])
        one_step()
        ctx.stats_reset()

    # ---- end to end: host (pinned) inputs in, all outputs back, every step ----------------
    outs_host = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.t.items()}
    h_host = torch.empty(n, dtype=torch.float32).pin_memory()
    h2d = sum(host[k].numel() * 4 for k in keys)
    d2h = sum(v.numel() * v.element_size() for v in outs_host.values()) + n * 4
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # The copies of step k+1 (host -> device) and of step k-1 (device -> host) overlap the
    # kernels of step k: two sets of device buffers, one copy stream per direction, events
    # between them.  Every step still moves all of its inputs in and all of its results out.
    # Inside a step the copies are ordered by need: positions, h and m arrive first (index and
    # density sweep start while v and u are still on their way), and the density sweep's results
    # leave while the force sweep runs -- which shortens what the first and the last step of the
    # timed region cannot overlap with anything.
    main = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    din = [d, {k: torch.empty_like(d[k]) for k in keys}]
    dout = [out, sph.StepBuffers(n)]
    dh = [h, torch.empty_like(h)]
    keys_a, keys_b = ("x", "y", "z", "h", "m"), ("vx", "vy", "vz", "u")
    outs_a = ("rho", "omega", "n_ngb")
    assert set(keys_a + keys_b) == set(keys)
    ev_in_a = [torch.cuda.Event() for _ in range(2)]
    ev_in_b = [torch.cuda.Event() for _ in range(2)]
    ev_dens = [torch.cuda.Event() for _ in range(2)]
    ev_comp = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def e2e_step(k):
        b = k & 1
        w_, o_, h_ = din[b], dout[b], dh[b]
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_comp[b])          # step k-2 no longer reads this input set
            for key in keys_a:
                w_[key].copy_(host[key], non_blocking=True)
            ev_in_a[b].record(s_in)
            for key in keys_b:
                w_[key].copy_(host[key], non_blocking=True)
            ev_in_b[b].record(s_in)
        main.wait_event(ev_in_a[b])
        main.wait_event(ev_out[b])               # step k-2's results have left this output set
        h_.copy_(w_["h"])
        ctx.build_cells(w_["x"], w_["y"], w_["z"], h_)
        ctx.density_h(w_["m"], h_, o_["rho"], o_["omega"], o_["n_ngb"])
        ev_dens[b].record(main)
        main.wait_event(ev_in_b[b])
        ctx.forces(w_["m"], w_["vx"], w_["vy"], w_["vz"], w_["u"], o_["rho"], h_, o_["omega"],
                   o_["ax"], o_["ay"], o_["az"], o_["dudt"], o_["mu_min"], o_["P"], o_["c"])
        ctx.timestep(h_, o_["c"], o_["ax"], o_["ay"], o_["az"], o_["mu_min"], o_["dt_i"], o_["dt_min"])
        ev_comp[b].record(main)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_dens[b])         # h, rho, Omega, n_i are final (the force sweep only reads them)
            h_host.copy_(h_, non_blocking=True)
            for key in outs_a:
                outs_host[key].copy_(o_[key], non_blocking=True)
            s_out.wait_event(ev_comp[b])
            for key, v in o_.t.items():
                if key not in outs_a:
                    outs_host[key].copy_(v, non_blocking=True)
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
    default_cfg = wname == "sedov_128^3" and not custom
    traffic, exe_frac, stale = ncu_numbers(names[dom]) if default_cfg else (None, None, None)
    frac_of = lambda fl, ms: fl / (ms * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=max(a.warmup, 3),
        ms_per_step=float(step_ms.mean()), higher_is_better=True, scaling="weak",
        vs_baseline=None, dtype="f32", data="synthetic",
        config=dict(workload=wname,
                    n_particles=n, kernel=a.kernel, n_ngb=a.n_ngb if custom else 64,
                    h_start="converged h of an untimed pass x U(0.98, 1.02); FLOP model of the roofline is "
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
                      traffic=traffic,
                      traffic_source="profiles/ncu_current.json (ncu --set full, dram bytes per launch of "
                                     + NCU_KERNEL_OF_CALL.get(names[dom], "-") + "; null when the CUDA "
                                     "sources changed since the capture)",
                      ncu_stale=stale,
                      peak_source="derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz",
                      measured_fma_peak=fma_peak, frac_of_measured_fma=ach / fma_peak,
                      useful_frac=ach / NOMINAL_FP32_TFLOPS,
                      executed_fp32_frac=exe_frac,
                      algorithmic_flops_per_launch=dom_flops,
                      frac_density_h=frac_of(f_dens, call_ms[1]), frac_forces=frac_of(f_force, call_ms[2]),
                      step_frac=(f_dens + f_force) / (float(step_ms.mean()) * 1e-3) / 1e12 /
                                NOMINAL_FP32_TFLOPS),
        e2e=dict(value=e2e_val, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                 ms_per_step=float(e2e_ms.item()) / K,
                 overlap="copies of steps k+1 / k-1 overlap the kernels of step k (two device "
                         "buffer sets, one copy stream per direction); inside a step x, y, z, h, m "
                         "arrive before v, u and the density results leave during the force sweep"),
        gpu_launches=KERNELS_PER_STEP * K, clocks=clocks)
    if av_line:
        line["av_variant"] = av_line
    if world == 1 and not a.no_cpu_baseline and not custom:   # the oracle sample is wendland_c2 / 64
        cb = oracle_sample(a.ref_nside, a.v_sigma)
        for k in ("seconds", "n"):
            cb.pop(k, None)
        line["cpu_baseline"] = cb
        if a.cpu_legs:
            line["cpu_baseline_legs"] = oracle_legs()
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    args = parse()
    if args.ncu_raw_csv:
        write_ncu_json(args.ncu_raw_csv)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)
