"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/sph.h declares; argument checks that need no device; the multi-rank reference arm."""
import ctypes as C
import json
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2511_11425_b200 import build, sph
    build.build()
    return sph.load()


def test_header_and_binding_name_the_same_symbols():
    from paper_2511_11425_b200 import sph
    assert _header_symbols() == sorted(sph.SYMBOLS)
    for name in ("sph_build_cells", "sph_density_h", "sph_forces", "sph_timestep"):
        assert name in sph.SYMBOLS      # the four calls BASELINE.json north_star fixes


def test_library_exports_every_declared_symbol(lib):
    for name in _header_symbols():
        assert hasattr(lib, name), name


def test_library_is_sm_100a_only():
    from paper_2511_11425_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_error_strings_and_null_checks_without_a_device(lib):
    assert lib.sph_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert lib.sph_strerror(code) not in (b"", b"unknown error")
    assert lib.sph_strerror(-99) == b"unknown error"
    # null context / null arguments are rejected before any CUDA call
    assert lib.sph_build_cells(None, 10, None, None, None, None) == -1
    assert lib.sph_density_h(None, None, None, None, None, None) == -1
    assert lib.sph_create(None, None, None, 10, None) == -1
    assert lib.sph_fp32_peak(None, C.c_float(1.0), None) == -1
    assert lib.sph_isentropic_u(None, 10, None, None, None) == -1
    assert lib.sph_block_predict(None, 10, 0, C.c_float(0.1), *([None] * 14)) == -1
    assert lib.sph_block_active(None, 10, 0, None, None) == -1
    assert lib.sph_block_kick(None, 10, 0, 3, C.c_float(0.1), *([None] * 12), 1) == -1


def test_binding_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_2511_11425_b200 import sph
    with pytest.raises(sph.SphError):
        sph.Sph(sph.Params(), sph.Box(), 16)
    with pytest.raises(sph.SphError):
        sph.fp32_peak(0.1)


def test_product_path_does_not_import_the_oracle():
    """Only tests/, __graft_entry__.smoke() and bench.py's baseline legs may touch oracle/."""
    pkg = os.path.join(ROOT, "paper_2511_11425_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "sph_oracle" not in txt and "liboracle" not in txt, f


def test_reference_arm_two_ranks_rank0_prints_one_line():
    """N > 1 path of `bench.py --impl reference`: launched like the driver does (torchrun,
    127.0.0.1), rank 0 alone runs the oracle sample and prints the JSON line."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731", os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--ref-nside", "12"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_replica_aggregation_gloo_world_size_2():
    """The only cross-rank step of bench.py: barrier, MAX of the per-rank time, summed work."""
    code = r'''
import os, torch, torch.distributed as dist
dist.init_process_group("gloo")
r = dist.get_rank()
t = torch.tensor([10.0 + 5.0 * r], dtype=torch.float64)
dist.barrier()
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.item() == 15.0
if r == 0:
    print("VALUE", dist.get_world_size() * 100.0 / t.item())
dist.destroy_process_group()
'''
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29732", "-c", code]
    # torchrun has no -c: write the snippet next to the test run
    path = os.path.join(ROOT, ".pytest_cache", "gloo_snippet.py")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    open(path, "w").write(code)
    cmd = cmd[:-2] + [path]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "VALUE 13.33" in r.stdout


def test_driver_floor_rung_matches_the_oracle():
    """Host logic of the block-step driver (which rungs a substep serves, for the FastGas
    threshold) against the oracle's loop, all substeps of three big steps, R = 0..6."""
    from oracle import sph_oracle as orc
    from paper_2511_11425_b200.integrate import floor_rung
    for R in range(7):
        for s in range(3 * 2 ** R + 1):
            assert floor_rung(s, R) == orc.block_floor_rung(s % 2 ** R, R) == orc.block_floor_rung(s, R)
