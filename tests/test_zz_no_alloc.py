"""sph_timestep_static (include/sph.h): the time-step criteria through the entry point that
allocates nothing -- its reduction scratch is a fixed array of the library image -- against
the existing path (sph_timestep of a context) on the outputs of a real density + force step,
two calls in a row with different sizes (the second smaller, so block minima of the first
call are still lying in the scratch behind the ones the second call writes).

Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2511_11425_b200 import workloads

TOL_DT = 1e-6   # the tolerance of the dt checks in test_gpu_parity.py (BASELINE.json north_star)


def _step(gu, w):
    """One density + force + dt step through the context: the inputs and the existing path's results."""
    from paper_2511_11425_b200 import sph
    d = gu.to_device(w)
    ctx = gu.make_ctx(w)
    out = sph.StepBuffers(int(w["n"]))
    h = d["h"].clone()
    sph.step(ctx, d, out, h)
    torch.cuda.synchronize()
    return ctx, out, h


def _outputs(w):
    n = int(w["n"])
    return (torch.full((n,), -1.0, dtype=torch.float32, device="cuda"),
            torch.full((1,), -1.0, dtype=torch.float32, device="cuda"))


def _static(sph, w, out, h, bufs=None):
    dt_i, dt_min = bufs if bufs is not None else _outputs(w)
    sph.timestep_static(h, out["c"], out["ax"], out["ay"], out["az"], out["mu_min"], dt_i, dt_min,
                        eta_cfl=0.3, eta_acc=0.2, av_alpha=float(w["av_alpha"]), av_beta=float(w["av_beta"]))
    torch.cuda.synchronize()
    return dt_i, dt_min


def _compare(out, dt_i, dt_min):
    ref_i, ref_min = out["dt_i"].double().cpu().numpy(), float(out["dt_min"].item())
    got_i = dt_i.double().cpu().numpy()
    assert np.isfinite(got_i).all() and (got_i > 0).all()
    assert (np.abs(got_i - ref_i) <= TOL_DT * ref_i).all()
    assert abs(float(dt_min.item()) - ref_min) <= TOL_DT * ref_min
    assert float(dt_min.item()) == float(dt_i.min().item())


@pytest.mark.gpu
def test_timestep_static_matches_the_context_path_on_two_calls_in_a_row():
    import gpu_util as gu
    from oracle import sph_oracle as orc
    from paper_2511_11425_b200 import sph
    # 64 000 particles = 15.6 blocks of 4096 (ragged tail), random velocities so that mu_min < 0
    w1 = workloads.sedov(nside=40, v_sigma=0.05)
    # 13 824 particles = 3.4 blocks: the scratch still holds twelve minima of the first call
    w2 = workloads.sedov(nside=24, v_sigma=0.2, seed=77)
    ctx1, out1, h1 = _step(gu, w1)
    ctx2, out2, h2 = _step(gu, w2)
    assert float(out2["dt_min"].item()) != float(out1["dt_min"].item())

    dt_i, dt_min = _static(sph, w1, out1, h1)
    _compare(out1, dt_i, dt_min)
    # ... and against the oracle (Eq. 26 in FP64 on the same inputs)
    _, op = gu.make_params(w1)
    odti, _ = orc.timestep(h1.cpu().numpy(), out1["c"].cpu().numpy(), out1["ax"].cpu().numpy(),
                           out1["ay"].cpu().numpy(), out1["az"].cpu().numpy(),
                           out1["mu_min"].cpu().numpy(), op)
    assert (np.abs(dt_i.double().cpu().numpy() - odti) <= TOL_DT * odti).all()

    # second call, straight after the first, smaller: stale scratch must not leak into the minimum;
    # and the call takes no device memory (the kernels were loaded by the first call)
    bufs = _outputs(w2)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    dt_i, dt_min = _static(sph, w2, out2, h2, bufs)
    assert torch.cuda.mem_get_info()[0] == free0
    _compare(out2, dt_i, dt_min)

    # and the first inputs once more
    again_i, again_min = _static(sph, w1, out1, h1)
    _compare(out1, again_i, again_min)
    del ctx1, ctx2


@pytest.mark.gpu
def test_timestep_static_rejects_sizes_beyond_the_scratch_and_bad_arguments():
    from paper_2511_11425_b200 import sph
    lib = sph.load()
    t = [torch.ones(64, dtype=torch.float32, device="cuda") for _ in range(8)]
    ptr = [C.c_void_p(x.data_ptr()) for x in t]
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = lib.sph_timestep_static(stream, sph.STATIC_MAX_N + 1, 0.3, 0.2, 1.0, 2.0, *ptr)
    assert rc == sph.SPH_EINVAL
    msg = lib.sph_static_last_error().decode()
    assert str(sph.STATIC_MAX_N) in msg and "sph_timestep" in msg
    assert lib.sph_timestep_static(stream, 0, 0.3, 0.2, 1.0, 2.0, *ptr) == sph.SPH_EINVAL
    assert lib.sph_timestep_static(stream, 64, 0.0, 0.2, 1.0, 2.0, *ptr) == sph.SPH_EINVAL
    assert lib.sph_timestep_static(stream, 64, 0.3, 0.2, 1.0, 2.0, *ptr[:7], None) == sph.SPH_EINVAL
    torch.cuda.synchronize()
    for x in t:                      # nothing was launched: the arrays are untouched
        assert bool((x == 1.0).all())
    # the binding refuses tensors of the wrong length before the library is called
    with pytest.raises(sph.SphError):
        sph.timestep_static(t[0], t[1], t[2], t[3], t[4], t[5], t[6][:32].contiguous(), t[7][:1].contiguous())
    # a valid call afterwards still works (n = 64: one partial block)
    sph.timestep_static(*t[:7], t[7][:1].contiguous())
    torch.cuda.synchronize()
    assert bool((t[6] > 0).all())
