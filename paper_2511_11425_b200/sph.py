"""Thin ctypes binding of the C-ABI CUDA library declared in include/sph.h.

Argument marshalling only: every step of the path runs in the library's kernels.  Torch is
used for device memory and the stream.  There is no CPU fallback: if the library is missing
or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SPH_B200_LIB") or os.path.join(_HERE, "libsph_b200.so")

SPH_OK, SPH_EINVAL, SPH_EBOX, SPH_ENOMEM, SPH_ECUDA, SPH_ESTALE, SPH_ENOSPC = 0, -1, -2, -3, -4, -5, -6

# every symbol include/sph.h declares (tests check the library exports exactly these)
SYMBOLS = ["sph_create", "sph_destroy", "sph_build_cells", "sph_density_h", "sph_forces",
           "sph_timestep", "sph_rungs", "sph_set_active", "sph_mark_neighbors",
           "sph_interface_correction", "sph_predict", "sph_kick", "sph_drift", "sph_isentropic_u", "sph_block_predict", "sph_block_active", "sph_block_kick", "sph_neighbors", "sph_stats", "sph_stats_reset", "sph_permutation",
           "sph_fp32_peak", "sph_timestep_static", "sph_static_last_error", "sph_strerror", "sph_last_error"]


class SphError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"sph error {code}: {text}")
        self.code = code


class _Box(C.Structure):
    _fields_ = [("lo", C.c_float * 3), ("len", C.c_float * 3), ("periodic", C.c_int32 * 3)]


class _Params(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("n_ngb", C.c_float), ("gamma", C.c_float),
                ("av_alpha", C.c_float), ("av_beta", C.c_float), ("av_eps", C.c_float),
                ("eta_cfl", C.c_float), ("eta_acc", C.c_float), ("h_tol", C.c_float),
                ("h_max_iter", C.c_int32), ("search_slack", C.c_float),
                ("cell_div_x", C.c_float), ("cell_div_yz", C.c_float), ("entropy", C.c_int32),
                ("tile", C.c_int32), ("tile_rows", C.c_int32), ("tile_cap", C.c_int32),
                ("tile_cap2", C.c_int32), ("tile_warps", C.c_int32), ("tile_forces", C.c_int32), ("tile_fcap", C.c_int32),
                ("tile_fwarps", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in (
        "dens_tested", "dens_listed", "dens_pairs", "dens_sweeps", "dens_recollect",
        "dens_overflow", "dens_nonconv", "dens_recheck", "force_tested", "force_pairs",
        "force_av_pairs", "n_cells", "grid_flags")] + [("reserved", C.c_int64 * 3)]


@dataclass
class Params:
    kernel: int = 1
    n_ngb: float = 64.0
    gamma: float = 5.0 / 3.0
    av_alpha: float = 1.0
    av_beta: float = 2.0
    av_eps: float = 0.01
    eta_cfl: float = 0.3
    eta_acc: float = 0.2
    h_tol: float = 0.0          # 0 -> library default
    h_max_iter: int = 0
    search_slack: float = 0.0
    cell_div_x: float = 0.0
    cell_div_yz: float = 0.0
    entropy: int = 0            # 1: dudt = Eq. (18) only, u advanced by isentropic_u
    tile: int = 0               # -1: staged-tile sweeps off (8-lanes-per-target kernels only)
    tile_rows: int = 0          # 0 -> library default
    tile_cap: int = 0
    tile_cap2: int = 0
    tile_warps: int = 0
    tile_forces: int = 0        # 1: force sweep on staged tiles (default: kept neighbour lists)
    tile_fcap: int = 0          # the force sweep's tile capacity and warps per bucket
    tile_fwarps: int = 0

    def c(self) -> _Params:
        return _Params(self.kernel, self.n_ngb, self.gamma, self.av_alpha, self.av_beta,
                       self.av_eps, self.eta_cfl, self.eta_acc, self.h_tol, self.h_max_iter,
                       self.search_slack, self.cell_div_x, self.cell_div_yz, int(self.entropy),
                       int(self.tile), int(self.tile_rows), int(self.tile_cap), int(self.tile_cap2), int(self.tile_warps),
                       int(self.tile_forces), int(self.tile_fcap), int(self.tile_fwarps))


@dataclass
class Box:
    lo: tuple = (0.0, 0.0, 0.0)
    len: tuple = (1.0, 1.0, 1.0)
    periodic: tuple = (1, 1, 1)

    def c(self) -> _Box:
        b = _Box()
        for d in range(3):
            b.lo[d], b.len[d], b.periodic[d] = float(self.lo[d]), float(self.len[d]), int(self.periodic[d])
        return b


_lib = None


def load():
    """dlopen the library (building it is __graft_entry__.build / python -m ...build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SphError(SPH_EINVAL, f"{LIB_PATH} missing: run `python -m paper_2511_11425_b200.build`")
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, fp = C.c_void_p, C.c_int64, C.c_int32, C.c_void_p  # device pointers as void*
    lib.sph_create.argtypes = [C.POINTER(vp), C.POINTER(_Params), C.POINTER(_Box), i64, vp]
    lib.sph_destroy.argtypes = [vp]
    lib.sph_destroy.restype = None
    lib.sph_build_cells.argtypes = [vp, i64, fp, fp, fp, fp]
    lib.sph_density_h.argtypes = [vp] + [fp] * 5
    lib.sph_forces.argtypes = [vp] + [fp] * 15
    lib.sph_timestep.argtypes = [vp] + [fp] * 8
    lib.sph_rungs.argtypes = [vp, fp, C.c_float, i32, fp]
    lib.sph_interface_correction.argtypes = [vp] + [fp] * 5 + [C.c_float] + [fp] * 3
    lib.sph_predict.argtypes = [vp, i64, fp, C.c_float] + [fp] * 12
    lib.sph_kick.argtypes = [vp, i64, fp, C.c_float] + [fp] * 8
    lib.sph_drift.argtypes = [vp, i64, fp, C.c_float] + [fp] * 6
    lib.sph_isentropic_u.argtypes = [vp, i64, fp, fp, fp]
    lib.sph_block_predict.argtypes = [vp, i64, i32, C.c_float] + [fp] * 14
    lib.sph_block_active.argtypes = [vp, i64, i32, fp, fp]
    lib.sph_block_kick.argtypes = [vp, i64, i32, i32, C.c_float] + [fp] * 12 + [i32]
    lib.sph_set_active.argtypes = [vp, fp]
    lib.sph_mark_neighbors.argtypes = [vp, fp, fp]
    lib.sph_neighbors.argtypes = [vp, fp, i32, fp, fp, i64, C.POINTER(i64)]
    lib.sph_stats.argtypes = [vp, C.POINTER(_Stats)]
    lib.sph_stats_reset.argtypes = [vp]
    lib.sph_permutation.argtypes = [vp, fp]
    lib.sph_fp32_peak.argtypes = [vp, C.c_float, C.POINTER(C.c_double)]
    lib.sph_timestep_static.argtypes = [vp, i64] + [C.c_float] * 4 + [fp] * 8
    lib.sph_static_last_error.argtypes = []
    lib.sph_static_last_error.restype = C.c_char_p
    lib.sph_strerror.argtypes = [C.c_int]
    lib.sph_strerror.restype = C.c_char_p
    lib.sph_last_error.argtypes = [vp]
    lib.sph_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("sph_destroy", "sph_strerror", "sph_last_error", "sph_static_last_error"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ptr(t: torch.Tensor, dtype, n=None):
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise SphError(SPH_EINVAL, f"expected a contiguous CUDA tensor of {dtype}")
    if n is not None and t.numel() != n:
        raise SphError(SPH_EINVAL, f"expected {n} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def fp32_peak(seconds: float = 1.0) -> float:
    """Measured FP32 FMA rate of the current device in TFLOP/s (sph_fp32_peak)."""
    if not torch.cuda.is_available():
        raise SphError(SPH_ECUDA, "no CUDA device")
    out = C.c_double(0.0)
    rc = load().sph_fp32_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), seconds,
                              C.byref(out))
    if rc:
        raise SphError(rc, load().sph_strerror(rc).decode())
    return out.value


STATIC_MAX_N = 16777216   # SPH_STATIC_MAX_N of include/sph.h


def timestep_static(h, c, ax, ay, az, mu_min, dt_i, dt_min, eta_cfl=0.3, eta_acc=0.2,
                    av_alpha=1.0, av_beta=2.0):
    """sph_timestep_static: the time-step criteria without a context and without any allocation
    (scratch in a fixed array of the library image; n <= STATIC_MAX_N).  Enqueued on torch's
    current stream of the current device."""
    if not torch.cuda.is_available():
        raise SphError(SPH_ECUDA, "no CUDA device: the SPH path has no CPU fallback")
    lib, n, f = load(), int(h.numel()), torch.float32
    args = [_ptr(t, f, n) for t in (h, c, ax, ay, az, mu_min, dt_i)] + [_ptr(dt_min, f, 1)]
    rc = lib.sph_timestep_static(C.c_void_p(torch.cuda.current_stream().cuda_stream), n,
                                 float(eta_cfl), float(eta_acc), float(av_alpha), float(av_beta), *args)
    if rc:
        raise SphError(rc, lib.sph_static_last_error().decode())


class Sph:
    """One sph_ctx.  All tensors: CUDA, contiguous, length n, caller order."""

    def __init__(self, params: Params, box: Box, n_max: int, stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise SphError(SPH_ECUDA, "no CUDA device: the SPH path has no CPU fallback")
        self.lib = load()
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.n_max = int(n_max)
        self.n = 0
        self._ctx = C.c_void_p()
        p, b = params.c(), box.c()
        rc = self.lib.sph_create(C.byref(self._ctx), C.byref(p), C.byref(b), self.n_max,
                                 C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise SphError(rc, self.lib.sph_strerror(rc).decode())

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.sph_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc:
            raise SphError(rc, self.lib.sph_last_error(self._ctx).decode() or
                           self.lib.sph_strerror(rc).decode())

    # ---- the four calls of the hot path -------------------------------------------------
    def build_cells(self, x, y, z, h):
        n = x.numel()
        f = torch.float32
        self._check(self.lib.sph_build_cells(self._ctx, n, _ptr(x, f, n), _ptr(y, f, n),
                                             _ptr(z, f, n), _ptr(h, f, n)))
        self.n = n

    def density_h(self, m, h_inout, rho, omega, n_ngb):
        n, f = self.n, torch.float32
        self._check(self.lib.sph_density_h(self._ctx, _ptr(m, f, n), _ptr(h_inout, f, n),
                                           _ptr(rho, f, n), _ptr(omega, f, n),
                                           _ptr(n_ngb, torch.int32, n)))

    def forces(self, m, vx, vy, vz, u, rho, h, omega, ax, ay, az, dudt, mu_min, P, c):
        n, f = self.n, torch.float32
        args = [_ptr(t, f, n) for t in (m, vx, vy, vz, u, rho, h, omega, ax, ay, az, dudt,
                                        mu_min, P, c)]
        self._check(self.lib.sph_forces(self._ctx, *args))

    def timestep(self, h, c, ax, ay, az, mu_min, dt_i, dt_min):
        n, f = self.n, torch.float32
        args = [_ptr(t, f, n) for t in (h, c, ax, ay, az, mu_min, dt_i)]
        self._check(self.lib.sph_timestep(self._ctx, *args, _ptr(dt_min, f, 1)))

    # ---- rungs (Eq. 27 + Saitoh-Makino limiter) ------------------------------------------
    def rungs(self, dt_i, dt0, max_rung, rung):
        n = self.n
        self._check(self.lib.sph_rungs(self._ctx, _ptr(dt_i, torch.float32, n), float(dt0),
                                       int(max_rung), _ptr(rung, torch.int32, n)))

    # ---- active set of a rung and the FastGas marking pass --------------
    def set_active(self, active):
        """active: uint8 tensor of n flags (caller order), or None for all particles."""
        ptr = _ptr(active, torch.uint8, self.n) if active is not None else None
        self._check(self.lib.sph_set_active(self._ctx, ptr))

    def mark_neighbors(self, src, mark):
        n = self.n
        self._check(self.lib.sph_mark_neighbors(self._ctx, _ptr(src, torch.uint8, n),
                                                _ptr(mark, torch.uint8, n)))

    # ---- interface correction (Eqs. 8-12) -------------------------------------------------
    def interface_correction(self, m, u, rho, h, mat, alpha, imbalance, rho_corr, P_corr=None):
        n, f = self.n, torch.float32
        self._check(self.lib.sph_interface_correction(
            self._ctx, _ptr(m, f, n), _ptr(u, f, n), _ptr(rho, f, n), _ptr(h, f, n),
            _ptr(mat, torch.int32, n) if mat is not None else None, float(alpha),
            _ptr(imbalance, f, n), _ptr(rho_corr, f, n),
            _ptr(P_corr, f, n) if P_corr is not None else None))

    # ---- time integration (Eqs. 19-25) ----------------------------------------------------
    def predict(self, dt, scale, vx, vy, vz, u, ax, ay, az, dudt, vxp, vyp, vzp, up):
        n, f = vx.numel(), torch.float32
        args = [_ptr(t, f, n) for t in (vx, vy, vz, u, ax, ay, az, dudt, vxp, vyp, vzp, up)]
        self._check(self.lib.sph_predict(self._ctx, n, _ptr(dt, f, 1), scale, *args))

    def kick(self, dt, scale, vx, vy, vz, u, ax, ay, az, dudt):
        n, f = vx.numel(), torch.float32
        args = [_ptr(t, f, n) for t in (vx, vy, vz, u, ax, ay, az, dudt)]
        self._check(self.lib.sph_kick(self._ctx, n, _ptr(dt, f, 1), scale, *args))

    def drift(self, dt, scale, x, y, z, vx, vy, vz):
        n, f = x.numel(), torch.float32
        args = [_ptr(t, f, n) for t in (x, y, z, vx, vy, vz)]
        self._check(self.lib.sph_drift(self._ctx, n, _ptr(dt, f, 1), scale, *args))

    def isentropic_u(self, rho_old, rho_new, u):
        """u *= (rho_new / rho_old)^(gamma-1), in place."""
        n, f = u.numel(), torch.float32
        self._check(self.lib.sph_isentropic_u(self._ctx, n, _ptr(rho_old, f, n), _ptr(rho_new, f, n),
                                              _ptr(u, f, n)))

    # ---- block time steps (reading R32) ----------------------
    def block_predict(self, s, delta, tnext, hk, vx, vy, vz, u, ax, ay, az, dudt, vxp, vyp, vzp, up):
        n, f = vx.numel(), torch.float32
        args = [_ptr(t, f, n) for t in (hk, vx, vy, vz, u, ax, ay, az, dudt, vxp, vyp, vzp, up)]
        self._check(self.lib.sph_block_predict(self._ctx, n, int(s), float(delta),
                                               _ptr(tnext, torch.int32, n), *args))

    def block_active(self, s, tnext, active):
        n = tnext.numel()
        self._check(self.lib.sph_block_active(self._ctx, n, int(s), _ptr(tnext, torch.int32, n),
                                              _ptr(active, torch.uint8, n)))

    def block_kick(self, s, max_rung, delta, rung_des, rung, tnext, hk, vx, vy, vz, u, ax, ay, az,
                   dudt, open=1):
        n, f, i = vx.numel(), torch.float32, torch.int32
        args = [_ptr(t, f, n) for t in (hk, vx, vy, vz, u, ax, ay, az, dudt)]
        self._check(self.lib.sph_block_kick(self._ctx, n, int(s), int(max_rung), float(delta),
                                            _ptr(rung_des, i, n), _ptr(rung, i, n),
                                            _ptr(tnext, i, n), *args, int(open)))

    # ---- diagnostics --------------------------------------------------------------------
    def neighbors(self, h, mode=0):
        """CSR lists (offsets int64[n+1], indices int32) at the prescribed h."""
        n = self.n
        off = torch.empty(n + 1, dtype=torch.int64, device=h.device)
        need = C.c_int64(0)
        self._check(self.lib.sph_neighbors(self._ctx, _ptr(h, torch.float32, n), mode,
                                           _ptr(off, torch.int64), None, 0, C.byref(need)))
        idx = torch.empty(max(need.value, 1), dtype=torch.int32, device=h.device)
        self._check(self.lib.sph_neighbors(self._ctx, _ptr(h, torch.float32, n), mode,
                                           _ptr(off, torch.int64), _ptr(idx, torch.int32),
                                           need.value, C.byref(need)))
        return off, idx[:need.value]

    def stats(self) -> dict:
        s = _Stats()
        self._check(self.lib.sph_stats(self._ctx, C.byref(s)))
        d = {k: int(getattr(s, k)) for k, _ in _Stats._fields_ if k != "reserved"}
        d["grid_dims"] = tuple(int(v) for v in s.reserved)
        return d

    def stats_reset(self):
        self._check(self.lib.sph_stats_reset(self._ctx))

    def permutation(self):
        p = torch.empty(self.n, dtype=torch.int32, device="cuda")
        self._check(self.lib.sph_permutation(self._ctx, _ptr(p, torch.int32, self.n)))
        return p


@dataclass
class StepBuffers:
    """Device arrays of one density + force step, allocated once."""
    n: int
    device: str = "cuda"
    t: dict = field(default_factory=dict)

    def __post_init__(self):
        f = dict(dtype=torch.float32, device=self.device)
        for k in ("rho", "omega", "ax", "ay", "az", "dudt", "mu_min", "P", "c", "dt_i"):
            self.t[k] = torch.empty(self.n, **f)
        self.t["n_ngb"] = torch.empty(self.n, dtype=torch.int32, device=self.device)
        self.t["dt_min"] = torch.empty(1, **f)

    def __getitem__(self, k):
        return self.t[k]


def step(ctx: Sph, w: dict, out: StepBuffers, h: torch.Tensor):
    """One pass of the whole hot path: build_cells -> density_h -> forces -> timestep.
    `w` holds the device tensors x, y, z, m, vx, vy, vz, u; `h` is updated in place."""
    ctx.build_cells(w["x"], w["y"], w["z"], h)
    ctx.density_h(w["m"], h, out["rho"], out["omega"], out["n_ngb"])
    ctx.forces(w["m"], w["vx"], w["vy"], w["vz"], w["u"], out["rho"], h, out["omega"],
               out["ax"], out["ay"], out["az"], out["dudt"], out["mu_min"], out["P"], out["c"])
    ctx.timestep(h, out["c"], out["ax"], out["ay"], out["az"], out["mu_min"], out["dt_i"],
                 out["dt_min"])


class StepGraph:
    """The whole hot path -- build_cells -> density_h -> forces -> timestep, about 26 kernel
    launches and a dozen memsets -- captured once in a CUDA graph and replayed with one launch:
    for problems so small that the launches, not the kernels, set the time of a step (config 1:
    4096 particles).  The context must live on a stream of its own (not the default stream):

        s = torch.cuda.Stream(); ctx = Sph(params, box, n, stream=s)
        g = StepGraph(ctx, w, out, h); g.replay()

    The graph holds the addresses of the tensors it was captured with: `w`, `out` and `h` must stay
    alive and are read / written in place by every replay (h: in the guess, out the solution).
    replay() enqueues on torch's current stream.  Argument marshalling only, like step()."""

    def __init__(self, ctx: Sph, w: dict, out: StepBuffers, h: torch.Tensor, warmup: int = 2):
        if ctx.stream.cuda_stream == torch.cuda.default_stream().cuda_stream:
            raise SphError(SPH_EINVAL, "StepGraph: create the context on a non-default stream")
        self.ctx, self.w, self.out, self.h = ctx, w, out, h
        cur = torch.cuda.current_stream()
        ctx.stream.wait_stream(cur)
        with torch.cuda.stream(ctx.stream):
            h0 = h.clone()
            for _ in range(max(int(warmup), 1)):      # module loading, function attributes
                h.copy_(h0)
                step(ctx, w, out, h)
            h.copy_(h0)
        ctx.stream.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=ctx.stream):
            step(ctx, w, out, h)
        h.copy_(h0)                                    # the capture itself runs nothing

    def replay(self):
        self.graph.replay()
