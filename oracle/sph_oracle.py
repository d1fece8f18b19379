"""ctypes front end of oracle/sph_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this module.  It holds no arithmetic of the method: it promotes the caller's FP32
arrays to FP64 exactly, calls the C functions and hands back numpy arrays.  The equations
and their PAPER.md citations are in sph_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile sph_oracle.c with gcc (OpenMP) into oracle/liboracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Box(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("len", C.c_double * 3), ("periodic", C.c_int32 * 3)]


class _Params(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("n_ngb", C.c_double), ("gamma", C.c_double),
                ("av_alpha", C.c_double), ("av_beta", C.c_double), ("av_eps", C.c_double),
                ("eta_cfl", C.c_double), ("eta_acc", C.c_double), ("entropy", C.c_int32)]


@dataclass
class Params:
    kernel: int = 1          # Wendland C2
    n_ngb: float = 64.0
    gamma: float = 5.0 / 3.0
    av_alpha: float = 1.0
    av_beta: float = 2.0
    av_eps: float = 0.01
    eta_cfl: float = 0.3
    eta_acc: float = 0.2
    entropy: int = 0         # 1: du/dt = Eq. (18) only (reading R31)

    def c(self) -> _Params:
        return _Params(self.kernel, self.n_ngb, self.gamma, self.av_alpha, self.av_beta,
                       self.av_eps, self.eta_cfl, self.eta_acc, int(self.entropy))


@dataclass
class Box:
    lo: tuple = (0.0, 0.0, 0.0)
    len: tuple = (1.0, 1.0, 1.0)
    periodic: tuple = (1, 1, 1)

    def c(self) -> _Box:
        b = _Box()
        for d in range(3):
            # FP32 box values are promoted exactly, like every other input
            b.lo[d] = float(np.float32(self.lo[d]))
            b.len[d] = float(np.float32(self.len[d]))
            b.periodic[d] = int(self.periodic[d])
        return b


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_w.restype = C.c_double
        _lib.orc_w.argtypes = [C.c_int, C.c_double]
        _lib.orc_dw.restype = C.c_double
        _lib.orc_dw.argtypes = [C.c_int, C.c_double]
        _lib.orc_dist2.restype = C.c_double
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _d(a):
    """Exact promotion to a contiguous FP64 array."""
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _p(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _targets(n, targets):
    if targets is None:
        return n, None
    t = np.ascontiguousarray(np.asarray(targets), dtype=np.int64)
    return len(t), t


def w(kernel: int, q: float) -> float:
    return lib().orc_w(int(kernel), float(q))


def dw(kernel: int, q: float) -> float:
    return lib().orc_dw(int(kernel), float(q))


def density(x, y, z, m, h_hint, box: Box, par: Params, targets=None, cells: bool = False,
            cell_side: float | None = None):
    """h (root of Eq. 6), rho (Eq. 5), Omega (Eq. 7), n_i.  Brute force unless cells=True."""
    x, y, z, m, hh = map(_d, (x, y, z, m, h_hint))
    n = len(x)
    b, p = box.c(), par.c()
    if cells:
        assert targets is None
        h = np.empty(n); rho = np.empty(n); om = np.empty(n); nn = np.empty(n, np.int32)
        nfb = C.c_int64(0)
        side = float(cell_side if cell_side is not None else 2.0 * 1.3 * hh.max())
        rc = lib().orc_density_cells(C.c_int64(n), _p(x), _p(y), _p(z), _p(m), _p(hh), C.byref(b),
                                     C.byref(p), C.c_double(side), _p(h), _p(rho), _p(om),
                                     _p(nn, C.c_int32), C.byref(nfb))
        if rc:
            raise RuntimeError(f"orc_density_cells failed: {rc}")
        return h, rho, om, nn
    nt, t = _targets(n, targets)
    h = np.empty(nt); rho = np.empty(nt); om = np.empty(nt); nn = np.empty(nt, np.int32)
    rc = lib().orc_density_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(m), _p(hh), C.byref(b),
                                 C.byref(p), C.c_int64(nt), _p(t, C.c_int64), _p(h), _p(rho),
                                 _p(om), _p(nn, C.c_int32))
    if rc:
        raise RuntimeError(f"orc_density_brute failed: {rc}")
    return h, rho, om, nn


def density_at_h(x, y, z, m, h, box: Box, par: Params, targets=None):
    """rho, Omega, n_i and the relative residual of Eq. (6) at a PRESCRIBED h (brute force)."""
    x, y, z, m, h = map(_d, (x, y, z, m, h))
    n = len(x)
    b, p = box.c(), par.c()
    nt, t = _targets(n, targets)
    rho = np.empty(nt); om = np.empty(nt); nn = np.empty(nt, np.int32); res = np.empty(nt)
    lib().orc_density_at_h_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(m), _p(h), C.byref(b),
                                 C.byref(p), C.c_int64(nt), _p(t, C.c_int64), _p(rho), _p(om),
                                 _p(nn, C.c_int32), _p(res))
    return rho, om, nn, res


def neighbors(x, y, z, h, box: Box, mode: int = 0, targets=None):
    """CSR neighbour lists at a prescribed h. mode 0 gather (self incl.), 1 gather-or-scatter."""
    x, y, z, h = map(_d, (x, y, z, h))
    n = len(x)
    b = box.c()
    nt, t = _targets(n, targets)
    off = np.zeros(nt + 1, np.int64)
    args = [C.c_int64(n), _p(x), _p(y), _p(z), _p(h), C.byref(b), C.c_int(mode), C.c_int64(nt),
            _p(t, C.c_int64), _p(off, C.c_int64)]
    lib().orc_neighbors_brute(*args, None)
    idx = np.empty(int(off[-1]), np.int64)
    lib().orc_neighbors_brute(*args, _p(idx, C.c_int64))
    return off, idx


def forces(x, y, z, m, vx, vy, vz, u, rho, h, omega, box: Box, par: Params, targets=None,
           cells: bool = False):
    """a, du/dt, mu_min and the normalisers Sa, Su (Eqs. 13-18). Returns a dict."""
    arrs = list(map(_d, (x, y, z, m, vx, vy, vz, u, rho, h, omega)))
    n = len(arrs[0])
    b, p = box.c(), par.c()
    nt, t = (n, None) if cells else _targets(n, targets)
    out = {k: np.empty(nt) for k in ("ax", "ay", "az", "dudt", "mu_min", "Sa", "Su")}
    npairs = np.empty(nt, np.int32)
    ptrs = [_p(a) for a in arrs]
    outs = [_p(out[k]) for k in ("ax", "ay", "az", "dudt", "mu_min", "Sa", "Su")]
    if cells:
        assert targets is None
        rc = lib().orc_forces_cells(C.c_int64(n), *ptrs, C.byref(b), C.byref(p),
                                    C.c_double(2.0 * float(arrs[9].max())), *outs,
                                    _p(npairs, C.c_int32))
    else:
        rc = lib().orc_forces_brute(C.c_int64(n), *ptrs, C.byref(b), C.byref(p), C.c_int64(nt),
                                    _p(t, C.c_int64), *outs, _p(npairs, C.c_int32))
    if rc:
        raise RuntimeError(f"orc_forces failed: {rc}")
    out["n_pairs"] = npairs
    return out


def eos(rho, u, gamma):
    rho, u = _d(rho), _d(u)
    P = np.empty_like(rho); c = np.empty_like(rho)
    lib().orc_eos(C.c_int64(len(rho)), _p(rho), _p(u), C.c_double(gamma), _p(P), _p(c))
    return P, c


def timestep(h, c, ax, ay, az, mu_min, par: Params):
    h, c, ax, ay, az, mu = map(_d, (h, c, ax, ay, az, mu_min))
    p = par.c()
    dti = np.empty_like(h)
    dtm = C.c_double(0)
    lib().orc_timestep(C.c_int64(len(h)), _p(h), _p(c), _p(ax), _p(ay), _p(az), _p(mu),
                       C.byref(p), _p(dti), C.byref(dtm))
    return dti, dtm.value


def axpy(a, x, y):
    """y + a x in FP64: the kick / predict update of Eqs. (19)-(24) with a = dt/2."""
    x, y = _d(x), _d(y)
    out = np.empty_like(x)
    lib().orc_axpy(C.c_int64(len(x)), C.c_double(a), _p(x), _p(y), _p(out))
    return out


def isentropic_u(rho_old, rho_new, u, gamma):
    """u (rho_new/rho_old)^(gamma-1): the isentropic update of PAPER.md:197 (reading R31)."""
    ro, rn, u = _d(rho_old), _d(rho_new), _d(u)
    out = np.empty_like(u)
    lib().orc_isentropic_u(C.c_int64(len(u)), C.c_double(gamma), _p(ro), _p(rn), _p(u), _p(out))
    return out


def drift(x, v, dt, lo, length, periodic):
    """Eq. (25) with the periodic wrap; returns the new coordinate array (FP64)."""
    x, v = _d(x).copy(), _d(v)
    lib().orc_drift(C.c_int64(len(x)), C.c_double(dt), _p(v), C.c_double(float(np.float32(lo))),
                    C.c_double(float(np.float32(length))), C.c_int(int(periodic)), _p(x))
    return x


def block_floor_rung(s: int, R: int) -> int:
    """Lowest rung whose steps begin at substep s (reading R32)."""
    f = lib().orc_block_floor_rung
    f.restype = C.c_int32
    return int(f(C.c_int64(int(s)), C.c_int32(int(R))))


def block_predict(s, delta, tnext, hk, base, rate):
    """Eqs. (19)-(20) per particle at substep s: base + ((s - tnext) delta + hk) rate."""
    tn = np.ascontiguousarray(tnext, np.int32)
    hk, base, rate = _d(hk), _d(base), _d(rate)
    out = np.empty_like(base)
    lib().orc_block_predict(C.c_int64(len(base)), C.c_int64(int(s)), C.c_double(delta),
                            _p(tn, C.c_int32), _p(hk), _p(base), _p(rate), _p(out))
    return out


def block_kick(s, R, delta, rung_des, rung, tnext, hk, q, rate, open=1):
    """Closing kick, rung change, opening kick of the particles with tnext == s
    (PAPER.md:245-259, 270); open=0: the closing kick alone.  q, rate: lists of arrays.
    Returns (rung, tnext, hk, q)."""
    rd = np.ascontiguousarray(rung_des, np.int32)
    rg = np.ascontiguousarray(rung, np.int32).copy()
    tn = np.ascontiguousarray(tnext, np.int32).copy()
    hk = _d(hk).copy()
    n, nq = len(rg), len(q)
    qq = np.ascontiguousarray(np.stack([_d(a) for a in q]).reshape(-1))
    rr = np.ascontiguousarray(np.stack([_d(a) for a in rate]).reshape(-1))
    lib().orc_block_kick(C.c_int64(n), C.c_int64(int(s)), C.c_int32(int(R)), C.c_double(delta),
                         _p(rd, C.c_int32), _p(rg, C.c_int32), _p(tn, C.c_int32), _p(hk),
                         C.c_int32(nq), _p(qq), _p(rr), C.c_int32(int(open)))
    return rg, tn, hk, [qq[k * n:(k + 1) * n].copy() for k in range(nq)]


def imbalance(x, y, z, m, h, mat, box: Box, par: Params, alpha: float, targets=None):
    """Kernel imbalance I_i of Eq. (8) (brute force).  mat: int material ids or None."""
    x, y, z, m, h = map(_d, (x, y, z, m, h))
    n = len(x)
    b, p = box.c(), par.c()
    nt, t = _targets(n, targets)
    out = np.empty(nt)
    mm = None if mat is None else np.ascontiguousarray(np.asarray(mat), dtype=np.int32)
    lib().orc_imbalance_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(m), _p(h),
                              _p(mm, C.c_int32) if mm is not None else None, C.byref(b),
                              C.byref(p), C.c_double(alpha), C.c_int64(nt), _p(t, C.c_int64),
                              _p(out))
    return out


def interface_correction(x, y, z, h, u, rho, imb, box: Box, par: Params, targets=None):
    """Eqs. (9)-(12) for the ideal gas (brute force): corrected rho, P and u (= c_v T)."""
    x, y, z, h, u, rho, imb = map(_d, (x, y, z, h, u, rho, imb))
    n = len(x)
    b, p = box.c(), par.c()
    nt, t = _targets(n, targets)
    rc = np.empty(nt); pc = np.empty(nt); uc = np.empty(nt)
    lib().orc_interface_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(h), _p(u), _p(rho), _p(imb),
                              C.byref(b), C.byref(p), C.c_int64(nt), _p(t, C.c_int64), _p(rc),
                              _p(pc), _p(uc))
    return rc, pc, uc


def rungs(dt_i, dt0, max_rung):
    """Eq. (27): smallest r >= 0 with 2^-r dt0 <= dt_i, capped at max_rung."""
    dt_i = _d(dt_i)
    out = np.empty(len(dt_i), np.int32)
    lib().orc_rungs(C.c_int64(len(dt_i)), _p(dt_i), C.c_double(float(np.float32(dt0))),
                    C.c_int32(int(max_rung)), _p(out, C.c_int32))
    return out


def rung_limiter(x, y, z, h, rung, box: Box, targets=None):
    """r_i >= r_j - 2 over the force pair set, one pass (brute force)."""
    x, y, z, h = map(_d, (x, y, z, h))
    n = len(x)
    b = box.c()
    nt, t = _targets(n, targets)
    rin = np.ascontiguousarray(np.asarray(rung), dtype=np.int32)
    out = np.empty(nt, np.int32)
    lib().orc_rung_limiter_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(h), C.byref(b),
                                 _p(rin, C.c_int32), C.c_int64(nt), _p(t, C.c_int64),
                                 _p(out, C.c_int32))
    return out


def mark_neighbors(x, y, z, h, src, box: Box):
    """FastGas marking pass: src itself plus everything on the interaction
    lists (force pair set) of the particles of src; brute force."""
    x, y, z, h = map(_d, (x, y, z, h))
    n = len(x)
    b = box.c()
    sin = np.ascontiguousarray(np.asarray(src) != 0, dtype=np.uint8)
    out = np.empty(n, np.uint8)
    lib().orc_mark_brute(C.c_int64(n), _p(x), _p(y), _p(z), _p(h), C.byref(b),
                         _p(sin, C.c_uint8), _p(out, C.c_uint8))
    return out
