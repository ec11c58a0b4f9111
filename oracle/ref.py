"""ctypes front end of the ORACLE (test infrastructure, not the product; see sc_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports paper_2010_11540_b200.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, List, Optional

import numpy as np

from .build import build

_lib = None

c_dp = C.POINTER(C.c_double)
c_ip = C.POINTER(C.c_int64)


class OrcGrid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("xmin", C.c_double), ("xmax", C.c_double),
                ("ymin", C.c_double), ("ymax", C.c_double), ("nbins", C.c_int32), ("smin", C.c_double),
                ("smax", C.c_double), ("fixed", C.c_int32), ("fixed_bits", C.c_int32),
                ("boundary", C.c_int32), ("long_kick", C.c_int32), ("interp", C.c_int32)]


class OrcBeam(C.Structure):
    _fields_ = [("gamma0", C.c_double), ("beta0", C.c_double), ("E0_eV", C.c_double), ("r_c", C.c_double),
                ("kappa", C.c_double), ("charge", C.c_int32), ("line_density", C.c_double),
                ("n_real", C.c_double), ("circumference", C.c_double)]


class OrcWork(C.Structure):
    _fields_ = [("Q", c_dp), ("Qi", c_ip), ("u", c_dp), ("Ex", c_dp), ("Ey", c_dp), ("cnt", c_ip),
                ("n_inside", C.c_int64)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_green_cell.restype = C.c_double
        _lib.orc_green_cell.argtypes = [C.c_double] * 4
        _lib.orc_lambda_at.restype = C.c_double
        _lib.orc_lambda_slope.restype = C.c_double
        _lib.orc_gather_scalar.restype = C.c_double
        _lib.orc_deposit_f64.restype = C.c_int64
        _lib.orc_deposit_fixed.restype = C.c_int64
    return _lib


def _dp(a: Optional[np.ndarray]):
    if a is None:
        return C.cast(None, c_dp)
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(c_dp)


def _ip(a: np.ndarray):
    assert a.dtype == np.int64 and a.flags.c_contiguous
    return a.ctypes.data_as(c_ip)


def grid_struct(g: Dict) -> OrcGrid:
    return OrcGrid(g["nx"], g["ny"], g["xmin"], g["xmax"], g["ymin"], g["ymax"], g.get("nbins", 0),
                   g.get("smin", 0.0), g.get("smax", 0.0), int(g.get("deposit_mode", 0) == 1), g.get("fixed_bits", 19),
                   int(g.get("boundary", 0)), int(g.get("long_kick", 0)), int(g.get("interp", 0)))


def beam_struct(b: Dict) -> OrcBeam:
    out = OrcBeam()
    lib().orc_beam_init(C.byref(out), C.c_double(b["kinetic_eV"]), C.c_double(b["mass_eV"]), C.c_int(b["charge"]),
                        C.c_double(b.get("line_density", 0.0)), C.c_double(b.get("n_real", 0.0)),
                        C.c_double(b.get("circumference", 0.0)))
    return out


class Work:
    """Caller-owned scratch + results of the last SC node on one grid."""

    def __init__(self, g: Dict):
        nc = g["nx"] * g["ny"]
        self.Q = np.zeros(nc)
        self.Qi = np.zeros(nc, np.int64)
        self.u = np.zeros(nc)
        self.Ex = np.zeros(nc)
        self.Ey = np.zeros(nc)
        self.cnt = np.zeros(max(1, g.get("nbins", 0)), np.int64)
        self.shape = (g["ny"], g["nx"])

    def struct(self) -> OrcWork:
        return OrcWork(_dp(self.Q), _ip(self.Qi), _dp(self.u), _dp(self.Ex), _dp(self.Ey), _ip(self.cnt), 0)


# ---------------------------------------------------------------- element maps (arrays in place)
def drift(p: Dict, L: float, gamma0: float):
    lib().orc_drift(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                    _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_double(L), C.c_double(gamma0))


def quad_matrix(k1: float, L: float) -> np.ndarray:
    M = np.zeros(8)
    lib().orc_quad_matrix(C.c_double(k1), C.c_double(L), _dp(M))
    return M


def linmap(p: Dict, M: np.ndarray, L: float, gamma0: float):
    M = np.ascontiguousarray(M, np.float64)
    lib().orc_linmap(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                     _dp(p.get("sigma")), _dp(p.get("psigma")), _dp(M), C.c_double(L), C.c_double(gamma0))


def cquad(p: Dict, k1: float, L: float, gamma0: float):
    lib().orc_cquad(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                    _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_double(k1), C.c_double(L), C.c_double(gamma0))


def xdrift(p: Dict, L: float, beta0: float):
    lib().orc_xdrift(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                     _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_double(L), C.c_double(beta0))


def sbend(p: Dict, L: float, h: float, beta0: float):
    lib().orc_sbend(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                    _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_double(L), C.c_double(h), C.c_double(beta0))


def sext(p: Dict, k2: float, L: float, gamma0: float):
    lib().orc_sext(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                   _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_double(k2), C.c_double(L), C.c_double(gamma0))


def mult(p: Dict, order: int, knl: float, ksl: float = 0.0):
    lib().orc_mult(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                   C.c_int(order), C.c_double(knl), C.c_double(ksl))


def rf(p: Dict, amp: float, h: float, circumference: float, phi0: float = 0.0):
    lib().orc_rf(C.c_int64(len(p["sigma"])), _dp(p["sigma"]), _dp(p["psigma"]), C.c_double(amp), C.c_double(h),
                 C.c_double(circumference), C.c_double(phi0))


# ---------------------------------------------------------------- SC node pieces
def deposit_f64(x, y, g: Dict):
    Q = np.zeros(g["nx"] * g["ny"])
    gs = grid_struct(g)
    n_in = lib().orc_deposit_f64(C.c_int64(len(x)), _dp(x), _dp(y), C.byref(gs), _dp(Q))
    return Q.reshape(g["ny"], g["nx"]), n_in


def deposit_fixed(x, y, g: Dict):
    Qi = np.zeros(g["nx"] * g["ny"], np.int64)
    gs = grid_struct(g)
    n_in = lib().orc_deposit_fixed(C.c_int64(len(x)), _dp(x), _dp(y), C.byref(gs), _ip(Qi))
    return Qi.reshape(g["ny"], g["nx"]), n_in


def lambda_hist(sigma, g: Dict) -> np.ndarray:
    cnt = np.zeros(g["nbins"], np.int64)
    gs = grid_struct(g)
    lib().orc_lambda_hist(C.c_int64(len(sigma)), _dp(sigma), C.byref(gs), _ip(cnt))
    return cnt


def lambda_at(sigma: float, g: Dict, cnt: np.ndarray, n_real: float, n: int) -> float:
    gs = grid_struct(g)
    return lib().orc_lambda_at(C.c_double(sigma), C.byref(gs), _ip(cnt), C.c_double(n_real), C.c_int64(n))


def lambda_slope(sigma: float, g: Dict, cnt: np.ndarray, n_real: float, n: int) -> float:
    gs = grid_struct(g)
    return lib().orc_lambda_slope(C.c_double(sigma), C.byref(gs), _ip(cnt), C.c_double(n_real), C.c_int64(n))


def gather_scalar(u: np.ndarray, g: Dict, x: float, y: float):
    """(inside, bilinear value of the node scalar u at (x, y))."""
    u = np.ascontiguousarray(u, np.float64).ravel()
    gs = grid_struct(g)
    inside = C.c_int(0)
    v = lib().orc_gather_scalar(C.byref(gs), _dp(u), C.c_double(x), C.c_double(y), C.byref(inside))
    return bool(inside.value), v


def green_cell(x: float, y: float, dx: float, dy: float) -> float:
    return lib().orc_green_cell(x, y, dx, dy)


def poisson(Q: np.ndarray, g: Dict, n_total: float, direct: bool = False) -> np.ndarray:
    """Open boundary (FFT convolution or the direct sum), or, for g["boundary"] == 1, the paper's pipe solver."""
    Q = np.ascontiguousarray(Q, np.float64).ravel()
    u = np.zeros_like(Q)
    gs = grid_struct(g)
    if int(g.get("boundary", 0)) == 1:
        fn = lib().orc_poisson_dirichlet
    else:
        fn = lib().orc_poisson_direct if direct else lib().orc_poisson_fft
    fn(C.byref(gs), _dp(Q), C.c_double(n_total), _dp(u))
    return u.reshape(g["ny"], g["nx"])


def field(u: np.ndarray, g: Dict):
    u = np.ascontiguousarray(u, np.float64).ravel()
    Ex = np.zeros_like(u)
    Ey = np.zeros_like(u)
    gs = grid_struct(g)
    lib().orc_field(C.byref(gs), _dp(u), _dp(Ex), _dp(Ey))
    return Ex.reshape(g["ny"], g["nx"]), Ey.reshape(g["ny"], g["nx"])


def gather(Ex, Ey, g: Dict, x: float, y: float):
    Ex = np.ascontiguousarray(Ex, np.float64).ravel()
    Ey = np.ascontiguousarray(Ey, np.float64).ravel()
    gs = grid_struct(g)
    ins = C.c_int(0)
    ex = C.c_double(0)
    ey = C.c_double(0)
    lib().orc_gather(C.byref(gs), _dp(Ex), _dp(Ey), C.c_double(x), C.c_double(y), C.byref(ins), C.byref(ex), C.byref(ey))
    return bool(ins.value), ex.value, ey.value


def gather_bicubic(u: np.ndarray, g: Dict, x: float, y: float):
    """(inside, u(x,y), -du/dx, -du/dy) of the bicubic surface of eqs. 28-29 (N4)."""
    u = np.ascontiguousarray(u, np.float64).ravel()
    gs = grid_struct(g)
    ins = C.c_int(0)
    uv, ex, ey = C.c_double(0), C.c_double(0), C.c_double(0)
    lib().orc_gather_bicubic(C.byref(gs), _dp(u), C.c_double(x), C.c_double(y), C.byref(ins), C.byref(uv),
                             C.byref(ex), C.byref(ey))
    return bool(ins.value), uv.value, ex.value, ey.value


def fft(re, im, inverse=False):
    re = np.array(re, np.float64)
    im = np.array(im, np.float64)
    lib().orc_fft(C.c_int(len(re)), _dp(re), _dp(im), C.c_int(int(inverse)))
    return re + 1j * im


def dft_naive(re, im, inverse=False):
    re = np.ascontiguousarray(re, np.float64)
    im = np.ascontiguousarray(im, np.float64)
    ore = np.zeros_like(re)
    oim = np.zeros_like(im)
    lib().orc_dft_naive(C.c_int(len(re)), _dp(re), _dp(im), _dp(ore), _dp(oim), C.c_int(int(inverse)))
    return ore + 1j * oim


def scnode(p: Dict, g: Dict, beam: Dict, L_sc: float, direct: bool = False) -> Work:
    w = Work(g)
    ws = w.struct()
    gs = grid_struct(g)
    bs = beam_struct(beam)
    rc = lib().orc_scnode(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                          _dp(p.get("sigma")), _dp(p.get("psigma")), C.byref(gs), C.byref(bs), C.c_double(L_sc),
                          C.c_int(int(direct)),
                          C.byref(ws))
    if rc:
        raise RuntimeError("orc_scnode failed")
    w.n_inside = ws.n_inside
    return w


def sc_kick(p: Dict, g: Dict, beam: Dict, L_sc: float, w: "Work") -> None:
    """Gather + kick IN PLACE on the arrays of p with the grids already in w (pins on prescribed fields)."""
    ws = w.struct()
    gs = grid_struct(g)
    bs = beam_struct(beam)
    lib().orc_sc_kick(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                      _dp(p.get("sigma")), _dp(p.get("psigma")), C.byref(gs), C.byref(bs), C.c_double(L_sc),
                      C.byref(ws))


def moments(p: Dict) -> np.ndarray:
    out = np.zeros(33)
    lib().orc_moments(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                      _dp(p.get("sigma")), _dp(p.get("psigma")), _dp(out))
    return out


# ---------------------------------------------------------------- whole loop
def track(kind, ipar, par, grids: List[Dict], beam: Dict, particles: Dict, n_turns: int = 0,
          stop_after_rows: int = -1, direct: bool = False):
    """Track COPIES of the particle arrays; returns (particles, [Work per grid])."""
    p = {k: (None if v is None else np.array(v, np.float64, copy=True)) for k, v in particles.items()}
    kind = np.ascontiguousarray(kind, np.int32)
    ipar = np.ascontiguousarray(ipar, np.int32)
    par = np.ascontiguousarray(par, np.float64)
    works = [Work(g) for g in grids]
    wss = (OrcWork * max(1, len(grids)))(*[w.struct() for w in works])
    gss = (OrcGrid * max(1, len(grids)))(*[grid_struct(g) for g in grids])
    bs = beam_struct(beam)
    rc = lib().orc_track(C.c_int64(len(p["x"])), _dp(p["x"]), _dp(p["px"]), _dp(p["y"]), _dp(p["py"]),
                         _dp(p.get("sigma")), _dp(p.get("psigma")), C.c_int64(len(kind)),
                         kind.ctypes.data_as(C.POINTER(C.c_int32)), ipar.ctypes.data_as(C.POINTER(C.c_int32)),
                         _dp(par), C.c_int32(len(grids)), gss, C.byref(bs), C.c_int64(n_turns),
                         C.c_int64(stop_after_rows), C.c_int(int(direct)), wss)
    if rc:
        raise RuntimeError("orc_track failed (bad table row, missing grid, or RF/lambda on a 4D beam)")
    for w, ws in zip(works, wss):
        w.n_inside = ws.n_inside
    return p, works


def track_workload(wl, n_turns: Optional[int] = None, stop_after_rows: int = -1, direct: bool = False):
    return track(wl.kind, wl.ipar, wl.par, wl.grids, wl.beam, wl.particles,
                 wl.n_turns if n_turns is None else n_turns, stop_after_rows, direct)
