"""The five BASELINE.json configurations as seeded synthetic inputs (see package docstring)."""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

# table row kinds (names follow SURVEY.md 8(b)); each side maps these to its own enum
DRIFT, LINMAP, MULT, RF, SCNODE, QUAD, CQUAD, SEXT, XDRIFT, SBEND = 0, 1, 2, 3, 4, 5, 6, 7, 8, 9
KIND_NAMES = {DRIFT: "DRIFT", LINMAP: "LINMAP", MULT: "MULT", RF: "RF", SCNODE: "SCNODE", QUAD: "QUAD", CQUAD: "CQUAD", SEXT: "SEXT", XDRIFT: "XDRIFT", SBEND: "SBEND"}

PROTON_MASS_EV = 938.27208816e6
KINETIC_EV = 3.0e9          # J-PARC MR injection energy, PAPER.md:318 (Table I)


@dataclass
class Workload:
    name: str
    kind: np.ndarray            # int32 [n_rows]
    ipar: np.ndarray            # int32 [n_rows]
    par: np.ndarray             # float64 [n_rows, 10]
    grids: List[Dict]
    beam: Dict
    particles: Dict[str, Optional[np.ndarray]]   # x, px, y, py, sigma, psigma (last two None for 4D)
    n_turns: int
    notes: Dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.particles["x"].shape[0])

    @property
    def n_rows(self) -> int:
        return int(self.kind.shape[0])

    @property
    def n_sc(self) -> int:
        return int((self.kind == SCNODE).sum())


def rows_to_arrays(rows: List[Tuple]) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """rows: list of (kind, ipar, [params...]) -> (kind, ipar, par[n,10])."""
    n = len(rows)
    kind = np.zeros(n, np.int32)
    ipar = np.zeros(n, np.int32)
    par = np.zeros((n, 10), np.float64)
    for r, (k, ip, p) in enumerate(rows):
        kind[r] = k
        ipar[r] = ip
        par[r, :len(p)] = p
    return kind, ipar, par


def make_grid(n: int, half: float, nbins: int = 0, smin: float = 0.0, smax: float = 0.0,
              deposit_mode: int = 0, fixed_bits: int = 19, ny: Optional[int] = None,
              half_y: Optional[float] = None) -> Dict:
    return dict(nx=int(n), ny=int(ny or n), xmin=-half, xmax=half, ymin=-(half_y or half), ymax=(half_y or half),
                nbins=int(nbins), smin=float(smin), smax=float(smax),
                deposit_mode=int(deposit_mode), fixed_bits=int(fixed_bits))


def make_beam_spec(line_density: float = 0.0, n_real: float = 0.0, circumference: float = 0.0) -> Dict:
    return dict(kinetic_eV=KINETIC_EV, mass_eV=PROTON_MASS_EV, charge=1,
                line_density=float(line_density), n_real=float(n_real), circumference=float(circumference))


# ------------------------------------------------------------------ random numbers
def rng_uniform(rng: np.random.Generator, n: int) -> np.ndarray:
    """53-bit uniforms in [0,1) from the PCG64 stream (numpy guarantees this stream's stability)."""
    return rng.random(n)


def rng_normal(rng: np.random.Generator, n: int) -> np.ndarray:
    """Box-Muller on the uniform stream (own transform: independent of numpy's normal sampler)."""
    u1 = rng_uniform(rng, n)
    u2 = rng_uniform(rng, n)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


def _trunc_pairs(rng, n: int, cut: float, npairs: int) -> np.ndarray:
    """n rows of 2*npairs standard normals with every pair (2k, 2k+1) rejected outside radius cut."""
    out = np.empty((0, 2 * npairs))
    while out.shape[0] < n:
        m = int((n - out.shape[0]) * 1.05) + 64
        g = rng_normal(rng, m * 2 * npairs).reshape(m, 2 * npairs)
        ok = np.ones(m, bool)
        for k in range(npairs):
            ok &= g[:, 2 * k] ** 2 + g[:, 2 * k + 1] ** 2 <= cut * cut
        out = np.concatenate([out, g[ok]], axis=0)
    return out[:n]


def _twiss_plane(u1, u2, sigma, beta, alpha):
    """normalised (u1,u2) -> (q, p) with rms sigma at a point with Twiss (beta, alpha)."""
    return sigma * u1, (sigma / beta) * (u2 - alpha * u1)


# ------------------------------------------------------------------ lattices
def _lattice_cfg1():
    f = 10.0 / np.sqrt(2.0)                  # 90 deg per cell, SURVEY 8d cfg1
    cell = [(MULT, 1, [1.0 / f, 0.0]), (DRIFT, 0, [10.0]), (MULT, 1, [-1.0 / f, 0.0]), (DRIFT, 0, [10.0]),
            (SCNODE, 0, [20.0])]
    return cell * 24, 480.0


def _lattice_cfg2():
    f1, f2 = 6.068730, 6.296936             # mu = (0.31, 0.29) 2 pi per 20 m cell, SURVEY 8d cfg2
    hqf = (MULT, 1, [0.5 / f1, 0.0])
    qd = (MULT, 1, [-1.0 / f2, 0.0])
    arm = [(DRIFT, 0, [5.0]), (SCNODE, 0, [5.0]), (DRIFT, 0, [5.0]), (SCNODE, 0, [5.0])]
    cell = [hqf, (MULT, 2, [0.5, 0.0])] + arm + [qd, (MULT, 2, [-0.5, 0.0])] + arm + [hqf]
    return cell * 72, 1440.0


K_F, K_D = 0.11526860, 0.11550173           # thick quads, tunes 21.35/21.44, SURVEY 8d cfg3 (probe p6)
CFG3_C = 1567.5                              # PAPER.md Table I ring; 216 quadrupoles
CFG3_H = 9
CFG3_TWISS = ((22.304, -1.939), (7.019, 0.707))   # (beta, alpha) x / y at the QF entrance (probe p6)


def _lattice_cfg3():
    l_last = CFG3_C / 216 - (1.5 + 0.5 + 1.0 + 1.5 + 1.5)
    rows = []
    for s in range(216):
        sign = 1.0 if s % 2 == 0 else -1.0
        k1 = K_F if s % 2 == 0 else -K_D
        rows += [(QUAD, 0, [k1, 1.5]), (DRIFT, 0, [0.5]), (MULT, 2, [sign * 0.05, 0.0]), (DRIFT, 0, [1.0]),
                 (MULT, 0, [0.0, 0.0]), (DRIFT, 0, [1.5]), (MULT, 3, [sign * 1.0, 0.0]), (DRIFT, 0, [1.5]),
                 (MULT, 0, [0.0, 0.0]), (DRIFT, 0, [l_last]), (SCNODE, 0, [CFG3_C / 216])]
    rows.append((RF, 0, [280.0e3, float(CFG3_H), 0.0]))
    return rows, CFG3_C


# ------------------------------------------------------------------ beams
def _beam_cfg1(rng, n):
    g = _trunc_pairs(rng, n, 4.0, 2)        # pair 0 = (x,y), pair 1 = (px,py): SURVEY A15
    return dict(x=3e-3 * g[:, 0], y=3e-3 * g[:, 1], px=0.3e-3 * g[:, 2], py=0.3e-3 * g[:, 3],
                sigma=None, psigma=None)


def _beam_cfg2(rng, n):
    g = rng_normal(rng, 4 * n).reshape(n, 4)
    r = rng_uniform(rng, n) ** 0.25          # uniform in the 4D unit ball
    u = g / np.linalg.norm(g, axis=1, keepdims=True) * r[:, None] * np.sqrt(6.0)
    return dict(x=4e-3 * u[:, 0], px=0.10365e-3 * u[:, 1], y=2e-3 * u[:, 2], py=0.47027e-3 * u[:, 3],
                sigma=None, psigma=None)


def _longitudinal(rng, n):
    g = _trunc_pairs(rng, n, 4.0, 1)
    return 15.0 * g[:, 0], 2e-3 * g[:, 1]


def _beam_cfg3(rng, n):
    g = _trunc_pairs(rng, n, 4.0, 2)        # pair 0 = (ux1, uy1) positions, pair 1 = (ux2, uy2)
    (bx, ax), (by, ay) = CFG3_TWISS
    x, px = _twiss_plane(g[:, 0], g[:, 2], 3e-3, bx, ax)
    y, py = _twiss_plane(g[:, 1], g[:, 3], 3e-3, by, ay)
    s, ps = _longitudinal(rng, n)
    return dict(x=x, px=px, y=y, py=py, sigma=s, psigma=ps)


def _beam_cfg5(rng, n):
    """80 % in a narrow round Gaussian spike (sigma0/8, cut at 4 sigma_spike => r < 0.5 sigma0),
    20 % in a hollow ring r in [2,3] sigma0 uniform in area."""
    s0 = 3e-3
    n_spike = (n * 4) // 5
    g = _trunc_pairs(rng, n_spike, 4.0, 1)
    ux = np.concatenate([g[:, 0] / 8.0, np.empty(n - n_spike)])
    uy = np.concatenate([g[:, 1] / 8.0, np.empty(n - n_spike)])
    rr = np.sqrt(4.0 + 5.0 * rng_uniform(rng, n - n_spike))
    th = 2.0 * np.pi * rng_uniform(rng, n - n_spike)
    ux[n_spike:] = rr * np.cos(th)
    uy[n_spike:] = rr * np.sin(th)
    perm = np.argsort(rng_uniform(rng, n), kind="stable")     # interleave spike and ring particles
    ux, uy = ux[perm], uy[perm]
    m = _trunc_pairs(rng, n, 4.0, 1)
    (bx, ax), (by, ay) = CFG3_TWISS
    x, px = _twiss_plane(ux, m[:, 0], s0, bx, ax)
    y, py = _twiss_plane(uy, m[:, 1], s0, by, ay)
    s, ps = _longitudinal(rng, n)
    return dict(x=x, px=px, y=y, py=py, sigma=s, psigma=ps)


# ------------------------------------------------------------------ public
def make_config(cfg: int, n: Optional[int] = None, n_turns: Optional[int] = None, grid_n: Optional[int] = None,
                deposit_mode: Optional[int] = None, fixed_bits: int = 19, seed: Optional[int] = None) -> Workload:
    """cfg in 1..5 (BASELINE.json configs[cfg-1]).  n / n_turns / grid_n override the config's size
    (decimated variants for tests); cfg 4 is cfg 3 with grid_n in {64,128,256,512}."""
    if cfg == 1:
        rows, C = _lattice_cfg1()
        n = n or 10_000
        rng = np.random.Generator(np.random.PCG64(seed or 1))
        parts = _beam_cfg1(rng, n)
        grids = [make_grid(grid_n or 64, 15e-3, deposit_mode=deposit_mode or 0, fixed_bits=fixed_bits)]
        beam = make_beam_spec(line_density=1e11, circumference=C)
        turns = 10
    elif cfg == 2:
        rows, C = _lattice_cfg2()
        n = n or 100_000
        rng = np.random.Generator(np.random.PCG64(seed or 2))
        parts = _beam_cfg2(rng, n)
        grids = [make_grid(grid_n or 128, 20e-3, deposit_mode=deposit_mode or 0, fixed_bits=fixed_bits)]
        beam = make_beam_spec(line_density=1.5e11, circumference=C)
        turns = 100
    elif cfg in (3, 4, 5):
        rows, C = _lattice_cfg3()
        half_bucket = C / (2 * CFG3_H)
        if cfg == 5:
            n = n or 10_000_000
            rng = np.random.Generator(np.random.PCG64(seed or 5))
            parts = _beam_cfg5(rng, n)
            gn, mode, turns = grid_n or 256, 1 if deposit_mode is None else deposit_mode, 100
        else:
            n = n or 1_000_000
            rng = np.random.Generator(np.random.PCG64(seed or 3))
            parts = _beam_cfg3(rng, n)
            gn, mode, turns = grid_n or 128, deposit_mode or 0, (1000 if cfg == 3 else 100)
        grids = [make_grid(gn, 24e-3, nbins=256, smin=-half_bucket, smax=half_bucket,
                           deposit_mode=mode, fixed_bits=fixed_bits)]
        beam = make_beam_spec(n_real=2e13, circumference=C)
    else:
        raise ValueError("cfg must be 1..5")
    kind, ipar, par = rows_to_arrays(rows)
    parts = {k: (None if v is None else np.ascontiguousarray(v, np.float64)) for k, v in parts.items()}
    return Workload(name=f"cfg{cfg}", kind=kind, ipar=ipar, par=par, grids=grids, beam=beam,
                    particles=parts, n_turns=n_turns or turns, notes=dict(cfg=cfg, seed=seed))
