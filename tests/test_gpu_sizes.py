"""GPU parity at the sizes and shapes of BASELINE.json configs 2-5: the grid sweep (64..512, both deposit modes; 256 and
512 exceed shared memory and take the windowed path) at the first nodes and after one WHOLE turn, the contention case
(cfg5) decimated and at its full 1e7 macroparticles, the full-size bench configuration (1e6 macroparticles, 128x128, the
launch configuration bench.py times), the long runs of SURVEY.md section 8(c) compared statistically (rms emittance,
rms tune spread; north_star: 1e-3 relative; oracle side stored under tests/golden/ by tests/golden/make_golden.py), the
1000-turn run of configs[2] (invariants), and the measurement behind the fixed-point allowance."""
import numpy as np
import pytest

from workloads import SCNODE, make_config

pytestmark = pytest.mark.gpu
NAMES = ("x", "px", "y", "py", "sigma", "psigma")


@pytest.fixture(scope="module")
def sc():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2010_11540_b200 as sc
    sc.load_library()
    return sc


def allowance(wl):
    """Fixed-point mode only ("fixed-point allowance"): 16 * 2^-s / N at 128 nodes per axis, times
    (nx/128)^2 on finer grids (a rounding-level coordinate difference flips a quantised fraction with probability ~ 1/dx,
    and a flipped weight perturbs the neighbouring field by ~ 1/dx)."""
    g = wl.grids[0]
    if g["deposit_mode"] != 1:
        return 0.0
    return 16 * 2.0 ** -g["fixed_bits"] / wl.n * max(1.0, g["nx"] / 128.0) ** 2


def rel_err(a, b):
    return float(np.abs(a - b).max() / max(np.sqrt(np.mean(b * b)), 1e-300))


def grid_err(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def check_node(sc, t, w, wl, mode):
    if mode == 1:
        assert np.array_equal(t.sc_get_grid(sc.SC_GRID_RHO_I64).ravel(), w.Qi)          # bit-exact
        s = wl.grids[0]["fixed_bits"]
        assert int(w.Qi.sum()) == w.n_inside << (2 * s)                                  # exact charge
    else:
        assert grid_err(t.sc_get_grid(sc.SC_GRID_RHO_F64).ravel(), w.Q) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_PHI).ravel(), w.u) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EX).ravel(), w.Ex) < 1e-10
    assert grid_err(t.sc_get_grid(sc.SC_GRID_EY).ravel(), w.Ey) < 1e-10
    assert np.array_equal(t.sc_get_grid(sc.SC_GRID_LAMBDA), w.cnt)
    assert t.sc_moments()[31] == wl.n - w.n_inside


@pytest.mark.parametrize("grid_n", [64, 128, 256, 512])
@pytest.mark.parametrize("mode", [0, 1])
def test_cfg4_grid_sweep(sc, orc, grid_n, mode):
    """cfg4: cfg3's beam and lattice on 64..512 grids: the node after 1 and after 3 segments (grids of the
    third node have seen two kicks), then the particles."""
    wl = make_config(4, n=40_009, grid_n=grid_n, deposit_mode=mode)
    nodes = np.flatnonzero(wl.kind == SCNODE)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    done = 0
    for k in (0, 2):
        rows = int(nodes[k]) + 1
        want, works = orc.track_workload(wl, stop_after_rows=rows)
        t.sc_step(rows - done)
        done = rows
        if k == 0 or mode == 0:
            check_node(sc, t, works[0], wl, mode)
        else:
            # after two kicks the coordinates differ by rounding (~1e-13 relative): now and then a quantised
            # fraction llrint(f 2^s) flips by one unit, which moves two weights by up to 2^s each; the total
            # stays exact because every inside particle contributes exactly 2^(2s)
            Qi = t.sc_get_grid(sc.SC_GRID_RHO_I64).ravel()
            assert int(Qi.sum()) == int(works[0].Qi.sum())
            assert np.abs(Qi - works[0].Qi).max() <= 8 << wl.grids[0]["fixed_bits"]
    got = t.sc_get_particles()
    tol = 1e-10 + allowance(wl)
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    t.close()


@pytest.mark.parametrize("n", [200_003, 10_000_000])
def test_cfg5_contention(sc, orc, n):
    """cfg5: 80 % of the particles on ~200 cells of a 256x256 grid, deterministic fixed-point deposit.
    Decimated and at the full 1e7 (first node: bit-exact grid, exact total charge, fields)."""
    wl = make_config(5, n=n)
    first = int(np.argmax(wl.kind == SCNODE)) + 1
    _, works = orc.track_workload(wl, stop_after_rows=first)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_step(first)
    check_node(sc, t, works[0], wl, 1)
    # the spike (smeared by the first segment's transport): 1.5 % of the 65536 cells hold most of the charge
    Q = works[0].Qi.astype(np.float64)
    assert np.sort(Q)[-1000:].sum() > 0.6 * Q.sum()
    t.close()


def test_cfg3_full_size_one_turn(sc, orc):
    """The bench configuration itself: 1e6 macroparticles, 128x128, fixed-point deposit, whole turns by graph
    replay (the launch configuration bench.py times).  First node bit-exact; one full turn within 1e-10."""
    wl = make_config(3, deposit_mode=1)
    assert wl.n == 1_000_000
    first = int(np.argmax(wl.kind == SCNODE)) + 1
    _, works = orc.track_workload(wl, stop_after_rows=first)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_step(first)
    check_node(sc, t, works[0], wl, 1)
    want, _ = orc.track_workload(wl, n_turns=1)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    tol = 1e-10 + allowance(wl)
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    mo, mg = orc.moments(want), t.sc_moments()
    # means against the rms of their coordinate, second moments against sqrt(var_r var_c), emittances relatively
    var = {}
    m = 7
    for r in range(6):
        for c in range(r, 6):
            var[(r, c)] = m
            m += 1
    rms = [np.sqrt(mo[var[(r, r)]]) for r in range(6)]
    for r in range(6):
        assert abs(mg[1 + r] - mo[1 + r]) < 1e-9 * rms[r]
        for c in range(r, 6):
            assert abs(mg[var[(r, c)]] - mo[var[(r, c)]]) < 1e-9 * rms[r] * rms[c]
    assert np.allclose(mg[28:31], mo[28:31], rtol=1e-8)
    # properties that hold at any size: second turn runs from the cached graph and stays finite, particle
    # count is conserved, nothing non-finite
    t.sc_track(2)
    m = t.sc_moments()
    assert m[0] == wl.n and m[32] == 0
    t.close()


@pytest.mark.parametrize("grid_n", [64, 128, 256, 512])
@pytest.mark.parametrize("mode", [0, 1])
def test_cfg4_one_whole_turn(sc, orc, grid_n, mode):
    """cfg4: one WHOLE turn (216 nodes) on every grid of the sweep, both deposit modes: all six coordinates within
    north_star's 1e-10 (fp64 deposit: no allowance; fixed point: + the flip allowance of DESIGN.md section 2).  256 and
    512 take the windowed deposit and the three-launch solver; 64 and 128 the field-window kernel."""
    wl = make_config(4, n=20_011, grid_n=grid_n, deposit_mode=mode)
    want, works = orc.track_workload(wl, n_turns=1)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    tol = 1e-10 + allowance(wl)
    for k in NAMES:
        assert rel_err(got[k], want[k]) < tol, (k, rel_err(got[k], want[k]))
    assert t.sc_moments()[31] == wl.n - works[0].n_inside
    t.close()


def _twin(wl, rel=1e-13, seed=78):
    """The same workload with every initial coordinate moved by `rel` relative (random signs): the level at which two
    correct implementations agree after a node (FFT summation order, fused multiply-adds)."""
    import copy
    rng = np.random.Generator(np.random.PCG64(seed))
    tw = copy.copy(wl)
    tw.particles = {k: (None if v is None else v * (1.0 + rel * rng.choice([-1.0, 1.0], size=v.shape))) for k, v in wl.particles.items()}
    return tw


def test_cfg5_one_turn_decimated(sc, orc):
    """cfg5 (spike + hollow ring, 256 x 256, fixed point) decimated to 2e5 macroparticles: per-particle coordinates
    after one whole turn.  80 % of the bunch charge sits in a spike two cells wide: its space-charge kicks are ~64 times
    cfg3's and the dynamics amplifies any difference enormously within a turn, so the comparison is made against what
    the ORACLE ITSELF does under a 1e-13 change of its input (the twin run): the GPU must stay within 10x of that, and
    north_star's 1e-10 + allowance is asserted on the first 8 segments, where it still can hold."""
    wl = make_config(5, n=200_003)
    nodes = np.flatnonzero(wl.kind == SCNODE)
    rows8 = int(nodes[7]) + 1
    want8, _ = orc.track_workload(wl, stop_after_rows=rows8)
    want, works = orc.track_workload(wl, n_turns=1)
    twin, _ = orc.track_workload(_twin(wl), n_turns=1)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_step(rows8)
    got8 = t.sc_get_particles()
    tol = 1e-10 + allowance(wl)
    for k in NAMES:
        assert rel_err(got8[k], want8[k]) < tol, (k, rel_err(got8[k], want8[k]))
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    for k in NAMES:
        own = rel_err(twin[k], want[k])                       # the oracle against itself, input moved by 1e-13
        assert rel_err(got[k], want[k]) < 10.0 * own + tol, (k, rel_err(got[k], want[k]), own)
    assert abs(t.sc_moments()[31] - (wl.n - works[0].n_inside)) <= 2
    t.close()


def _golden(name):
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)) as f:
        return json.load(f)


def test_cfg5_full_size_one_turn(sc):
    """cfg5 at its full 1e7 macroparticles, one whole turn, in the launch configuration bench.py --cfg 5 times: 1024
    sampled particles and the moments against the oracle's (tests/golden/cfg5_full.json, written by
    tests/golden/make_golden.py from the oracle alone: its turn takes five minutes of one core).  Tolerance as in
    test_cfg5_one_turn_decimated: 10x what the oracle's own twin run (input moved by 1e-13) differs by."""
    gold = _golden("cfg5_full.json")
    wl = make_config(5)
    assert wl.n == gold["n"] == 10_000_000
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(1)
    got = t.sc_get_particles()
    idx = np.array(gold["index"])
    tol = 1e-10 + allowance(wl)
    for k in NAMES:
        want = np.array(gold["particles"][k])
        own = np.abs(np.array(gold["twin"]["particles"][k]) - want).max() / gold["rms"][k]
        err = np.abs(got[k][idx] - want).max() / gold["rms"][k]
        assert err < 10.0 * own + tol, (k, err, own)
    mg, mo = t.sc_moments(), np.array(gold["moments"])
    assert mg[0] == wl.n and mg[32] == 0
    assert abs(mg[31] - (wl.n - gold["n_inside_last_node"])) <= 2
    assert np.allclose(mg[28:31], mo[28:31], rtol=1e-7)
    t.close()


def _tunes(snaps, beta, alpha):
    """Turn-averaged phase advance per turn in Floquet-normalised coordinates."""
    q = np.stack([s[0] for s in snaps])
    p = np.stack([s[1] for s in snaps])
    phi = np.arctan2(-(beta * p + alpha * q), q)
    d = np.mod(np.diff(phi, axis=0), 2 * np.pi)
    return d.mean(axis=0) / (2 * np.pi)


def _long_run(sc, gold, planes, strict=False):
    """strict=True: north_star's 1e-3 on every statistic, no twin-based widening; the measured deviations are printed (pytest -s)
    and the largest of them returned."""
    wl = make_config(gold["cfg"], n=gold["n"], deposit_mode=gold["deposit_mode"])
    if "n_real" in gold:
        wl.beam["n_real"] = gold["n_real"]
    nt = gold["n_tagged"]
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    snaps, emit = [], {}
    for turn in range(1, gold["turns"] + 1):
        t.sc_track(1)
        g = t.sc_get_particles()
        snaps.append(tuple(g[k][:nt].copy() for k in ("x", "px", "y", "py")))
        if str(turn) in gold["emittances"]:
            emit[str(turn)] = t.sc_moments()[28:31]
    m = t.sc_moments()
    assert m[0] == wl.n and m[32] == 0
    t.close()
    # north_star: 1e-3 relative.  Where the dynamics is chaotic (cfg3's literal intensity) two runs
    # that differ by rounding decorrelate particle by particle, and the statistics of 1e5 macroparticles then differ by
    # sampling noise.  The oracle's own twin runs (initial coordinates moved by one unit in the last place, independent sign
    # patterns: "twin" and the ensemble "twins" of the stored file) measure that noise: s = rms over the members of their
    # relative deviation from the unperturbed oracle run (for the emittances: the largest such rms up to that turn), and the
    # bound is the larger of 1e-3 and 4 s ("Tolerances").  cfg2 is not chaotic (twin deviation 1e-11 after
    # 100 turns): there 1e-3 stands.
    members = ([gold["twin"]] if gold.get("twin") else []) + gold.get("twins", [])

    def rms_dev(get, want):
        return float(np.sqrt(np.mean([((get(m) - want) / want) ** 2 for m in members]))) if members else 0.0

    def bound(floor_rms):
        return 1e-3 if strict else max(1e-3, 4.0 * floor_rms)

    measured = {}
    floor = [0.0] * planes
    for turn, want in gold["emittances"].items():                 # rms emittances along the run, every plane tracked
        for pl in range(planes):
            floor[pl] = max(floor[pl], rms_dev(lambda m: m["emittances"][turn][pl], want[pl]))
            dev = abs(emit[turn][pl] - want[pl]) / want[pl]
            measured[f"emittance[{pl}]"] = max(measured.get(f"emittance[{pl}]", 0.0), dev)
            assert dev < bound(floor[pl]), (turn, pl, emit[turn][pl], want[pl], floor[pl])
    for (a, b, name) in ((0, 1, "x"), (2, 3, "y")):               # per-particle tunes of the tagged particles
        tw = gold["tunes"][name]
        tg = _tunes([(s[a], s[b]) for s in snaps], tw["beta"], tw["alpha"])
        f_s = rms_dev(lambda m: m["tunes"][name]["rms_spread"], tw["rms_spread"])
        f_m = rms_dev(lambda m: m["tunes"][name]["mean"], tw["mean"])
        measured[f"tune_rms_spread[{name}]"] = abs(tg.std() - tw["rms_spread"]) / tw["rms_spread"]
        measured[f"tune_mean[{name}]"] = abs(tg.mean() - tw["mean"]) / abs(tw["mean"])
        assert measured[f"tune_rms_spread[{name}]"] < bound(f_s), (name, tg.std(), tw["rms_spread"], f_s)
        assert measured[f"tune_mean[{name}]"] < bound(f_m), (name, tg.mean(), tw["mean"], f_m)
    floors = {f"emittance[{pl}]": floor[pl] for pl in range(planes)}
    print("long run cfg%d%s: measured relative deviation from the oracle (largest over the run) " % (gold["cfg"], " n_real=%g" % gold["n_real"] if "n_real" in gold else "") +
          ", ".join(f"{k}={v:.2e}" for k, v in measured.items()) + "; twin rms deviation of the emittances " +
          ", ".join(f"{k}={v:.2e}" for k, v in floors.items()))
    return measured


def test_long_run_statistics_cfg2_literal(sc):
    """BASELINE.json configs[1] as written: 1e5 macroparticles, 128 x 128, 100 turns (the paper's tune-shift regime).
    rms emittances every 10 turns and the mean and rms spread of the per-particle tunes within
    north_star's 1e-3 of the oracle's (tests/golden/long_cfg2.json, written by the oracle alone: nine minutes of a core)."""
    _long_run(sc, _golden("long_cfg2.json"), 2)


def test_long_run_statistics_cfg3_1e5_200_turns(sc):
    """configs[2] decimated to 1e5 macroparticles at the config's bunch charge, 200 turns, fixed-point deposit
    (SURVEY.md section 8(c)): emittances of all three planes every 10 turns, tune mean and rms spread, 1e-3."""
    _long_run(sc, _golden("long_cfg3.json"), 3)


def test_long_run_statistics_cfg3_paper_regime(sc):
    """The 6D path -- cfg3's lattice with RF, the 256-bin line density and 216 nodes per turn, 1e5 macroparticles, 200 turns,
    fixed-point deposit -- at a bunch charge of 2.3e12, the paper's tune-shift regime, where
    the motion is regular: the oracle's own twin run (initial coordinates moved by one unit in the last place) stays far
    below 1e-3, so north_star's tolerance can be asked for as stated.  STRICT 1e-3 on the rms emittances of all three planes
    every 10 turns and on the mean and rms spread of the per-particle tunes; no twin-based widening."""
    gold = _golden("long_cfg3_paper.json")
    tw = gold["twin"]
    for turn, want in gold["emittances"].items():         # the regime is not chaotic: shown by the stored twin, not assumed
        for pl in range(3):
            assert abs(tw["emittances"][turn][pl] - want[pl]) < 1e-4 * want[pl]
    measured = _long_run(sc, gold, 3, strict=True)
    assert max(measured.values()) < 1e-3


def test_ten_turns_fixed_point_paper_regime(sc, orc):
    """north_star's 10-turn tolerance (1e-8 per particle) on the 6D path in FIXED-POINT deposit mode -- the mode bench.py times --
    at the paper-regime bunch charge: 20 000 macroparticles of cfg3's beam, 10 whole turns (2160 nodes), all six coordinates.
    The fixed-point flip allowance of DESIGN.md section 2 is added as in every fixed-mode tracking test."""
    wl = make_config(3, n=20_000, deposit_mode=1)
    wl.beam["n_real"] = 2.3e12
    want, _ = orc.track_workload(wl, n_turns=10)
    t = sc.Tracker.from_workload(wl)
    t.sc_load_particles(wl.particles)
    t.sc_track(10)
    got = t.sc_get_particles()
    t.close()
    tol = 1e-8 + allowance(wl)
    errs = {k: rel_err(got[k], want[k]) for k in NAMES}
    print("10 turns, fixed point, n_real 2.3e12: " + ", ".join(f"{k}={v:.2e}" for k, v in errs.items()) + f" (tolerance {tol:.2e})")
    for k in NAMES:
        assert errs[k] < tol, (k, errs[k])


def test_cfg3_thousand_turns_invariants(sc):
    """configs[2] literally: 1e6 macroparticles, 1000 turns (GPU only: the oracle would need four hours).  What holds
    at any size: particle count conserved, nothing non-finite, the deterministic deposit reproduces the run bit for bit
    (compared over 100 turns), emittance growth bounded (the literal intensity is far beyond the paper's regime: the beam
    blows up in the first turns and then evolves slowly; numbers recorded in DESIGN.md section 5)."""
    wl = make_config(3, deposit_mode=1)
    runs = []
    for rep in range(2):
        t = sc.Tracker.from_workload(wl)
        t.sc_load_particles(wl.particles)
        t.sc_track(100)
        runs.append(t.sc_get_particles())
        if rep == 1:
            m100 = t.sc_moments()
            t.sc_track(900)
            m = t.sc_moments()
            assert m[0] == wl.n and m[32] == 0
            assert m[31] < 0.05 * wl.n                        # particles outside the grid at the last node
            assert 0.9 * m100[28] < m[28] < 1.5 * m100[28] and 0.9 * m100[29] < m[29] < 1.5 * m100[29]
            print("cfg3 1000 turns: eps_x %.6e eps_y %.6e eps_s %.6e n_outside %d non-finite %d" % (m[28], m[29], m[30], m[31], m[32]))
        t.close()
    for k in NAMES:
        assert np.array_equal(runs[0][k], runs[1][k]), k


def test_fixed_point_allowance_is_measured(sc, orc):
    """DESIGN.md section 2, "fixed-point allowance": after transport the two sides' coordinates differ by rounding, so a
    quantised fraction llrint(f 2^s) now and then lands on the other side of a tie; every flip moves one particle's weight
    by 2^-s between two neighbouring cells (total charge stays exact).  Measured here after the 216 segments of one turn,
    at the LAST node, before its kick: number of differing cells, their size, and the coordinate error, against the
    allowance 16 * 2^-s / n that the fixed-mode tracking tests add to north_star's 1e-10."""
    for n, max_cells, err_budget in ((20_000, 40, 0.05), (1_000_000, 2000, 0.75)):
        wl = make_config(3, n=n, deposit_mode=1)
        s = wl.grids[0]["fixed_bits"]
        last = int(np.flatnonzero(wl.kind == SCNODE)[-1]) + 1
        want, works = orc.track_workload(wl, stop_after_rows=last)
        t = sc.Tracker.from_workload(wl)
        t.sc_load_particles(wl.particles)
        t.sc_step(last)
        got = t.sc_get_particles()
        d = t.sc_get_grid(sc.SC_GRID_RHO_I64).ravel() - works[0].Qi
        assert int(d.sum()) == 0                                            # charge exact whatever flipped
        assert np.count_nonzero(d) <= max_cells, np.count_nonzero(d)        # 4 cells per flip
        assert np.abs(d).max() <= 4 << s                                    # a few units of 2^s per cell
        tol = 1e-10 + 16 * 2.0 ** -s / n
        worst = max(rel_err(got[k], want[k]) for k in NAMES)
        assert worst < err_budget * tol, (n, worst, tol)                    # measured: 4e-13 (no flip) and 7e-11
        t.close()


