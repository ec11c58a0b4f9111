"""Seeded synthetic inputs (lattice tables, grids, beams) shaped like the paper's workloads.

This module serves BOTH the oracle (oracle/) and the CUDA path (paper_2010_11540_b200/): it only
*describes* inputs -- table rows as (kind, ipar, 10 parameters), grid/beam specs as plain dicts,
particle coordinates as numpy arrays -- and holds none of the method's arithmetic (no transfer
maps, no deposit, no Poisson solve, no kick).  Optics numbers a recipe needs (focal lengths,
quadrupole strengths, Twiss parameters at the injection point) are constants taken from
SURVEY.md section 8(d) (they were obtained with throw-away numpy probes) and are cited there.

The paper's own workload is the J-PARC Main Ring tracked from a SAD lattice (PAPER.md:312-342,
Tables I/II); that lattice is not available, so the five configurations of BASELINE.json stand in
for it (same sizes: 1e4-1e7 macroparticles, 64^2-512^2 grids, hundreds to thousands of table rows
per turn, 3 GeV protons, C = 1567.5 m, h = 9).  See DESIGN.md "Input recipe".
"""
from .configs import (DRIFT, LINMAP, MULT, RF, SCNODE, QUAD, CQUAD, SEXT, XDRIFT, SBEND, KIND_NAMES, Workload, make_config,
                      make_grid, make_beam_spec, rows_to_arrays, rng_uniform, rng_normal)

__all__ = ["DRIFT", "LINMAP", "MULT", "RF", "SCNODE", "QUAD", "CQUAD", "SEXT", "XDRIFT", "SBEND", "KIND_NAMES", "Workload", "make_config",
           "make_grid", "make_beam_spec", "rows_to_arrays", "rng_uniform", "rng_normal"]
