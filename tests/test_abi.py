"""CPU-side checks of the C-ABI boundary (no GPU, no compute calls): the library builds, loads and
exports every symbol include/sc_track.h declares; the POD layouts the binding marshals match the
header; host-side validation answers with error codes (never exceptions); and without a CUDA device
the product path fails loudly instead of falling back to anything."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2010_11540_b200 as sc
from paper_2010_11540_b200 import binding, build
from workloads import make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sc_track.h")


@pytest.fixture(scope="module")
def lib():
    build.build()
    return sc.load_library()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sc_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert {"sc_create", "sc_load_particles", "sc_track", "sc_moments", "sc_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/sc_track.h but not exported"
    assert sorted(sc.EXPORTS) == names, "binding.EXPORTS and the header disagree"


def test_pod_layouts_match_the_header():
    assert C.sizeof(binding.sc_elem) == 88                    # int32 kind, ipar + 10 doubles
    assert binding.sc_elem.p.offset == 8
    assert C.sizeof(binding.sc_grid) == 88                    # + int32 boundary, long_kick, interp, padding
    assert binding.sc_grid.boundary.offset == 72
    assert binding.sc_grid.interp.offset == 80
    assert C.sizeof(binding.sc_beam) == 48


def test_pod_sizes_match_the_compiled_library(lib):
    out = (C.c_int32 * 3)()
    assert lib.sc_abi_sizes(out, 3) == 0
    assert list(out) == [C.sizeof(binding.sc_elem), C.sizeof(binding.sc_grid), C.sizeof(binding.sc_beam)]


def _args(wl, grids=None, nmax=None):
    el = binding._elems(wl.kind, wl.ipar, wl.par)
    gr = binding._grids(grids if grids is not None else wl.grids)
    return el, wl.n_rows, gr, len(grids if grids is not None else wl.grids), nmax or wl.n


def test_workspace_bytes_covers_the_particle_store(lib):
    wl = make_config(3, n=1000)
    el, nr, gr, ng, nmax = _args(wl, nmax=1_000_000)
    out = C.c_int64(0)
    assert lib.sc_workspace_bytes(el, nr, gr, ng, nmax, C.byref(out)) == 0
    assert out.value >= 6 * 8 * 1_000_000 + 128 * 128 * 8 * 4
    assert out.value < 6 * 8 * 1_000_000 + 64 * 1024 * 1024


@pytest.mark.parametrize("patch,code", [
    (dict(nx=100), -5),                 # not a power of two: SC_EUNSUPPORTED
    (dict(nx=1024), -5),
    (dict(xmax=-1.0), -1),              # empty extent: SC_EINVAL
    (dict(nbins=5000), -1),
    (dict(deposit_mode=7), -1),
    (dict(deposit_mode=1, fixed_bits=21), -1),
    (dict(boundary=2), -1),
    (dict(interp=2), -1),
])
def test_validation_codes(lib, patch, code):
    wl = make_config(1, n=16)
    g = dict(wl.grids[0], **patch)
    el, nr, gr, ng, nmax = _args(wl, grids=[g])
    out = C.c_int64(0)
    assert lib.sc_workspace_bytes(el, nr, gr, ng, nmax, C.byref(out)) == code
    assert lib.sc_last_error(None)       # a message, never NULL


def test_fixed_point_overflow_is_rejected(lib):
    """int64 accumulators: max_particles * 2^(2 fixed_bits) must stay below 2^63 (every particle in one cell)."""
    wl = make_config(1, n=16)
    out = C.c_int64(0)
    for bits, nmax, code in ((20, 8_388_607, 0), (20, 8_388_608, -1), (19, 33_554_431, 0), (19, 33_554_432, -1)):
        g = dict(wl.grids[0], deposit_mode=1, fixed_bits=bits)
        el, nr, gr, ng, _ = _args(wl, grids=[g])
        assert lib.sc_workspace_bytes(el, nr, gr, ng, nmax, C.byref(out)) == code, (bits, nmax)


def test_bad_table_rows_are_rejected(lib):
    wl = make_config(1, n=16)
    kind = wl.kind.copy(); kind[3] = 99
    el = binding._elems(kind, wl.ipar, wl.par)
    gr = binding._grids(wl.grids)
    out = C.c_int64(0)
    assert lib.sc_workspace_bytes(el, wl.n_rows, gr, 1, 16, C.byref(out)) == -1
    ipar = wl.ipar.copy(); ipar[np.argmax(wl.kind == 4)] = 3         # SCNODE -> grid that does not exist
    el = binding._elems(wl.kind, ipar, wl.par)
    assert lib.sc_workspace_bytes(el, wl.n_rows, gr, 1, 16, C.byref(out)) == -1
    assert lib.sc_workspace_bytes(None, 0, gr, 1, 16, C.byref(out)) == -1


def test_null_handles_are_safe(lib):
    lib.sc_destroy(None)
    assert lib.sc_track(None, 1) == -1
    assert lib.sc_kernel_launches(None) == 0
    assert lib.sc_last_error(None) is not None


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product fails loudly (SC_ECUDA from the C call, RuntimeError from the
    binding); it never routes through the oracle or any CPU path."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    wl = make_config(1, n=16)
    with pytest.raises(RuntimeError):
        sc.Tracker.from_workload(wl)
    el, nr, gr, ng, nmax = _args(wl)
    h = C.c_void_p()
    bm = binding._beam(wl.beam)
    rc = lib.sc_create(C.byref(h), el, nr, gr, ng, C.byref(bm), nmax, None, 0, None, 0)
    assert rc == -3 and not h.value
    assert b"no CPU fallback" in lib.sc_last_error(None)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2010_11540_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+\"[^\"]*oracle", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2010_11540_b200|#include\s+\"[^\"]*csrc", text, flags=re.M), f
