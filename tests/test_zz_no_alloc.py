"""sc_moments_static: the beam moments for callers that cannot allocate device memory.

Who those callers are: sc_moments() lives on a context, and a context lives in a device workspace that somebody must
allocate.  A diagnostics hook in a process whose allocator has already claimed the whole GPU for its pool, or a beam
monitor that runs while tracking streams are busy (cudaMalloc and cudaFree hold up every stream of the device), can do
neither.  sc_moments_static() takes particle arrays that are already on the GPU and keeps its per-CTA partial sums in
an array compiled into the library (0.66 MiB per GPU), which is why it has a size limit, SC_MOMENTS_STATIC_MAX_PARTICLES.

What is checked here: its 33 results against sc_moments() of a context holding the same particles -- the existing path,
which the other GPU tests compare with the oracle -- within the tolerances tests/test_gpu_sizes.py uses for moments
(means within 1e-9 of the coordinate's rms, second moments within 1e-9 of the product of the two rms values, emittances
1e-8 relative), on two calls in a row: the second call sees fewer particles than the first, so it finds the first
call's partial sums and completion counters still in the shared array and must not be affected by them.  A third call
covers the 4D beam.  Repeating a call must give the same bits.  The size limit and the argument checks answer with an
error code and a message before any device work, so that part runs without a GPU.

The file is named so that pytest collects it last: a failure here must not hide the parity tests under `pytest -x`.  It
does not depend on what ran before it (the first call on a device does its own one-time set-up) and passes alone in a
fresh process as well as at the end of the whole suite."""
import ctypes as C

import numpy as np
import pytest

from workloads import make_config

NAMES = ("x", "px", "y", "py", "sigma", "psigma")


def _lib():
    import paper_2010_11540_b200 as sc
    from paper_2010_11540_b200 import build
    build.build()
    return sc, sc.load_library()


def test_sizes_beyond_the_built_in_scratch_are_refused():
    """n above the limit, n < 1, missing pointers and a lone sigma are refused with SC_EINVAL and a message (no device
    work happens before these checks, so no GPU is needed)."""
    sc, lib = _lib()
    limit = sc.SC_MOMENTS_STATIC_MAX_PARTICLES
    assert limit == 1 << 24
    fake = C.c_void_p(4096)          # never dereferenced: the checks come first
    rc = lib.sc_moments_static(fake, fake, fake, fake, fake, fake, limit + 1, fake, None)
    assert rc == -1
    msg = lib.sc_last_error(None).decode()
    assert "SC_MOMENTS_STATIC_MAX_PARTICLES" in msg and str(limit) in msg and str(limit + 1) in msg
    assert lib.sc_moments_static(fake, fake, fake, fake, fake, fake, 0, fake, None) == -1
    assert lib.sc_moments_static(fake, fake, fake, fake, fake, None, 10, fake, None) == -1
    assert "sigma" in lib.sc_last_error(None).decode()
    assert lib.sc_moments_static(None, fake, fake, fake, fake, fake, 10, fake, None) == -1
    assert lib.sc_moments_static(fake, fake, fake, fake, fake, fake, 10, None, None) == -1


def _existing_path(sc, tracker, particles):
    """sc_moments() of a context that holds exactly these particles (no tracking: the moments of the arrays as given)."""
    tracker.sc_load_particles(particles)
    return tracker.sc_moments()


def _assert_moments_agree(got, want, ncoord):
    """The tolerances of tests/test_gpu_sizes.py::test_cfg3_full_size_one_turn for moments."""
    idx, m = {}, 7
    for r in range(6):
        for c in range(r, 6):
            idx[(r, c)] = m
            m += 1
    assert got[0] == want[0]
    rms = [np.sqrt(want[idx[(r, r)]]) for r in range(6)]
    for r in range(ncoord):
        assert abs(got[1 + r] - want[1 + r]) <= 1e-9 * rms[r], ("mean", r, got[1 + r], want[1 + r])
        for c in range(r, ncoord):
            assert abs(got[idx[(r, c)]] - want[idx[(r, c)]]) <= 1e-9 * rms[r] * rms[c], ("second moment", r, c)
    for r in range(ncoord, 6):          # absent coordinates count as zero on both paths
        assert got[1 + r] == 0.0 and want[1 + r] == 0.0
        for c in range(6):
            assert got[idx[(min(r, c), max(r, c))]] == 0.0
    npl = ncoord // 2
    assert np.allclose(got[28:28 + npl], want[28:28 + npl], rtol=1e-8, atol=0.0)
    assert np.all(got[28 + npl:31] == 0.0)
    assert got[31] == 0.0                # no context, no node: documented
    assert got[32] == want[32] == 0.0    # nothing non-finite


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    sc, _ = _lib()

    # cfg3's 6D bunch (the bench workload's beam), a ragged count spanning 49 CTA chunks of 4096 and a tail
    wl = make_config(3, n=200_003, deposit_mode=1)
    first = {k: np.ascontiguousarray(wl.particles[k]) for k in NAMES}
    # the second call: fewer particles (18 chunks), displaced and stretched so that every moment differs from the first's
    n2 = 70_001
    second = {k: np.ascontiguousarray(1.7 * first[k][::-1][:n2] + 0.3 * np.sqrt(np.mean(first[k] ** 2))) for k in NAMES}

    t = sc.Tracker.from_workload(wl)
    want1 = _existing_path(sc, t, first)
    want2 = _existing_path(sc, t, second)
    t.close()

    dev1 = {k: torch.from_numpy(v).cuda() for k, v in first.items()}
    dev2 = {k: torch.from_numpy(v).cuda() for k, v in second.items()}
    out1 = torch.full((sc.SC_N_MOMENTS,), float("nan"), dtype=torch.float64, device="cuda")
    out2 = torch.full((sc.SC_N_MOMENTS,), float("nan"), dtype=torch.float64, device="cuda")
    out1_again = torch.full((sc.SC_N_MOMENTS,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()

    # two calls in a row on one stream, nothing in between; then the first one once more
    sc.sc_moments_static(dev1, out1)
    sc.sc_moments_static(dev2, out2)
    sc.sc_moments_static(dev1, out1_again)
    torch.cuda.synchronize()
    got1, got2, got1_again = out1.cpu().numpy(), out2.cpu().numpy(), out1_again.cpu().numpy()

    assert want1[0] == 200_003 and want2[0] == n2
    _assert_moments_agree(got1, want1, 6)
    _assert_moments_agree(got2, want2, 6)
    assert np.array_equal(got1, got1_again), "a repeated call must give the same bits, whatever ran in between"
    # the inputs are read only
    for k in NAMES:
        assert np.array_equal(dev1[k].cpu().numpy(), first[k])


@pytest.mark.gpu
def test_4d_beam_and_a_single_chunk():
    """cfg2's coasting 4D beam (sigma = psigma = NULL) after a 6D call, and a beam smaller than one CTA's chunk."""
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    sc, _ = _lib()
    wl = make_config(2, n=50_021)
    four = {k: (None if wl.particles.get(k) is None else np.ascontiguousarray(wl.particles[k])) for k in NAMES}
    assert four["sigma"] is None and four["psigma"] is None
    t = sc.Tracker.from_workload(wl)
    want = _existing_path(sc, t, four)
    tiny = {k: (None if v is None else v[:37].copy()) for k, v in four.items()}
    want_tiny = _existing_path(sc, t, tiny)
    t.close()

    dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in four.items()}
    dev_tiny = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in tiny.items()}
    out = torch.full((sc.SC_N_MOMENTS,), float("nan"), dtype=torch.float64, device="cuda")
    out_tiny = torch.full((sc.SC_N_MOMENTS,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    sc.sc_moments_static(dev, out)
    sc.sc_moments_static(dev_tiny, out_tiny)
    torch.cuda.synchronize()
    _assert_moments_agree(out.cpu().numpy(), want, 4)
    _assert_moments_agree(out_tiny.cpu().numpy(), want_tiny, 4)
