"""Thin ctypes binding of libsc_track (include/sc_track.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for exactly two
things: the device workspace (one uint8 tensor from the caching allocator, handed to sc_create)
and the CUDA stream the library works on.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SC_TRACK_LIB") or os.path.join(_HERE, "libsc_track.so")   # SC_TRACK_LIB: another build of the same library (the checked one)

SC_DRIFT, SC_LINMAP, SC_MULT, SC_RF, SC_SCNODE, SC_QUAD, SC_CQUAD, SC_SEXT, SC_XDRIFT, SC_SBEND = 0, 1, 2, 3, 4, 5, 6, 7, 8, 9
SC_DEPOSIT_F64, SC_DEPOSIT_FIXED = 0, 1
SC_GRID_RHO_F64, SC_GRID_RHO_I64, SC_GRID_PHI, SC_GRID_EX, SC_GRID_EY, SC_GRID_LAMBDA = range(6)
SC_N_MOMENTS = 33
SC_MOMENTS_STATIC_MAX_PARTICLES = 1 << 24
SC_FLAG_NO_PDL = 1
SC_FLAG_FUSED_POISSON = 2
SC_FLAG_NO_FIELD_WINDOW = 4
SC_FLAG_BLOCK_FFT_POISSON = 8
SC_FLAG_WARP_FFT_POISSON = 16
SC_REPLAY_TURN, SC_REPLAY_PUSH, SC_REPLAY_POISSON, SC_REPLAY_EMPTY = 0, 1, 2, 3
SC_BOUNDARY_OPEN, SC_BOUNDARY_PIPE = 0, 1
SC_INTERP_BILINEAR, SC_INTERP_BICUBIC = 0, 1
ERRORS = {0: "SC_OK", -1: "SC_EINVAL", -2: "SC_ENOMEM", -3: "SC_ECUDA", -4: "SC_ESTATE", -5: "SC_EUNSUPPORTED"}

EXPORTS = ["sc_workspace_bytes", "sc_create", "sc_load_particles", "sc_track", "sc_step", "sc_get_particles",
           "sc_get_grid", "sc_moments", "sc_moments_static", "sc_profile_turn", "sc_profile_replay", "sc_profile_copy", "sc_get_constants", "sc_kernel_launches", "sc_abi_sizes", "sc_last_error", "sc_destroy"]


class sc_elem(C.Structure):
    _fields_ = [("kind", C.c_int32), ("ipar", C.c_int32), ("p", C.c_double * 10)]


class sc_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("xmin", C.c_double), ("xmax", C.c_double),
                ("ymin", C.c_double), ("ymax", C.c_double), ("nbins", C.c_int32), ("smin", C.c_double),
                ("smax", C.c_double), ("deposit_mode", C.c_int32), ("fixed_bits", C.c_int32),
                ("boundary", C.c_int32), ("long_kick", C.c_int32), ("interp", C.c_int32)]


class sc_beam(C.Structure):
    _fields_ = [("kinetic_eV", C.c_double), ("mass_eV", C.c_double), ("charge", C.c_int32),
                ("line_density", C.c_double), ("n_real", C.c_double), ("circumference", C.c_double)]


class ScError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


_lib = None
c_dp = C.POINTER(C.c_double)


def load_library() -> C.CDLL:
    """dlopen libsc_track.so (built in-tree by paper_2010_11540_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2010_11540_b200.build` "
                          "(there is no CPU fallback for the CUDA path)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
    lib.sc_workspace_bytes.argtypes = [C.POINTER(sc_elem), i64, C.POINTER(sc_grid), i32, i64, C.POINTER(i64)]
    lib.sc_create.argtypes = [C.POINTER(vp), C.POINTER(sc_elem), i64, C.POINTER(sc_grid), i32, C.POINTER(sc_beam),
                              i64, vp, i64, vp, u64]
    lib.sc_load_particles.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i32]
    lib.sc_track.argtypes = [vp, i64]
    lib.sc_step.argtypes = [vp, i64]
    lib.sc_get_particles.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32]
    lib.sc_get_grid.argtypes = [vp, i32, i32, vp, i64]
    lib.sc_moments.argtypes = [vp, c_dp, i32]
    lib.sc_moments_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp]
    lib.sc_get_constants.argtypes = [vp, c_dp, i32]
    lib.sc_profile_turn.argtypes = [vp, c_dp, i32]
    lib.sc_profile_replay.argtypes = [vp, i32, i32, vp, i64, c_dp, i32]
    lib.sc_profile_copy.argtypes = [vp, i32, vp, i64, c_dp, i32]
    lib.sc_kernel_launches.argtypes = [vp]
    lib.sc_kernel_launches.restype = i64
    lib.sc_last_error.argtypes = [vp]
    lib.sc_last_error.restype = C.c_char_p
    lib.sc_destroy.argtypes = [vp]
    lib.sc_destroy.restype = None
    for name in EXPORTS:
        if name not in ("sc_kernel_launches", "sc_last_error", "sc_destroy"):
            getattr(lib, name).restype = C.c_int
    lib.sc_abi_sizes.argtypes = [C.POINTER(C.c_int32), i32]
    sizes = (C.c_int32 * 3)()
    if lib.sc_abi_sizes(sizes, 3) or list(sizes) != [C.sizeof(sc_elem), C.sizeof(sc_grid), C.sizeof(sc_beam)]:
        raise ImportError(f"{LIB_PATH} was built from another include/sc_track.h (struct sizes {list(sizes)}): rebuild it")
    _lib = lib
    return lib


def _elems(kind, ipar, par) -> C.Array:
    n = len(kind)
    arr = (sc_elem * n)()
    for r in range(n):
        arr[r].kind = int(kind[r])
        arr[r].ipar = int(ipar[r])
        for k in range(10):
            arr[r].p[k] = float(par[r][k])
    return arr


def _grids(grids: Sequence[Dict]) -> C.Array:
    arr = (sc_grid * max(1, len(grids)))()
    for i, g in enumerate(grids):
        arr[i] = sc_grid(g["nx"], g["ny"], g["xmin"], g["xmax"], g["ymin"], g["ymax"], g.get("nbins", 0),
                         g.get("smin", 0.0), g.get("smax", 0.0), g.get("deposit_mode", 0), g.get("fixed_bits", 19),
                         g.get("boundary", 0), g.get("long_kick", 0), g.get("interp", 0))
    return arr


def _beam(b: Dict) -> sc_beam:
    return sc_beam(b["kinetic_eV"], b["mass_eV"], b["charge"], b.get("line_density", 0.0), b.get("n_real", 0.0),
                   b.get("circumference", 0.0))


def sc_moments_static(p: Dict, out, stream=None) -> None:
    """sc_moments_static of include/sc_track.h: the 33 moments of particle arrays that are already on the GPU, for
    callers that must not allocate device memory (no context, no workspace; the partial sums go into an array built
    into the library, which limits n to SC_MOMENTS_STATIC_MAX_PARTICLES).  p: dict x, px, y, py, sigma, psigma of
    contiguous torch CUDA float64 tensors (sigma and psigma None for a 4D beam); out: a torch CUDA float64 tensor of
    at least SC_N_MOMENTS elements, written asynchronously on `stream` (default: torch's current stream).  This wrapper
    only marshals pointers: it allocates nothing either.  Calls that can overlap on the GPU must be ordered by the
    caller (they share the built-in array)."""
    import torch
    lib = load_library()
    names = ("x", "px", "y", "py", "sigma", "psigma")
    ptrs = []
    n = int(p["x"].shape[0])
    for k in names:
        a = p.get(k)
        if a is None:
            ptrs.append(C.c_void_p(0))
        else:
            if not (a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and a.shape[0] == n):
                raise ValueError(f"{k}: contiguous CUDA float64 tensor of {n} elements expected")
            ptrs.append(C.c_void_p(a.data_ptr()))
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= SC_N_MOMENTS):
        raise ValueError("out: contiguous CUDA float64 tensor of at least SC_N_MOMENTS elements expected")
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib.sc_moments_static(*ptrs, n, C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc:
        raise ScError(rc, lib.sc_last_error(None).decode())


class Tracker:
    """sc_create ... sc_destroy as an object.  Particle arrays go in and out as numpy (host) arrays or
    torch CUDA tensors (device pointers, no host round trip)."""

    def __init__(self, kind, ipar, par, grids: List[Dict], beam: Dict, max_particles: int, stream=None, flags: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2010_11540_b200 needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self._torch = torch
        self.grids = [dict(g) for g in grids]
        self.n_rows = len(kind)
        self.max_particles = int(max_particles)
        self._el = _elems(kind, ipar, par)
        self._gr = _grids(grids)
        self._bm = _beam(beam)
        nbytes = C.c_int64(0)
        rc = self.lib.sc_workspace_bytes(self._el, self.n_rows, self._gr, len(grids), self.max_particles, C.byref(nbytes))
        if rc:
            raise ScError(rc, self.lib.sc_last_error(None).decode())
        # device memory and stream come from torch (plumbing); a dedicated stream so that whole turns
        # can be captured into CUDA graphs (the legacy default stream cannot be captured)
        self.stream = stream if stream is not None else torch.cuda.Stream()
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device="cuda")
        base = (self.workspace.data_ptr() + 255) & ~255
        self.stream.wait_stream(torch.cuda.current_stream())
        h = C.c_void_p()
        rc = self.lib.sc_create(C.byref(h), self._el, self.n_rows, self._gr, len(grids), C.byref(self._bm),
                                self.max_particles, C.c_void_p(base), nbytes.value, C.c_void_p(self.stream.cuda_stream), int(flags))
        if rc:
            raise ScError(rc, self.lib.sc_last_error(None).decode())
        self.h = h
        self.n = 0
        self.sixd = False

    @classmethod
    def from_workload(cls, wl, max_particles: Optional[int] = None, stream=None, flags: int = 0) -> "Tracker":
        return cls(wl.kind, wl.ipar, wl.par, wl.grids, wl.beam, max_particles or wl.n, stream, flags)

    def _check(self, rc: int):
        if rc:
            raise ScError(rc, self.lib.sc_last_error(self.h).decode())

    # ---- the C calls, same names
    def sc_load_particles(self, p: Dict):
        """p: dict x, px, y, py, sigma, psigma of numpy float64 arrays (host) or torch CUDA float64
        tensors (device); sigma/psigma None for a 4D beam."""
        torch = self._torch
        names = ("x", "px", "y", "py", "sigma", "psigma")
        on_dev = isinstance(p["x"], torch.Tensor)
        ptrs, keep = [], []
        for k in names:
            a = p.get(k)
            if a is None:
                ptrs.append(C.c_void_p(0))
            elif on_dev:
                assert a.is_cuda and a.dtype == torch.float64 and a.is_contiguous()
                keep.append(a)
                ptrs.append(C.c_void_p(a.data_ptr()))
            else:
                a = np.ascontiguousarray(a, np.float64)
                keep.append(a)
                ptrs.append(C.c_void_p(a.ctypes.data))
        n = int(keep[0].shape[0])
        if on_dev:
            self.stream.wait_stream(torch.cuda.current_stream())
        self._check(self.lib.sc_load_particles(self.h, *ptrs, n, int(on_dev)))
        if on_dev:
            self.stream.synchronize()      # the source tensors may be freed by the caller
        self.n = n
        self.sixd = p.get("sigma") is not None

    def sc_track(self, n_turns: int):
        self._check(self.lib.sc_track(self.h, int(n_turns)))

    def sc_step(self, n_rows: int):
        self._check(self.lib.sc_step(self.h, int(n_rows)))

    def sc_get_particles(self, device: bool = False) -> Dict:
        names = ("x", "px", "y", "py", "sigma", "psigma")
        ncoord = 6 if self.sixd else 4
        out: Dict = {k: None for k in names}
        ptrs = []
        if device:
            torch = self._torch
            with torch.cuda.stream(self.stream):
                for k in names[:ncoord]:
                    out[k] = torch.empty(self.n, dtype=torch.float64, device="cuda")
            ptrs = [C.c_void_p(out[k].data_ptr()) if out[k] is not None else C.c_void_p(0) for k in names]
        else:
            for k in names[:ncoord]:
                out[k] = np.empty(self.n, np.float64)
            ptrs = [C.c_void_p(out[k].ctypes.data) if out[k] is not None else C.c_void_p(0) for k in names]
        self._check(self.lib.sc_get_particles(self.h, *ptrs, int(device)))
        return out

    def sc_get_grid(self, which: int, grid_id: int = 0) -> np.ndarray:
        g = self.grids[grid_id]
        if which == SC_GRID_LAMBDA:
            out = np.zeros(max(1, g.get("nbins", 0)), np.int64)
            self._check(self.lib.sc_get_grid(self.h, grid_id, which, C.c_void_p(out.ctypes.data), out.nbytes))
            return out[:g.get("nbins", 0)]
        dt = np.int64 if which == SC_GRID_RHO_I64 else np.float64
        out = np.zeros((g["ny"], g["nx"]), dt)
        self._check(self.lib.sc_get_grid(self.h, grid_id, which, C.c_void_p(out.ctypes.data), out.nbytes))
        return out

    def sc_moments(self) -> np.ndarray:
        out = np.zeros(SC_N_MOMENTS)
        self._check(self.lib.sc_moments(self.h, out.ctypes.data_as(c_dp), SC_N_MOMENTS))
        return out

    def sc_profile_turn(self) -> Dict[str, float]:
        out = np.zeros(5)
        self._check(self.lib.sc_profile_turn(self.h, out.ctypes.data_as(c_dp), 5))
        return dict(push_ms=out[0], n_push=int(out[1]), poisson_ms=out[2], n_poisson=int(out[3]), turn_ms=out[4])

    def _scratch(self):
        """device scratch for the measurement hooks: 8 bytes x coordinates x n (rounded up to even), from torch"""
        nbytes = 8 * (6 if self.sixd else 4) * (self.n + 2) + 256
        if getattr(self, "_scr", None) is None or self._scr.numel() < nbytes:
            self._scr = self._torch.empty(nbytes, dtype=self._torch.uint8, device="cuda")
            self._torch.cuda.current_stream().synchronize()
        base = (self._scr.data_ptr() + 255) & ~255
        return C.c_void_p(base), self._scr.numel() - 256

    def sc_profile_replay(self, mode: int, reps: int = 5) -> Dict[str, float]:
        out = np.zeros(7)
        ptr, nb = self._scratch()
        self._check(self.lib.sc_profile_replay(self.h, int(mode), int(reps), ptr, nb, out.ctypes.data_as(c_dp), 7))
        return dict(turn_ms=out[0], n_kernels=int(out[1]), n_nodes=int(out[2]), n_outside=out[3], reps=int(out[4]), n=int(out[5]),
                    n_psigma_stores=int(out[6]))

    def sc_profile_copy(self, reps: int = 5) -> Dict[str, float]:
        out = np.zeros(2)
        ptr, nb = self._scratch()
        self._check(self.lib.sc_profile_copy(self.h, int(reps), ptr, nb, out.ctypes.data_as(c_dp), 2))
        return dict(copy_ms=out[0], bytes=out[1])

    def sc_get_constants(self) -> Dict[str, float]:
        out = np.zeros(6)
        self._check(self.lib.sc_get_constants(self.h, out.ctypes.data_as(c_dp), 6))
        return dict(zip(("gamma0", "beta0", "E0_eV", "r_c", "kappa", "circumference"), out))

    def sc_kernel_launches(self) -> int:
        return int(self.lib.sc_kernel_launches(self.h))

    def synchronize(self):
        self.stream.synchronize()

    def sc_destroy(self):
        if getattr(self, "h", None) is not None and self.h:
            self.stream.synchronize()
            self.lib.sc_destroy(self.h)
            self.h = None

    close = sc_destroy

    def __del__(self):
        try:
            self.sc_destroy()
        except Exception:
            pass
