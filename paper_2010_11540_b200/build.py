"""Build libsc_track.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_2010_11540_b200.build          # -> paper_2010_11540_b200/libsc_track.so

nvcc cross-compiles without a GPU.  -lineinfo keeps ncu's source page mapped to csrc/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsc_track.so")
SOURCES = ["sc_track.cu", "sc_moments_static.cu"]
DEPS = ["sc_track.cu", "sc_moments_static.cu", "sc_host.h", "sc_device.cuh", "k_push.cuh", "k_poisson.cuh", "k_poisson_fused.cuh", "k_poisson_warp.cuh", "k_poisson_cluster.cuh", "k_moments.cuh",
        os.path.join("..", "..", "include", "sc_track.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


LIB_CHECK = os.path.join(HERE, "libsc_track_check.so")
LIB_TRACE = os.path.join(HERE, "libsc_track_trace.so")


def build(force: bool = False, verbose: bool = False, check: bool = False, trace: bool = False) -> str:
    """check=True: the checked build (-DSC_CHECK: device-side index assertions, sc_device.cuh) -> libsc_track_check.so.
    trace=True: the tracing build (-DSC_TRACE: global-timer stamps at the kernels' phase boundaries, read by
    paper_2010_11540_b200.trace) -> libsc_track_trace.so."""
    if check or trace:
        cmd = [_nvcc()] + NVCC_FLAGS + ["-DSC_CHECK" if check else "-DSC_TRACE", "-o", LIB_CHECK if check else LIB_TRACE] + [os.path.join(CSRC, s) for s in SOURCES]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        return LIB_CHECK if check else LIB_TRACE
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    with open(os.path.join(HERE, "ptxas_info.txt"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv, check="--check" in sys.argv, trace="--trace" in sys.argv))
