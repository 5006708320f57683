"""Build libepr.so (hand-written CUDA, sm_100a) in-tree with nvcc.  `python -m paper_2601_22793_b200.build`.

Every translation unit is compiled to an object in parallel (the FFT kernels are instantiated in
FFT_GROUPS units from the same source, -DEPR_FFT_GROUP=g), then linked into one shared library."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libepr.so")
FFT_GROUPS = 11
# (source, object stem, extra flags)
UNITS = [("epr_api.cu", "epr_api", []), ("epr_kernels.cu", "epr_kernels", []), ("epr_fftd.cu", "epr_fftd", []),
         ("epr_general.cu", "epr_general", []), ("epr_fftgen.cu", "epr_fftgen", []),
         ("epr_static.cu", "epr_static", [])] + \
        [("epr_fftk.cu", f"epr_fftk_g{g}", [f"-DEPR_FFT_GROUP={g}"]) for g in range(FFT_GROUPS)]
HEADERS = ["epr_internal.h", "epr_math.cuh", "epr_fft.cuh", "epr_tma.cuh", os.path.join("..", "..", "include", "epr.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _newest_header():
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _compile(unit, nvcc, force, verbose, hdr_t):
    src, stem, extra = unit
    obj = os.path.join(OBJ, stem + ".o")
    src_p = os.path.join(CSRC, src)
    if not force and os.path.exists(obj) and os.path.getmtime(obj) > max(os.path.getmtime(src_p), hdr_t):
        return obj, ""
    cmd = [nvcc] + NVCC_FLAGS + os.environ.get("EPR_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + extra + ["-c", src, "-o", obj]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src} {extra}:\n" + res.stdout + res.stderr)
    return obj, res.stderr


def build(force=False, verbose=False, dev=False):
    """Compile what is missing or older than its sources, link, return the library path.
    dev=True: developer build with FFT group 0 only (2048, 16, 32) — seconds instead of a minute; never ship it."""
    os.makedirs(OBJ, exist_ok=True)
    nvcc = os.environ.get("NVCC", "nvcc")
    hdr_t = _newest_header()
    units = UNITS
    if dev:
        units = [u for u in UNITS if u[0] != "epr_fftk.cu" or u[1].endswith("_g0")]
        units = [(s, st + "_dev", ex + ["-DEPR_FFT_DEV"]) if s == "epr_fftd.cu" else (s, st, ex) for s, st, ex in units]
    with ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 4)) as ex:
        results = list(ex.map(lambda u: _compile(u, nvcc, force, verbose, hdr_t), units))
    objs = [o for o, _ in results]
    if verbose:
        sys.stderr.write("".join(log for _, log in results))
    if True:  # always relink: a dev and a full build share the output name
        res = subprocess.run([nvcc, "-shared", "-o", LIB] + objs, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, dev="--dev" in sys.argv))
