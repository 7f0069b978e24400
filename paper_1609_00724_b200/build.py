"""In-tree build of libqsl.so (hand-written CUDA for sm_100a) with nvcc.  `python -m paper_1609_00724_b200.build`."""
from __future__ import annotations

import concurrent.futures
import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libqsl.so")
PEAKS_SRC = os.path.join(HERE, "peaks", "peaks.cu")       # bench utility, a library of its own (include/qsl_peaks.h)
PEAKS_LIB = os.path.join(HERE, "libqsl_peaks.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-DQSL_TARGET_ARCH=100", "-I" + os.path.join(ROOT, "include"), "-I" + CSRC]
NVCC_FLAGS += os.environ.get("QSL_NVCC_EXTRA", "").split()      # e.g. -DQSL_T2_MIN_BLOCKS=2 for tuning experiments


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stamp() -> str:
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(CSRC, "*.cu*")) + [PEAKS_SRC, os.path.join(ROOT, "include", "qsl.h"),
                     os.path.join(ROOT, "include", "qsl_peaks.h")]):
        h.update(f.encode()); h.update(open(f, "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp_file = os.path.join(OBJ, "stamp")
    stamp = _stamp()
    if (not force and os.path.exists(LIB) and os.path.exists(PEAKS_LIB) and os.path.exists(stamp_file)
            and open(stamp_file).read() == stamp):
        return LIB
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    nvcc = _nvcc()

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
        if verbose and (r.stdout or r.stderr):
            print(r.stdout, r.stderr, file=sys.stderr)
        return obj

    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, len(srcs) + 1)) as ex:
        objs = list(ex.map(compile_one, srcs + [PEAKS_SRC]))
    for lib, parts in ((LIB, objs[:-1]), (PEAKS_LIB, objs[-1:])):
        r = subprocess.run([nvcc, "-shared", "-o", lib, *parts], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link of %s failed:\n%s\n%s" % (lib, r.stdout, r.stderr))
    with open(stamp_file, "w") as f:
        f.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
