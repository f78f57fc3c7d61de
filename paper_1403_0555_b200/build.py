"""Build libu1gf.so (the CUDA path) in-tree with nvcc for sm_100a.

`python -m paper_1403_0555_b200.build [--force]` or via __graft_entry__.build().  nvcc cross-compiles without a
GPU; the .so is git-ignored but travels to the GPU box with the gpurun snapshot.

Ablation knobs: the environment variable U1GF_NVCC_DEFINES (e.g. "-DU1GF_LANES_R6_BRANCH -DU1GF_LANES_FIN_PRE=1")
is appended to the nvcc command line and forces a rebuild; the knobs are documented where they are used in csrc/ and
the commands that used them are recorded under profiles/.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libu1gf.so")
SOURCES = ["orbit.cu", "relax_generic.cu", "relax_lanes.cu", "relax_stream.cu", "count_copies.cu", "discovery.cu", "check_fp.cu", "peaks.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]
EXTRA_DEFINES = os.environ.get("U1GF_NVCC_DEFINES", "").split()


def _deps_mtime():
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".h") or f.endswith(".cuh")]
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "u1gf.h"))
    return max(os.path.getmtime(h) for h in hdrs)


def _compile(src, force, hdr_m):
    s = os.path.join(CSRC, src)
    o = os.path.join(OBJ, src.replace(".cu", ".o"))
    if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), hdr_m):
        return o, False
    log = o + ".log"
    with open(log, "w") as f:
        subprocess.run(["nvcc", *NVCC_FLAGS, *EXTRA_DEFINES, "-c", s, "-o", o], check=True, stdout=f, stderr=subprocess.STDOUT)
    return o, True


def build(force: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "defines.txt")
    old = open(stamp).read() if os.path.exists(stamp) else ""
    if old != " ".join(EXTRA_DEFINES):     # a different set of knobs than the objects were built with
        force = True
        with open(stamp, "w") as f:
            f.write(" ".join(EXTRA_DEFINES))
    hdr_m = _deps_mtime()
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        res = list(ex.map(lambda s: _compile(s, force, hdr_m), SOURCES))
    if force or any(r[1] for r in res) or not os.path.exists(LIB):
        subprocess.run(["nvcc", "-shared", "-o", LIB, *[r[0] for r in res],
                        "-gencode", "arch=compute_100a,code=sm_100a"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
