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
LIB = os.path.join(HERE, "libu1gf.so")                   # the method: include/u1gf.h
LIB_MEASURE = os.path.join(HERE, "libu1gf_measure.so")   # roofline probes: include/u1gf_measure.h (not the method)
SOURCES = ["common.cu", "orbit.cu", "relax_generic.cu", "relax_lanes.cu", "relax_stream.cu", "relax_tma.cu", "count_copies.cu",
           "discovery.cu", "check_fp.cu", "host_calls.cu", "ensemble.cu", "merge.cu", "readout.cu"]
MEASURE_SOURCES = [("common.cu", "common_measure.o", ["-DU1GF_MEASURE_LIB"]), ("peaks.cu", "peaks.o", [])]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]
EXTRA_DEFINES = os.environ.get("U1GF_NVCC_DEFINES", "").split()


def _deps_mtime():
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".h") or f.endswith(".cuh")]
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "u1gf.h"))
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "u1gf_measure.h"))
    return max(os.path.getmtime(h) for h in hdrs)


def _compile(src, force, hdr_m, obj=None, extra=(), objdir=None):
    s = os.path.join(CSRC, src)
    o = os.path.join(objdir or OBJ, obj or src.replace(".cu", ".o"))
    if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), hdr_m):
        return o, False
    log = o + ".log"
    with open(log, "w") as f:
        r = subprocess.run(["nvcc", *NVCC_FLAGS, *EXTRA_DEFINES, *extra, "-c", s, "-o", o], stdout=f, stderr=subprocess.STDOUT)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n" + open(log).read()[-4000:])
    return o, True


def _link(lib, objs):
    subprocess.run(["nvcc", "-shared", "-o", lib, *objs, "-gencode", "arch=compute_100a,code=sm_100a"], check=True)


def build(force: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "defines.txt")
    old = open(stamp).read() if os.path.exists(stamp) else ""
    if old != " ".join(EXTRA_DEFINES):     # a different set of knobs than the objects were built with
        force = True
        with open(stamp, "w") as f:
            f.write(" ".join(EXTRA_DEFINES))
    hdr_m = _deps_mtime()
    jobs = [(src, None, ()) for src in SOURCES] + [(src, obj, tuple(extra)) for src, obj, extra in MEASURE_SOURCES]
    with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
        res = list(ex.map(lambda j: _compile(j[0], force, hdr_m, j[1], j[2]), jobs))
    main, meas = res[:len(SOURCES)], res[len(SOURCES):]
    if force or any(r[1] for r in main) or not os.path.exists(LIB):
        _link(LIB, [r[0] for r in main])
    if force or any(r[1] for r in meas) or not os.path.exists(LIB_MEASURE):
        _link(LIB_MEASURE, [r[0] for r in meas])
    return LIB


def build_variant(name: str, defines, sources=("relax_lanes.cu",)) -> str:
    """libu1gf_<name>.so: the method library with `sources` recompiled under extra -D flags (the other objects are
    those of the regular build).  Used by tests that need a compile-time knob (the R6 redo path)."""
    build()
    vdir = os.path.join(OBJ, "variant_" + name)
    os.makedirs(vdir, exist_ok=True)
    hdr_m = _deps_mtime()
    objs = []
    for src in SOURCES:
        if src in sources:
            objs.append(_compile(src, False, hdr_m, extra=tuple(defines), objdir=vdir)[0])
        else:
            objs.append(os.path.join(OBJ, src.replace(".cu", ".o")))
    lib = os.path.join(HERE, f"libu1gf_{name}.so")
    if not os.path.exists(lib) or any(os.path.getmtime(o) > os.path.getmtime(lib) for o in objs):
        _link(lib, objs)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
