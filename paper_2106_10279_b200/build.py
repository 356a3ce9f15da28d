"""Builds paper_2106_10279_b200/libmadflow_b200.so (the C-ABI library of include/mf.h) in-tree with nvcc for
sm_100a.  No GPU is needed to build (nvcc cross-compiles).

    python -m paper_2106_10279_b200.build [--force] [--verbose]

Steps: (1) csrc/gen_me.py, csrc/gen_coop.py and csrc/gen_coop3.py write the straight-line matrix-element code (the role of the paper's exporter
plugin); (2) nvcc compiles csrc/madflow_b200.cu into the shared library.
"""
import glob
import importlib.util
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmadflow_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _sources():
    return (glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")) +
            glob.glob(os.path.join(CSRC, "*.py")) + [os.path.join(os.path.dirname(HERE), "include", "mf.h")])


def generate():
    """runs the build-time generators: gen_me.py (straight-line matrix elements) and gen_coop.py (the
    cooperative g g -> t tbar g g program); both only rewrite their header when its text changes"""
    out = []
    if CSRC not in sys.path:
        sys.path.insert(0, CSRC)          # gen_coop imports gen_me
    for name in ("gen_me", "gen_coop", "gen_coop3", "gen_cta5", "gen_qq_colour"):
        spec = importlib.util.spec_from_file_location(name, os.path.join(CSRC, name + ".py"))
        mod = importlib.util.module_from_spec(spec)
        sys.modules[name] = mod
        spec.loader.exec_module(mod)
        out.append(mod.main())
    return out


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _sources())


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    generate()
    extra = os.environ.get("MF_NVCC_EXTRA", "").split()        # e.g. -DMF_COOP_GROUP=2 (tuning experiments)
    cmd = [NVCC] + FLAGS + extra + ["-o", LIB, os.path.join(CSRC, "madflow_b200.cu")]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed (see %s)" % log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
