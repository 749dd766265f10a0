"""Build libgmapp.so in-tree for sm_100a: ten translation units compiled in parallel, then linked.

Stand-alone on purpose (no import of the binding: api.py refuses to import while the library is missing):
    python paper_2606_12579_b200/build_lib.py [--force]
nvcc cross-compiles without a GPU."""
import os
import subprocess
import sys

_PKG = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_PKG, "csrc")
_INCLUDE = os.path.join(os.path.dirname(_PKG), "include")
SO = os.path.join(_PKG, "libgmapp.so")
TUS = ["gmapp.cu", "gmapp_wide.cu"] + ["gmapp_x2_%s%s%s.cu" % (h, x, m) for m in ("", "_mv") for h in ("cf", "apf") for x in ("", "_x")]
NVCC = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
        "-diag-suppress", "128"]          # 128: "loop is not reachable" in the if-constant branches of the templates


def nvcc_commands(out: str = SO, extra=(), objdir=None):
    """The compile commands (one per translation unit) and the link command."""
    objdir = objdir or os.path.join(_PKG, "build")
    objs = [os.path.join(objdir, tu.replace(".cu", ".o")) for tu in TUS]
    compiles = [[*NVCC, "-I", _INCLUDE, *extra, "-c", "-o", o, os.path.join(_CSRC, tu)] for tu, o in zip(TUS, objs)]
    link = [*NVCC, "-shared", "-o", out, *objs]
    return compiles, link


def stale() -> bool:
    srcs = [os.path.join(_CSRC, f) for f in os.listdir(_CSRC)] + [os.path.join(_INCLUDE, "gmapp.h")]
    return not os.path.exists(SO) or os.path.getmtime(SO) < max(os.path.getmtime(f) for f in srcs)


def build(force: bool = False, extra=(), out: str = SO) -> str:
    if force or out != SO or stale():
        compiles, link = nvcc_commands(out=out, extra=extra)
        os.makedirs(os.path.join(_PKG, "build"), exist_ok=True)
        procs = [subprocess.Popen(c) for c in compiles]
        rcs = [p.wait() for p in procs]
        if any(rcs):
            raise subprocess.CalledProcessError(max(rcs), compiles[rcs.index(max(rcs))])
        subprocess.check_call(link)
    return out


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print(SO)
