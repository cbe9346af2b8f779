"""In-tree builds (no JIT cache) of the sm_100a libraries with nvcc.

  librt.so      paper_2404_17630_b200/csrc/*.cu      the product: C-ABI of include/rt.h
  _meshgen.so   paper_2404_17630_b200/inputs/csrc    input generator (host OpenMP + device)

(The C oracle has its own oracle/build.py; nothing here touches oracle/.)
`python -m paper_2404_17630_b200.build [rt|meshgen|all]`.  A target is rebuilt when
any of its sources is newer than the library.
"""
import glob
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2404_17630_b200")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]

RT_SO = os.path.join(PKG, "librt.so")
MESHGEN_SO = os.path.join(PKG, "inputs", "_meshgen.so")


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build_rt(force=False, verbose=False):
    src = sorted(glob.glob(os.path.join(PKG, "csrc", "*.cu")))
    dep = src + glob.glob(os.path.join(PKG, "csrc", "*.cuh")) + glob.glob(os.path.join(ROOT, "include", "*.h"))
    if force or _stale(RT_SO, dep):
        out = _run([NVCC, "-O3", "-std=c++17", "-lineinfo", "-Xptxas", "-v", *ARCH, "-shared", "-Xcompiler", "-fPIC",
                    "-I", os.path.join(ROOT, "include"), "-o", RT_SO, *src, "-lcudart"])
        if verbose:
            print(out)
    return RT_SO


def build_meshgen(force=False):
    d = os.path.join(PKG, "inputs", "csrc")
    src = [os.path.join(d, "meshgen.cu")]
    dep = src + [os.path.join(d, "voronoi_cell.h")]
    if force or _stale(MESHGEN_SO, dep):
        _run([NVCC, "-O2", "-std=c++17", "-lineinfo", *ARCH, "-shared", "-Xcompiler", "-fPIC,-fopenmp",
              "-o", MESHGEN_SO, *src, "-lcudart", "-lgomp"])
    return MESHGEN_SO


def build_all(force=False):
    return build_rt(force), build_meshgen(force)


if __name__ == "__main__":
    what = sys.argv[1] if len(sys.argv) > 1 else "all"
    force = "--force" in sys.argv
    if what in ("rt", "all"):
        print(build_rt(force, verbose=True))
    if what in ("meshgen", "all"):
        print(build_meshgen(force))
