"""In-tree build of the two shared libraries (no pip, no JIT cache):

  libxy_levy.so   host-only Levy-graph builder / colouring   (g++)
  libxy_b200.so   the C-ABI hot-path library, sm_100a only   (nvcc -gencode arch=compute_100a,code=sm_100a)

Both are rebuilt only when a source is newer than the library (libxy_b200.so: per translation unit, objects in build/).  __graft_entry__.build() calls
build_all(); the bindings call the per-library functions lazily and fail loudly if a build fails.
"""
import os
import shutil
import subprocess

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
INCLUDE = os.path.join(ROOT, "include")

LEVY_LIB = os.path.join(PKG, "libxy_levy.so")
XY_LIB = os.path.join(PKG, "libxy_b200.so")

NVCC_ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _stale(lib, sources):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(s) > t for s in sources)


def _sources(patterns):
    out = []
    for d, exts in patterns:
        for f in sorted(os.listdir(d)):
            if f.endswith(exts):
                out.append(os.path.join(d, f))
    return out


def build_levy(force=False, verbose=False):
    src = [os.path.join(CSRC, "levy_graph.cpp")]
    deps = src + [os.path.join(INCLUDE, "xy_levy.h")]
    if force or _stale(LEVY_LIB, deps):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-Wall", "-Wextra",
               "-I", INCLUDE, *src, "-o", LEVY_LIB]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
    return LEVY_LIB


def nvcc_path():
    for p in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if p and os.path.exists(p):
            return p
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def build_xy(force=False, verbose=False, extra_flags=()):
    """nvcc every csrc/*.cu into build/*.o (in parallel: the kernel instantiations are spread over xy_inst_*.cu so that
    they compile side by side) and link libxy_b200.so.  An object is rebuilt when its source or any header is newer."""
    from concurrent.futures import ThreadPoolExecutor
    srcs = _sources([(CSRC, (".cu",))])
    hdrs = _sources([(CSRC, (".cuh", ".h")), (INCLUDE, (".h",))])
    if not force and not _stale(XY_LIB, srcs + hdrs):
        return XY_LIB
    objdir = os.path.join(PKG, "build")
    os.makedirs(objdir, exist_ok=True)
    nvcc = nvcc_path()
    flags = [*NVCC_ARCH, "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v" if verbose else "-O3",
             "-I", INCLUDE, "-I", CSRC, *extra_flags]

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        if force or _stale(obj, [src, *hdrs]):
            cmd = [nvcc, *flags, "-c", src, "-o", obj]
            if verbose:
                print(" ".join(cmd), flush=True)
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode != 0:
                print(r.stdout + r.stderr, flush=True)
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=max(1, min(len(srcs), os.cpu_count() or 1))) as pool:
        objs = list(pool.map(compile_one, srcs))
    if force or _stale(XY_LIB, objs):
        cmd = [nvcc, *NVCC_ARCH, "-shared", *objs, "-o", XY_LIB, "-lcudart"]
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.run(cmd, check=True)
    return XY_LIB


def build_all(force=False, verbose=False):
    return build_levy(force, verbose), build_xy(force, verbose)
