"""Builds libcloak.so (the C-ABI CUDA library) and synth/libcloaksynth.so in-tree with nvcc for sm_100a.

`python -m paper_2606_18400_b200.build` or `__graft_entry__.build()`.  nvcc cross-compiles without a GPU.
"""
import glob
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-cudart", "static", "--expt-relaxed-constexpr"]


def _stale(out, srcs):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(s) > t for s in srcs)


def _compile_objects(srcs, deps, incs, objdir, verbose):
    os.makedirs(objdir, exist_ok=True)
    objs, procs = [], []
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s) + ".o")
        objs.append(o)
        if _stale(o, [s] + deps):
            cmd = [NVCC] + FLAGS + incs + ["-c", s, "-o", o]
            if verbose:
                print(" ".join(cmd), flush=True)
            procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for s, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {s}:\n{out}")
        if verbose and out.strip():
            print(out)
    return objs


def build_lib(verbose=False, force=False):
    csrc = os.path.join(PKG, "csrc")
    srcs = sorted(glob.glob(os.path.join(csrc, "*.cu")))
    deps = sorted(glob.glob(os.path.join(csrc, "*.cuh"))) + [os.path.join(ROOT, "include", "cloak.h")]
    out = os.path.join(PKG, "libcloak.so")
    if force or _stale(out, srcs + deps):
        objs = _compile_objects(srcs, deps, ["-I", os.path.join(ROOT, "include"), "-I", csrc],
                                os.path.join(PKG, "build"), verbose)
        subprocess.check_call([NVCC, "-shared", "-cudart", "static", "-o", out] + objs)
    return out


def build_synth(verbose=False, force=False):
    sdir = os.path.join(ROOT, "synth")
    srcs = sorted(glob.glob(os.path.join(sdir, "csrc", "*.cu")))
    out = os.path.join(sdir, "libcloaksynth.so")
    if force or _stale(out, srcs):
        objs = _compile_objects(srcs, [], [], os.path.join(sdir, "build"), verbose)
        subprocess.check_call([NVCC, "-shared", "-cudart", "static", "-o", out] + objs)
    return out


if __name__ == "__main__":
    v = "-v" in sys.argv
    print(build_lib(verbose=v, force="-f" in sys.argv))
    print(build_synth(verbose=v, force="-f" in sys.argv))
