"""Compile helper for the input-generator libraries (host C++ and the CUDA fill kernels).

Holds no method arithmetic; see workloads/__init__.py.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build_host(force=False):
    src = os.path.join(HERE, "gen.cpp")
    out = os.path.join(HERE, "libstreami_workloads_host.so")
    if force or _stale(out, [src]):
        cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-fopenmp", src, "-o", out + ".tmp"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)
    return out


def build_cuda(force=False):
    src = os.path.join(HERE, "fill.cu")
    out = os.path.join(HERE, "libstreami_workloads_cuda.so")
    if force or _stale(out, [src]):
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
               "-std=c++17", "-Xcompiler", "-fPIC", "-shared", src, "-o", out + ".tmp"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)
    return out
