"""Build libstreami_b200.so in-tree with nvcc for sm_100a (no torch involved).

-fmad=false: the formula sheet fixes every fused multiply-add explicitly
(__fmaf_rn); the compiler must not contract anything else.  Defaults -prec-div=true
-prec-sqrt=true -ftz=false are kept; never -use_fast_math.
"""
import concurrent.futures
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libstreami_b200.so")
UNITS = ["api_field.cu", "api_trace.cu", "api_rounds.cu", "api_mesh.cu", "api_noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off"]


def _sources():
    hdr = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdr.append(os.path.join(os.path.dirname(HERE), "include", "streami.h"))
    return hdr


def _compile(unit, verbose):
    src = os.path.join(CSRC, unit)
    obj = os.path.join(CSRC, unit.replace(".cu", ".o"))
    deps = [src] + _sources()
    if os.path.exists(obj) and all(os.path.getmtime(d) <= os.path.getmtime(obj) for d in deps):
        return obj
    cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (unit, r.stdout, r.stderr))
    if verbose:
        print(r.stderr)
    return obj


def build(force=False, verbose=False):
    if force:
        for u in UNITS:
            o = os.path.join(CSRC, u.replace(".cu", ".o"))
            if os.path.exists(o):
                os.remove(o)
    with concurrent.futures.ThreadPoolExecutor(len(UNITS)) as ex:
        objs = list(ex.map(lambda u: _compile(u, verbose), UNITS))
    if force or not os.path.exists(SO) or any(os.path.getmtime(o) > os.path.getmtime(SO) for o in objs):
        cmd = ["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", SO + ".tmp"] + objs
        subprocess.run(cmd, check=True)
        os.replace(SO + ".tmp", SO)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
