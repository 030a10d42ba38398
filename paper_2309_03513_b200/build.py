"""Build libtddft_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2309_03513_b200.build [-j N] [--force]
"""
import argparse
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libtddft_b200.so")
NVCC = os.environ.get("NVCC", "nvcc")
FLAGS = ["-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
NGROUPS = 8


def _units():
    units = []
    for name in ("api.cu", "extensions.cu", "davidson.cu", "kernels.cu", "contract.cu", "gemm.cu", "gram_static.cu", "fft_dispatch.cu", "fft_fused.cu"):
        units.append((os.path.join(CSRC, name), os.path.join(OBJ, name[:-3] + ".o"), []))
    units.append((os.path.join(CSRC, "plan.cpp"), os.path.join(OBJ, "plan.o"), ["-x", "cu"]))
    for g in range(NGROUPS):
        units.append((os.path.join(CSRC, "fft_inst.cu"), os.path.join(OBJ, "fft_inst_%d.o" % g), ["-DTD_GROUP=%d" % g]))
    return units


def _newest_header():
    t = 0.0
    for d in (CSRC, os.path.join(HERE, "..", "include")):
        for f in os.listdir(d):
            if f.endswith((".h", ".cuh")):
                t = max(t, os.path.getmtime(os.path.join(d, f)))
    return t


def build(jobs=None, force=False, verbose=True):
    os.makedirs(OBJ, exist_ok=True)
    hdr = _newest_header()
    todo = []
    for src, obj, extra in _units():
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr):
            todo.append((src, obj, extra))

    def compile_one(u):
        src, obj, extra = u
        cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return u, r

    if todo:
        with ThreadPoolExecutor(max_workers=jobs or os.cpu_count() or 4) as ex:
            for u, r in ex.map(compile_one, todo):
                if verbose:
                    print("nvcc", os.path.basename(u[1]), "ok" if r.returncode == 0 else "FAILED", flush=True)
                if r.returncode != 0:
                    sys.stderr.write(r.stdout + r.stderr)
                    raise RuntimeError("nvcc failed on %s" % u[0])
    objs = [o for _, o, _ in _units()]
    if todo or not os.path.exists(LIB):
        cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
        if verbose:
            print("linked", LIB, flush=True)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("-j", type=int, default=None)
    ap.add_argument("--force", action="store_true")
    a = ap.parse_args()
    build(a.j, a.force)
