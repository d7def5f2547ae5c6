"""Builds libfr_b200.so in-tree with nvcc for sm_100a (no torch involved).

    python -m paper_1312_1638_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfr_b200.so")
CPP = ["fr_basis.cpp", "fr_mesh.cpp"]
CU = ["fr_api.cu", "fr_generic.cu", "fr_tensor.cu", "fr_hex_tma.cu", "fr_hex_fluxdiv_tma.cu", "fr_hex_interp_tma.cu", "fr_element.cu", "fr_rk.cu", "fr_peaks.cu", "fr_mixed.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".hpp", ".cuh"))]
    hdrs.append(os.path.join(HERE, "..", "include", "fr.h"))
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for src in CPP + CU:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, src + ".o")
        objs.append(o)
        if force or _stale(o, [s] + hdrs):
            if src.endswith(".cpp"):
                cmd = ["g++", "-O2", "-fPIC", "-fopenmp", "-std=gnu++17", "-c", s, "-o", o]
            else:
                cmd = [NVCC, "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v" if verbose else "-warn-spills"] + ARCH + ["-c", s, "-o", o]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError("compiling %s failed:\n%s" % (src, out))
        if verbose and out:
            print(out)
    if force or procs or _stale(LIB, objs):
        cmd = [NVCC, "-shared", "-o", LIB] + objs + ARCH + ["-Xcompiler", "-fopenmp", "-lquadmath", "-lgomp"]
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if r.returncode != 0:
            raise RuntimeError("linking libfr_b200.so failed:\n" + r.stdout)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
