"""Builds csrc/libmeg6.so for sm_100a with nvcc (in-tree, so that it travels with the repo snapshot)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(CSRC, "libmeg6.so")
SOURCES = sorted(f for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))
HEADER = os.path.join(HERE, "..", "include", "meg6.h")


def needs_build():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [HEADER]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = "nvcc"
    arch = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC"]
    if verbose:
        arch.append("-Xptxas=-v")
    arch += os.environ.get("MEG6_NVCC_FLAGS", "").split()
    objs = []
    # the metric kernels are compiled without FMA contraction (see meg6_geom.cuh); the rest with it
    for src, extra in (("meg6_geom.cu", ["-fmad=false"]), ("meg6.cu", [])):
        obj = os.path.join(CSRC, src[:-3] + ".o")
        r = subprocess.run([nvcc] + arch + extra + ["-c", "-o", obj, os.path.join(CSRC, src)],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s%s" % (src, r.stdout, r.stderr))
        if verbose:
            print(r.stderr)
        objs.append(obj)
    r = subprocess.run([nvcc, "-shared", "-o", SO] + objs, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
