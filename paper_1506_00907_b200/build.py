"""Builds libdgrtm.so (the C-ABI library of include/dgrtm.h) in-tree for sm_100a.

    python -m paper_1506_00907_b200.build [--force] [--orders 1,2,3,4,5,6]

One translation unit per DG order (kernels_inst.cu with -DDG_ORDER=N, float and double each),
compiled in parallel with nvcc; host runtime with g++; linked with nvcc -shared (static cudart).
Objects go to paper_1506_00907_b200/build/, the library next to this file.
"""
import argparse
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdgrtm.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC = os.path.join(CUDA_HOME, "bin", "nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CUDA_SOURCES = ["fma_bench.cu", "noalloc.cu", "trace_pack.cu"]
HOST_SOURCES = ["refelem.cpp", "mesh_setup.cpp", "api_core.cpp", "api_bind.cpp", "api_step.cpp",
                "api_rtm.cpp", "api_get.cpp"]


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def _headers():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    hs.append(os.path.join(HERE, "..", "include", "dgrtm.h"))
    return hs


def _run(cmd):
    p = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if p.returncode != 0:
        raise RuntimeError("command failed: %s\n%s" % (" ".join(cmd), p.stdout))
    return p.stdout


def build(force=False, orders=(1, 2, 3, 4, 5, 6), verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    hdr_time = _newest(_headers())
    jobs = []
    objs = []
    for n in orders:
        src = os.path.join(CSRC, "kernels_inst.cu")
        obj = os.path.join(OBJ, "kernels_order%d.o" % n)
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr_time, os.path.getmtime(src)):
            jobs.append([NVCC, "-std=c++17", "-O3", *ARCH, "-lineinfo", "-Xptxas", "-v", "-DDG_ORDER=%d" % n,
                         "-Xcompiler", "-fPIC", "-c", src, "-o", obj])
    for name in CUDA_SOURCES:          # order-independent device code
        src = os.path.join(CSRC, name)
        obj = os.path.join(OBJ, name.replace(".cu", ".o"))
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr_time, os.path.getmtime(src)):
            jobs.append([NVCC, "-std=c++17", "-O3", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC", "-c", src, "-o", obj])
    missing = [n for n in range(1, 7) if n not in orders]
    stub = os.path.join(OBJ, "kernels_missing.cpp")
    if missing:   # partial builds (development): unresolved orders return no table
        with open(stub, "w") as fh:
            fh.write('#include "%s"\nnamespace dgrtm {\n' % os.path.join(CSRC, "kernels.h"))
            for n in missing:
                fh.write("const KernelTable* dg_kernel_table_order%d(int) { return nullptr; }\n" % n)
            fh.write("}\n")
        obj = os.path.join(OBJ, "kernels_missing.o")
        objs.append(obj)
        jobs.append(["g++", "-std=c++17", "-O2", "-fPIC", "-I", os.path.join(CUDA_HOME, "include"), "-c", stub, "-o", obj])
    for name in HOST_SOURCES:
        src = os.path.join(CSRC, name)
        obj = os.path.join(OBJ, name.replace(".cpp", ".o"))
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr_time, os.path.getmtime(src)):
            jobs.append(["g++", "-std=c++17", "-O2", "-fPIC", "-Wall", "-pthread", "-I", os.path.join(CUDA_HOME, "include"),
                         "-c", src, "-o", obj])
    logs = []
    if jobs:
        with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            logs = list(ex.map(_run, jobs))
    if verbose:
        for lg in logs:
            sys.stdout.write(lg)
    if jobs or force or not os.path.exists(LIB):
        _run([NVCC, "-shared", *ARCH, "-o", LIB, *objs, "-lquadmath", "-lpthread"])
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--orders", default="1,2,3,4,5,6")
    ap.add_argument("--verbose", action="store_true")
    a = ap.parse_args()
    print(build(a.force, tuple(int(x) for x in a.orders.split(",")), a.verbose))
