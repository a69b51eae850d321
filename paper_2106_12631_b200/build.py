"""In-tree build with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2106_12631_b200.build [--force] [-v]

One object per .cu (compiled in parallel), linked into paper_2106_12631_b200/libmg_b200.so (the product, include/mg.h)
and paper_2106_12631_b200/libmg_probe.so (the ALU microbenchmarks bench.py prints, include/mg_probe.h).
"""
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmg_b200.so")
PROBE_LIB = os.path.join(HERE, "libmg_probe.so")
SOURCES = ["mg_api.cu", "rng_rambo.cu", "me_eemumu.cu", "me_ggtt.cu", "me_ggttg.cu", "me_ggttgg.cu", "me_qqtt.cu", "me_tables.cu", "xsec.cu"]
PROBE_SOURCES = ["alu_peak.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--fmad=true"]


def _newest_header():
    t = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            if f.endswith((".h", ".cuh")):
                t = max(t, os.path.getmtime(os.path.join(root, f)))
    return t


def _compile(src, force, hdr_time):
    obj = os.path.join(OBJ, src[:-3] + ".o")
    path = os.path.join(CSRC, src)
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(path), hdr_time):
        return obj, ""
    r = subprocess.run(["nvcc"] + NVCC_FLAGS + ["-c", path, "-o", obj], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    return obj, r.stderr


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    hdr_time = _newest_header()
    srcs = SOURCES + PROBE_SOURCES
    with concurrent.futures.ThreadPoolExecutor(max_workers=len(srcs)) as ex:
        results = list(ex.map(lambda s: _compile(s, force, hdr_time), srcs))
    objs = [o for o, _ in results]
    log = "".join(l for _, l in results)
    if log:
        with open(os.path.join(OBJ, "ptxas.log"), "a") as f:
            f.write(log)
    for lib, n0, n1 in ((LIB, 0, len(SOURCES)), (PROBE_LIB, len(SOURCES), len(srcs))):
        o = objs[n0:n1]
        if force or not os.path.exists(lib) or any(os.path.getmtime(x) > os.path.getmtime(lib) for x in o):
            subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64", "-o", lib] + o)
    if verbose and log:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
