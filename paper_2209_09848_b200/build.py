"""Build paper_2209_09848_b200/libtno_mf.so (CUDA, sm_100a only) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtno_mf.so")
CU = ["api.cu", "tables.cu", "search_generic.cu", "search_sep.cu", "topk.cu", "inject.cu", "best.cu", "background.cu", "scatter.cu"]
CPP = ["plan.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "--fmad=true", "-Xcompiler", "-fPIC,-O2,-ffp-contract=off", "-Xptxas", "-v"]


def _newer(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + \
           [os.path.join(HERE, "..", "include", "tno_mf.h"), os.path.abspath(__file__)]
    if not force and not _newer(LIB, deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    logs = []
    for f in CU + CPP:
        src = os.path.join(CSRC, f)
        obj = os.path.join(bdir, f + ".o")
        objs.append(obj)
        if not force and not _newer(obj, deps):
            continue
        cmd = [nvcc] + NVCC_FLAGS + ["-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        logs.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed on " + f)
    cmd = [nvcc, "-shared", "-o", LIB + ".tmp"] + objs + ["-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    with open(os.path.join(bdir, "ptxas.log"), "a") as fh:
        fh.write("\n".join(logs))
    if verbose:
        sys.stderr.write("\n".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
