"""Build paper_2209_09848_b200/libtno_mf.so (CUDA, sm_100a only) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtno_mf.so")
CU = ["api.cu", "tables.cu", "search_generic.cu", "search_sep.cu", "topk.cu", "inject.cu", "best.cu", "background.cu", "scatter.cu",
      "local_z_static.cu", "debug.cu"]
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
    # sanitizer / debug builds: TNO_MF_HOST_FLAGS="-fsanitize=address -fsanitize=undefined" (no commas inside a flag: -Xcompiler splits on them) instruments the host code
    # (planner, ABI), TNO_MF_NVCC_FLAGS="-DTNO_DEBUG_CHECKS" adds flags for nvcc itself (profiles/r2_sanitizers.md)
    host_extra = os.environ.get("TNO_MF_HOST_FLAGS", "")
    nvcc_extra = os.environ.get("TNO_MF_NVCC_FLAGS", "").split()
    flags = list(NVCC_FLAGS) + nvcc_extra
    if host_extra:
        flags[flags.index("-fPIC,-O2,-ffp-contract=off")] += "," + ",".join(host_extra.split())
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
        cmd = [nvcc] + flags + ["-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        logs.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed on " + f)
    # (the arch again at the link step: without it nvcc adds an empty device-link stub for its default architecture)
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp"] + objs + \
          ["-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    if host_extra:
        cmd += ["-Xcompiler", ",".join(host_extra.split())]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    with open(os.path.join(bdir, "ptxas.log"), "a") as fh:
        fh.write("\n".join(logs))
    if verbose:
        sys.stderr.write("\n".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
