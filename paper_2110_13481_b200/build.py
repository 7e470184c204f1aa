"""Builds the CUDA shared library libdlr_b200.so in-tree (sm_100a only):  python -m paper_2110_13481_b200.build
The rank-templated kernels are compiled once per supported rank, in parallel."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdlr_b200.so")
RANKS = (5, 8, 10, 15, 20)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC"] + os.environ.get("DLR_NVCC_EXTRA", "").split()     # e.g. -DDLR_ENABLE_TUNE for experiments


def _newer(target, deps):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "dlr.h"))
    jobs = []
    for r in RANKS:
        jobs.append((os.path.join(CSRC, "rank_inst.cu"), os.path.join(OBJ, f"rank_{r}.o"), [f"-DDLR_RANK={r}"]))
    jobs.append((os.path.join(CSRC, "api.cu"), os.path.join(OBJ, "api.o"), []))
    jobs.append((os.path.join(CSRC, "noalloc.cu"), os.path.join(OBJ, "noalloc.o"), []))

    def run(job):
        src, obj, extra = job
        if not force and _newer(obj, [src] + hdrs):
            return
        cmd = [NVCC] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
        list(ex.map(run, jobs))
    objs = [j[1] for j in jobs]
    # stand-alone peak probe (fp64 and L2/HBM peaks quoted by bench.py and DESIGN.md): python -m ... build, then ./peak_probe
    probe_src, probe = os.path.join(CSRC, "peak_probe.cu"), os.path.join(HERE, "peak_probe")
    if force or not _newer(probe, [probe_src]):
        res = subprocess.run([NVCC] + FLAGS[:5] + ["-o", probe, probe_src], capture_output=True, text=True)
        if res.returncode:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed: peak_probe.cu")
    if force or not _newer(LIB, objs):
        cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-lcudart"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
