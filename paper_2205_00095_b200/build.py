"""Build libdgrhd.so (the C-ABI CUDA library of include/dgrhd.h) in-tree for sm_100a.

    python -m paper_2205_00095_b200.build [--force]

nvcc cross-compiles without a GPU.  The fused stage kernel is instantiated once per (ndim, EOS)
pair in its own translation unit (csrc/stage_inst.cu) so the objects build in parallel.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libdgrhd.so")
OBJ = os.path.join(HERE, "build")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _sources():
    deps = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))]
    deps.append(os.path.join(ROOT, "include", "dgrhd.h"))
    return deps


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    deps = _sources()
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps)):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    jobs = [([nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "dgrhd.cu"), "-o",
              os.path.join(OBJ, "dgrhd.o")], os.path.join(OBJ, "dgrhd.o"))]
    for nd in (1, 2, 3):
        for eos in (0, 1):
            o = os.path.join(OBJ, f"stage_{nd}_{eos}.o")
            jobs.append(([nvcc, *NVCC_FLAGS, f"-DDG_INST_ND={nd}", f"-DDG_INST_EOS={eos}", "-c",
                          os.path.join(CSRC, "stage_inst.cu"), "-o", o], o))
    extra = os.environ.get("DGRHD_NVCC_EXTRA", "").split()      # kernel-tuning experiments only
    for j in jobs:
        j[0][1:1] = extra
    if verbose:
        for j in jobs:
            j[0].insert(1, "-Xptxas=-v")

    def run(job):
        r = subprocess.run(job[0], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(job[0]) + "\n" + r.stdout + r.stderr)
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        logs = list(ex.map(run, jobs))
    if verbose:
        sys.stderr.write("\n".join(logs))
    link = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB,
            *[j[1] for j in jobs]]
    r = subprocess.run(link, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: " + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
