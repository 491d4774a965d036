"""Build libdgrhd.so (the C-ABI CUDA library of include/dgrhd.h) in-tree for sm_100a.

    python -m paper_2205_00095_b200.build [--force] [-v] [--debug-asserts]

nvcc cross-compiles without a GPU.  The fused stage kernel is instantiated once per (ndim, EOS,
Riemann flux) triple in its own translation unit (csrc/stage_inst.cu) so the objects build in parallel.
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


def build(force: bool = False, verbose: bool = False, debug_asserts: bool = False) -> str:
    """debug_asserts: compile with -DDG_DEBUG_ASSERTS (every shared-memory slot index and halo offset of
    the fused kernel is bounds-checked and a failed check traps): the stand-in for compute-sanitizer,
    which is closed on this GPU pool.  Always rebuilds; rebuild with force=True afterwards."""
    deps = _sources()
    force = force or debug_asserts
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps)):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    jobs = [([nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "dgrhd.cu"), "-o",
              os.path.join(OBJ, "dgrhd.o")], os.path.join(OBJ, "dgrhd.o"))]
    for nd in (3, 2, 1):                                     # the slowest translation units first
        for eos in (0, 1):
            for rs in (0, 1):                                    # HLL, HLLC
                o = os.path.join(OBJ, f"stage_{nd}_{eos}{rs}.o")
                jobs.append(([nvcc, *NVCC_FLAGS, f"-DDG_INST_ND={nd}", f"-DDG_INST_EOS={eos}",
                              f"-DDG_INST_RS={rs}", "-c", os.path.join(CSRC, "stage_inst.cu"), "-o", o], o))
    if debug_asserts:                                            # bounds / ownership checks in the kernels
        for j in jobs:
            j[0].insert(1, "-DDG_DEBUG_ASSERTS")
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
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug_asserts="--debug-asserts" in sys.argv))
