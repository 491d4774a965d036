"""Build libdgrhd.so (the C-ABI CUDA library of include/dgrhd.h) in-tree for sm_100a.

    python -m paper_2205_00095_b200.build [--force] [-v] [--debug-asserts]

nvcc cross-compiles without a GPU.  The fused stage kernel is instantiated once per (ndim, EOS,
Riemann flux) triple in its own translation unit (csrc/stage_inst.cu) so the objects build in parallel.

The library proves what it was built from: a hash of csrc/ and include/dgrhd.h is compiled into the string
dgrhd_version() returns ("dgrhd 0.3 (sm_100a) src=<hash>", "+asserts" appended for the debug build).
build() reuses an existing library only when that string, read from the file's bytes, carries the hash of the
sources as they are now; LAST_MODE says which happened ("compiled" / "reused").  The bounds-checked debug build
goes to a file of its own, libdgrhd_dbg.so, which the binding loads only when DGRHD_DEBUG_ASSERTS=1 is set, so a
debug build can never be picked up by a later plain build, test or benchmark.
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libdgrhd.so")
LIB_DBG = os.path.join(HERE, "libdgrhd_dbg.so")
OBJ = os.path.join(HERE, "build")
VERSION_HEAD = b"dgrhd 0.3 (sm_100a) src="
LAST_MODE = None                                   # "compiled" | "reused", set by build()

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


def source_hash() -> str:
    """sha256 over the names and bytes of every file the library is compiled from (16 hex digits)."""
    h = hashlib.sha256()
    for f in _sources():
        h.update(os.path.basename(f).encode() + b"\0")
        with open(f, "rb") as fh:
            h.update(fh.read())
        h.update(b"\0")
    return h.hexdigest()[:16]


def stage_kernel_hash() -> str:
    """Hash of the sources the fused stage kernel is compiled from.  bench.py's per-DOF constants (executed flop,
    DRAM bytes) come from an ncu capture of that kernel and are valid only for the sources they were taken on."""
    h = hashlib.sha256()
    for name in ("stage_kernel.cuh", "physics.cuh", "stage_inst.cu"):
        with open(os.path.join(CSRC, name), "rb") as fh:
            h.update(name.encode() + b"\0" + fh.read() + b"\0")
    return h.hexdigest()[:16]


def library_version(path: str) -> str:
    """The dgrhd_version() string of a built library, read from the file's bytes (no dlopen: a library that
    is about to be rebuilt must not already be mapped into this process).  '' if there is none."""
    try:
        with open(path, "rb") as fh:
            blob = fh.read()
    except OSError:
        return ""
    i = blob.find(VERSION_HEAD)
    if i < 0:
        return ""
    return blob[i:blob.index(b"\0", i)].decode(errors="replace")


def build(force: bool = False, verbose: bool = False, debug_asserts: bool = False) -> str:
    """debug_asserts: compile with -DDG_DEBUG_ASSERTS (every shared-memory slot index and halo offset of
    the fused kernel is bounds-checked and a failed check traps) into libdgrhd_dbg.so: the stand-in for
    compute-sanitizer, which is closed on this GPU pool.  Run the tests against it with DGRHD_DEBUG_ASSERTS=1."""
    global LAST_MODE
    lib = LIB_DBG if debug_asserts else LIB
    obj_dir = OBJ + ("_dbg" if debug_asserts else "")
    src = source_hash()
    want = VERSION_HEAD.decode() + src + ("+asserts" if debug_asserts else "")
    if not force and library_version(lib) == want:
        LAST_MODE = "reused"
        return lib
    os.makedirs(obj_dir, exist_ok=True)
    nvcc = _nvcc()
    jobs = [([nvcc, *NVCC_FLAGS, f'-DDG_SRC_HASH="{src}"', "-c", os.path.join(CSRC, "dgrhd.cu"), "-o",
              os.path.join(obj_dir, "dgrhd.o")], os.path.join(obj_dir, "dgrhd.o"))]
    # the con2prim comparison variants: no FMA contraction, so that Brent's path matches the oracle's (c2p_variant.cu)
    jobs.append(([nvcc, *NVCC_FLAGS, "-fmad=false", "-c", os.path.join(CSRC, "c2p_variant.cu"), "-o",
                  os.path.join(obj_dir, "c2p_variant.o")], os.path.join(obj_dir, "c2p_variant.o")))
    for nd in (3, 2, 1):                                     # the slowest translation units first
        for eos in (0, 1):
            for rs in (0, 1):                                    # HLL, HLLC
                o = os.path.join(obj_dir, f"stage_{nd}_{eos}{rs}.o")
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
    link = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib,
            *[j[1] for j in jobs]]
    r = subprocess.run(link, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: " + r.stdout + r.stderr)
    if library_version(lib) != want:
        raise RuntimeError(f"built {lib} reports {library_version(lib)!r}, expected {want!r}")
    LAST_MODE = "compiled"
    return lib


if __name__ == "__main__":
    out = build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug_asserts="--debug-asserts" in sys.argv)
    print(f"{out}\nbuild_mode: {LAST_MODE}  version: {library_version(out)}")
