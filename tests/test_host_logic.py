"""CPU-only checks of the host logic: the C-ABI library loads and exports every symbol declared in
include/dgrhd.h, argument errors are caught before any launch, the binding refuses to run without
a device (no CPU fallback), and bench.py's multi-rank aggregation (gloo, world_size 2)."""
import ctypes
import json
import os
import re
import subprocess
import sys

import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2205_00095_b200 import build
    return ctypes.CDLL(build.build())


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "dgrhd.h")).read()
    names = set(re.findall(r"\b(dgrhd_[a-z0-9_]+)\s*\(", hdr))
    assert {"dgrhd_create", "dgrhd_set_state", "dgrhd_rhs", "dgrhd_enforce_physicality", "dgrhd_cfl_dt",
            "dgrhd_step", "dgrhd_con2prim_batch"} <= names
    L = _lib()
    for n in names:
        assert hasattr(L, n), n
    from paper_2205_00095_b200 import binding
    assert set(binding.EXPORTS) == names


def test_library_proves_what_it_was_built_from():
    """dgrhd_version() carries the hash of the sources the library was compiled from; build() reuses a library
    only when that hash matches, and the bounds-checked debug build is a different file behind an env switch."""
    from paper_2205_00095_b200 import build, binding as b
    path = build.build()
    assert build.LAST_MODE in ("compiled", "reused") and path == build.LIB != build.LIB_DBG
    v = b.dgrhd_version()
    assert v == build.library_version(path) and v.endswith("src=" + build.source_hash())
    assert build.library_version(os.path.join(ROOT, "README.md")) == ""
    r = subprocess.run([sys.executable, "-c", "from paper_2205_00095_b200 import binding; print(binding.LIB_PATH)"],
                       capture_output=True, text=True, cwd=ROOT, env=dict(os.environ, DGRHD_DEBUG_ASSERTS="1"))
    assert r.stdout.strip() == build.LIB_DBG


def test_argument_errors_are_detected_without_a_device():
    from paper_2205_00095_b200 import binding as b
    L = b.lib()
    assert b"sm_100a" in L.dgrhd_version()
    good = b.make_config(2, [8, 8], [0, 0], [1, 1], [0, 1], 2, 1, 0.0)
    assert b.dgrhd_workspace_bytes(good) >= (3 * 5 + 2) * 8 * 8 * 9 * 8      # 3 states + 2 pressure buffers

    def mutated(**kw):
        c = b.make_config(1, [8], [0], [1], [0], 2, 0, 5 / 3)
        for k, v in kw.items():
            if isinstance(v, tuple):
                getattr(c, k)[v[0]] = v[1]
            else:
                setattr(c, k, v)
        return c

    assert b.dgrhd_workspace_bytes(mutated()) > 0
    for bad in (mutated(ndim=4), mutated(ndim=0), mutated(xmax=(0, -1.0)), mutated(order_p=5), mutated(gamma_ad=1.0),
                mutated(bc=(0, 7)), mutated(eos=3), mutated(rk_stages=4), mutated(nelem=(0, 0)), mutated(nelem=(1, 2)),
                mutated(eps_q=-1.0), b.make_config(3, [2048] * 3, [0] * 3, [1] * 3, [0] * 3, 3, 0, 5 / 3),
                # periodic at one end of an axis only, either way round; a Dirichlet ghost state that is not finite
                b.make_config(1, [8], [0], [1], [(1, 0)], 2, 0, 5 / 3), b.make_config(1, [8], [0], [1], [(0, 2)], 2, 0, 5 / 3),
                b.make_config(1, [8], [0], [1], [3], 2, 0, 5 / 3,
                              bc_state={(0, 0): [1, float("nan"), 0, 0, 1], (0, 1): [1, 0, 0, 0, 1]}),
                b.make_config(1, [8], [0], [1], [(3, 1)], 2, 0, 5 / 3, bc_state={(0, 0): [1, 0, float("inf"), 0, 1]})):
        assert b.dgrhd_workspace_bytes(bad) == 0
    assert b._bc_code((1, 0)) == -1 and b._bc_code((0, 0)) == 0 and b._bc_code((2, 2)) == 2 and b._bc_code((1, 3)) == 1 + 256 * 3
    assert b.dgrhd_workspace_bytes(b.make_config(1, [8], [0], [1], [(3, 1)], 2, 0, 5 / 3,
                                                 bc_state={(0, 0): [1, 0.2, 0, 0, 1]})) > 0
    h = ctypes.c_void_p()
    assert L.dgrhd_create(ctypes.byref(good), None, 0, None, ctypes.byref(h)) == b.EINVAL
    assert b"workspace" in L.dgrhd_last_error(None)
    assert L.dgrhd_con2prim_batch(9, 1.5, 4, None, None, None, None) == b.EINVAL
    assert L.dgrhd_con2prim_batch(0, 1.5, -1, None, None, None, None) == b.EINVAL
    assert L.dgrhd_con2prim_batch(0, 1.5, 0, None, None, None, None) == b.OK       # n = 0 is a no-op
    assert L.dgrhd_step(None, 1.0, 1, None) == b.EINVAL


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the behaviour WITHOUT a device")
def test_no_cpu_fallback():
    from paper_2205_00095_b200 import binding as b
    with pytest.raises(b.DgrhdError) as e:
        b.Context(b.make_config(1, [8], [0], [1], [0], 2, 0, 5 / 3))
    assert e.value.code == b.ECUDA
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1"], capture_output=True, text=True)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def _rank(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    secs = bench.max_over_ranks(0.5 + rank, "cpu")          # rank 1 is the slow one
    q.put((rank, secs, bench.aggregate_value(world, 1000, 4, secs)))
    dist.barrier()
    dist.destroy_process_group()


def test_bench_multi_rank_aggregation_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_rank, args=(r, 2, 29713, q)) for r in range(2)]
    [p.start() for p in ps]
    res = sorted(q.get(timeout=120) for _ in ps)
    [p.join(60) for p in ps]
    for rank, secs, val in res:
        assert secs == 1.5                                    # max over ranks
        assert val == 2 * 1000 * 3 * 4 / 1.5                  # replicas: all ranks' units / max time


def test_reference_arm_prints_one_json_line_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""
