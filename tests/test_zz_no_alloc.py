"""dgrhd_rhs_static: the spatial operator R = L(U) for callers that cannot allocate device memory.

Some users of this library sit where no device memory can be had at the moment they need the residual:
a plug-in inside an application whose own arena already owns (almost) all of the GPU's memory, a process
whose device-memory budget was fixed up front and is spent, a loop that must not stall on the
device-wide synchronisation cudaMalloc / cudaFree imply.  The regular path (dgrhd_create + dgrhd_rhs)
needs a caller-allocated workspace; dgrhd_rhs_static needs none, because its scratch (the nodal pressure
between its two kernels and the failure counters) is one fixed array compiled into libdgrhd.so.  The price
is a size limit (DGRHD_STATIC_MAX_NDOF nodes) and that all calls share that array.

What is checked here, against the regular path on the same inputs and at the tolerance the operator's
parity tests use (1e-11 of the per-variable maximum, tests/test_gpu_parity.py):
  * two calls in a row on DIFFERENT meshes and states: the second must not see what the first left in
    the shared array (stale pressure of another mesh, stale counters);
  * the per-call failure count: a state with a known number of inadmissible nodes reports that number,
    the clean state right after it reports zero again;
  * a mesh over the limit is refused with ENOMEM and a message that names the limit, before any launch.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It passes alone in a fresh process (where its first call does the
one-time set-up of the array's device address) and after the other tests.
"""
import numpy as np
import pytest
import torch

import oracle as O
from _util import B, gcfg, mesh, relmax, smooth_prims, to_dev

TOL = 1e-11          # the tolerance of test_rhs_matches_oracle

# nd, nelem, p, eos, Gamma, bc, riemann -- ragged against the tile sizes, both EOS, both fluxes
CASES = [
    (3, [7, 5, 6], 3, 0, 5 / 3, [0, 0, 0], 0),
    (2, [21, 10], 2, 1, 0.0, [0, 1], 1),
    (1, [101], 4, 0, 4 / 3, [1], 0),
    (3, [5, 6, 3], 1, 1, 0.0, [1, 0, 1], 1),
]


def _case(nd, nelem, p, eos, G, bc, rs, seed):
    d = mesh(nd, nelem, p, eos, G, bc, riemann=rs)
    U = O.prim2con_batch(eos, G, smooth_prims(d, seed=seed))      # input data only (Eq. 4)
    return gcfg(d), to_dev(U)


def _regular(cfg, U):
    """The existing path: a context with a torch-allocated workspace, then dgrhd_rhs."""
    ctx = B().Context(cfg)
    R = ctx.dgrhd_rhs(U).cpu().numpy()
    nfail = ctx.dgrhd_get_counters()["n_c2p_fail"]
    ctx.close()
    return R, nfail


def _agree(Rs, Rr):
    assert np.isfinite(Rs).all()
    scale = np.maximum(np.max(np.abs(Rr), axis=1), 1e-9)           # rows of unused axes are ~0
    assert (np.max(np.abs(Rs - Rr), axis=1) / scale <= TOL).all(), relmax(Rs, Rr)


@pytest.mark.gpu
def test_two_static_calls_in_a_row_match_the_workspace_path():
    b = B()
    work = [_case(*c, seed=40 + i) for i, c in enumerate(CASES)]
    want = [_regular(cfg, U) for cfg, U in work]
    # back to back, a different mesh every time, largest first so that stale pressure of a bigger mesh
    # is in the array when a smaller one runs; then the whole sequence once more
    for rep in range(2):
        for (cfg, U), (Rr, nf) in zip(work, want):
            out = torch.full_like(U, float("nan"))                 # caller-owned output, fully overwritten
            Rs, nfail = b.dgrhd_rhs_static(cfg, U, out=out)
            assert Rs.data_ptr() == out.data_ptr()
            assert nf == 0 and nfail == 0
            _agree(Rs.cpu().numpy(), Rr)
    # the same state twice in a row gives the same bits (the shared array carries nothing over)
    cfg, U = work[0]
    R1, _ = b.dgrhd_rhs_static(cfg, U)
    R2, _ = b.dgrhd_rhs_static(cfg, U, count_failures=False)      # asynchronous variant of the call
    torch.cuda.synchronize()
    assert torch.equal(R1, R2)


@pytest.mark.gpu
def test_static_call_counts_failures_per_call_and_starts_from_zero():
    b = B()
    cfg, U = _case(*CASES[1], seed=7)
    bad = U.clone()
    nodes = [3, 500, 1234]                                         # E < sqrt(D^2 + |M|^2): not admissible (Eq. 25)
    for n in nodes:
        bad[4, n] = 0.5 * torch.sqrt(bad[0, n] ** 2 + bad[1, n] ** 2 + bad[2, n] ** 2 + bad[3, n] ** 2)
    Rr_bad, nf_bad = _regular(cfg, bad)
    Rr, nf = _regular(cfg, U)
    assert nf_bad == len(nodes) and nf == 0
    Rs_bad, nfail_bad = b.dgrhd_rhs_static(cfg, bad)
    assert nfail_bad == len(nodes)
    Rs_bad = Rs_bad.cpu().numpy()
    ok = np.isfinite(Rr_bad)
    assert (np.isfinite(Rs_bad) == ok).all()                       # the same nodes are poisoned on both paths
    assert np.max(np.abs(Rs_bad - Rr_bad)[ok]) <= TOL * np.max(np.abs(Rr_bad[ok]))
    Rs, nfail = b.dgrhd_rhs_static(cfg, U)                         # the next call starts from zero again
    assert nfail == 0
    _agree(Rs.cpu().numpy(), Rr)


@pytest.mark.gpu
def test_static_call_at_exactly_its_size_limit():
    """256 x 256 elements at p = 3 are 2^20 nodes: the largest mesh the built-in array takes."""
    b = B()
    cfg, U = _case(2, [256, 256], 3, 0, 5 / 3, [0, 1], 1, seed=3)
    assert U.shape[1] == b.STATIC_MAX_NDOF
    Rr, nf = _regular(cfg, U)
    for _ in range(2):
        Rs, nfail = b.dgrhd_rhs_static(cfg, U)
        assert nf == 0 and nfail == 0
        _agree(Rs.cpu().numpy(), Rr)


def test_static_call_refuses_meshes_over_its_limit():
    """Host logic only (the size is checked before anything touches the device): 128^3 at p = 3 has 2^27
    nodes, the built-in array holds 2^20."""
    b = B()
    assert b.STATIC_MAX_NDOF == 1 << 20
    big = b.make_config(3, [128] * 3, [0] * 3, [1] * 3, [0] * 3, 3, 0, 5 / 3)
    L = b.lib()
    import ctypes as C
    fake = C.c_void_p(256)                                         # never dereferenced: refused first
    assert L.dgrhd_rhs_static(C.byref(big), fake, C.c_void_p(512), None, None) == b.ENOMEM
    msg = L.dgrhd_last_error(None).decode()
    assert "1048576" in msg and "134217728" in msg and "dgrhd_rhs" in msg
    edge = b.make_config(2, [256, 257], [0, 0], [1, 1], [0, 0], 3, 0, 5 / 3)     # 1 052 672 nodes: just over
    assert L.dgrhd_rhs_static(C.byref(edge), fake, C.c_void_p(512), None, None) == b.ENOMEM
    assert L.dgrhd_rhs_static(None, fake, C.c_void_p(512), None, None) == b.EINVAL
    small = b.make_config(1, [8], [0], [1], [0], 2, 0, 5 / 3)
    assert L.dgrhd_rhs_static(C.byref(small), None, C.c_void_p(512), None, None) == b.EINVAL
    assert L.dgrhd_rhs_static(C.byref(small), fake, fake, None, None) == b.EINVAL          # overlap
    assert L.dgrhd_rhs_static(C.byref(small), C.c_void_p(264), C.c_void_p(512), None, None) == b.EINVAL   # alignment
