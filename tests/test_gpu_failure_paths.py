"""Failure paths of the C ABI on the GPU: a state on which no recovery succeeds (CFL mode cannot form a time
step), and misaligned state pointers.  Numerical trouble is counted, never silent; argument errors are
refused before any launch (include/dgrhd.h, conventions)."""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle as O
from _util import B, gcfg, mesh, smooth_prims, to_dev

pytestmark = pytest.mark.gpu


def _inadmissible(d, seed=1):
    """A smooth state with E = sqrt(D^2 + |M|^2) / 2 at every node: Eq. 25 fails everywhere."""
    U = O.prim2con_batch(d["eos"], d["gamma_ad"], smooth_prims(d, seed=seed))
    U[4] = 0.5 * np.sqrt(U[0] ** 2 + U[1] ** 2 + U[2] ** 2 + U[3] ** 2)
    return U


@pytest.mark.parametrize("nd,nelem,p,eos,G", [(1, [16], 2, 0, 5 / 3), (2, [6, 5], 3, 1, 0.0), (3, [3, 2, 4], 1, 0, 4 / 3)])
def test_state_without_a_wave_speed_is_counted_and_reported(nd, nelem, p, eos, G):
    b = B()
    d = mesh(nd, nelem, p, eos, G, [0] * nd)
    U = _inadmissible(d)
    ctx = b.Context(gcfg(d))
    ctx.dgrhd_set_state(to_dev(U))
    assert ctx.dgrhd_get_counters(reset=True)["n_c2p_fail"] == U.shape[1]     # every node failed, every node counted
    for Ux in (None, to_dev(U)):                                           # internal state / caller state
        with pytest.raises(b.DgrhdError) as e:
            ctx.dgrhd_cfl_dt(0.3, Ux)
        assert e.value.code == b.ESTATE and "wave speed" in str(e.value)
    ctx.dgrhd_step(-0.3, 2)                                                 # asynchronous form: counted only
    c = ctx.dgrhd_get_counters()
    assert c["n_bad_dt"] == 2 and c["n_stages"] == 2 * 3
    with pytest.raises(b.DgrhdError) as e:                                  # with a time read-back: reported
        ctx.dgrhd_step(-0.3, 3, t=0.0)
    assert e.value.code == b.ESTATE and "3 step(s)" in str(e.value)
    assert ctx.dgrhd_get_counters()["n_bad_dt"] == 5
    # a fixed time step needs no wave speed: no bad step is counted, however useless the state
    ctx.dgrhd_get_counters(reset=True)
    assert ctx.dgrhd_step(1e-3, 1, t=0.0) == pytest.approx(1e-3)
    assert ctx.dgrhd_get_counters()["n_bad_dt"] == 0
    ctx.close()


def test_a_good_state_after_a_bad_one_steps_normally():
    b = B()
    d = mesh(2, [6, 5], 2, 0, 5 / 3, [0, 1])
    good = O.prim2con_batch(0, 5 / 3, smooth_prims(d, seed=2))
    ctx = b.Context(gcfg(d))
    ctx.dgrhd_set_state(to_dev(_inadmissible(d)))
    with pytest.raises(b.DgrhdError):
        ctx.dgrhd_step(-0.3, 1, t=0.0)
    ctx.dgrhd_set_state(to_dev(good))
    ctx.dgrhd_get_counters(reset=True)
    t = ctx.dgrhd_step(-0.3, 2, t=0.0)
    Uo, to, _ = O.step(O.make_config(d["ndim"], d["nelem"], d["xmin"], d["xmax"], d["bc"], d["order_p"], d["eos"],
                                     d["gamma_ad"]), good, -0.3, 2)
    assert abs(t - to) <= 1e-12 * to and ctx.dgrhd_get_counters()["n_bad_dt"] == 0
    Ug = ctx.dgrhd_get_state().cpu().numpy()
    assert (np.max(np.abs(Ug - Uo), axis=1) <= 1e-11 * np.max(np.abs(Uo), axis=1).clip(1e-9)).all()
    ctx.close()


def test_misaligned_state_pointers_are_refused():
    """State rows move with 16-byte accesses: a pointer at an odd multiple of 8 bytes is EINVAL, nothing runs."""
    b = B()
    L = b.lib()
    for lim in (0, 1):
        d = mesh(2, [4, 3], 2, 0, 5 / 3, [0, 0], shock_limiter=lim, moe_alpha=1e-3 * lim)
        ctx = b.Context(gcfg(d))
        big = torch.zeros(5 * ctx.ndof + 2, dtype=torch.float64, device="cuda")
        mis = C.c_void_p(big.data_ptr() + 8)
        ok = C.c_void_p(ctx.new_state().data_ptr())
        assert L.dgrhd_rhs(ctx._h, mis, ok) == b.EINVAL and b"16-byte" in L.dgrhd_last_error(ctx._h)
        assert L.dgrhd_rhs(ctx._h, ok, mis) == b.EINVAL
        assert L.dgrhd_enforce_physicality(ctx._h, mis, None, None, None) == b.EINVAL
        assert b"16-byte" in L.dgrhd_last_error(ctx._h)
        if lim:
            assert L.dgrhd_shock_limiter(ctx._h, mis, None) == b.EINVAL
        else:
            assert L.dgrhd_shock_limiter(ctx._h, ok, None) == b.ESTATE        # created without a limiter
        assert float(big.abs().sum()) == 0.0                                   # nothing was written
        ctx.close()
