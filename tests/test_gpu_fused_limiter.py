"""The physicality-enforcing operator INSIDE the fused stage kernel, with cells
actually limited, against the oracle's step -- the code path bench.py times.  Inputs: the config-5
recipe (`inputs.box3d`, near-vacuum cells under a fast flow) and its 2D companion (`inputs.box2d`) at
sizes the oracle finishes in a second, spanning several tiles with ragged tails; every (ndim, p)
instantiation that has more than one thread group shape is covered (3D p=1..4, 2D p=2..4, both EOS).

  one RK1 step (one stage: combine + operator on identical inputs): activation count exact (R13e),
      state to 1e-11 in the max norm (the initial states have P/E >~ 5e-5, reading R16);
  three SSPRK3 steps (9 stages, limited nodes present in the stage inputs): state to 1e-9; the
      activation counts are compared and their difference printed (R16: marginal cells may flip).
"""
import numpy as np
import pytest

import oracle as O
from paper_2205_00095_b200 import inputs as I

from _util import B, cellmax, gcfg, ocfg, relmax, to_dev

pytestmark = pytest.mark.gpu

# three limited SSPRK3 steps: global max norm / cell-local norm (tests/_util.py), within 100x of the achieved values
TOL_GLOBAL, TOL_LOCAL = 2e-11, 1e-10     # achieved over the 11 instantiations: <= 2.1e-13 / <= 1.9e-12

CASES = {
    "3d_p3_n8": lambda: I.box3d(0, n=8, p=3, kmax=1),
    "3d_p3_n16": lambda: I.box3d(0, n=16, p=3, kmax=2),
    "3d_p3_n7_ragged": lambda: I.box3d(3, n=7, p=3, kmax=1),
    "3d_p4_n4": lambda: I.box3d(0, n=4, p=4, kmax=1),
    "3d_p2_n6": lambda: I.box3d(0, n=6, p=2, kmax=1),
    "3d_p1_n7": lambda: I.box3d(2, n=7, p=1, kmax=1),
    "2d_p2_24x20": lambda: I.box2d(0, 24, 20, 2, 1),
    "2d_p3_9x7": lambda: I.box2d(0, 9, 7, 3, 1),
    "2d_p4_9x8": lambda: I.box2d(3, 9, 8, 4, 1),
    "2d_p2_tm_20x14": lambda: I.box2d(2, 20, 14, 2, 1, eos=I.EOS_TM, gamma_ad=0.0),
    "2d_p2_outflow_24x20": lambda: I.box2d(0, 24, 20, 2, 1, bc=(I.BC_OUTFLOW, I.BC_PERIODIC)),
}


def run_both(d, U, stages, nsteps):
    Uo, to, cnt_o = O.step(ocfg(d, rk_stages=stages), U, -0.3, nsteps)
    ctx = B().Context(gcfg(d, rk_stages=stages))
    ctx.dgrhd_set_state(to_dev(U))
    tg = ctx.dgrhd_step(-0.3, nsteps, t=0.0)
    Ug = ctx.dgrhd_get_state().cpu().numpy()
    return Uo, to, cnt_o, Ug, tg, ctx.dgrhd_get_counters()


@pytest.mark.parametrize("name", list(CASES))
def test_one_stage_with_limited_cells_matches_oracle_exactly_in_flags(name):
    d, W = CASES[name]()
    U = O.prim2con_batch(d["eos"], d["gamma_ad"], W.numpy())
    Uo, to, cnt_o, Ug, tg, c = run_both(d, U, 1, 1)
    assert cnt_o[0] > 0, "the case must exercise the operator"
    assert abs(tg - to) <= 1e-13 * to
    assert (c["n_flagged"], c["n_bad_mean"], c["n_c2p_fail"]) == tuple(cnt_o)
    err = relmax(Ug, Uo)
    assert err.max() <= 1e-11, err


@pytest.mark.parametrize("name", list(CASES))
def test_three_ssprk3_steps_with_limited_cells_match_oracle(name):
    d, W = CASES[name]()
    U = O.prim2con_batch(d["eos"], d["gamma_ad"], W.numpy())
    Uo, to, cnt_o, Ug, tg, c = run_both(d, U, 3, 3)
    assert cnt_o[0] > 0 and cnt_o[1] == c["n_bad_mean"] == 0 and cnt_o[2] == c["n_c2p_fail"] == 0
    assert np.isfinite(Ug).all() and abs(tg - to) <= 1e-11 * to
    err = relmax(Ug, Uo)
    nn = (d["order_p"] + 1) ** d["ndim"]
    loc = cellmax(Ug, Uo, d["nelem"][:d["ndim"]], nn)
    dflag = c["n_flagged"] - cnt_o[0]
    print(f"{name}: max-norm rel. diff {err.max():.2e}, cell-local {loc.max():.2e}, activations {cnt_o[0]} (oracle) {dflag:+d} (CUDA - oracle)")
    assert err.max() <= TOL_GLOBAL and loc.max() <= TOL_LOCAL, (err, loc)
    assert abs(dflag) <= 2                       # achieved: +0 on every instantiation


def test_conserved_integrals_of_a_periodic_box_drift_at_roundoff_only():
    """Discrete conservation of the CUDA path (the operator preserves cell averages;
    the interface flux is single-valued): sum_e sum_i w_i U_i of D and E over a periodic box after
    three limited SSPRK3 steps equals its initial value to rounding."""
    d, W = I.box3d(0, n=8, p=3, kmax=1)
    U = O.prim2con_batch(d["eos"], d["gamma_ad"], W.numpy())
    _, w1, _ = O.gll(4)
    w3 = (w1[None, None, :] * w1[None, :, None] * w1[:, None, None]).reshape(-1)
    ctx = B().Context(gcfg(d))
    ctx.dgrhd_set_state(to_dev(U))
    ctx.dgrhd_step(-0.3, 3)
    Ug = ctx.dgrhd_get_state().cpu().numpy()
    assert ctx.dgrhd_get_counters()["n_flagged"] > 0
    for v in (0, 4):
        s0 = (U[v].reshape(-1, 64) * w3).sum()
        s1 = (Ug[v].reshape(-1, 64) * w3).sum()
        assert abs(s1 - s0) <= 1e-13 * abs(s0), (v, s0, s1)
