"""Parity of the CUDA path (through the C ABI, libdgrhd.so) with the CPU oracle, element by element
on the same seeded inputs.  Tolerances are the ones BASELINE.json's north_star states, made concrete
in DESIGN.md "Parity statements":
  con2prim          R6 norm: |d rho|/rho, |d|u||/|u|, direction error <= 1e-10; |dP| <= 1e-10 P + 1e-13 E
  per-stage residual max|R_gpu - R_cpu| / max|R_cpu| <= 1e-11 per variable
  limiter           flags bit-exact; s and U to 1e-11
  10 steps, smooth  max-norm relative <= 1e-9
"""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2205_00095_b200 import inputs as I

pytestmark = pytest.mark.gpu

from _util import B, DEV, gcfg, mesh, ocfg, relmax, smooth_prims, to_dev  # noqa: E402


# ------------------------------------------------------------------------------------------------
# library surface
# ------------------------------------------------------------------------------------------------
def test_library_reports_version_and_rejects_bad_arguments():
    b = B()
    assert "sm_100a" in b.dgrhd_version()
    bad = b.make_config(1, [0], [0.0], [1.0], [0], 2, 0, 5 / 3)
    assert b.dgrhd_workspace_bytes(bad) == 0
    with pytest.raises(b.DgrhdError):
        b.Context(bad)
    ctx = b.Context(gcfg(mesh(1, [8], 2, 0, 5 / 3)))
    with pytest.raises(b.DgrhdError) as e:          # no state yet
        ctx.dgrhd_step(1e-3, 1)
    assert e.value.code == b.ESTATE
    U = ctx.new_state()
    with pytest.raises(b.DgrhdError) as e:          # overlap
        ctx.dgrhd_rhs(U, U)
    assert e.value.code == b.EINVAL
    with pytest.raises(b.DgrhdError):
        b.dgrhd_con2prim_batch(7, 1.5, U)
    ctx.close()


# ------------------------------------------------------------------------------------------------
# con2prim / prim2con  (config 3 domain; spans many blocks and a ragged tail)
# ------------------------------------------------------------------------------------------------
def c2p_errors(Wg, Wo, Uo):
    rho_e = np.abs(Wg[0] - Wo[0]) / Wo[0]
    ug, uo = np.sqrt((Wg[1:4] ** 2).sum(0)), np.sqrt((Wo[1:4] ** 2).sum(0))
    u_e = np.abs(ug - uo) / np.maximum(uo, 1e-300)
    dir_e = np.sqrt((((Wg[1:4] / np.maximum(ug, 1e-300)) - (Wo[1:4] / np.maximum(uo, 1e-300))) ** 2).sum(0))
    p_ok = np.abs(Wg[4] - Wo[4]) <= 1e-10 * Wo[4] + 1e-13 * Uo[4]
    return rho_e, u_e, dir_e, p_ok


@pytest.mark.parametrize("eos,G", [(0, 4.0 / 3.0), (0, 5.0 / 3.0), (1, 0.0)])
def test_con2prim_batch_matches_oracle(eos, G):
    n = (1 << 17) + 37
    Wt = I.c2p_states(3, n).numpy()
    Uo = O.prim2con_batch(eos, G, Wt)
    Wo, sto = O.con2prim_batch(eos, G, Uo)
    st = torch.full((n,), -1, dtype=torch.int32, device=DEV)
    Wg = B().dgrhd_con2prim_batch(eos, G, to_dev(Uo), status=st).cpu().numpy()
    assert np.array_equal(st.cpu().numpy(), sto)
    assert (sto == 0).all()
    rho_e, u_e, dir_e, p_ok = c2p_errors(Wg, Wo, Uo)
    assert rho_e.max() <= 1e-10 and u_e.max() <= 1e-10 and dir_e.max() <= 1e-10
    assert p_ok.all()


@pytest.mark.parametrize("eos,G", [(0, 5.0 / 3.0), (1, 0.0)])
def test_prim2con_batch_matches_oracle(eos, G):
    n = 50_001
    Wt = I.c2p_states(5, n).numpy()
    Uo = O.prim2con_batch(eos, G, Wt)
    Ug = B().dgrhd_prim2con_batch(eos, G, to_dev(Wt)).cpu().numpy()
    assert np.max(np.abs(Ug - Uo) / np.abs(Uo).max(0)) <= 1e-14


@pytest.mark.parametrize("eos,G", [(0, 5.0 / 3.0), (1, 0.0)])
def test_con2prim_edge_cases(eos, G):
    b = B()
    # n = 0 is a no-op
    e = torch.empty(5, 0, dtype=torch.float64, device=DEV)
    assert b.dgrhd_con2prim_batch(eos, G, e).shape == (5, 0)
    # zero momentum, tiny momentum (Eq. 60 branch), inadmissible states (status 1, NaN out)
    U = np.array([[1.0, 0, 0, 0, 2.5], [1.0, 1e-7, 0, 0, 1.8], [2.0, 0, -3e-6, 1e-6, 2.9],
                  [-1.0, 0, 0, 0, 1.0], [1.0, 2.0, 0, 0, 1.5], [1.0, 0.1, 0, 0, np.nan]]).T.copy()
    Wo, sto = O.con2prim_batch(eos, G, U)
    st = torch.zeros(U.shape[1], dtype=torch.int32, device=DEV)
    Wg = b.dgrhd_con2prim_batch(eos, G, to_dev(U), status=st).cpu().numpy()
    assert np.array_equal(st.cpu().numpy(), sto) and list(sto) == [0, 0, 0, 1, 1, 1]
    assert np.isnan(Wg[:, 3:]).all()
    # relative 1e-10 on every primitive, u included: with the Newton polish of the Taub-Matthews root
    # (reading R7b) the velocity is recovered to full relative accuracy down to |u| ~ 1e-7
    np.testing.assert_allclose(Wg[:, :3], Wo[:, :3], rtol=1e-10, atol=1e-300)


WIDE = dict(n=(1 << 16) + 13, lor=(0.0, 4.0), theta=(-10.0, 6.0), rho=(-6.0, 2.0), qmin=1e-10)


def wide_states(seed):
    """Seeded primitives far outside config 3's domain: Lorentz factor 1..1e4, Theta = P/rho 1e-10..1e6."""
    rng = np.random.default_rng(seed)
    n = WIDE["n"]
    lor = 10.0 ** rng.uniform(*WIDE["lor"], n)
    theta = 10.0 ** rng.uniform(*WIDE["theta"], n)
    rho = 10.0 ** rng.uniform(*WIDE["rho"], n)
    umag = np.sqrt((lor - 1.0) * (lor + 1.0))
    d = rng.normal(size=(3, n))
    d /= np.sqrt((d ** 2).sum(0))
    return np.vstack([rho[None], umag * d, (rho * theta)[None]]), lor


@pytest.mark.parametrize("eos,G", [(0, 4.0 / 3.0), (0, 5.0 / 3.0), (1, 0.0)])
def test_con2prim_wide_domain_matches_oracle_and_exact_primitives(eos, G):
    """Outside the comfortable domain: gamma up to 1e4, Theta from 1e-10 to 1e6,
    kept where the admissibility margin (E - sqrt(D^2+|M|^2))/E is >= 1e-10 (below that the pressure
    has no correct digit in fp64, reading R6).  Both sides are held to the exactly known primitives in
    the conditioning-aware norm of R6 (errors grow like eps gamma^2), to each other in twice that, and
    must agree on the status of every state; Taub-Matthews fallbacks are counted."""
    b = B()
    W, lor = wide_states(17 + eos)
    U = O.prim2con_batch(eos, G, W)
    margin = (U[4] - np.sqrt(U[0] ** 2 + (U[1:4] ** 2).sum(0))) / U[4]
    keep = margin >= WIDE["qmin"]
    assert keep.sum() > 0.5 * W.shape[1]
    W, U, lor = W[:, keep], np.ascontiguousarray(U[:, keep]), lor[keep]
    Wo, sto = O.con2prim_batch(eos, G, U)
    b.dgrhd_tm_fallback_count(reset=True)
    st = torch.full((U.shape[1],), -1, dtype=torch.int32, device=DEV)
    Wg = b.dgrhd_con2prim_batch(eos, G, to_dev(U), status=st).cpu().numpy()
    nfall = b.dgrhd_tm_fallback_count()
    assert np.array_equal(st.cpu().numpy(), sto) and (sto == 0).all()
    tol = 1e-10 + 1e-14 * lor ** 2                      # ~ 45 eps gamma^2
    umag = np.sqrt((W[1:4] ** 2).sum(0))
    for X in (Wo, Wg):                                  # each side against the exact primitives
        assert (np.abs(X[0] / W[0] - 1) <= tol).all()
        assert (np.abs(np.sqrt((X[1:4] ** 2).sum(0)) / umag - 1) <= tol).all()
        assert (np.abs(X[4] - W[4]) <= 1e-10 * W[4] + 1e-13 * U[4]).all()
    rho_e, u_e, dir_e, _ = c2p_errors(Wg, Wo, U)        # and against each other
    assert (rho_e <= 2 * tol).all() and (u_e <= 2 * tol).all() and (dir_e <= 2 * tol).all()
    assert (np.abs(Wg[4] - Wo[4]) <= 2e-10 * Wo[4] + 2e-13 * U[4]).all()
    print(f"eos {eos}: {U.shape[1]} states, gamma <= {lor.max():.3g}, Taub-Matthews fallbacks {nfall}")
    assert nfall <= U.shape[1] // 100


def test_taub_matthews_fallback_is_taken_and_counted_when_the_fast_route_cannot_converge():
    """The convergence test after the Newton polish (Newton on the cubic is not guaranteed
    to converge) and its double-precision fallback: over the whole wide domain above the fast route
    converges and the count stays 0; here E/D ~ 1e170 overflows the cubic's coefficients in any fp64
    evaluation, so the polish cannot converge: the state takes the fallback, is counted, and ends with
    the same status as the oracle's closed form (2: no positive finite pressure).  A normal state in
    the same batch is untouched."""
    b = B()
    U = np.array([[1e-170, 0.5, 0, 0, 1.0], [1e-200, 0.3, 0.2, 0, 1.0], [1.0, 0.5, 0, 0, 2.0]]).T.copy()
    Wo, sto = O.con2prim_batch(1, 0.0, U)
    b.dgrhd_tm_fallback_count(reset=True)
    st = torch.full((3,), -1, dtype=torch.int32, device=DEV)
    Wg = b.dgrhd_con2prim_batch(1, 0.0, to_dev(U), status=st).cpu().numpy()
    assert np.array_equal(st.cpu().numpy(), sto) and list(sto) == [2, 2, 0]
    assert b.dgrhd_tm_fallback_count(reset=True) == 2
    assert b.dgrhd_tm_fallback_count() == 0
    np.testing.assert_allclose(Wg[:, 2], Wo[:, 2], rtol=1e-12)


def test_con2prim_batch_host_wrapper_chunks():
    b = B()
    n = 10_007
    Wt = I.c2p_states(9, n).numpy()
    Uo = O.prim2con_batch(0, 4 / 3, Wt)
    Wo, _ = O.con2prim_batch(0, 4 / 3, Uo)
    Uh = torch.from_numpy(Uo).pin_memory()
    Wh = torch.empty_like(Uh).pin_memory()
    stage = torch.empty(80 * 3000, dtype=torch.uint8, device=DEV)      # forces 4 chunks
    b.dgrhd_con2prim_batch_host(0, 4 / 3, Uh, Wh, stage)
    rho_e, u_e, dir_e, p_ok = c2p_errors(Wh.numpy(), Wo, Uo)
    assert rho_e.max() <= 1e-10 and u_e.max() <= 1e-10 and p_ok.all()


# ------------------------------------------------------------------------------------------------
# spatial operator R = L(U)
# ------------------------------------------------------------------------------------------------
RHS_CASES = [
    # nd, nelem (ragged against the tile sizes), p, eos, Gamma, bc
    (1, [256], 2, 0, 5 / 3, [1]), (1, [67], 1, 0, 4 / 3, [0]), (1, [70], 3, 1, 0.0, [0]),
    (1, [101], 4, 0, 5 / 3, [1]), (1, [300], 0, 0, 5 / 3, [0]), (1, [1], 2, 0, 5 / 3, [0]),
    (2, [21, 10], 2, 1, 0.0, [0, 1]), (2, [9, 7], 3, 0, 5 / 3, [1, 0]), (2, [18, 6], 1, 0, 4 / 3, [0, 0]),
    (2, [5, 3], 4, 1, 0.0, [1, 1]), (2, [40, 9], 0, 0, 5 / 3, [0, 0]),
    (3, [5, 3, 3], 3, 0, 5 / 3, [0, 0, 0]), (3, [6, 5, 3], 2, 1, 0.0, [0, 1, 0]),
    (3, [5, 6, 3], 1, 0, 4 / 3, [1, 1, 1]), (3, [3, 2, 2], 4, 0, 5 / 3, [0, 0, 1]),
    (3, [9, 9, 5], 0, 1, 0.0, [0, 0, 0]), (3, [1, 1, 1], 3, 0, 5 / 3, [0, 0, 0]),
]


@pytest.mark.parametrize("nd,nelem,p,eos,G,bc", RHS_CASES)
def test_rhs_matches_oracle(nd, nelem, p, eos, G, bc):
    d = mesh(nd, nelem, p, eos, G, bc)
    W = smooth_prims(d, seed=nd * 10 + p)
    U = O.prim2con_batch(eos, G, W)
    Ro, nf = O.rhs(ocfg(d), U)
    ctx = B().Context(gcfg(d))
    Rg = ctx.dgrhd_rhs(to_dev(U)).cpu().numpy()
    assert nf == 0 and ctx.dgrhd_get_counters()["n_c2p_fail"] == 0
    assert np.isfinite(Rg).all()
    err = relmax(Rg, Ro)
    active = np.max(np.abs(Ro), axis=1) > 1e-9          # rows that are identically ~0 (unused axes)
    assert (err[active] <= 1e-11).all(), err
    assert np.max(np.abs(Rg - Ro)[~active], initial=0.0) <= 1e-11


def test_rhs_first_stage_of_config1_and_discontinuous_data():
    """Config 1's initial state (P/E >~ 5e-5, R16) over several seeds: jumps exercise every HLL branch."""
    for seed in range(6):
        d, W = I.riemann1d(seed)
        U = O.prim2con_batch(d["eos"], d["gamma_ad"], W.numpy())
        Ro, _ = O.rhs(ocfg(d), U)
        Rg = B().Context(gcfg(d)).dgrhd_rhs(to_dev(U)).cpu().numpy()
        err = relmax(Rg, Ro)
        assert (err[[0, 1, 4]] <= 1e-11).all(), (seed, err)


def test_rhs_supersonic_faces_take_the_upwind_branches():
    d = mesh(1, [40], 2, 0, 5 / 3, [1])
    W = smooth_prims(d, 3, amp=0.1)
    for sgn in (+1.0, -1.0):
        Wb = W.copy()
        Wb[1] = sgn * 3.0 + 0.1 * W[1]               # u = gamma v = 3: faster than sound everywhere
        U = O.prim2con_batch(0, 5 / 3, Wb)
        Ro, _ = O.rhs(ocfg(d), U)
        Rg = B().Context(gcfg(d)).dgrhd_rhs(to_dev(U)).cpu().numpy()
        assert (relmax(Rg, Ro)[[0, 1, 4]] <= 1e-11).all()


# ------------------------------------------------------------------------------------------------
# physicality-enforcing operator: flags bit-exact, s and U to 1e-11
# ------------------------------------------------------------------------------------------------
LIM_CASES = [(1, [300], 2, 0, 5 / 3), (1, [77], 4, 1, 0.0), (2, [33, 20], 2, 1, 0.0),
             (2, [15, 9], 3, 0, 5 / 3), (3, [9, 8, 7], 3, 0, 5 / 3), (3, [7, 6, 5], 1, 0, 4 / 3),
             (3, [4, 3, 3], 4, 1, 0.0), (2, [50, 11], 0, 0, 5 / 3)]


@pytest.mark.parametrize("nd,nelem,p,eos,G", LIM_CASES)
def test_enforce_physicality_matches_oracle(nd, nelem, p, eos, G):
    d = mesh(nd, nelem, p, eos, G)
    nn = (p + 1) ** nd
    W = smooth_prims(d, seed=7 + p)
    W[0] *= np.exp(3.0 * np.sin(np.arange(W.shape[1]) * 0.37))       # strong density contrast
    U = O.prim2con_batch(eos, G, W)
    Ubad, cells = I.limiter_stress(torch.from_numpy(U), nn, seed=11, frac=0.2)
    Ubad = Ubad.numpy()
    if p == 0:                                                       # single node: the mean is the node
        Ubad = U.copy()
    Uo, flag_o, s_o, cnt_o = O.enforce_physicality(ocfg(d), Ubad)
    ctx = B().Context(gcfg(d))
    Ug = to_dev(Ubad)
    flag_g, s_g, cnt_g = ctx.dgrhd_enforce_physicality(Ug)
    assert np.array_equal(flag_g.cpu().numpy(), flag_o)              # cell-wise activation: exact
    assert cnt_g == tuple(cnt_o)
    if p > 0:
        assert cnt_o[0] >= len(cells) * 0.9
    np.testing.assert_allclose(s_g.cpu().numpy(), s_o, rtol=1e-11, atol=1e-13)
    Ug = Ug.cpu().numpy()
    un = flag_o.repeat(nn) == 0
    assert np.array_equal(Ug[:, un], Ubad[:, un])                    # untouched cells bit-identical
    scale = np.abs(Uo).max(axis=0) + 1e-300
    assert np.max(np.abs(Ug - Uo) / scale) <= 1e-11
    # idempotent: a second application flags nothing, except the cells whose mean is itself
    # inadmissible (flattened to that mean, R13d), which it flags and counts again
    _, _, cnt2 = ctx.dgrhd_enforce_physicality(to_dev(Ug))
    assert cnt2 == (cnt_o[1], cnt_o[1])


def test_enforce_physicality_inadmissible_mean_is_flattened_and_counted():
    d = mesh(1, [10], 2, 0, 5 / 3)
    W = smooth_prims(d, 1)
    U = O.prim2con_batch(0, 5 / 3, W)
    U[4, 6:9] = 0.5 * U[0, 6:9]                                      # whole cell 2 below rest mass
    Uo, flag_o, s_o, cnt_o = O.enforce_physicality(ocfg(d), U)
    ctx = B().Context(gcfg(d))
    Ug = to_dev(U)
    flag_g, s_g, cnt_g = ctx.dgrhd_enforce_physicality(Ug)
    assert cnt_g == tuple(cnt_o) == (1, 1)
    assert s_g.cpu().numpy()[2] == 0.0 and np.array_equal(flag_g.cpu().numpy(), flag_o)
    np.testing.assert_allclose(Ug.cpu().numpy(), Uo, rtol=1e-13)


# ------------------------------------------------------------------------------------------------
# CFL step
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nd,nelem,p,eos,G", [(1, [100], 2, 0, 5 / 3), (2, [12, 9], 2, 1, 0.0),
                                              (3, [5, 4, 3], 3, 0, 5 / 3)])
def test_cfl_dt_matches_oracle(nd, nelem, p, eos, G):
    d = mesh(nd, nelem, p, eos, G)
    U = O.prim2con_batch(eos, G, smooth_prims(d, 5))
    dto = O.cfl_dt(ocfg(d), U, 0.3)
    ctx = B().Context(gcfg(d))
    Ud = to_dev(U)
    assert abs(ctx.dgrhd_cfl_dt(0.3, Ud) - dto) <= 1e-13 * dto
    ctx.dgrhd_set_state(Ud)
    assert abs(ctx.dgrhd_cfl_dt(0.3) - dto) <= 1e-13 * dto


# ------------------------------------------------------------------------------------------------
# dgrhd_step: SSP-RK stages with the operator after every stage (R15), dt on the device (R11)
# ------------------------------------------------------------------------------------------------
STEP_CASES = [(1, [64], 2, 0, 4 / 3, 3), (1, [50], 1, 0, 5 / 3, 2), (1, [40], 0, 1, 0.0, 1),
              (2, [12, 10], 2, 1, 0.0, 3), (3, [5, 4, 4], 3, 0, 5 / 3, 3), (2, [9, 6], 3, 0, 5 / 3, 3)]


@pytest.mark.parametrize("nd,nelem,p,eos,G,stages", STEP_CASES)
def test_ten_steps_on_smooth_problems_match_oracle(nd, nelem, p, eos, G, stages):
    d = mesh(nd, nelem, p, eos, G, rk_stages=stages)
    U = O.prim2con_batch(eos, G, smooth_prims(d, seed=21 + nd))
    Uo, to, cnt_o = O.step(ocfg(d), U, -0.3, 10)
    ctx = B().Context(gcfg(d))
    ctx.dgrhd_set_state(to_dev(U))
    tg = ctx.dgrhd_step(-0.3, 10, t=0.0)
    Ug = ctx.dgrhd_get_state().cpu().numpy()
    assert abs(tg - to) <= 1e-12 * to
    err = relmax(Ug, Uo)
    active = np.max(np.abs(Uo), axis=1) > 1e-12
    assert (err[active] <= 1e-9).all(), err
    c = ctx.dgrhd_get_counters()
    assert c["n_stages"] == 10 * stages and c["n_c2p_fail"] == cnt_o[2] == 0
    assert c["n_flagged"] == cnt_o[0] and c["n_bad_mean"] == cnt_o[1]
    # primitives of the internal state are those of the state
    Wg = ctx.dgrhd_get_prims().cpu().numpy()                         # con2prim of the CUDA state itself
    Wo, _ = O.con2prim_batch(eos, G, Ug)
    rho_e, u_e, dir_e, p_ok = c2p_errors(Wg, Wo, Ug)                 # R6 norm
    assert rho_e.max() <= 1e-10 and u_e.max() <= 1e-10 and p_ok.all()


def test_fixed_dt_steps_and_split_calls_agree():
    d = mesh(1, [48], 2, 0, 5 / 3)
    U = O.prim2con_batch(0, 5 / 3, smooth_prims(d, 2))
    Uo, to, _ = O.step(ocfg(d), U, 2e-4, 6)
    b = B()
    c1, c2 = b.Context(gcfg(d)), b.Context(gcfg(d))
    c1.dgrhd_set_state(to_dev(U))
    c2.dgrhd_set_state(to_dev(U))
    t1 = c1.dgrhd_step(2e-4, 6, t=0.0)
    t2 = 0.0
    for _ in range(6):
        t2 = c2.dgrhd_step(2e-4, 1, t=t2)
    assert abs(t1 - to) < 1e-15 and abs(t2 - to) < 1e-15
    U1, U2 = c1.dgrhd_get_state(), c2.dgrhd_get_state()
    assert torch.equal(U1, U2)                                        # deterministic
    assert (relmax(U1.cpu().numpy(), Uo)[[0, 1, 4]] <= 1e-10).all()


def test_config1_riemann_50_steps_limiter_active():
    """Config 1 (BASELINE.json configs[0]): parity of a shocked, limited run.  Limited nodes hug the
    admissibility boundary where the residual is ill-conditioned (R16): the state is compared in the
    max norm at 1e-12 (achieved over the three seeds: 1.2e-14) and the activation counts, which could differ
    at marginal cells, are held to 2 cells in total (achieved: identical) -- both are reported."""
    worst, dflag = 0.0, 0
    for seed in range(3):
        d, W = I.riemann1d(seed)
        U = O.prim2con_batch(d["eos"], d["gamma_ad"], W.numpy())
        Uo, to, cnt_o = O.step(ocfg(d), U, -0.3, 50)
        ctx = B().Context(gcfg(d))
        ctx.dgrhd_set_state(to_dev(U))
        tg = ctx.dgrhd_step(-0.3, 50, t=0.0)
        Ug = ctx.dgrhd_get_state().cpu().numpy()
        c = ctx.dgrhd_get_counters()
        assert np.isfinite(Ug).all() and c["n_bad_mean"] == 0 == cnt_o[1]
        assert abs(tg - to) <= 1e-9 * to
        worst = max(worst, relmax(Ug, Uo)[[0, 1, 4]].max())
        dflag += abs(c["n_flagged"] - cnt_o[0])
    print(f"config1: worst max-norm rel. diff {worst:.3e}, activation-count diff {dflag}")
    assert worst <= 1e-12 and dflag <= 2


def test_entropy_wave_converges_at_order_p_plus_1_on_gpu():
    """Config 2 (BASELINE.json configs[1]) run entirely on the CUDA path: L1(rho) error vs the exact
    solution has order p+1."""
    b = B()
    for p, nes in [(1, [32, 64, 128]), (2, [16, 32, 64])]:
        errs = []
        for ne in nes:
            d, W, x, phi = I.wave1d(1, ne, p)
            ctx = b.Context(gcfg(d))
            U = b.dgrhd_prim2con_batch(d["eos"], d["gamma_ad"], W.to(DEV))
            ctx.dgrhd_set_state(U)
            nsteps = int(np.ceil(2.0 / (0.1 * (1.0 / ne) / (2 * p + 1))))
            ctx.dgrhd_step(2.0 / nsteps, nsteps)
            rho = ctx.dgrhd_get_prims()[0].cpu()
            exact = I.wave1d_exact(x, 2.0, phi)[0]
            errs.append(float((rho - exact).abs().mean()))
        orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
        assert (np.abs(orders - (p + 1)) < 0.35).all(), (p, errs, orders)


def test_cuda_graph_replay_is_bit_identical_and_cuts_launch_overhead():
    """dgrhd_step through the captured per-step graph (default) vs plain launches: same bits; on
    config 1 (768 DOF, launch-latency bound) the time per step is reported."""
    import time
    b = B()
    d, W = I.riemann1d(0)
    U = b.dgrhd_prim2con_batch(d["eos"], d["gamma_ad"], W.to(DEV))
    res, us = [], []
    for graph in (1, 0):
        ctx = b.Context(gcfg(d))
        ctx.dgrhd_set_option(b.OPT_CUDA_GRAPH, graph)
        ctx.dgrhd_set_state(U)
        ctx.dgrhd_step(-0.3, 5)                       # CFL mode, dt on the device
        ctx.dgrhd_step(1e-4, 3)                       # fixed dt: graph re-captured
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.dgrhd_step(-0.3, 200)
        torch.cuda.synchronize()
        us.append((time.perf_counter() - t0) / 200 * 1e6)
        res.append(ctx.dgrhd_get_state())
        assert ctx.dgrhd_get_counters()["n_stages"] == 3 * 208
    assert torch.equal(res[0], res[1])
    print(f"config 1: {us[0]:.1f} us/step with the CUDA graph, {us[1]:.1f} us/step with plain launches")


def test_tm_slow_flows_recovered_to_full_relative_accuracy_on_gpu():
    """The CUDA Taub-Matthews route (single-precision closed form + three Newton steps on Eq. 61,
    DESIGN.md R7b) against exactly known primitives and against the oracle, |u| in [1e-9, 1e-1]."""
    rng = np.random.default_rng(4)
    n = 20011
    umag = 10.0 ** rng.uniform(-9, -1, n)
    dirn = rng.normal(size=(3, n)); dirn /= np.sqrt((dirn ** 2).sum(0))
    rho = 10.0 ** rng.uniform(-3, 2, n)
    P = rho * 10.0 ** rng.uniform(-6, 3, n)
    W = np.vstack([rho[None], umag * dirn, P[None]])
    U = O.prim2con_batch(1, 0.0, W)
    Wo, _ = O.con2prim_batch(1, 0.0, U)
    st = torch.zeros(n, dtype=torch.int32, device=DEV)
    Wg = B().dgrhd_con2prim_batch(1, 0.0, to_dev(U), status=st).cpu().numpy()
    assert int(st.max()) == 0
    ug = np.sqrt((Wg[1:4] ** 2).sum(0))
    assert np.max(np.abs(ug / umag - 1)) < 2e-12
    assert np.max(np.abs(Wg[0] / rho - 1)) < 1e-14
    rho_e, u_e, dir_e, p_ok = c2p_errors(Wg, Wo, U)
    assert rho_e.max() <= 1e-10 and u_e.max() <= 1e-10 and dir_e.max() <= 1e-10 and p_ok.all()
