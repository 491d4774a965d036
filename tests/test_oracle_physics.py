"""Pins for the oracle's pointwise physics (O1-O3) and basis tables (O4).

Each test checks ``oracle/`` against something other than itself: a closed form, a textbook
identity, a tensor-transformation law, a numerical Jacobian, a 50-digit solve of an independent
formulation, or a claim printed in PAPER.md (fixtures in tests/golden/).
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle as O
from paper_2205_00095_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")
EOSES = [(O.EOS_IDEAL, 4.0 / 3.0), (O.EOS_IDEAL, 5.0 / 3.0), (O.EOS_TM, 0.0)]


# ------------------------------------------------------------------ O4: GLL tables ------------
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5])
def test_gll_quadrature_and_derivative(N):
    x, w, D = O.gll(N)
    assert abs(w.sum() - 2.0) < 1e-15
    assert np.allclose(x, -x[::-1], atol=1e-16) and np.allclose(w, w[::-1], atol=1e-16)
    # GLL with N nodes integrates degree <= 2N-3 exactly (N=1: midpoint rule, degree 1)
    maxdeg = 1 if N == 1 else 2 * N - 3
    for k in range(maxdeg + 1):
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(np.dot(w, x ** k) - exact) < 2e-15, (N, k)
    if N > 1:   # ... and not degree 2N-2
        k = 2 * N - 2
        assert abs(np.dot(w, x ** k) - 2.0 / (k + 1)) > 1e-3
    # D[q,i] = l_i'(x_q): exact derivative of every polynomial of degree <= N-1
    for k in range(N):
        f = x ** k
        df = k * x ** (k - 1) if k > 0 else np.zeros(N)
        assert np.allclose(D @ f, df, atol=5e-14), (N, k)
    # summation by parts: w_i D_ij + w_j D_ji = delta_ip delta_jp - delta_i0 delta_j0
    if N > 1:
        B = np.zeros((N, N)); B[0, 0] = -1.0; B[-1, -1] = 1.0
        Q = w[:, None] * D
        assert np.allclose(Q + Q.T, B, atol=5e-15)
    # the node positions used by the input generator are the same points
    assert np.allclose(x, I.node_positions(N), atol=1e-16)


# ------------------------------------------------------------------ O1: EOS -------------------
@pytest.mark.parametrize("eos,G", EOSES)
def test_sound_speed_is_eq6_of_enthalpy(eos, G):
    """Eq. 9 / Eq. 11 must equal Eq. 6 applied to Eq. 8 / Eq. 10 (derivatives by 30-digit FD)."""
    mp.mp.dps = 40
    rng = np.random.default_rng(1)
    for _ in range(40):
        rho = 10.0 ** rng.uniform(-6, 2)
        P = rho * 10.0 ** rng.uniform(-6, 3)

        def h(r, p):
            th = p / r
            if eos == O.EOS_IDEAL:
                return 1 + mp.mpf(G) / (mp.mpf(G) - 1) * th
            return mp.mpf(5) / 2 * th + mp.mpf(3) / 2 * mp.sqrt(th * th + mp.mpf(4) / 9)
        r, p = mp.mpf(rho), mp.mpf(P)
        dh_drho = mp.diff(lambda q: h(q, p), r)
        dh_dP = mp.diff(lambda q: h(r, q), p)
        n = r * dh_dP - 1
        cs2 = -r / (n * h(r, p)) * dh_drho                  # Eq. 6
        assert abs(O.cs2(eos, G, rho, P) / float(cs2) - 1) < 1e-13
        assert abs(O.enthalpy(eos, G, rho, P) / float(h(r, p)) - 1) < 1e-15


def test_taub_matthews_identities_and_limits():
    for th in [1e-8, 1e-3, 0.1, 1.0, 30.0, 1e4]:
        h = O.enthalpy(O.EOS_TM, 0.0, 1.0, th)
        assert abs((h - th) * (h - 4 * th) - 1.0) < 1e-13 * max(1.0, h * h)   # (h-Th)(h-4Th)=1
        geq = (h - 1) / (h - 1 - th)                                        # Eq. 12
        assert 4.0 / 3.0 - 1e-9 < geq < 5.0 / 3.0 + 1e-9
    # cold limit: Gamma_eq -> 5/3, cs^2 -> (5/3) Theta;  hot limit: Gamma_eq -> 4/3, cs^2 -> 1/3
    th = 1e-9
    h = O.enthalpy(O.EOS_TM, 0.0, 1.0, th)
    assert abs((h - 1) / th - 2.5) < 1e-6                     # h-1 = Gamma/(Gamma-1) Th with 5/3
    assert abs(O.cs2(O.EOS_TM, 0.0, 1.0, th) / (5.0 / 3.0 * th) - 1) < 1e-6
    assert abs(O.cs2(O.EOS_TM, 0.0, 1.0, 1e8) - 1.0 / 3.0) < 1e-7
    assert abs(O.enthalpy(O.EOS_TM, 0.0, 1.0, 1e8) / (4e8) - 1) < 1e-7
    # ideal: cold cs^2 -> Gamma Theta, hot cs^2 -> Gamma-1
    assert abs(O.cs2(O.EOS_IDEAL, 5 / 3, 1.0, 1e-9) / (5 / 3 * 1e-9) - 1) < 1e-8
    assert abs(O.cs2(O.EOS_IDEAL, 4 / 3, 1.0, 1e9) - 1.0 / 3.0) < 1e-8


# ------------------------------------------------------------------ O1: Eq. 2 and Eq. 4 -------
@pytest.mark.parametrize("eos,G", EOSES)
def test_prim2con_and_flux_are_the_boosted_stress_energy_tensor(eos, G):
    """[E, M; M, momentum flux] = Lambda T_rest Lambda^T and [D, D-flux] = Lambda N_rest for a
    perfect fluid (T_rest = diag(rho h - P, P, P, P), N_rest = (rho,0,0,0)): pins Eq. 2 and Eq. 4
    (signs, factors of gamma, which index carries the pressure) against plain matrix algebra."""
    rng = np.random.default_rng(2)
    for _ in range(50):
        rho = 10.0 ** rng.uniform(-3, 2)
        P = rho * 10.0 ** rng.uniform(-3, 2)
        u = rng.normal(size=3) * 10.0 ** rng.uniform(-2, 1)
        g = math.sqrt(1 + u @ u)
        v = u / g
        h = O.enthalpy(eos, G, rho, P)
        L = np.eye(4)                                  # boost from the rest frame to velocity v
        L[0, 0] = g
        L[0, 1:] = L[1:, 0] = g * v
        L[1:, 1:] += (g - 1) * np.outer(v, v) / (v @ v)
        T = L @ np.diag([rho * h - P, P, P, P]) @ L.T
        Nvec = L @ np.array([rho, 0, 0, 0])
        W = np.array([rho, *u, P])
        U = O.prim2con(eos, G, W)
        scale = T[0, 0]
        assert abs(U[0] - Nvec[0]) < 1e-13 * Nvec[0]
        assert np.allclose(U[1:4], T[0, 1:], atol=1e-13 * scale)
        assert abs(U[4] - T[0, 0]) < 1e-13 * scale
        for d in range(3):
            F = O.flux(eos, G, W, d)
            assert abs(F[0] - Nvec[1 + d]) < 1e-13 * Nvec[0]
            assert np.allclose(F[1:4], T[1 + d, 1:], atol=1e-13 * scale)
            assert abs(F[4] - T[0, 1 + d]) < 1e-13 * scale


def test_prim2con_rest_frame_closed_form():
    # at rest: D = rho, M = 0, E = rho + P/(Gamma-1) for the ideal gas (internal energy)
    U = O.prim2con(O.EOS_IDEAL, 5.0 / 3.0, [2.0, 0, 0, 0, 3.0])
    assert np.allclose(U, [2.0, 0, 0, 0, 2.0 + 3.0 / (2.0 / 3.0)], atol=1e-15)


# ------------------------------------------------------------------ Eq. 21-22 -----------------
def _num_jacobian_eigs(eos, G, W, d):
    U0 = O.prim2con(eos, G, W)

    def F(U):
        Wp, st, _ = O.con2prim(eos, G, U)
        assert st == 0
        return O.flux(eos, G, Wp, d)
    J = np.zeros((5, 5))
    for k in range(5):
        hk = 1e-6 * max(abs(U0[k]), 0.1 * U0[4])
        Up, Um = U0.copy(), U0.copy()
        Up[k] += hk; Um[k] -= hk
        J[:, k] = (F(Up) - F(Um)) / (2 * hk)
    return np.sort(np.linalg.eigvals(J).real)


@pytest.mark.parametrize("eos,G", EOSES)
def test_wavespeeds_are_extreme_eigenvalues_of_flux_jacobian(eos, G):
    rng = np.random.default_rng(3)
    for _ in range(20):
        rho = 10.0 ** rng.uniform(-1, 1)
        P = rho * 10.0 ** rng.uniform(-2, 1)
        u = rng.normal(size=3) * 10.0 ** rng.uniform(-1, 0.5)
        W = np.array([rho, *u, P])
        for d in range(3):
            ev = _num_jacobian_eigs(eos, G, W, d)
            lm, lp = O.wavespeeds(eos, G, W, d)
            vd = u[d] / math.sqrt(1 + u @ u)
            assert abs(ev[0] - lm) < 2e-6 and abs(ev[-1] - lp) < 2e-6
            assert np.allclose(ev[1:4], vd, atol=2e-5)        # triple middle eigenvalue v_d


@pytest.mark.parametrize("eos,G", EOSES)
def test_wavespeeds_closed_forms(eos, G):
    # at rest: +-cs;  purely normal flow: relativistic velocity addition (v +- cs)/(1 +- v cs)
    cs = math.sqrt(O.cs2(eos, G, 1.3, 0.7))
    lm, lp = O.wavespeeds(eos, G, [1.3, 0, 0, 0, 0.7], 1)
    assert abs(lm + cs) < 1e-15 and abs(lp - cs) < 1e-15
    v = 0.6
    u = v / math.sqrt(1 - v * v)
    lm, lp = O.wavespeeds(eos, G, [1.3, 0, u, 0, 0.7], 1)
    assert abs(lp - (v + cs) / (1 + v * cs)) < 1e-14
    assert abs(lm - (v - cs) / (1 - v * cs)) < 1e-14
    # transverse direction of the same flow: symmetric pair
    lm, lp = O.wavespeeds(eos, G, [1.3, 0, u, 0, 0.7], 0)
    assert abs(lm + lp) < 1e-15 and 0 < lp < cs


# ------------------------------------------------------------------ HLL (R9) ------------------
@pytest.mark.parametrize("eos,G", EOSES)
def test_hll_consistency_upwinding_and_jump_conditions(eos, G):
    rng = np.random.default_rng(4)
    for _ in range(30):
        WL = np.array([10 ** rng.uniform(-1, 1), *rng.normal(size=3) * 0.5, 10 ** rng.uniform(-2, 1)])
        WR = np.array([10 ** rng.uniform(-1, 1), *rng.normal(size=3) * 0.5, 10 ** rng.uniform(-2, 1)])
        d = int(rng.integers(3))
        Fc = O.flux(eos, G, WL, d)                                                  # F^(W,W)=F(W)
        assert np.allclose(O.hll(eos, G, WL, WL, d), Fc, rtol=0, atol=4e-16 * np.abs(Fc).max())
        F = O.hll(eos, G, WL, WR, d)
        lL = min(O.wavespeeds(eos, G, WL, d)[0], O.wavespeeds(eos, G, WR, d)[0])    # Eq. 23
        lR = max(O.wavespeeds(eos, G, WL, d)[1], O.wavespeeds(eos, G, WR, d)[1])    # Eq. 24
        UL, UR = O.prim2con(eos, G, WL), O.prim2con(eos, G, WR)
        FL, FR = O.flux(eos, G, WL, d), O.flux(eos, G, WR, d)
        if lL < 0 < lR:
            # integral (Rankine-Hugoniot) form: one intermediate state U* joins both outer waves
            Us_L = UL + (F - FL) / lL
            Us_R = UR + (F - FR) / lR
            assert np.allclose(Us_L, Us_R, rtol=0, atol=1e-12 * max(UL[4], UR[4]) / min(-lL, lR))
    # supersonic to the right / left picks the upwind flux exactly
    fast = 5.0
    WL = np.array([1.0, fast, 0, 0, 0.01]); WR = np.array([0.5, fast, 0.1, 0, 0.02])
    assert np.array_equal(O.hll(0, 5 / 3, WL, WR, 0), O.flux(0, 5 / 3, WL, 0))
    WL[1] = WR[1] = -fast
    assert np.array_equal(O.hll(0, 5 / 3, WL, WR, 0), O.flux(0, 5 / 3, WR, 0))
    # mirror symmetry: reflecting the problem flips the sign of the mass/energy/normal-momentum flux
    WL = np.array([1.0, 0.3, 0.2, -0.1, 1.0]); WR = np.array([0.3, -0.4, 0.1, 0.2, 0.2])
    F = O.hll(1, 0.0, WL, WR, 0)
    mir = lambda W: np.array([W[0], -W[1], W[2], W[3], W[4]])
    Fm = O.hll(1, 0.0, mir(WR), mir(WL), 0)
    assert np.allclose(Fm, [-F[0], F[1], -F[2], -F[3], -F[4]], atol=1e-15)


# ------------------------------------------------------------------ O2/O3: con2prim -----------
def _mp_con2prim(eos, G, U, dps=50):
    """Independent formulation at 50 digits: solve for the pressure (Schneider et al. style):
    v = M/(E+P), gamma = 1/sqrt(1-v^2), rho = D/gamma, residual = rho h(rho,P) gamma^2 - (E+P)."""
    mp.mp.dps = dps
    D, E = mp.mpf(float(U[0])), mp.mpf(float(U[4]))
    M = mp.sqrt(sum(mp.mpf(float(m)) ** 2 for m in U[1:4]))

    def hfun(rho, P):
        th = P / rho
        if eos == O.EOS_IDEAL:
            return 1 + mp.mpf(G) / (mp.mpf(G) - 1) * th
        return mp.mpf(5) / 2 * th + mp.mpf(3) / 2 * mp.sqrt(th * th + mp.mpf(4) / 9)

    def res(P):
        v = M / (E + P)
        g = 1 / mp.sqrt(1 - v * v)
        rho = D / g
        return rho * hfun(rho, P) * g * g - (E + P)
    lo = max(mp.mpf(0), M - E) + mp.mpf(10) ** (-45) * E
    hi = 2 * E
    P = mp.findroot(res, (lo, hi), solver="anderson", tol=mp.mpf(10) ** (-70), maxsteps=400,
                    verify=False)
    P = mp.findroot(res, P, tol=mp.mpf(10) ** (-90), maxsteps=100, verify=False)  # Newton polish
    v = M / (E + P)
    g = 1 / mp.sqrt(1 - v * v)
    return D / g, g * v, P


@pytest.mark.parametrize("eos,G", [(O.EOS_IDEAL, 4.0 / 3.0), (O.EOS_IDEAL, 5.0 / 3.0), (O.EOS_TM, 0.0)])
def test_con2prim_matches_50_digit_pressure_solve(eos, G):
    W = I.c2p_states(7, 120).numpy()
    U = O.prim2con_batch(eos, G, W)
    for k in range(W.shape[1]):
        Wk, st, _ = O.con2prim(eos, G, U[:, k])
        assert st == 0
        rho, umag, P = _mp_con2prim(eos, G, U[:, k])
        g2 = 1 + float(umag) ** 2
        # conditioning-aware bounds (R6): rho,|u| ~ eps*gamma^2, P absolute ~ eps*E
        assert abs(Wk[0] / float(rho) - 1) < 40 * 2.2e-16 * g2 + 1e-14
        assert abs(np.linalg.norm(Wk[1:4]) / float(umag) - 1) < 40 * 2.2e-16 * g2 + 5e-12 * (eos == 1)
        assert abs(Wk[4] - float(P)) < 1e-10 * float(P) + 1e-14 * U[4, k]


@pytest.mark.parametrize("eos,G", [(O.EOS_IDEAL, 4.0 / 3.0), (O.EOS_TM, 0.0)])
def test_con2prim_round_trip_config3_domain(eos, G):
    """prim -> con (Eq. 4) -> prim with exactly known primitives (protocol of PAPER.md:405)."""
    W = I.c2p_states(11, 20000).numpy()
    U = O.prim2con_batch(eos, G, W)
    W2, st = O.con2prim_batch(eos, G, U)
    assert st.max() == 0
    g2 = 1 + (W[1:4] ** 2).sum(0)
    umag, umag2 = np.sqrt((W[1:4] ** 2).sum(0)), np.sqrt((W2[1:4] ** 2).sum(0))
    beta, beta2 = umag / np.sqrt(g2), umag2 / np.sqrt(1 + umag2 ** 2)
    assert np.max(np.abs(beta2 - beta)) < 2e-14                       # velocity itself: ~eps
    assert np.max(np.abs(W2[0] / W[0] - 1) / g2) < 50 * 2.2e-16
    assert np.max(np.abs(umag2 / np.maximum(umag, 1e-300) - 1) / g2) < (50 if eos == 0 else 5e4) * 2.2e-16
    dirn, dirn2 = W[1:4] / umag, W2[1:4] / umag2
    assert np.max(np.abs(dirn - dirn2)) < 1e-14
    assert np.max(np.abs(W2[4] - W[4]) / U[4]) < 5e-15                # |dP|/E ~ eps
    assert np.max(np.abs(W2[4] / W[4] - 1)) < 1e-5                    # plain relative P: cancellation


def test_tm_both_cubic_branches_are_exercised_and_agree():
    """Eq. 69 (d<0) and Eq. 71 (d>=0) both occur over the config-3 domain and both round-trip."""
    W = I.c2p_states(5, 4000).numpy()
    U = O.prim2con_batch(O.EOS_TM, 0.0, W)
    xi = np.sqrt((U[1:4] ** 2).sum(0)) / U[0]; eta = U[4] / U[0]
    den = ((eta - xi) * (eta + xi)) ** 2; s = eta ** 2 + xi ** 2; br = 4 * s - (xi ** 2 + 1)
    c1 = (s * br - 14 * xi ** 2 * eta ** 2) / (2 * den); c2 = (br ** 2 - 57 * xi ** 2 * eta ** 2) / (16 * den)
    c3 = -9 * xi ** 2 * eta ** 2 / (16 * den)
    d = ((3 * c2 - c1 ** 2) / 9) ** 3 + ((9 * c1 * c2 - 27 * c3 - 2 * c1 ** 3) / 54) ** 2
    assert (d < 0).sum() > 100 and (d >= 0).sum() > 100
    W2, st = O.con2prim_batch(O.EOS_TM, 0.0, U)
    g2 = 1 + (W[1:4] ** 2).sum(0)
    for mask in (d < 0, d >= 0):
        assert st[mask].max() == 0
        assert np.max(np.abs(W2[0, mask] / W[0, mask] - 1) / g2[mask]) < 50 * 2.2e-16


def test_tm_recovers_slow_flows_to_full_relative_accuracy():
    """Reading R7b: as gamma -> 1 the closed-form root of Eq. 61 (W = gamma^2 - 1 = |u|^2) carries an
    absolute error ~1e-16, i.e. no correct digits of u below |u| ~ 1e-8; with one Newton correction on
    the cubic the round trip from exactly known primitives recovers u to ~1e-13 relative over
    |u| in [1e-9, 1e-1], for cold and hot gas alike (Fig. 2 protocol :405)."""
    rng = np.random.default_rng(4)
    n = 4000
    umag = 10.0 ** rng.uniform(-9, -1, n)
    dirn = rng.normal(size=(3, n)); dirn /= np.sqrt((dirn ** 2).sum(0))
    rho = 10.0 ** rng.uniform(-3, 2, n)
    P = rho * 10.0 ** rng.uniform(-6, 3, n)
    W = np.vstack([rho[None], umag * dirn, P[None]])
    U = O.prim2con_batch(O.EOS_TM, 0.0, W)
    W2, st = O.con2prim_batch(O.EOS_TM, 0.0, U)
    assert st.max() == 0
    u2 = np.sqrt((W2[1:4] ** 2).sum(0))
    assert np.max(np.abs(u2 / umag - 1)) < 2e-12
    assert np.max(np.abs(W2[0] / rho - 1)) < 1e-14
    assert np.max(np.abs(W2[4] - P) / (P + 1e-3 * U[4])) < 1e-11


def test_ideal_newton_iteration_claims_of_the_paper():
    """tests/golden/con2prim_iteration_claims.txt: on the Fig. 2 grid the
    iterative ideal solver reaches (near) machine precision in velocity with 6 iterations for
    Lorentz factors below 10 and with 12 iterations for all Lorentz factors up to 100."""
    claims = []
    for line in open(os.path.join(GOLD, "con2prim_iteration_claims.txt")):
        if line.strip() and not line.startswith("#"):
            nit, gmax, tol = line.split()[:3]
            claims.append((int(nit), float(gmax), float(tol)))
    assert len(claims) == 2
    Wg, lor = I.fig2_grid()
    Wg, lor = Wg.numpy(), lor.numpy()
    beta = np.sqrt((lor - 1) * (lor + 1)) / lor
    for G in (4.0 / 3.0, 5.0 / 3.0):
        U = O.prim2con_batch(O.EOS_IDEAL, G, Wg)
        for nit, gmax, tol in claims:
            for k in np.nonzero(lor <= gmax)[0]:
                Wk, st = O.con2prim_ideal_fixed(G, U[:, k], nit)
                b = Wk[1] / math.sqrt(1 + Wk[1] ** 2)
                if beta[k] == 0.0:
                    assert b == 0.0
                else:
                    assert abs(b / beta[k] - 1) < tol, (G, nit, lor[k], b, beta[k])
        # the adaptive stopping rule (R3) lands on the same root and within 16 iterations
        for k in range(Wg.shape[1]):
            Wk, st, nit = O.con2prim(O.EOS_IDEAL, G, U[:, k])
            assert st == 0 and nit <= 16
            if beta[k] > 0:
                assert abs(Wk[1] / math.sqrt(1 + Wk[1] ** 2) / beta[k] - 1) < 5e-15


def test_small_xi_series_eq60_matches_newton_across_the_switch():
    G = 5.0 / 3.0
    for th in (1e-6, 1e-2, 10.0):
        for umag in (0.99e-4, 0.5e-4, 1e-6, 1e-9):      # xi ~ h*u straddles/below 1e-4
            W = np.array([1.0, umag * 0.6, -umag * 0.8, 0.0, th])
            U = O.prim2con(O.EOS_IDEAL, G, W)
            Wa, st, nit = O.con2prim(O.EOS_IDEAL, G, U)
            Wb, stb = O.con2prim_ideal_fixed(G, U, 12)  # pure Newton (bypasses Eq. 60)
            assert st == 0 and stb == 0
            assert np.allclose(Wa[1:4], Wb[1:4], rtol=2e-15, atol=0)
            assert np.allclose(Wa[1:4], W[1:4], rtol=5e-15, atol=0)
            assert abs(Wa[4] - W[4]) < 1e-15 * U[4] * 10
    # zero momentum: exactly at rest
    U = O.prim2con(O.EOS_IDEAL, G, [2.0, 0, 0, 0, 0.5])
    Wz, st, _ = O.con2prim(O.EOS_IDEAL, G, U)
    assert st == 0 and np.all(Wz[1:4] == 0) and Wz[0] == 2.0 and abs(Wz[4] - 0.5) < 1e-15
    Wz, st, _ = O.con2prim(O.EOS_TM, 0.0, O.prim2con(O.EOS_TM, 0.0, [2.0, 0, 0, 0, 0.5]))
    assert st == 0 and np.all(Wz[1:4] == 0) and abs(Wz[0] - 2.0) < 1e-15 and abs(Wz[4] - 0.5) < 1e-14


@pytest.mark.parametrize("eos,G", [(O.EOS_IDEAL, 5.0 / 3.0), (O.EOS_TM, 0.0)])
def test_con2prim_rejects_inadmissible_states(eos, G):
    for U in ([-1.0, 0, 0, 0, 1.0], [1.0, 2.0, 0, 0, 2.0], [1.0, 0, 0, 0, 0.5],
              [1.0, 0.1, 0, 0, float("nan")]):
        W, st, _ = O.con2prim(eos, G, U)
        assert st == 1 and np.all(np.isnan(W))


# ------------------------------------------------------------------------------------------------
# HLLC interface flux (SURVEY.md 8(f).1; PAPER.md:126, :161 ref [34]) -- pins that do not restate it
# ------------------------------------------------------------------------------------------------
def _random_pair(rng, eos):
    def one():
        rho, P = 10.0 ** rng.uniform(-2, 1), 10.0 ** rng.uniform(-3, 1)
        v = rng.uniform(-0.6, 0.6, 3)
        g = 1.0 / np.sqrt(1.0 - v @ v)
        return np.array([rho, *(g * v), P])
    return one(), one()


@pytest.mark.parametrize("eos,G", [(0, 5.0 / 3.0), (0, 4.0 / 3.0), (1, 0.0)])
def test_hllc_star_states_satisfy_the_jump_conditions_of_all_three_waves(eos, G):
    """Rankine-Hugoniot across lambda_L, lambda* and lambda_R, the integral (consistency) relation, the
    contact conditions m* = (E* + p*) lambda* with ONE p* on both sides, and lambda_L <= lambda* <= lambda_R:
    a dropped term or wrong sign in any star-state formula breaks one of them."""
    rng = np.random.default_rng(3)
    for _ in range(400):
        WL, WR = _random_pair(rng, eos)
        for d in range(3):
            F, ls, UsL, UsR = O.hllc(eos, G, WL, WR, d)
            lmL, lpL = O.wavespeeds(eos, G, WL, d)
            lmR, lpR = O.wavespeeds(eos, G, WR, d)
            lL, lR = min(lmL, lmR), max(lpL, lpR)
            UL, UR = O.prim2con(eos, G, WL), O.prim2con(eos, G, WR)
            FL, FR = O.flux(eos, G, WL, d), O.flux(eos, G, WR, d)
            assert lL - 1e-14 <= ls <= lR + 1e-14
            Uh = (lR * UR - lL * UL + FL - FR) / (lR - lL)
            sc = np.abs(UL) + np.abs(UR) + 1e-300
            assert np.max(np.abs((ls - lL) * UsL + (lR - ls) * UsR - (lR - lL) * Uh) / sc) < 1e-12
            FsL, FsR = FL + lL * (UsL - UL), FR + lR * (UsR - UR)          # RH across the outer waves
            assert np.max(np.abs(FsR - FsL - ls * (UsR - UsL)) / sc) < 1e-12   # RH across the contact
            # one pressure on both sides of the contact, from either side's normal-momentum flux:
            # F*_m = m* lambda* + p*  and  F*_E = m* ;  m* = (E* + p*) lambda*
            m = 1 + d
            pL, pR = FsL[m] - UsL[m] * ls, FsR[m] - UsR[m] * ls
            assert abs(pL - pR) <= 1e-11 * max(abs(pL), 1e-3)
            for Us, p in ((UsL, pL), (UsR, pR)):
                assert abs(Us[m] - (Us[4] + p) * ls) <= 1e-11 * max(abs(Us[4]), 1e-3)


def test_hllc_is_consistent_upwinds_and_mirrors():
    rng = np.random.default_rng(5)
    for eos, G in ((0, 5.0 / 3.0), (1, 0.0)):
        for _ in range(50):
            WL, WR = _random_pair(rng, eos)
            for d in range(3):
                F, _, _, _ = O.hllc(eos, G, WL, WL, d)                     # F(W, W) = F(W)
                np.testing.assert_allclose(F, O.flux(eos, G, WL, d), rtol=1e-12, atol=1e-14)
                Fm, _, _, _ = O.hllc(eos, G, WR * [1, -1, -1, -1, 1], WL * [1, -1, -1, -1, 1], d)
                F, _, _, _ = O.hllc(eos, G, WL, WR, d)                     # mirror image
                np.testing.assert_allclose(Fm, -F * [1, -1, -1, -1, 1], rtol=1e-11, atol=1e-13)
        Ws = np.array([1.0, 3.0, 0.2, 0.0, 0.5])                           # supersonic to the right
        F, _, _, _ = O.hllc(eos, G, Ws, Ws * [0.5, 1, 1, 1, 0.7], 0)
        np.testing.assert_allclose(F, O.flux(eos, G, Ws, 0), rtol=1e-14)


@pytest.mark.parametrize("eos,G", [(0, 5.0 / 3.0), (1, 0.0)])
def test_hllc_preserves_an_isolated_contact_exactly_while_hll_smears_it(eos, G):
    """Equal velocity and pressure, a density jump: the exact flux at the interface is the upwind one.
    HLLC returns it to rounding (the point of the third wave); the two-wave HLL flux does not."""
    for vx in (0.3, -0.45):
        g = 1.0 / np.sqrt(1.0 - vx * vx - 0.04)
        WL = np.array([1.0, g * vx, g * 0.2, 0.0, 0.7])
        WR = np.array([0.05, g * vx, g * 0.2, 0.0, 0.7])
        exact = O.flux(eos, G, WL if vx > 0 else WR, 0)
        F, ls, _, _ = O.hllc(eos, G, WL, WR, 0)
        assert abs(ls - vx) < 1e-13
        np.testing.assert_allclose(F, exact, rtol=1e-12, atol=1e-14)
        assert np.max(np.abs(O.hll(eos, G, WL, WR, 0) - exact)) > 1e-3


# ------------------------------------------------------------------------------------------------
# The paper's comparison variants of con2prim: ideal analytic quartic, TM Brent
# ------------------------------------------------------------------------------------------------
def _variant_claims():
    out = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "con2prim_variant_claims.txt")):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            out[k] = [float(x) for x in v]
    return out


def _beta_err(Wv, W, lor):
    beta = W[1] / lor
    bv = Wv[1] / np.sqrt(1.0 + Wv[1] ** 2)
    return np.abs(bv - beta) / np.maximum(beta, 1e-300)


@pytest.mark.parametrize("G", [5.0 / 3.0, 4.0 / 3.0])
def test_ideal_analytic_quartic_reproduces_the_accuracy_the_paper_reports(G):
    """Fig. 2's protocol on the restated Eq. 39-57: ~1e-15 below gamma = 3, a power-law loss to ~1e-10
    at gamma = 100 -- and the true beta is a root of the quartic with the restored
    beta^3 term (a wrong coefficient or sign in Eq. 40-53 moves every error to O(1))."""
    cl = _variant_claims()
    W, lor = I.fig2_grid(25)
    W, lor = W.numpy(), lor.numpy()
    U = O.prim2con_batch(0, G, W)
    Wv, st = O.con2prim_variant_batch(0, 1, G, U)
    assert (st == 0).all()
    err = _beta_err(Wv, W, lor)
    mov = W[1] > 0
    lo, hi = mov & (lor < 3.0), lor > 90.0
    assert np.median(err[lo]) <= 5 * cl["ideal_analytic_err_below_gamma_3"][0] and err[lo].max() <= 1e-13
    assert 1e-13 <= err[hi].max() <= 3 * cl["ideal_analytic_err_at_gamma_100"][0]
    # power law: the median error grows monotonically over decades of gamma
    med = [np.median(err[mov & (lor >= a) & (lor < b)]) for a, b in ((1, 3), (3, 10), (10, 30), (30, 101))]
    assert all(m2 > 2 * m1 for m1, m2 in zip(med, med[1:]))
    # the iterative solver of the hot path is at machine precision on the same grid
    W0, _ = O.con2prim_batch(0, G, U)
    assert _beta_err(W0, W, lor)[mov].max() <= 5e-15
    # rest of the primitives at a benign point
    k = int(np.argmin(np.abs(lor - 2.0)))
    np.testing.assert_allclose(Wv[[0, 1], k], W[[0, 1], k], rtol=1e-12)


def test_tm_brent_converges_to_the_analytic_root_and_needs_the_iterations_the_paper_reports():
    cl = _variant_claims()
    W, lor = I.fig2_grid(25)
    W, lor = W.numpy(), lor.numpy()
    U = O.prim2con_batch(1, 0.0, W)
    mov = W[1] > 0
    Wa, _ = O.con2prim_batch(1, 0.0, U)
    errs = {}
    for mi in (5, 25, 50):
        Wv, st = O.con2prim_variant_batch(1, 1, 0.0, U, mi)
        errs[mi] = _beta_err(Wv, W, lor)[mov].max()
    assert errs[50] <= 5e-15 and _beta_err(Wa, W, lor)[mov].max() <= 5e-15      # both at machine precision
    assert errs[int(cl["tm_brent_min_iterations_to_match"][0])] > 1e-3          # 5 iterations are not enough
    assert errs[25] > errs[50]                                                  # nor 25 everywhere (Fig. 2)
    its = [O.con2prim_variant(1, 1, 0.0, U[:, i], 100)[2] for i in range(0, U.shape[1], 7)]
    assert min(i for i in its if i > 0) > 5 and max(its) > 15                   # ">5 and up to >15"
    # re-bracketing: a root far above gamma = 200
    Wf = np.array([1.0, 5e3, 0.0, 0.0, 0.1])
    Wr, st, _ = O.con2prim_variant(1, 1, 0.0, O.prim2con(1, 0.0, Wf), 100)
    assert st == 0 and abs(Wr[1] / Wf[1] - 1) < 1e-8
    # inadmissible input is rejected like in the hot-path solvers
    assert O.con2prim_variant(1, 1, 0.0, [1.0, 2.0, 0, 0, 1.5])[1] == 1
    assert O.con2prim_variant(0, 1, 5 / 3, [1.0, 2.0, 0, 0, 1.5])[1] == 1
