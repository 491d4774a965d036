"""CPU oracle for the DG-RHD stage -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes/numpy wrapper over ``oracle/dgrhd_oracle.c`` (plain fp64 C written from PAPER.md).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package.  It imports nothing from ``paper_2205_00095_b200``.
All arrays are numpy float64 in the canonical layout ``X[5, ndof]`` (see dgrhd_oracle.h).
"""
import ctypes as C
import numpy as np

from .build import build as _build

EOS_IDEAL, EOS_TM = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_DIRICHLET = 0, 1, 2, 3
RIEMANN_HLL, RIEMANN_HLLC = 0, 1


class Config(C.Structure):
    _fields_ = [("ndim", C.c_int), ("nelem", C.c_int64 * 3), ("xmin", C.c_double * 3),
                ("xmax", C.c_double * 3), ("bc", C.c_int * 3), ("order_p", C.c_int),
                ("eos", C.c_int), ("gamma_ad", C.c_double), ("rk_stages", C.c_int),
                ("eps_q", C.c_double), ("delta_s", C.c_double), ("riemann", C.c_int),
                ("shock_limiter", C.c_int), ("moe_alpha", C.c_double),
                ("bc_state", C.c_double * 5 * 2 * 3)]


def _bc_code(b):
    """int (both ends) or (lo, hi) -> lo + 256*hi (hi = 0: same as lo).  Periodic (0) is a property of the
    whole axis: a pair with periodic at one end only is refused."""
    if isinstance(b, (tuple, list)):
        lo, hi = int(b[0]), int(b[1])
        if lo != hi and 0 in (lo, hi):
            raise ValueError(f"boundary pair {b}: periodic at one end only")
        return lo + 256 * (hi if hi != lo else 0)
    return int(b)


def make_config(ndim, nelem, xmin, xmax, bc, order_p, eos, gamma_ad, rk_stages=3,
                eps_q=1e-12, delta_s=1e-10, riemann=0, bc_state=None, shock_limiter=0, moe_alpha=0.0):
    c = Config()
    c.ndim = ndim
    for d in range(3):
        c.nelem[d] = int(nelem[d]) if d < ndim else 1
        c.xmin[d] = float(xmin[d]) if d < ndim else 0.0
        c.xmax[d] = float(xmax[d]) if d < ndim else 1.0
        c.bc[d] = _bc_code(bc[d]) if d < ndim else 0
    c.order_p, c.eos, c.gamma_ad, c.rk_stages = order_p, eos, gamma_ad, rk_stages
    c.eps_q, c.delta_s = eps_q, delta_s
    c.riemann = int(riemann)
    c.shock_limiter, c.moe_alpha = int(shock_limiter), float(moe_alpha)
    for (d, side), W in (bc_state or {}).items():      # {(axis, side): [rho, ux, uy, uz, P]}
        for v in range(5):
            c.bc_state[d][side][v] = float(W[v])
    return c


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_enthalpy.restype = C.c_double
        L.orc_enthalpy.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_cs2.restype = C.c_double
        L.orc_cs2.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_limiter_node_s.restype = C.c_double
        L.orc_limiter_node_s.argtypes = [_dp, _dp, C.c_double]
        L.orc_cfl_dt.restype = C.c_double
        L.orc_cfl_dt.argtypes = [C.POINTER(Config), _dp, C.c_double]
        L.orc_ndof.restype = C.c_int64
        L.orc_ndof.argtypes = [C.POINTER(Config)]
        L.orc_step.argtypes = [C.POINTER(Config), _dp, C.c_double, C.c_int, _dp,
                               C.POINTER(C.c_int64)]
        L.orc_prim2con_batch.argtypes = [C.c_int, C.c_double, C.c_int64, _dp, _dp]
        L.orc_con2prim_batch.argtypes = [C.c_int, C.c_double, C.c_int64, _dp, _dp,
                                         C.POINTER(C.c_int)]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _v5(x):
    a = np.ascontiguousarray(x, dtype=np.float64)
    assert a.shape == (5,)
    return a


def num_threads():
    return int(lib().orc_num_threads())


def gll(N):
    x, w, D = np.zeros(N), np.zeros(N), np.zeros((N, N))
    lib().orc_gll(C.c_int(N), _p(x), _p(w), _p(D))
    return x, w, D


def enthalpy(eos, G, rho, P):
    return lib().orc_enthalpy(eos, G, rho, P)


def cs2(eos, G, rho, P):
    return lib().orc_cs2(eos, G, rho, P)


def prim2con(eos, G, W):
    U = np.zeros(5)
    lib().orc_prim2con(C.c_int(eos), C.c_double(G), _p(_v5(W)), _p(U))
    return U


def flux(eos, G, W, d):
    F = np.zeros(5)
    lib().orc_flux(C.c_int(eos), C.c_double(G), _p(_v5(W)), C.c_int(d), _p(F))
    return F


def wavespeeds(eos, G, W, d):
    lm, lp = C.c_double(), C.c_double()
    lib().orc_wavespeeds(C.c_int(eos), C.c_double(G), _p(_v5(W)), C.c_int(d), C.byref(lm),
                         C.byref(lp))
    return lm.value, lp.value


def hllc(eos, G, WL, WR, d):
    """Returns (F, lambda*, U*_L, U*_R)."""
    F, UsL, UsR = np.zeros(5), np.zeros(5), np.zeros(5)
    ls = C.c_double()
    lib().orc_hllc(C.c_int(eos), C.c_double(G), _p(_v5(WL)), _p(_v5(WR)), C.c_int(d), _p(F), C.byref(ls),
                   _p(UsL), _p(UsR))
    return F, ls.value, UsL, UsR


def hll(eos, G, WL, WR, d):
    F = np.zeros(5)
    lib().orc_hll(C.c_int(eos), C.c_double(G), _p(_v5(WL)), _p(_v5(WR)), C.c_int(d), _p(F))
    return F


def con2prim(eos, G, U):
    W = np.zeros(5)
    nit = C.c_int()
    st = lib().orc_con2prim(C.c_int(eos), C.c_double(G), _p(_v5(U)), _p(W), C.byref(nit))
    return W, int(st), nit.value


def con2prim_ideal_fixed(G, U, niter):
    W = np.zeros(5)
    st = lib().orc_con2prim_ideal_fixed(C.c_double(G), _p(_v5(U)), _p(W), C.c_int(niter))
    return W, int(st)


def prim2con_batch(eos, G, W):
    W = np.ascontiguousarray(W, dtype=np.float64)
    U = np.empty_like(W)
    lib().orc_prim2con_batch(eos, G, W.shape[1], _p(W), _p(U))
    return U


def con2prim_batch(eos, G, U):
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.empty_like(U)
    st = np.zeros(U.shape[1], dtype=np.int32)
    lib().orc_con2prim_batch(eos, G, U.shape[1], _p(U), _p(W), st.ctypes.data_as(C.POINTER(C.c_int)))
    return W, st


def con2prim_variant(eos, variant, G, U, max_iter=50):
    """variant 1: ideal EOS analytic quartic / Taub-Matthews Brent.  Returns (W, status, iterations)."""
    W = np.zeros(5)
    nit = C.c_int()
    st = lib().orc_con2prim_variant(C.c_int(eos), C.c_int(variant), C.c_double(G), _p(_v5(U)), _p(W),
                                    C.c_int(max_iter), C.byref(nit))
    return W, int(st), nit.value


def con2prim_variant_batch(eos, variant, G, U, max_iter=50):
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.empty_like(U)
    st = np.zeros(U.shape[1], dtype=np.int32)
    lib().orc_con2prim_variant_batch(C.c_int(eos), C.c_int(variant), C.c_double(G), C.c_int64(U.shape[1]),
                                     _p(U), _p(W), st.ctypes.data_as(C.POINTER(C.c_int)), C.c_int(max_iter))
    return W, st


def admissible(U, eps=0.0):
    return bool(lib().orc_admissible(_p(_v5(U)), C.c_double(eps)))


def limiter_node_s(Ubar, Ui, eps_q):
    return lib().orc_limiter_node_s(_p(_v5(Ubar)), _p(_v5(Ui)), eps_q)


def ndof(cfg):
    return int(lib().orc_ndof(C.byref(cfg)))


def rhs(cfg, U):
    U = np.ascontiguousarray(U, dtype=np.float64)
    R = np.empty_like(U)
    nf = C.c_int64(0)
    lib().orc_rhs(C.byref(cfg), _p(U), _p(R), C.byref(nf))
    return R, nf.value


def enforce_physicality(cfg, U):
    """Returns (U_limited, flag[n_e] uint8, s[n_e], (n_flagged, n_bad_mean)); U is not modified."""
    U = np.array(U, dtype=np.float64, order="C", copy=True)
    nn = (cfg.order_p + 1) ** cfg.ndim
    ne = U.shape[1] // nn
    flag = np.zeros(ne, dtype=np.uint8)
    s = np.zeros(ne)
    cnt = (C.c_int64 * 2)(0, 0)
    lib().orc_enforce_physicality(C.byref(cfg), _p(U), flag.ctypes.data_as(C.POINTER(C.c_ubyte)),
                                  _p(s), cnt)
    return U, flag, s, (cnt[0], cnt[1])


def shock_limiter(cfg, U):
    """Returns (U_limited, theta[n_e], n_limited); U is not modified."""
    U = np.array(U, dtype=np.float64, order="C", copy=True)
    nn = (cfg.order_p + 1) ** cfg.ndim
    theta = np.zeros(U.shape[1] // nn)
    lib().orc_shock_limiter.restype = C.c_int64
    n = lib().orc_shock_limiter(C.byref(cfg), _p(U), _p(theta))
    return U, theta, int(n)


def cfl_dt(cfg, U, cfl):
    U = np.ascontiguousarray(U, dtype=np.float64)
    return lib().orc_cfl_dt(C.byref(cfg), _p(U), cfl)


def step(cfg, U, dt, nsteps, t=0.0):
    """dt > 0 fixed; dt <= 0: CFL number -dt.  Returns (U_new, t_new, (n_flagged, n_bad_mean,
    n_c2p_fail))."""
    U = np.array(U, dtype=np.float64, order="C", copy=True)
    tt = C.c_double(t)
    cnt = (C.c_int64 * 3)(0, 0, 0)
    lib().orc_step(C.byref(cfg), _p(U), dt, nsteps, C.cast(C.byref(tt), _dp), cnt)
    return U, tt.value, (cnt[0], cnt[1], cnt[2])


# ---------------------------------------------------------------------------------------------
# Norm used by the parity tests and by smoke() (no method arithmetic)
# ---------------------------------------------------------------------------------------------
def cell_local_ratio(a, b, nelem, nn):
    """Cell-local error norm for multi-scale states: per variable and cell, max over the cell's nodes of |a - b|
    divided by the max of |b| over the cell AND its face neighbours (no wrap: at a mesh face the neighbourhood is
    just smaller, which only makes the norm stricter).  The three momentum rows share the scale |M| (a component
    that vanishes locally has no scale of its own), floored at 1e-6 of the neighbourhood's energy density (same
    units, c = 1) so that fluid at rest, whose momentum is rounding noise around zero, has a scale at all.  Unlike relmax, which divides by the GLOBAL maximum, this does
    not let a near-vacuum cell hide a large relative error behind a dense cell elsewhere.  Returns [5, n_elem]."""
    a, b = np.asarray(a), np.asarray(b)
    nd = len(nelem)
    ne = int(np.prod(nelem))
    err = np.abs(a - b).reshape(5, ne, nn).max(2)
    sc = np.abs(b).reshape(5, ne, nn).max(2)
    sc[1:4] = np.maximum(np.sqrt((b[1:4] ** 2).sum(0)).reshape(ne, nn).max(1), 1e-6 * sc[4])[None, :]
    grid = sc.reshape((5,) + tuple(reversed([int(n) for n in nelem])))          # [5, (nz,) (ny,) nx]
    nb = grid.copy()
    for ax in range(1, nd + 1):
        pad = [(0, 0)] * (nd + 1)
        pad[ax] = (1, 1)
        g = np.pad(grid, pad, mode="edge")
        lo = np.take(g, range(0, grid.shape[ax]), axis=ax)
        hi = np.take(g, range(2, grid.shape[ax] + 2), axis=ax)
        nb = np.maximum(nb, np.maximum(lo, hi))
    return err / np.maximum(nb.reshape(5, ne), 1e-300)
