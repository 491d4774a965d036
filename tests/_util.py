"""Helpers shared by the GPU parity tests: configuration marshalling for both sides, device transfer,
norms and seeded smooth test fields (input data only, no method arithmetic)."""
import numpy as np
import torch

import oracle as O
from paper_2205_00095_b200 import inputs as I

DEV = "cuda"
KEYS = ("ndim", "nelem", "xmin", "xmax", "bc", "order_p", "eos", "gamma_ad", "rk_stages", "eps_q",
        "delta_s", "riemann", "bc_state", "shock_limiter", "moe_alpha")


def B():
    from paper_2205_00095_b200 import binding
    return binding


def ocfg(d, **kw):
    d = {"riemann": 0, "bc_state": None, "shock_limiter": 0, "moe_alpha": 0.0, **d, **kw}
    return O.make_config(*[d[k] for k in KEYS])


def gcfg(d, **kw):
    d = {"riemann": 0, "bc_state": None, "shock_limiter": 0, "moe_alpha": 0.0, **d, **kw}
    return B().make_config(*[d[k] for k in KEYS])


def to_dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(DEV).contiguous()


def relmax(a, b):
    """max|a-b| / max|b| per variable (rows)."""
    a, b = np.asarray(a), np.asarray(b)
    return np.max(np.abs(a - b), axis=1) / np.maximum(np.max(np.abs(b), axis=1), 1e-300)


cell_local_ratio = O.cell_local_ratio          # the cell-local error norm (oracle/__init__.py, test infrastructure)


def cellmax(a, b, nelem, nn):
    """max over cells of cell_local_ratio, per variable."""
    return cell_local_ratio(a, b, nelem, nn).max(1)


def smooth_prims(cfgd, seed, amp=0.3):
    """Smooth, bounded, seeded primitive field on the mesh of cfgd (pure input data)."""
    nd, N = cfgd["ndim"], cfgd["order_p"] + 1
    rng = np.random.default_rng(seed)
    ph = rng.uniform(0, 2 * np.pi, size=(5, 3))
    ax = [I.axis_coords(cfgd["xmin"][d], cfgd["xmax"][d], cfgd["nelem"][d], N).numpy() for d in range(nd)]
    L = [cfgd["xmax"][d] - cfgd["xmin"][d] for d in range(nd)]
    if nd == 1:
        X = [ax[0]]
    elif nd == 2:
        yy, xx = np.meshgrid(ax[1], ax[0], indexing="ij")
        X = [xx, yy]
    else:
        zz, yy, xx = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
        X = [xx, yy, zz]
    s = [sum(np.sin(2 * np.pi * (X[d] - cfgd["xmin"][d]) / L[d] + ph[v, d]) for d in range(nd)) / nd
         for v in range(5)]
    Wg = np.stack([1.0 + amp * s[0], 0.8 * amp * s[1], 0.8 * amp * s[2] * (nd > 1),
                   0.8 * amp * s[3] * (nd > 2), 0.7 + 0.5 * amp * s[4]])
    W = I.grid_to_canonical(torch.from_numpy(Wg), cfgd["nelem"][:nd], N)
    return W.contiguous().numpy()


def mesh(nd, nelem, p, eos, G, bc=None, **kw):
    lo = [0.0, -0.5, 0.25][:nd]
    hi = [1.0, 1.0, 1.0][:nd]
    return I._cfg(nd, nelem, lo, hi, bc or [I.BC_PERIODIC] * nd, p, eos, G, **kw)


def sub_box(U, nelem, nn, org, m):
    """The m^d-element sub-mesh of the canonical state U[5, ndof] with corner element `org`
    (periodic wrap), as a canonical state of its own.  Pure index shuffling."""
    nd = len(nelem)
    idx = [(org[d] + np.arange(m)) % nelem[d] for d in range(nd)]
    if nd == 1:
        e = idx[0]
    elif nd == 2:
        e = (idx[0][None, :] + nelem[0] * idx[1][:, None]).reshape(-1)
    else:
        e = (idx[0][None, None, :] + nelem[0] * (idx[1][None, :, None] + nelem[1] * idx[2][:, None, None])).reshape(-1)
    cols = (e[:, None] * nn + np.arange(nn)[None, :]).reshape(-1)
    return U[:, cols], e


def interior_mask(m, nd, margin):
    """Boolean mask over the m^d elements of a sub-box: True at least `margin` elements from its rim."""
    a = np.arange(m)
    ok = (a >= margin) & (a < m - margin)
    if nd == 1:
        return ok
    if nd == 2:
        return (ok[None, :] & ok[:, None]).reshape(-1)
    return (ok[None, None, :] & ok[None, :, None] & ok[:, None, None]).reshape(-1)
