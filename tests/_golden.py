"""Reader of tests/golden/moe_limiter_cases.txt (hand-worked cases of the shock limiter, reading R18): pure text
parsing, no method arithmetic.  Used by the oracle pin (CPU) and by the GPU test that holds the CUDA path to the
same hand-worked numbers."""
import os
from fractions import Fraction

import numpy as np

VARS = {"D": 0, "Mx": 1, "My": 2, "Mz": 3, "E": 4}
BCS = {"periodic": 0, "outflow": 1}


def _vals(text):
    return [float(Fraction(tok)) for tok in text.replace("|", " ").split()]


def moe_cases():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "moe_limiter_cases.txt")
    cases, cur = [], None
    for raw in open(path):
        line = raw.split("#", 1)[0].strip()
        if not line:
            continue
        key, _, rest = line.partition(" ")
        if key == "case":
            cur = {"name": rest.strip(), "U": {}, "out": {}}
            cases.append(cur)
        elif key in ("ndim", "p"):
            cur[key] = int(rest)
        elif key == "nelem":
            cur["nelem"] = [int(t) for t in rest.split()]
        elif key == "bc":
            cur["bc"] = BCS[rest.strip()]
        elif key == "alpha":
            cur["alpha"] = float(Fraction(rest.strip()))
        elif key == "theta":
            cur["theta"] = np.array(_vals(rest))
        elif key == "out":
            var, _, vals = rest.strip().partition(" ")
            cur["out"][VARS[var]] = np.array(_vals(vals))
        elif key in VARS:
            cur["U"][VARS[key]] = np.array(_vals(rest))
        else:
            raise ValueError(f"{path}: unknown key {key!r}")
    for c in cases:
        ne = int(np.prod(c["nelem"]))
        ndof = ne * (c["p"] + 1) ** c["ndim"]
        U = np.zeros((5, ndof))
        for v, x in c["U"].items():
            assert x.size == ndof, (c["name"], v, x.size, ndof)
            U[v] = x
        assert c["theta"].size == ne and all(x.size == ndof for x in c["out"].values()), c["name"]
        c["state"] = U
        nd = c["ndim"]
        c["cfg"] = dict(ndim=nd, nelem=c["nelem"], xmin=[0.0] * nd, xmax=[1.0] * nd, bc=[c["bc"]] * nd,
                        order_p=c["p"], eos=0, gamma_ad=5.0 / 3.0, rk_stages=3, eps_q=1e-12, delta_s=1e-10,
                        riemann=0, bc_state=None, shock_limiter=1, moe_alpha=c["alpha"])
    return cases
