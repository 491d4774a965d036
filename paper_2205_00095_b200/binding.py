"""Thin ctypes binding over libdgrhd.so (include/dgrhd.h) -- argument marshalling only.

Every function has the name of the C entry point it calls; tensors are torch CUDA float64 tensors
whose ``data_ptr()`` is handed through (PyTorch is used for device memory and streams only).  There
is no CPU fallback: if the library is missing or a call fails, a ``DgrhdError`` is raised.
"""
import ctypes as C
import os

import torch

EOS_IDEAL, EOS_TAUB_MATTHEWS = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_DIRICHLET = 0, 1, 2, 3
RIEMANN_HLL, RIEMANN_HLLC = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, 1, 2, 3, 4
OPT_CUDA_GRAPH = 0
C2P_DEFAULT, C2P_ALTERNATE = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
# DGRHD_DEBUG_ASSERTS=1 selects the bounds-checked debug build (python -m paper_2205_00095_b200.build --debug-asserts)
LIB_PATH = os.path.join(_HERE, "libdgrhd_dbg.so" if os.environ.get("DGRHD_DEBUG_ASSERTS") == "1" else "libdgrhd.so")


class DgrhdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dgrhd error {code}: {msg}")
        self.code = code


class Config(C.Structure):
    """dgrhd_config of include/dgrhd.h."""
    _fields_ = [("ndim", C.c_int), ("nelem", C.c_int64 * 3), ("xmin", C.c_double * 3),
                ("xmax", C.c_double * 3), ("bc", C.c_int * 3), ("order_p", C.c_int),
                ("eos", C.c_int), ("gamma_ad", C.c_double), ("rk_stages", C.c_int),
                ("eps_q", C.c_double), ("delta_s", C.c_double), ("riemann", C.c_int),
                ("shock_limiter", C.c_int), ("moe_alpha", C.c_double),
                ("bc_state", C.c_double * 5 * 2 * 3)]


def _bc_code(b):
    """int (both ends) or (lo, hi) -> DGRHD_BC_PAIR(lo, hi); periodic at exactly one end has no encoding
    and gives -1, which the library rejects as an invalid configuration."""
    if isinstance(b, (tuple, list)):
        lo, hi = int(b[0]), int(b[1])
        if lo == hi:
            return lo
        return -1 if BC_PERIODIC in (lo, hi) else lo + 256 * hi
    return int(b)


def make_config(ndim, nelem, xmin, xmax, bc, order_p, eos, gamma_ad, rk_stages=3, eps_q=1e-12,
                delta_s=1e-10, riemann=0, bc_state=None, shock_limiter=0, moe_alpha=0.0):
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
    for (d, side), W in (bc_state or {}).items():      # {(axis, end): [rho, ux, uy, uz, P]}
        for v in range(5):
            c.bc_state[d][side][v] = float(W[v])
    return c


_lib = None
_vp, _dp, _i64p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)

EXPORTS = ("dgrhd_workspace_bytes", "dgrhd_create", "dgrhd_destroy", "dgrhd_set_state",
           "dgrhd_get_state", "dgrhd_get_prims", "dgrhd_rhs", "dgrhd_enforce_physicality",
           "dgrhd_cfl_dt", "dgrhd_step", "dgrhd_get_counters", "dgrhd_con2prim_batch",
           "dgrhd_prim2con_batch", "dgrhd_con2prim_batch_host", "dgrhd_run_host", "dgrhd_tm_fallback_count", "dgrhd_probe_fp64", "dgrhd_con2prim_batch_variant", "dgrhd_shock_limiter",
           "dgrhd_set_option", "dgrhd_last_error", "dgrhd_version", "dgrhd_rhs_static")


def lib():
    """Load libdgrhd.so (hard error if it has not been built: python -m paper_2205_00095_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise DgrhdError(ECUDA, f"{LIB_PATH} not built; run python -m paper_2205_00095_b200.build "
                                    "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.dgrhd_workspace_bytes.restype = C.c_size_t
        L.dgrhd_workspace_bytes.argtypes = [C.POINTER(Config)]
        L.dgrhd_create.argtypes = [C.POINTER(Config), _vp, C.c_size_t, _vp, C.POINTER(_vp)]
        L.dgrhd_destroy.argtypes = [_vp]
        L.dgrhd_set_option.argtypes = [_vp, C.c_int, C.c_int]
        L.dgrhd_set_state.argtypes = [_vp, _vp]
        L.dgrhd_get_state.argtypes = [_vp, _vp]
        L.dgrhd_get_prims.argtypes = [_vp, _vp]
        L.dgrhd_rhs.argtypes = [_vp, _vp, _vp]
        L.dgrhd_rhs_static.argtypes = [C.POINTER(Config), _vp, _vp, _i64p, _vp]
        L.dgrhd_enforce_physicality.argtypes = [_vp, _vp, _vp, _vp, _i64p]
        L.dgrhd_cfl_dt.argtypes = [_vp, _vp, C.c_double, _dp]
        L.dgrhd_shock_limiter.argtypes = [_vp, _vp, _vp]
        L.dgrhd_step.argtypes = [_vp, C.c_double, C.c_int, _dp]
        L.dgrhd_get_counters.argtypes = [_vp, _i64p, C.c_int]
        L.dgrhd_con2prim_batch.argtypes = [C.c_int, C.c_double, C.c_int64, _vp, _vp, _vp, _vp]
        L.dgrhd_tm_fallback_count.argtypes = [_i64p, C.c_int, _vp]
        L.dgrhd_con2prim_batch_variant.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int64, _vp, _vp, _vp,
                                                   C.c_int, _vp]
        L.dgrhd_probe_fp64.argtypes = [_vp, _dp, _dp, _vp]
        L.dgrhd_prim2con_batch.argtypes = [C.c_int, C.c_double, C.c_int64, _vp, _vp, _vp]
        L.dgrhd_con2prim_batch_host.argtypes = [C.c_int, C.c_double, C.c_int64, _vp, _vp, _vp,
                                                C.c_size_t, _vp]
        L.dgrhd_run_host.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _dp]
        L.dgrhd_last_error.restype = C.c_char_p
        L.dgrhd_last_error.argtypes = [_vp]
        L.dgrhd_version.restype = C.c_char_p
        _lib = L
    return _lib


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, rows=None):
    if t is None:
        return None
    assert t.is_contiguous(), "tensor must be contiguous"
    if rows is not None:
        assert t.dtype == torch.float64 and t.shape[0] == rows, "expected float64 [5, n]"
    return C.c_void_p(t.data_ptr())


def _check(code, ctx=None):
    if code != OK:
        raise DgrhdError(code, lib().dgrhd_last_error(ctx).decode())


def dgrhd_version():
    return lib().dgrhd_version().decode()


def dgrhd_workspace_bytes(cfg):
    return int(lib().dgrhd_workspace_bytes(C.byref(cfg)))


class Context:
    """Owner of a dgrhd_ctx and of its workspace tensor; methods carry the C names."""

    def __init__(self, cfg, device="cuda"):
        if isinstance(cfg, dict):
            cfg = make_config(**cfg)
        self.cfg = cfg
        self.n_nodes = (cfg.order_p + 1) ** cfg.ndim
        self.n_elem = 1
        for d in range(cfg.ndim):
            self.n_elem *= cfg.nelem[d]
        self.ndof = self.n_elem * self.n_nodes
        nbytes = dgrhd_workspace_bytes(cfg)
        if nbytes == 0:
            raise DgrhdError(EINVAL, "invalid configuration")
        if not torch.cuda.is_available():
            raise DgrhdError(ECUDA, "no CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._h = C.c_void_p()
        self._stream = torch.cuda.current_stream(self.device)
        _check(lib().dgrhd_create(C.byref(cfg), C.c_void_p(self.workspace.data_ptr()), nbytes,
                                  C.c_void_p(self._stream.cuda_stream), C.byref(self._h)))

    def close(self):
        if self._h:
            lib().dgrhd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def dgrhd_set_option(self, option, value):
        _check(lib().dgrhd_set_option(self._h, option, value), self._h)

    def new_state(self):
        return torch.empty(5, self.ndof, dtype=torch.float64, device=self.device)

    def dgrhd_set_state(self, U):
        _check(lib().dgrhd_set_state(self._h, _ptr(U, 5)), self._h)

    def dgrhd_get_state(self, out=None):
        out = self.new_state() if out is None else out
        _check(lib().dgrhd_get_state(self._h, _ptr(out, 5)), self._h)
        return out

    def dgrhd_get_prims(self, out=None):
        out = self.new_state() if out is None else out
        _check(lib().dgrhd_get_prims(self._h, _ptr(out, 5)), self._h)
        return out

    def dgrhd_rhs(self, U, out=None):
        out = self.new_state() if out is None else out
        _check(lib().dgrhd_rhs(self._h, _ptr(U, 5), _ptr(out, 5)), self._h)
        return out

    def dgrhd_enforce_physicality(self, U=None, want_flags=True, sync=True):
        """In place on U (None = internal state).  Returns (flag[n_e] uint8, s[n_e], counters)."""
        flag = s = None
        if want_flags:
            flag = torch.empty(self.n_elem, dtype=torch.uint8, device=self.device)
            s = torch.empty(self.n_elem, dtype=torch.float64, device=self.device)
        cnt = (C.c_int64 * 2)(0, 0)
        _check(lib().dgrhd_enforce_physicality(self._h, _ptr(U, 5) if U is not None else None,
                                               _ptr(flag), _ptr(s), cnt if sync else None), self._h)
        return flag, s, (int(cnt[0]), int(cnt[1]))

    def dgrhd_shock_limiter(self, U):
        """In place on U.  Returns theta[n_e]."""
        theta = torch.empty(self.n_elem, dtype=torch.float64, device=self.device)
        _check(lib().dgrhd_shock_limiter(self._h, _ptr(U, 5), _ptr(theta)), self._h)
        return theta

    def dgrhd_cfl_dt(self, cfl, U=None):
        dt = C.c_double()
        _check(lib().dgrhd_cfl_dt(self._h, _ptr(U, 5) if U is not None else None, cfl, C.byref(dt)),
               self._h)
        return dt.value

    def dgrhd_step(self, dt, nsteps=1, t=None):
        """dt > 0 fixed; dt < 0: CFL number -dt.  t (float) -> returns the advanced time (syncs)."""
        if t is None:
            _check(lib().dgrhd_step(self._h, dt, nsteps, None), self._h)
            return None
        tt = C.c_double(t)
        _check(lib().dgrhd_step(self._h, dt, nsteps, C.byref(tt)), self._h)
        return tt.value

    def dgrhd_run_host(self, U_host_in, U_host_out, dt, nsteps, t=0.0):
        """Host (pinned) buffers in and out around nsteps steps; synchronises."""
        tt = C.c_double(t)
        _check(lib().dgrhd_run_host(self._h, C.c_void_p(U_host_in.data_ptr()),
                                    C.c_void_p(U_host_out.data_ptr()), dt, nsteps, C.byref(tt)),
               self._h)
        return tt.value

    def dgrhd_get_counters(self, reset=False):
        out = (C.c_int64 * 8)()
        _check(lib().dgrhd_get_counters(self._h, out, int(reset)), self._h)
        return dict(n_flagged=out[0], n_bad_mean=out[1], n_c2p_fail=out[2], n_stages=out[3],
                    n_tm_fallback=out[4], n_bad_dt=out[5], n_shock_limited=out[6])


STATIC_MAX_NDOF = 1 << 20          # DGRHD_STATIC_MAX_NDOF of include/dgrhd.h


def dgrhd_rhs_static(cfg, U, out=None, count_failures=True):
    """R = L(U) through the entry point that needs no context and no workspace: its scratch is an array
    built into libdgrhd.so (at most STATIC_MAX_NDOF nodes; a larger mesh raises DgrhdError ENOMEM).  It is
    meant for callers that cannot allocate device memory at that point (a plug-in whose host application
    owns all of the GPU's memory, a process with a spent memory budget, a loop that must not stall on
    cudaMalloc); the C call allocates nothing.  This wrapper only marshals: when `out` is None it asks
    torch for the output tensor, so pass your own `out` if torch must not allocate either.  Calls share the
    one array: do not let two of them overlap on the GPU.  Returns (R, n_c2p_fail of this call), or
    (R, None) without synchronising when count_failures is False."""
    out = torch.empty_like(U) if out is None else out
    nfail = C.c_int64(-1)
    _check(lib().dgrhd_rhs_static(C.byref(cfg), _ptr(U, 5), _ptr(out, 5),
                                  C.byref(nfail) if count_failures else None, _stream()))
    return out, (int(nfail.value) if count_failures else None)


def dgrhd_con2prim_batch(eos, gamma_ad, U, W=None, status=None):
    W = torch.empty_like(U) if W is None else W
    _check(lib().dgrhd_con2prim_batch(eos, gamma_ad, U.shape[1], _ptr(U, 5), _ptr(W, 5),
                                      _ptr(status), _stream()))
    return W


def dgrhd_con2prim_batch_variant(eos, variant, gamma_ad, U, W=None, status=None, max_iter=50):
    W = torch.empty_like(U) if W is None else W
    _check(lib().dgrhd_con2prim_batch_variant(eos, variant, gamma_ad, U.shape[1], _ptr(U, 5), _ptr(W, 5),
                                              _ptr(status), max_iter, _stream()))
    return W


def dgrhd_tm_fallback_count(reset=False):
    out = C.c_int64()
    _check(lib().dgrhd_tm_fallback_count(C.byref(out), int(reset), _stream()))
    return out.value


def dgrhd_probe_fp64():
    """(sustained FP64 FMA TFLOP/s of the current device, nominal max SM clock in MHz)."""
    scratch = torch.zeros(1, dtype=torch.float64, device="cuda")
    tf, mhz = C.c_double(), C.c_double()
    _check(lib().dgrhd_probe_fp64(_ptr(scratch), C.byref(tf), C.byref(mhz), _stream()))
    return tf.value, mhz.value


def dgrhd_prim2con_batch(eos, gamma_ad, W, U=None):
    U = torch.empty_like(W) if U is None else U
    _check(lib().dgrhd_prim2con_batch(eos, gamma_ad, W.shape[1], _ptr(W, 5), _ptr(U, 5), _stream()))
    return U


def dgrhd_con2prim_batch_host(eos, gamma_ad, U_host, W_host, stage):
    """U_host/W_host: CPU (pinned) float64 [5, n]; stage: CUDA uint8 staging tensor."""
    _check(lib().dgrhd_con2prim_batch_host(eos, gamma_ad, U_host.shape[1],
                                           C.c_void_p(U_host.data_ptr()),
                                           C.c_void_p(W_host.data_ptr()),
                                           C.c_void_p(stage.data_ptr()), stage.numel(), _stream()))
    return W_host
