"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path, and therefore holds
none of the method's arithmetic: it only draws seeded random numbers and evaluates the workload's
*primitive* fields W = [rho, ux, uy, uz, P] (u = gamma*v) at the nodal coordinates.
Conserved states are produced from W by each side's own Eq. 4 (``oracle.prim2con_batch`` in tests,
``dgrhd_prim2con_batch`` in the product).  The only table here is where the nodes sit inside an
element (needed to sample a field), not the weights or derivative matrices of the method.

All random draws use a CPU ``torch.Generator`` seeded by the caller, so the same seed gives the same
input on any device; the (possibly large) field evaluation then runs on ``device``.
Layout: W[5, ndof], ndof index = e*n_n + n, e = ix + nx*(iy + ny*iz), n = i + N*(j + N*k).
"""
import math

import torch

EOS_IDEAL, EOS_TM = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_DIRICHLET = 0, 1, 2, 3
RIEMANN_HLL, RIEMANN_HLLC = 0, 1

# positions of the N = p+1 nodes on [-1, 1] (Gauss-Lobatto-Legendre, reading R1)
_NODES = {
    1: [0.0],
    2: [-1.0, 1.0],
    3: [-1.0, 0.0, 1.0],
    4: [-1.0, -math.sqrt(1.0 / 5.0), math.sqrt(1.0 / 5.0), 1.0],
    5: [-1.0, -math.sqrt(3.0 / 7.0), 0.0, math.sqrt(3.0 / 7.0), 1.0],
}

F64 = torch.float64


def node_positions(N):
    return list(_NODES[N])


def axis_coords(xmin, xmax, ne, N, device="cpu"):
    """Global coordinates of the ne*N nodes along one axis, index = ie*N + i."""
    h = (xmax - xmin) / ne
    xi = torch.tensor(_NODES[N], dtype=F64, device=device)
    ie = torch.arange(ne, dtype=F64, device=device)
    return (xmin + h * (ie[:, None] + 0.5 * (xi[None, :] + 1.0))).reshape(-1)


def grid_to_canonical(F, nelem, N):
    """F[..., (z), (y), x] on the global node grid (fastest = x) -> [..., ndof] canonical."""
    nd = len(nelem)
    lead = F.shape[:-nd]
    if nd == 1:
        return F.reshape(*lead, -1)
    if nd == 2:
        nx, ny = nelem
        G = F.reshape(*lead, ny, N, nx, N)          # iy, j, ix, i
        L = len(lead)
        return G.permute(*range(L), L + 0, L + 2, L + 1, L + 3).reshape(*lead, -1)
    nx, ny, nz = nelem
    G = F.reshape(*lead, nz, N, ny, N, nx, N)       # iz, k, iy, j, ix, i
    L = len(lead)
    return G.permute(*range(L), L + 0, L + 2, L + 4, L + 1, L + 3, L + 5).reshape(*lead, -1)


def _u_from_v(v):
    """u = gamma v for a [3, n] three-velocity (parameterisation of the input)."""
    g = 1.0 / torch.sqrt(1.0 - (v * v).sum(0))
    return v * g


def _cfg(ndim, nelem, xmin, xmax, bc, p, eos, gamma_ad, **kw):
    d = dict(ndim=ndim, nelem=list(nelem), xmin=list(xmin), xmax=list(xmax), bc=list(bc),
             order_p=p, eos=eos, gamma_ad=gamma_ad, rk_stages=3, eps_q=1e-12, delta_s=1e-10,
             riemann=RIEMANN_HLL, bc_state=None, shock_limiter=0, moe_alpha=0.0)
    d.update(kw)
    return d


# ---------------------------------------------------------------------------------------------
# config 1: 1D Riemann problem with seeded left/right states (shape of PAPER.md:537-583)
# ---------------------------------------------------------------------------------------------
def riemann1d(seed, ne=256, p=2, device="cpu", states=None):
    g = torch.Generator().manual_seed(int(seed))
    r = torch.rand(6, generator=g, dtype=F64)
    if states is None:
        rho = 10.0 ** (-1.0 + 2.0 * r[0:2])
        P = 10.0 ** (-3.0 + 4.0 * r[2:4])
        vx = -0.5 + r[4:6]
        vy = torch.zeros(2, dtype=F64)
    else:   # explicit (rho, vx, vy, P) left/right, e.g. the paper's Eq. 85-89
        (rl, vxl, vyl, pl), (rr, vxr, vyr, pr) = states
        rho = torch.tensor([rl, rr], dtype=F64)
        vx = torch.tensor([vxl, vxr], dtype=F64)
        vy = torch.tensor([vyl, vyr], dtype=F64)
        P = torch.tensor([pl, pr], dtype=F64)
    N = p + 1
    side = (torch.arange(ne) >= ne // 2).long().repeat_interleave(N)     # by element
    v = torch.stack([vx[side], vy[side], torch.zeros(ne * N, dtype=F64)])
    W = torch.cat([rho[side][None], _u_from_v(v), P[side][None]]).to(device)
    cfg = _cfg(1, [ne], [0.0], [1.0], [BC_OUTFLOW], p, EOS_IDEAL, 5.0 / 3.0)
    return cfg, W.contiguous()


# The five 1D Riemann problems of PAPER.md:537-583 as printed (Eq. 85-89): (rho, vx, vy, P) left and
# right of x = 0.5 on [0,1], adiabatic index, end time; tests 1-4 Dirichlet at both ends, test 5 a
# uniform state with a reflecting wall at x = 1.
PAPER_RIEMANN_1D = {
    1: dict(L=(10.0, 0.0, 0.0, 40.0 / 3.0), R=(1.0, 0.0, 0.0, 2.0 / 3.0 * 1e-6), gamma_ad=5.0 / 3.0, t_end=0.4),
    2: dict(L=(1.0, 0.0, 0.0, 1e3), R=(1.0, 0.0, 0.0, 1e-2), gamma_ad=5.0 / 3.0, t_end=0.4),
    3: dict(L=(1.0, 0.0, 0.0, 1e3), R=(1.0, 0.0, 0.99, 1e-2), gamma_ad=5.0 / 3.0, t_end=0.4),
    4: dict(L=(1.0, 0.01, 0.0, 1.0), R=(0.125, 0.01, 0.0, 0.1), gamma_ad=4.0 / 3.0, t_end=0.4),
    5: dict(L=(1.0, 0.99999, 0.0, 0.01), R=(1.0, 0.99999, 0.0, 0.01), gamma_ad=4.0 / 3.0, t_end=1.5),
}


def paper_riemann1d(k, ne=256, p=2, device="cpu", riemann=RIEMANN_HLL):
    """Problem k = 1..5 of PAPER.md:537-583 (Eq. 85-89) with the paper's boundary conditions."""
    pr = PAPER_RIEMANN_1D[k]
    cfg, W = riemann1d(0, ne=ne, p=p, device=device, states=(pr["L"], pr["R"]))

    def prim(s):                       # (rho, vx, vy, P) -> [rho, ux, uy, uz, P]
        g = 1.0 / math.sqrt(1.0 - s[1] ** 2 - s[2] ** 2)
        return [s[0], g * s[1], g * s[2], 0.0, s[3]]

    cfg.update(gamma_ad=pr["gamma_ad"], riemann=riemann,
               bc=[(BC_DIRICHLET, BC_REFLECT if k == 5 else BC_DIRICHLET)],
               bc_state={(0, 0): prim(pr["L"]), (0, 1): prim(pr["R"])})
    return cfg, W, pr["t_end"]


# The three 2D Riemann problems of PAPER.md:603-680 as printed (Eq. 91-106): (rho, vx, vy, P) in the four
# quadrants Q1 = [0,1]x[0,1], Q2 = [-1,0]x[0,1], Q3 = [-1,0]x[-1,0], Q4 = [0,1]x[-1,0]; Gamma = 5/3,
# transmissive boundaries on all sides, evolved to t = 0.8.
PAPER_RIEMANN_2D = {
    1: ((0.035145216124503, 0.0, 0.0, 0.162931056509027), (0.1, 0.7, 0.0, 1.0), (0.5, 0.0, 0.0, 1.0), (0.1, 0.0, 0.7, 1.0)),
    2: ((0.5, 0.5, -0.5, 5.0), (1.0, 0.5, 0.5, 5.0), (3.0, -0.5, 0.5, 5.0), (1.5, -0.5, -0.5, 5.0)),
    3: ((1.0, 0.0, 0.0, 1.0), (0.5771, -0.3529, 0.0, 0.4), (1.0, -0.3529, -0.3529, 1.0), (0.5771, 0.0, -0.3529, 0.4)),
}


def paper_riemann2d(k, n=64, p=1, device="cpu", riemann=RIEMANN_HLLC):
    """Problem k = 1..3 of PAPER.md:603-680 (Eq. 95-106) on n x n elements of [-1,1]^2, by element."""
    N = p + 1
    q = torch.tensor(PAPER_RIEMANN_2D[k], dtype=F64)                      # [quadrant, (rho, vx, vy, P)]
    hi = (torch.arange(n) >= n // 2).long().repeat_interleave(N)          # 1 in the upper half of an axis
    # quad[y-node, x-node]: y > 0 & x > 0 -> Q1 (0), y > 0 & x < 0 -> Q2 (1), y < 0 & x < 0 -> Q3 (2), else Q4 (3)
    quad = torch.tensor([[2, 3], [1, 0]])[hi[:, None], hi[None, :]]
    vals = q[quad]                                                        # [ny*N, nx*N, 4]
    v = torch.stack([vals[..., 1], vals[..., 2], torch.zeros_like(vals[..., 1])]).reshape(3, -1)
    Wg = torch.cat([vals[..., 0].reshape(1, -1), _u_from_v(v), vals[..., 3].reshape(1, -1)])
    W = grid_to_canonical(Wg.reshape(5, n * N, n * N), [n, n], N).to(device)
    cfg = _cfg(2, [n, n], [-1.0, -1.0], [1.0, 1.0], [BC_OUTFLOW, BC_OUTFLOW], p, EOS_IDEAL, 5.0 / 3.0,
               riemann=riemann)
    return cfg, W.contiguous(), 0.8


# ---------------------------------------------------------------------------------------------
# config 2: 1D smooth density (entropy) wave, exact solution rho = 1 + A sin(2 pi (x - v t) + phi)
# ---------------------------------------------------------------------------------------------
def wave1d(seed, ne, p, amp=1e-4, vx=0.5, device="cpu"):
    g = torch.Generator().manual_seed(int(seed))
    phi = float(2.0 * math.pi * torch.rand(1, generator=g, dtype=F64))
    N = p + 1
    x = axis_coords(0.0, 1.0, ne, N)
    W = wave1d_exact(x, 0.0, phi, amp, vx).to(device)
    cfg = _cfg(1, [ne], [0.0], [1.0], [BC_PERIODIC], p, EOS_IDEAL, 4.0 / 3.0)
    return cfg, W.contiguous(), x, phi


def wave1d_exact(x, t, phi, amp=1e-4, vx=0.5):
    rho = 1.0 + amp * torch.sin(2.0 * math.pi * (x - vx * t) + phi)
    v = torch.stack([torch.full_like(x, vx), torch.zeros_like(x), torch.zeros_like(x)])
    return torch.cat([rho[None], _u_from_v(v), torch.ones_like(x)[None]])


# ---------------------------------------------------------------------------------------------
# config 3: con2prim batch (shape of PAPER.md:405/:435)
# ---------------------------------------------------------------------------------------------
def c2p_states(seed, n, device="cpu", chunk=1 << 22):
    """rho log-uniform [1e-6,1e2], Theta=P/rho log-uniform [1e-6,1e3], Lorentz factor log-uniform
    [1,100], isotropic direction.  Drawn on the CPU generator in fixed-size chunks so that a prefix
    of a larger batch equals the smaller batch."""
    g = torch.Generator().manual_seed(int(seed))
    W = torch.empty(5, n, dtype=F64, device=device)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        r = torch.rand(3, chunk, generator=g, dtype=F64)[:, :m]
        nrm = torch.randn(3, chunk, generator=g, dtype=F64)[:, :m]
        rho = 10.0 ** (-6.0 + 8.0 * r[0])
        theta = 10.0 ** (-6.0 + 9.0 * r[1])
        lor = 10.0 ** (2.0 * r[2])
        umag = torch.sqrt((lor - 1.0) * (lor + 1.0))
        dirn = nrm / torch.sqrt((nrm * nrm).sum(0))
        W[:, s:s + m] = torch.cat([rho[None], umag * dirn, (rho * theta)[None]]).to(device)
    return W


def fig2_grid(ng=25):
    """The 25x25 grid of PAPER.md:405 in c=1 units: D... rho=1, P/(rho c^2) from 1e5/9e16 to
    1e10/9e16 (log-spaced), Lorentz factor 1..100 (log-spaced), velocity along x."""
    c2 = 9.0e16
    P = torch.logspace(5, 10, ng, dtype=F64) / c2
    lor = torch.logspace(0, 2, ng, dtype=F64)
    PP, LL = torch.meshgrid(P, lor, indexing="ij")
    PP, LL = PP.reshape(-1), LL.reshape(-1)
    umag = torch.sqrt((LL - 1.0) * (LL + 1.0))
    z = torch.zeros_like(PP)
    return torch.stack([torch.ones_like(PP), umag, z, z, PP]), LL


# ---------------------------------------------------------------------------------------------
# config 4: 2D relativistic Kelvin-Helmholtz (shape of PAPER.md:683, :729)
# ---------------------------------------------------------------------------------------------
def kh2d(seed, nx=512, ny=1024, p=2, device="cpu"):
    g = torch.Generator().manual_seed(int(seed))
    phi = float(2.0 * math.pi * torch.rand(1, generator=g, dtype=F64))
    N = p + 1
    x = axis_coords(-0.5, 0.5, nx, N, device)[None, :]
    y = axis_coords(-1.0, 1.0, ny, N, device)[:, None]
    th = torch.tanh(y / 0.01)
    vx = (0.5 * th).expand(ny * N, nx * N)
    rho = (0.55 + 0.45 * th).expand(ny * N, nx * N)
    vy = 0.01 * torch.sin(2.0 * math.pi * x + phi) * torch.exp(-(y / 0.1) ** 2)
    v = torch.stack([vx, vy, torch.zeros_like(vy)]).reshape(3, -1)
    Wg = torch.cat([rho.reshape(1, -1), _u_from_v(v), torch.ones(1, v.shape[1], dtype=F64,
                                                                 device=device)])
    W = grid_to_canonical(Wg.reshape(5, ny * N, nx * N), [nx, ny], N)
    cfg = _cfg(2, [nx, ny], [-0.5, -1.0], [0.5, 1.0], [BC_PERIODIC, BC_OUTFLOW], p, EOS_TM, 0.0)
    return cfg, W.contiguous()


# ---------------------------------------------------------------------------------------------
# config 5: 3D periodic box, random-phase band-limited velocity over log-normal density
# ---------------------------------------------------------------------------------------------
def _band_field(g, nf, kmax, coords, device):
    """nf independent real unit-variance fields sum_{0<|k|<=kmax} a cos(2 pi k.x + phi_k) on the
    tensor grid coords = (x, y, z); returns [nf, nz, ny, nx]."""
    K = torch.arange(-kmax, kmax + 1, dtype=F64)
    kz, ky, kx = torch.meshgrid(K, K, K, indexing="ij")
    k2 = kx * kx + ky * ky + kz * kz
    mask = (k2 > 0) & (k2 <= kmax * kmax)
    phase = 2.0 * math.pi * torch.rand(nf, *mask.shape, generator=g, dtype=F64)
    nmode = float(mask.sum())
    amp = math.sqrt(2.0 / nmode)                  # sum over all k (both signs) of a cos(): var = 1
    c = (amp * mask.to(F64))[None] * torch.exp(1j * phase)            # [nf, kz, ky, kx]
    c = c.to(device)
    Kd = K.to(device)
    ex, ey, ez = (torch.exp(2j * math.pi * Kd[:, None] * xc[None, :]) for xc in coords)
    A = torch.einsum("fzyx,zc->fcyx", c, ez)      # [nf, Z, ky, kx]
    A = torch.einsum("fcyx,yb->fcbx", A, ey)      # [nf, Z, Y, kx]
    out = torch.empty(nf, ez.shape[1], ey.shape[1], ex.shape[1], dtype=F64, device=device)
    for f in range(nf):                           # one field at a time bounds the complex temporaries
        out[f] = torch.matmul(A[f], ex).real
    return out


def box3d(seed, n=128, p=3, kmax=8, device="cpu", sigma=2.0, vrms=0.6, vcap=0.99,
          rho_floor=1e-6, p_over_rho=0.01):
    g = torch.Generator().manual_seed(int(seed))
    N = p + 1
    xc = axis_coords(0.0, 1.0, n, N, device)
    coords = (xc, xc, xc)
    vg = _band_field(g, 3, kmax, coords, device) * (vrms / math.sqrt(3.0))
    gg = _band_field(g, 1, kmax, coords, device)
    vmag = torch.sqrt((vg * vg).sum(0, keepdim=True))
    vg = vg * torch.clamp(vcap / vmag, max=1.0)
    rho = torch.clamp(torch.exp(sigma * gg), min=rho_floor)
    del gg, vmag
    v = vg.reshape(3, -1)
    Wg = torch.cat([rho.reshape(1, -1), _u_from_v(v), p_over_rho * rho.reshape(1, -1)])
    del vg, v
    W = grid_to_canonical(Wg.reshape(5, n * N, n * N, n * N), [n, n, n], N)
    cfg = _cfg(3, [n, n, n], [0.0] * 3, [1.0] * 3, [BC_PERIODIC] * 3, p, EOS_IDEAL, 5.0 / 3.0)
    return cfg, W.contiguous()


def box2d(seed, nx=32, ny=32, p=2, kmax=1, device="cpu", eos=EOS_IDEAL, gamma_ad=5.0 / 3.0, sigma=2.0,
          vrms=0.6, vcap=0.99, rho_floor=1e-6, p_over_rho=0.01, bc=(BC_PERIODIC, BC_PERIODIC)):
    """2D companion of config 5 (same recipe evaluated on the plane z = 0.3125 of the 3D band-limited
    fields, all three velocity components kept): exercises the physicality operator of the 2D
    kernels, which config 4's smooth shear layer never triggers."""
    g = torch.Generator().manual_seed(int(seed))
    N = p + 1
    coords = (axis_coords(0.0, 1.0, nx, N, device), axis_coords(0.0, 1.0, ny, N, device),
              torch.tensor([0.3125], dtype=F64, device=device))
    vg = _band_field(g, 3, kmax, coords, device)[:, 0] * (vrms / math.sqrt(3.0))
    gg = _band_field(g, 1, kmax, coords, device)[:, 0]
    vmag = torch.sqrt((vg * vg).sum(0, keepdim=True))
    vg = vg * torch.clamp(vcap / vmag, max=1.0)
    rho = torch.clamp(torch.exp(sigma * gg), min=rho_floor)
    v = vg.reshape(3, -1)
    Wg = torch.cat([rho.reshape(1, -1), _u_from_v(v), p_over_rho * rho.reshape(1, -1)])
    W = grid_to_canonical(Wg.reshape(5, ny * N, nx * N), [nx, ny], N)
    cfg = _cfg(2, [nx, ny], [0.0] * 2, [1.0] * 2, list(bc), p, eos, gamma_ad)
    return cfg, W.contiguous()


def limiter_stress(U, n_nodes, seed, frac=0.05):
    """Companion input 5L: overwrite 1-3 nodes in a seeded `frac` of the cells of the conserved
    state U[5, ndof] with inadmissible values (D < 0, or E = 0.9 sqrt(D^2+|M|^2)).  Pure data
    editing (no method arithmetic beyond building the bad value)."""
    g = torch.Generator().manual_seed(int(seed))
    U = U.clone()
    ne = U.shape[1] // n_nodes
    ncell = max(1, int(frac * ne))
    cells = torch.randperm(ne, generator=g)[:ncell]
    for c in cells.tolist():
        k = int(torch.randint(1, min(3, n_nodes) + 1, (1,), generator=g))
        nodes = torch.randperm(n_nodes, generator=g)[:k]
        for nn_ in nodes.tolist():
            j = c * n_nodes + nn_
            if float(torch.rand(1, generator=g)) < 0.5:
                U[0, j] = -0.1 * abs(float(U[0, j]))
            else:
                m = math.sqrt(float(U[0, j]) ** 2 + float((U[1:4, j] ** 2).sum()))
                U[4, j] = 0.9 * m
    return U, cells
