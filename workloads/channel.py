"""Problem descriptions (plain data) and seeded initial states.  See workloads/__init__.py.

Recipe (stands in for the paper's pressure-driven channel, P:L102,
whose fields the paper does not print): mesh [0,2]x[0,1]; endpoint-inclusive uniform velocity
nodes with trapezoid weights; xmin FIXED(rho=1.0), xmax FIXED(rho=0.8), ymin/ymax diffuse WALL
at T=1; omega=0.81; mu_ref from Kn; CFL 0.8; initial primitives = linear density drop times
seeded smooth +-eps noise; W = cons(prim) analytically, f = Maxwellian of prim at the nodes.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

BC_PERIODIC, BC_FIXED, BC_WALL = 0, 1, 2


@dataclasses.dataclass
class Problem:
    """Everything ``ugks_init`` needs, as plain data.  bcs = [xmin, xmax, ymin, ymax], each
    (type, rho, U, V, T)."""
    I: int
    J: int
    x0: float
    x1: float
    y0: float
    y1: float
    u: np.ndarray
    wu: np.ndarray
    v: np.ndarray
    wv: np.ndarray
    omega: float = 0.81
    mu_ref: float = 0.0          # <= 0: derive from Kn inside the library
    Kn: float = 0.1
    Pr: float = 1.0
    K_int: int = 0
    bcs: list = dataclasses.field(default_factory=lambda: [(BC_PERIODIC, 1, 0, 0, 1)] * 4)
    cfl: float = 0.8
    steps: int = 1
    name: str = ""
    seed: int = 0
    eps: tuple = (0.01, 0.01, 0.01, 0.01)   # (rho, U, V, T) noise amplitudes
    rho_drop: float = 0.1                   # rho = (1 - rho_drop * x) * (1 + eps n)

    @property
    def Nu(self): return len(self.u)

    @property
    def Nv(self): return len(self.v)

    @property
    def N(self): return len(self.u) * len(self.v)

    @property
    def points(self): return self.I * self.J * self.N

    @property
    def dx(self): return (self.x1 - self.x0) / self.I

    @property
    def dy(self): return (self.y1 - self.y0) / self.J


def trapezoid_grid(n: int, a: float):
    """Endpoint-inclusive uniform nodes on [-a, a] with trapezoid weights h*(1/2,1,...,1,1/2) (AMB-16)."""
    u = -a + 2.0 * a * np.arange(n, dtype=np.float64) / (n - 1)
    h = 2.0 * a / (n - 1)
    w = np.full(n, h)
    w[0] = w[-1] = 0.5 * h
    return u, w


_CHANNEL_BCS = [(BC_FIXED, 1.0, 0.0, 0.0, 1.0), (BC_FIXED, 0.8, 0.0, 0.0, 1.0),
                (BC_WALL, 1.0, 0.0, 0.0, 1.0), (BC_WALL, 1.0, 0.0, 0.0, 1.0)]

# name: (I, J, Nu=Nv, half-width a, Kn, steps, eps)   -- BASELINE.json configs[0..4]
_SPECS = {
    "C1": (32, 16, 16, 4.0, 0.1, 10, (0.01, 0.01, 0.01, 0.01)),
    "C2": (128, 64, 28, 5.0, 0.05, 200, (0.01, 0.01, 0.01, 0.01)),
    "C3": (512, 256, 28, 5.0, 0.01, 100, (0.01, 0.01, 0.01, 0.01)),
    "C4": (1024, 512, 40, 6.0, 0.1, 50, (0.01, 0.01, 0.01, 0.01)),
    "C5": (128, 64, 200, 20.0, 1.0, 50, (0.0, 0.05, 0.05, 0.0)),
}
CONFIGS = tuple(_SPECS)


def channel_config(name: str, I: int | None = None, J: int | None = None, Nuv: int | None = None) -> Problem:
    """BASELINE.json config ``name`` ("C1".."C5"); I/J/Nuv override sizes (reduced parity cases)."""
    I0, J0, n0, a, Kn, steps, eps = _SPECS[name]
    n = Nuv or n0
    u, wu = trapezoid_grid(n, a)
    v, wv = trapezoid_grid(n, a)
    return Problem(I=I or I0, J=J or J0, x0=0.0, x1=2.0, y0=0.0, y1=1.0, u=u, wu=wu, v=v, wv=wv,
                   omega=0.81, mu_ref=0.0, Kn=Kn, bcs=list(_CHANNEL_BCS), cfl=0.8, steps=steps,
                   name=name, seed=181008137 + int(name[1]), eps=eps, rho_drop=0.1)


_PAPER_MESHES = {"M1": (40, 20), "M2": (80, 40), "M3": (120, 60), "M4": (160, 80)}     # P:L110-117 Table 1


def paper_mesh(name: str, nuv: int = 29) -> Problem:
    """The paper's own shapes: mesh M1..M4 of Table 1 with an odd nuv x nuv velocity grid (29, 49, 69:
    P:L115-117, L140; a node at u = 0 and at v = 0), Kn = 0.1, same channel recipe as C1..C5.  The paper does not
    state its velocity range or quadrature rule (AMB-16): [-5, 5]^2, [-6, 6]^2, [-7, 7]^2 with trapezoid weights here."""
    I, J = _PAPER_MESHES[name]
    a = {29: 5.0, 49: 6.0, 69: 7.0}.get(nuv, 5.0)
    u, wu = trapezoid_grid(nuv, a)
    v, wv = trapezoid_grid(nuv, a)
    return Problem(I=I, J=J, x0=0.0, x1=2.0, y0=0.0, y1=1.0, u=u, wu=wu, v=v, wv=wv, omega=0.81, mu_ref=0.0, Kn=0.1,
                   bcs=list(_CHANNEL_BCS), cfl=0.8, steps=10000, name=f"{name}-{nuv}", seed=181008137 + 10 * int(name[1]) + nuv,
                   eps=(0.01, 0.01, 0.01, 0.01), rho_drop=0.1)


def periodic_box(I: int, J: int, Nu: int, Nv: int, a: float = 5.0, Kn: float = 0.1, seed: int = 1,
                 eps=(0.05, 0.05, 0.05, 0.05), lx: float = 1.0, ly: float = 1.0, cfl: float = 0.8,
                 mu_ref: float = 0.0, bu: float | None = None) -> Problem:
    """Fully periodic box used by the invariants tests (conservation, fixed point, symmetry)."""
    u, wu = trapezoid_grid(Nu, a if bu is None else bu)
    v, wv = trapezoid_grid(Nv, a)
    return Problem(I=I, J=J, x0=0.0, x1=lx, y0=0.0, y1=ly, u=u, wu=wu, v=v, wv=wv, Kn=Kn, mu_ref=mu_ref,
                   bcs=[(BC_PERIODIC, 1, 0, 0, 1)] * 4, cfl=cfl, name="box", seed=seed, eps=eps, rho_drop=0.0)


def smooth_noise(p: Problem, rng: np.random.Generator) -> np.ndarray:
    """n_F(x,y) at cell centres, max-abs 1:  sum_{p,q=1..3} A_pq sin(2 pi p x/Lx + phi) sin(2 pi q y/(2 Ly) + theta)."""
    A = rng.uniform(-1.0, 1.0, (3, 3))
    phi = rng.uniform(0.0, 2.0 * math.pi, (3, 3))
    th = rng.uniform(0.0, 2.0 * math.pi, (3, 3))
    periodic = p.bcs[2][0] == BC_PERIODIC
    x = p.x0 + (np.arange(p.I) + 0.5) * p.dx
    y = p.y0 + (np.arange(p.J) + 0.5) * p.dy
    X, Y = np.meshgrid(x, y)            # [J][I]
    Lx, Ly = p.x1 - p.x0, p.y1 - p.y0
    n = np.zeros_like(X)
    for a in range(3):
        for b in range(3):
            ky = (2.0 if periodic else 1.0) * math.pi * (b + 1) / Ly      # periodic boxes get whole waves
            n += A[a, b] * np.sin(2.0 * math.pi * (a + 1) * (X - p.x0) / Lx + phi[a, b]) * np.sin(ky * (Y - p.y0) + th[a, b])
    return n / np.max(np.abs(n))


def maxwellian_field(p: Problem, rho, U, V, T, out: np.ndarray | None = None) -> np.ndarray:
    """f[J][I][Nv][Nu] = rho (lam/pi) exp(-lam((u-U)^2 + (v-V)^2)), lam = 1/T  (Eq. (1))."""
    J, I = rho.shape
    f = out if out is not None else np.empty((J, I, p.Nv, p.Nu))
    lam = 1.0 / T
    for j in range(J):                   # row by row: bounded temporaries at C4 size
        du = p.u[None, None, :] - U[j][:, None, None]
        dv = p.v[None, :, None] - V[j][:, None, None]
        f[j] = (rho[j] * lam[j] / math.pi)[:, None, None] * np.exp(-lam[j][:, None, None] * (du * du + dv * dv))
    return f


def initial_state(p: Problem, want_f: bool = True, out_f: np.ndarray | None = None):
    """Seeded primitives -> (W[J][I][4], f[J][I][Nv][Nu], prim[J][I][4]) for problem ``p`` (AMB-18)."""
    rng = np.random.default_rng(p.seed)
    n = [smooth_noise(p, rng) for _ in range(4)]          # order rho, U, V, T
    x = p.x0 + (np.arange(p.I) + 0.5) * p.dx
    rho = (1.0 - p.rho_drop * x)[None, :] * (1.0 + p.eps[0] * n[0])
    U = p.eps[1] * n[1]
    V = p.eps[2] * n[2]
    T = 1.0 + p.eps[3] * n[3]
    lam = 1.0 / T
    W = np.stack([rho, rho * U, rho * V, 0.5 * rho * (U * U + V * V) + rho / (2.0 * lam)], axis=-1)
    prim = np.stack([rho, U, V, lam], axis=-1)
    f = maxwellian_field(p, rho, U, V, T, out=out_f) if want_f else None
    return np.ascontiguousarray(W), f, prim
