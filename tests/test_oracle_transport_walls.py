"""Pins P10-P15 of DESIGN.md: free-transport limit by brute force, diffuse walls, channel sanity,
stiff regime.  CPU only."""
import numpy as np
import pytest

import workloads
from oracle import Oracle
from tests.util import cons_of_prim, err_f


def _brute_force_free_transport(p, f, dt):
    """Exact upwind advection of the van Leer piecewise-linear reconstruction, face by face, written
    independently of the oracle: during [0,dt] the particles of velocity n crossing a face are those of the
    upwind cell within distance |n| dt of it; for a linear profile their mean is the profile at the middle of
    that segment.  Periodic in both directions.  f[J][I][Nv][Nu]."""
    J, I, Nv, Nu = f.shape
    out = f.copy()
    for axis, (d, vel) in enumerate([(p.dy, p.v), (p.dx, p.u)]):          # axis 0: y (j), axis 1: x (i)
        n = vel[:, None] * np.ones((1, Nu)) if axis == 0 else np.ones((Nv, 1)) * vel[None, :]
        fm, fp = np.roll(f, 1, axis), np.roll(f, -1, axis)
        sm, sp = (f - fm) / d, (fp - f) / d
        with np.errstate(divide="ignore", invalid="ignore"):
            sig = np.where(sm * sp > 0, 2 * sm * sp / (sm + sp), 0.0)
        # face between cell c-1 (L) and c (R), stored at index c
        fL, sL = np.roll(f, 1, axis), np.roll(sig, 1, axis)
        xs = -0.5 * n * dt                                                 # middle of the swept segment, face at 0
        fromL = fL + sL * (0.5 * d + xs)                                   # L's centre is at -d/2
        fromR = f + sig * (-0.5 * d + xs)                                  # R's centre is at +d/2
        up = np.where(n > 0, fromL, np.where(n < 0, fromR, 0.5 * (fromL + fromR)))
        swept = n * dt * up                                                # per unit face length
        out += (swept - np.roll(swept, -1, axis)) / d
    return out


@pytest.mark.parametrize("nuv", [(8, 8), (9, 7)])
def test_P10_free_transport_limit_brute_force(nuv):
    """north_star: as tau -> infinity the update reduces to exact upwind free transport (4x4 mesh).
    Rough data so the limiter is active; (9,7) has u = 0 and v = 0 nodes (H(0) = 1/2, P13)."""
    p = workloads.periodic_box(4, 4, nuv[0], nuv[1], a=4.0, mu_ref=7.310334e14, seed=2, bu=3.0)
    rng = np.random.default_rng(42)
    W, f, _ = workloads.initial_state(p)
    f = f * rng.uniform(0.2, 1.8, f.shape)                                 # rough in space and velocity
    o = Oracle(p)
    o.set_state(W, f)
    o.step(1)
    expect = _brute_force_free_transport(p, f, o.dt)
    assert err_f(expect, f) > 1e-2                                         # a real change
    assert err_f(o.f(), expect) < 2e-14


def _closed_box(I, J, n, a=6.0, Kn=0.1, Tw=1.0):
    u, wu = workloads.trapezoid_grid(n, a)
    wall = (workloads.BC_WALL, 1.0, 0.0, 0.0, Tw)
    return workloads.Problem(I=I, J=J, x0=0.0, x1=1.0, y0=0.0, y1=1.0, u=u, wu=wu, v=u.copy(), wv=wu.copy(),
                             Kn=Kn, bcs=[wall] * 4, cfl=0.8, seed=9, eps=(0.05, 0.05, 0.05, 0.05), rho_drop=0.0)


@pytest.mark.parametrize("n", [16, 17])
def test_P11_closed_box_conserves_mass(n):
    """O9: the diffuse wall returns exactly the mass that hits it."""
    p = _closed_box(6, 5, n)
    W, f, _ = workloads.initial_state(p)
    o = Oracle(p)
    o.set_state(W, f)
    m0 = W[..., 0].sum()
    o.step(5)
    Wn = o.W()
    assert abs(Wn[..., 0].sum() - m0) < 2e-15 * m0
    assert np.max(np.abs(Wn - W)) > 1e-4
    # each wall face: zero mass flux, and the stage output reports a sane rho_w
    FW, Ff, st = o.face_flux(1, 2, 0)
    assert abs(FW[0]) < 1e-17 and 0.5 < st[38] < 2.0
    FW, Ff, st = o.face_flux(0, p.I, 3)
    assert abs(FW[0]) < 1e-17 and 0.5 < st[38] < 2.0


@pytest.mark.parametrize("n,tol", [(16, 2e-8), (28, 1e-15), (40, 1e-15)])
def test_P12_wall_equilibrium_is_a_fixed_point_to_quadrature_error(n, tol):
    p = _closed_box(4, 4, n, Tw=1.0)
    ones = np.ones((p.J, p.I))
    f = workloads.maxwellian_field(p, ones, 0 * ones, 0 * ones, ones)
    W = np.broadcast_to(cons_of_prim(np.array([1.0, 0, 0, 1.0])), (p.J, p.I, 4)).copy()
    o = Oracle(p)
    o.set_state(W, f)
    o.step(1)
    assert np.max(np.abs(o.W() - W)) < tol
    assert err_f(o.f(), f) < max(tol, 1e-15) * 10


def test_wall_momentum_and_energy_flux_signs():
    """A gas at rest pushes on the wall: the x-momentum flux through the xmax wall is +p*ell*dt, through
    the xmin wall it is also +p*ell*dt (signed along +x); a hot wall returns more energy than it receives."""
    p = _closed_box(4, 4, 40, a=7.0, Tw=1.0)
    ones = np.ones((p.J, p.I))
    f = workloads.maxwellian_field(p, ones, 0 * ones, 0 * ones, ones)
    W = np.broadcast_to(cons_of_prim(np.array([1.0, 0, 0, 1.0])), (p.J, p.I, 4)).copy()
    o = Oracle(p)
    o.set_state(W, f)
    pres = 0.5                                                   # p = rho/(2 lam)
    for (d, i, j, comp, ell) in [(0, p.I, 1, 1, p.dy), (0, 0, 1, 1, p.dy), (1, 1, p.J, 2, p.dx), (1, 1, 0, 2, p.dx)]:
        FW, _, _ = o.face_flux(d, i, j)
        assert abs(FW[comp] - pres * ell * o.dt) < 1e-13, (d, i, j, FW)
        assert abs(FW[0]) < 1e-17 and abs(FW[3]) < 1e-15
    hot = _closed_box(4, 4, 40, a=7.0, Tw=1.5)
    oh = Oracle(hot)
    oh.set_state(W, f)
    FW, _, _ = oh.face_flux(0, hot.I, 1)
    assert FW[3] < -1e-5 and abs(FW[0]) < 1e-17                  # net energy flows from the hot wall into the gas


def test_P14_channel_sanity():
    """C1: stays finite; the pressure drop drives the gas toward the low-density side (mean U > 0)."""
    p = workloads.channel_config("C1")
    W, f, _ = workloads.initial_state(p)
    o = Oracle(p)
    o.set_state(W, f)
    o.step(10)
    Wn, fn = o.W(), o.f()
    assert np.all(np.isfinite(fn)) and np.all(np.isfinite(Wn))
    assert np.mean(Wn[..., 1] / Wn[..., 0]) > 1e-3
    assert 0.75 < Wn[..., 0].min() and Wn[..., 0].max() < 1.05


def test_P15_stiff_regime_is_stable_and_relaxes_to_equilibrium():
    """dt/tau ~ 1e3: the asymptotic-preserving branch (Mt1 ~ dt - tau, implicit Eq. (3))."""
    p = workloads.periodic_box(6, 6, 16, 16, a=6.0, Kn=1e-5, seed=4, eps=(0.02, 0.02, 0.02, 0.02))
    W, f, _ = workloads.initial_state(p)
    rng = np.random.default_rng(0)
    f = f * rng.uniform(0.9, 1.1, f.shape)                       # start off-equilibrium
    o = Oracle(p)
    o.set_state(W, f)
    tau = 2 * o.mu_ref
    assert o.dt / tau > 100
    o.step(20)
    Wn, fn = o.W(), o.f()
    assert np.all(np.isfinite(fn)) and Wn[..., 0].min() > 0.9 and Wn[..., 0].max() < 1.1
    # Eq. (3) is trapezoidal: the non-equilibrium part is multiplied by (1-x/2)/(1+x/2) -> -1 per step, so it
    # neither grows nor decays fast; it must stay bounded by its initial size
    rho = Wn[..., 0]; U = Wn[..., 1] / rho; V = Wn[..., 2] / rho
    T = 2 * (Wn[..., 3] - 0.5 * rho * (U * U + V * V)) / rho
    g = workloads.maxwellian_field(p, rho, U, V, T)
    rho0 = W[..., 0]; U0 = W[..., 1] / rho0; V0 = W[..., 2] / rho0
    T0 = 2 * (W[..., 3] - 0.5 * rho0 * (U0 * U0 + V0 * V0)) / rho0
    g0 = workloads.maxwellian_field(p, rho0, U0, V0, T0)
    assert err_f(fn, g) < 1.05 * err_f(f, g0)
