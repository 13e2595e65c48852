"""Pins P6-P9, P13 of DESIGN.md: what the physics fixes about a whole oracle step.  CPU only."""
import numpy as np
import pytest

import workloads
from oracle import Oracle
from oracle import binding as ob
from tests.util import cons_of_prim, err_f


def _uniform_state(p, prim):
    rho, U, V, lam = prim
    J, I = p.J, p.I
    ones = np.ones((J, I))
    f = workloads.maxwellian_field(p, rho * ones, U * ones, V * ones, ones / lam)
    W = np.broadcast_to(cons_of_prim(np.array(prim)), (J, I, 4)).copy()
    return W, f


@pytest.mark.parametrize("nuv", [(16, 16), (29, 29), (12, 17)])
def test_P6_uniform_maxwellian_is_a_fixed_point(nuv):
    """north_star: a uniform Maxwellian is a steady fixed point (periodic box).  W must not move at
    all (analytic moments, zero slopes); f moves only by round-off.  29x29 has u=0, v=0 nodes (P13)."""
    p = workloads.periodic_box(6, 5, nuv[0], nuv[1], a=6.0, Kn=0.05)
    prim = (0.9, 0.31, -0.12, 1.2)
    W, f = _uniform_state(p, prim)
    o = Oracle(p)
    o.set_state(W, f)
    o.step(3)
    assert np.max(np.abs(o.W() - W)) < 1e-15
    assert err_f(o.f(), f) < 5e-16
    assert np.all(o.residual() < 1e-15)


@pytest.mark.parametrize("nuv,kn", [((16, 16), 0.1), ((29, 29), 0.1), ((16, 20), 1e-4)])
def test_P7_conservation_in_a_periodic_box(nuv, kn):
    """north_star: mass, momentum, energy conserved to 1e-13 relative in a periodic box."""
    p = workloads.periodic_box(8, 6, nuv[0], nuv[1], a=6.0, Kn=kn, seed=3)
    W, f, _ = workloads.initial_state(p)
    o = Oracle(p)
    o.set_state(W, f)
    tot0 = W.reshape(-1, 4).sum(0)
    o.step(5)
    Wn = o.W()
    tot = Wn.reshape(-1, 4).sum(0)
    assert np.max(np.abs(Wn - W)) > 1e-4            # something did happen
    assert abs(tot[0] - tot0[0]) < 1e-13 * tot0[0]
    assert abs(tot[3] - tot0[3]) < 1e-13 * tot0[3]
    assert abs(tot[1] - tot0[1]) < 1e-13 * tot0[0] and abs(tot[2] - tot0[2]) < 1e-13 * tot0[0]
    # the f-moment totals follow W only to quadrature accuracy of the velocity grid
    Wf = o.W_of_f().reshape(-1, 4).sum(0)
    assert abs(Wf[0] - tot[0]) < 1e-6 * tot[0]


def test_P8_homogeneous_relaxation_closed_form():
    """Spatially uniform non-equilibrium f, periodic: fluxes cancel, W is constant and Eq. (3) gives
    f^n - g = ((1 - x/2)/(1 + x/2))^n (f^0 - g), x = dt/tau."""
    p = workloads.periodic_box(4, 4, 20, 20, a=7.0, Kn=0.02)
    prim_a, prim_b = np.array([0.6, 0.5, 0.0, 1.0]), np.array([0.4, -0.4, 0.3, 0.7])
    Wa, fa = _uniform_state(p, prim_a)
    Wb, fb = _uniform_state(p, prim_b)
    W, f = Wa + Wb, fa + fb                      # bimodal: far from a Maxwellian
    prim = ob.prim_of_W(W[0, 0])
    g = workloads.maxwellian_field(p, *[np.full((p.J, p.I), v) for v in (prim[0], prim[1], prim[2], 1 / prim[3])])
    o = Oracle(p)
    o.set_state(W, f)
    x = o.dt / ob.tau(o.mu_ref, p.omega, prim[0], prim[3])
    assert 0.01 < x < 10
    n = 7
    o.step(n)
    assert np.max(np.abs(o.W() - W)) < 2e-15
    fac = ((1 - x / 2) / (1 + x / 2)) ** n
    expect = g + fac * (f - g)
    assert err_f(o.f(), expect) < 5e-15


def _transpose_problem(p):
    q = workloads.Problem(I=p.J, J=p.I, x0=p.y0, x1=p.y1, y0=p.x0, y1=p.x1, u=p.v, wu=p.wv, v=p.u, wv=p.wu,
                          omega=p.omega, mu_ref=p.mu_ref, Kn=p.Kn, cfl=p.cfl,
                          bcs=[_swapUV(p.bcs[2]), _swapUV(p.bcs[3]), _swapUV(p.bcs[0]), _swapUV(p.bcs[1])])
    return q


def _swapUV(bc):
    return (bc[0], bc[1], bc[3], bc[2], bc[4])


@pytest.mark.parametrize("kind", ["periodic", "channel", "odd"])
def test_P9_transpose_symmetry_y_code_equals_x_code(kind):
    """Swap x<->y, u<->v, I<->J, rhoU<->rhoV: the result must transpose (pins the y-face path, the
    local-frame swap P and the tangential terms against the x-face path)."""
    if kind == "periodic":
        p = workloads.periodic_box(7, 5, 14, 18, a=5.0, Kn=0.05, seed=5, bu=6.0, lx=1.3, ly=0.7)
    elif kind == "odd":
        p = workloads.periodic_box(5, 6, 13, 9, a=5.0, Kn=0.5, seed=6, bu=5.5)
    else:
        p = workloads.channel_config("C1", I=9, J=6, Nuv=14)
        p.bcs[0] = (workloads.BC_FIXED, 1.0, 0.05, -0.02, 1.1)
    W, f, _ = workloads.initial_state(p)
    q = _transpose_problem(p)
    Wq = np.ascontiguousarray(W.transpose(1, 0, 2)[..., [0, 2, 1, 3]])
    fq = np.ascontiguousarray(f.transpose(1, 0, 3, 2))
    a, b = Oracle(p), Oracle(q)
    assert abs(a.dt - b.dt) < 1e-18
    a.set_state(W, f); b.set_state(Wq, fq)
    a.step(3); b.step(3)
    assert np.max(np.abs(a.W() - b.W().transpose(1, 0, 2)[..., [0, 2, 1, 3]])) < 1e-15
    assert err_f(b.f().transpose(1, 0, 3, 2), a.f()) < 1e-15
    assert np.max(np.abs(a.W() - W)) > 1e-5


def test_P9_mirror_symmetry():
    """x -> -x, u -> -u: pins the upwind selection H, the half-range moments ML/MR and a_L/a_R."""
    p = workloads.channel_config("C1", I=8, J=5, Nuv=12)
    W, f, _ = workloads.initial_state(p)
    q = workloads.channel_config("C1", I=8, J=5, Nuv=12)
    q.bcs = [p.bcs[1], p.bcs[0], p.bcs[2], p.bcs[3]]
    Wq = np.ascontiguousarray(W[:, ::-1, :] * np.array([1, -1, 1, 1.0]))
    fq = np.ascontiguousarray(f[:, ::-1, :, ::-1])
    a, b = Oracle(p), Oracle(q)
    a.set_state(W, f); b.set_state(Wq, fq)
    a.step(3); b.step(3)
    assert np.max(np.abs(a.W() - b.W()[:, ::-1, :] * np.array([1, -1, 1, 1.0]))) < 1e-15
    assert err_f(b.f()[:, ::-1, :, ::-1], a.f()) < 1e-15


def test_threads_do_not_change_the_result_and_one_by_one_matches_full_step():
    p = workloads.channel_config("C1", I=10, J=7, Nuv=10)
    W, f, _ = workloads.initial_state(p)
    a, b = Oracle(p), Oracle(p, threads=4)
    a.set_state(W, f); b.set_state(W, f)
    cells = [(0, 0), (9, 6), (4, 3), (0, 3), (5, 0)]
    one = [a.cell_update(i, j) for (i, j) in cells]
    a.step(2); b.step(2)
    assert np.array_equal(a.f(), b.f()) and np.array_equal(a.W(), b.W())
    c = Oracle(p); c.set_state(W, f); c.step(1)
    fc, Wc = c.f(), c.W()
    for (i, j), (Wn, fn) in zip(cells, one):
        assert np.array_equal(Wn, Wc[j, i]) and np.array_equal(fn, fc[j, i])


def test_api_errors():
    p = workloads.periodic_box(4, 4, 8, 8)
    o = Oracle(p)
    with pytest.raises(ob.OracleError):
        o.step(1)                                  # no state yet
    bad = workloads.periodic_box(4, 4, 8, 8); bad.Pr = 0.7
    with pytest.raises(ob.OracleError):
        Oracle(bad)
    bad = workloads.periodic_box(4, 4, 8, 8); bad.bcs = [(0, 1, 0, 0, 1), (2, 1, 0, 0, 1), (0, 1, 0, 0, 1), (0, 1, 0, 0, 1)]
    with pytest.raises(ob.OracleError):
        Oracle(bad)                                # periodic must be paired
