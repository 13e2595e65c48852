"""Pins P20-P22 of DESIGN.md: NEXT-1, the tangential slope of f in the free-transport part of the face solution
(readings O3t / O8t; Eq. (2), "b (tangential)", ref [2] of the paper).  CPU only.

The oracle option ``tangential`` reconstructs the initial state of Eq. (2) in both directions, f0(x,y) = f0 + sigma0 x +
theta0 y on the upwind side; along the characteristic through the face centre that adds -Mt5 t theta0 to the time integral
of the free-transport part.  None of the pins retypes that term: P20 integrates the reconstruction over the swept
parallelogram by brute-force sampling, P21 compares with the exact solution of collisionless transport, P22 are invariants
(conservation, fixed point, x<->y transposition, S5/S7 vs S8 consistency) that a one-sided or mis-signed theta would break.
"""
import math

import numpy as np
import pytest

import workloads
from oracle import Oracle
from tests.util import err_f


def _van_leer(f, d, axis):
    sm, sp = (f - np.roll(f, 1, axis)) / d, (np.roll(f, -1, axis) - f) / d
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(sm * sp > 0, 2 * sm * sp / (sm + sp), 0.0)


def _brute_force_swept_transport(p, f, dt, nsamp=6):
    """Free transport of the piecewise-LINEAR 2-D reconstruction L_c(x,y) = f_c + sx (x - x_c) + sy (y - y_c) (van Leer slopes
    in both directions), face by face: the particles of velocity (u, v) that cross a face during [0, dt] fill the
    parallelogram spanned by the face and -(u, v) dt; their number is |normal velocity| dt x (face length) x (mean of the
    upwind cell's reconstruction over that parallelogram), the mean taken by sampling nsamp x nsamp points.  Periodic."""
    J, I, Nv, Nu = f.shape
    U = np.broadcast_to(p.u[None, :], (Nv, Nu))
    V = np.broadcast_to(p.v[:, None], (Nv, Nu))
    sx, sy = _van_leer(f, p.dx, 1), _van_leer(f, p.dy, 0)
    out = f.copy()
    ss = (np.arange(nsamp) + 0.5) / nsamp                                      # midpoints along the face and along time
    for axis, d, ell, n, t in ((1, p.dx, p.dy, U, V), (0, p.dy, p.dx, V, U)):  # x-faces (normal u), y-faces (normal v)
        def mean_from(cell_f, cell_sn, cell_st, xc):
            """mean of the reconstruction of a cell whose centre is at normal offset xc from the face, over the parallelogram"""
            acc = np.zeros_like(cell_f)
            for a in ss:                                                       # position along the face, in (-ell/2, ell/2)
                for b in ss:                                                   # time fraction
                    xn = -n * dt * b - xc                                      # normal coordinate relative to the cell centre
                    xt = ell * (a - 0.5) - t * dt * b                          # tangential coordinate relative to the cell centre
                    acc += cell_f + cell_sn * xn + cell_st * xt
            return acc / (nsamp * nsamp)
        sn, st = (sx, sy) if axis == 1 else (sy, sx)
        fromL = mean_from(np.roll(f, 1, axis), np.roll(sn, 1, axis), np.roll(st, 1, axis), -0.5 * d)   # L's centre at -d/2
        fromR = mean_from(f, sn, st, 0.5 * d)
        up = np.where(n > 0, fromL, np.where(n < 0, fromR, 0.5 * (fromL + fromR)))
        swept = n * dt * up                                                    # per unit face length, signed along +axis
        out += (swept - np.roll(swept, -1, axis)) / d
    return out


@pytest.mark.parametrize("nuv", [(8, 8), (9, 7)])
def test_P20_oblique_free_transport_brute_force(nuv):
    """tau -> infinity, rough data (both limiters active), 4x4 periodic mesh: one step equals the swept-parallelogram
    transport of the 2-D reconstruction.  (9,7) has u = 0 and v = 0 nodes."""
    p = workloads.periodic_box(4, 4, nuv[0], nuv[1], a=4.0, mu_ref=7.310334e14, seed=2, bu=3.0, lx=1.0, ly=0.8)
    rng = np.random.default_rng(43)
    W, f, _ = workloads.initial_state(p)
    f = f * rng.uniform(0.2, 1.8, f.shape)
    o = Oracle(p, tangential=True)
    o.set_state(W, f)
    o.step(1)
    expect = _brute_force_swept_transport(p, f, o.dt)
    o0 = Oracle(p)
    o0.set_state(W, f)
    o0.step(1)
    assert err_f(o0.f(), expect) > 3e-4                                        # the theta term is not a no-op here
    assert err_f(o.f(), expect) < 5e-14


def _collisionless_error(I, tangential, tend=0.2):
    """L1 error against the exact solution f(x, y, t) = f(x - u t, y - v t, 0) of collisionless transport of a smooth
    periodic density wave along the diagonal (one oblique velocity pair dominates: 2 x 2 velocity grid)."""
    u = np.array([-0.7, 1.0]); wu = np.array([0.5, 0.5])
    v = np.array([-0.4, 0.6]); wv = np.array([0.5, 0.5])
    p = workloads.Problem(I=I, J=I, x0=0.0, x1=1.0, y0=0.0, y1=1.0, u=u, wu=wu, v=v, wv=wv, mu_ref=7.310334e14,
                          bcs=[(workloads.BC_PERIODIC, 1, 0, 0, 1)] * 4, cfl=0.8, name="free")
    xc = (np.arange(I) + 0.5) / I
    X, Y = np.meshgrid(xc, xc)

    def prof(x, y):                                                            # cell averages ~ point values + O(h^2): same order
        return 1.0 + 0.3 * np.sin(2 * math.pi * x) * np.cos(2 * math.pi * y) + 0.2 * np.sin(2 * math.pi * (x + y))
    f = np.empty((I, I, 2, 2))
    for m in range(2):
        for k in range(2):
            f[:, :, m, k] = prof(X, Y) * (1.0 + 0.1 * k + 0.05 * m)
    w = wv[:, None] * wu[None, :]
    W = np.stack([(f * w).sum((2, 3)), (f * w * u[None, :]).sum((2, 3)), (f * w * v[:, None]).sum((2, 3)),
                  (f * w * 0.5 * (u[None, :] ** 2 + v[:, None] ** 2)).sum((2, 3))], axis=-1)
    W[..., 3] += 1.0                                                           # keeps lambda > 0 (W does not feed back as tau -> inf)
    o = Oracle(p, threads=8, tangential=tangential)
    o.set_state(W, f)
    n = int(math.ceil(tend / o.dt))
    o.step(n)
    t = n * o.dt
    err = 0.0
    fo = o.f()
    for m in range(2):
        for k in range(2):
            exact = prof(X - u[k] * t, Y - v[m] * t) * (1.0 + 0.1 * k + 0.05 * m)
            err += np.mean(np.abs(fo[:, :, m, k] - exact))
    return err / 4


def test_P21_collisionless_oblique_transport_is_second_order_and_better_with_theta():
    e1 = [_collisionless_error(I, True) for I in (16, 32, 64)]
    e0 = [_collisionless_error(I, False) for I in (16, 32, 64)]
    assert e1[1] / e1[2] > 3.3 and e1[0] / e1[1] > 2.5, e1                    # second order with the 2-D reconstruction
    assert e1[2] < 0.8 * e0[2], (e1, e0)                                       # and more accurate than the normal-only scheme


def test_P22_invariants_with_tangential_slopes():
    """conservation to 1e-13, uniform fixed point, x<->y transposition, and sum_q w psi F_q = F_W per face."""
    p = workloads.periodic_box(8, 6, 12, 10, a=5.0, Kn=0.05, seed=5, bu=6.0, lx=1.3, ly=0.7)
    W, f, _ = workloads.initial_state(p)
    o = Oracle(p, tangential=True)
    o.set_state(W, f)
    # per-face consistency of F_W (S5 analytic + S7 discrete) with the moments of F_q (S8), on a grid fine enough for the
    # quadrature error of the Maxwellian part (P19): theta must enter both, with the same sign and weight
    pc = workloads.periodic_box(12, 12, 28, 28, a=6.0, Kn=0.05, seed=7)
    Wc, fc, _ = workloads.initial_state(pc)
    oc, on = Oracle(pc, tangential=True), Oracle(pc)
    oc.set_state(Wc, fc); on.set_state(Wc, fc)
    w = pc.wv[:, None] * pc.wu[None, :]
    U, V = np.broadcast_to(pc.u[None, :], w.shape), np.broadcast_to(pc.v[:, None], w.shape)
    moved = 0.0
    for d, i, j in ((0, 3, 2), (1, 5, 4), (0, 0, 0), (1, 7, 0)):
        FW, Ff, st = oc.face_flux(d, i, j)
        S = np.array([np.sum(w * q * Ff) for q in (np.ones_like(w), U, V, 0.5 * (U * U + V * V))])
        scale = (pc.dy if d == 0 else pc.dx) * oc.dt * st[4]
        assert np.max(np.abs(S - FW)) < 1e-7 * scale
        moved = max(moved, float(np.max(np.abs(FW - on.face_flux(d, i, j)[0]))) / scale)
    assert moved > 1e-6                                                        # theta changes the macroscopic flux
    tot0 = W.reshape(-1, 4).sum(0)
    o.step(5)
    tot = o.W().reshape(-1, 4).sum(0)
    assert np.all(np.abs(tot - tot0) < 1e-13 * tot0[0])
    # transposition: swap x<->y, u<->v
    q = workloads.Problem(I=p.J, J=p.I, x0=p.y0, x1=p.y1, y0=p.x0, y1=p.x1, u=p.v, wu=p.wv, v=p.u, wv=p.wu, Kn=p.Kn,
                          bcs=list(p.bcs), cfl=p.cfl)
    Wt = np.ascontiguousarray(W.transpose(1, 0, 2)[..., [0, 2, 1, 3]])
    ft = np.ascontiguousarray(f.transpose(1, 0, 3, 2))
    ot = Oracle(q, tangential=True)
    ot.set_state(Wt, ft)
    ot.step(5)
    assert err_f(np.ascontiguousarray(ot.f().transpose(1, 0, 3, 2)), o.f()) < 1e-14
    # uniform Maxwellian: all slopes vanish, nothing moves
    ones = np.ones((p.J, p.I))
    fu = workloads.maxwellian_field(p, 0.9 * ones, 0.3 * ones, -0.1 * ones, ones / 1.2)
    Wu = np.broadcast_to(np.array([0.9, 0.27, -0.09, 0.5 * 0.9 * 0.1 + 0.9 / 2.4]), (p.J, p.I, 4)).copy()
    o.set_state(Wu, fu)
    o.step(3)
    assert np.max(np.abs(o.W() - Wu)) < 1e-15 and err_f(o.f(), fu) < 5e-16
