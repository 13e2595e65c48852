"""Pins P1-P5 of DESIGN.md: the oracle's closed-form pieces against independent mathematics
(numerical quadrature, finite differences, limits).  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import integrate

import workloads
from oracle import binding as ob

PRIMS = [(1.0, 0.0, 0.0, 1.0), (0.8, 0.3, -0.2, 1.3), (1.7, -0.9, 0.45, 0.6), (0.3, 2.0, 1.0, 2.5)]


def _g1(n, U, lam):                       # 1-D normalised Gaussian factor of the Maxwellian
    return math.sqrt(lam / math.pi) * math.exp(-lam * (n - U) ** 2)


@pytest.mark.parametrize("prim", PRIMS)
def test_P1_half_and_full_range_moments_vs_quadrature(prim):
    """O4: <n^p> over n>0, n<0 and the whole line, p = 0..6, against scipy.integrate.quad."""
    rho, U, V, lam = prim
    ML, MR, Mu, Mv = ob.gauss_moments(prim)
    for p in range(7):
        qL = integrate.quad(lambda n: n ** p * _g1(n, U, lam), 0, np.inf, epsabs=1e-13, epsrel=1e-12)[0]
        qR = integrate.quad(lambda n: n ** p * _g1(n, U, lam), -np.inf, 0, epsabs=1e-13, epsrel=1e-12)[0]
        qV = integrate.quad(lambda t: t ** p * _g1(t, V, lam), -np.inf, np.inf, epsabs=1e-13, epsrel=1e-12)[0]
        scale = max(1.0, abs(qL), abs(qR))
        assert abs(ML[p] - qL) < 2e-9 * scale, (p, ML[p], qL)
        assert abs(MR[p] - qR) < 2e-9 * scale, (p, MR[p], qR)
        assert abs(Mv[p] - qV) < 2e-9 * max(1.0, abs(qV)), (p, Mv[p], qV)
        assert Mu[p] == ML[p] + MR[p]


@pytest.mark.parametrize("prim", PRIMS)
def test_P1_moment_vectors_vs_2d_quadrature(prim):
    """O4: T_X[c](alpha,beta) = <n^a t^b psi (c.psi)> against a dense 2-D tensor quadrature."""
    rho, U, V, lam = prim
    c = np.array([0.3, -0.7, 0.2, 0.11])
    sig = 1.0 / math.sqrt(2 * lam)
    n = np.linspace(U - 12 * sig, U + 12 * sig, 2401)
    t = np.linspace(V - 12 * sig, V + 12 * sig, 2401)
    wn = np.full_like(n, n[1] - n[0]); wn[[0, -1]] *= 0.5
    wt = np.full_like(t, t[1] - t[0]); wt[[0, -1]] *= 0.5
    gn = np.sqrt(lam / np.pi) * np.exp(-lam * (n - U) ** 2) * wn
    gt = np.sqrt(lam / np.pi) * np.exp(-lam * (t - V) ** 2) * wt
    nz = np.argmin(np.abs(n))               # the half-range split needs a node at exactly n = 0
    n = n - n[nz]
    gn = np.sqrt(lam / np.pi) * np.exp(-lam * (n - U) ** 2) * wn
    Hn = {"Mu": np.ones_like(n), "ML": (n > 0) + 0.5 * (n == 0), "MR": (n < 0) + 0.5 * (n == 0)}
    Nn, Tt = np.meshgrid(n, t, indexing="ij")
    psi = [np.ones_like(Nn), Nn, Tt, 0.5 * (Nn ** 2 + Tt ** 2)]
    cpsi = sum(ci * p for ci, p in zip(c, psi))
    for X in ("Mu", "ML", "MR"):
        G = (gn * Hn[X])[:, None] * gt[None, :]
        for (a, b) in [(0, 0), (1, 0), (2, 0), (0, 1), (1, 1)]:
            got = ob.moment_T(prim, X, c, a, b)
            got_m = ob.moment_T(prim, X, None, a, b)
            GP = G * Nn ** a * Tt ** b
            for r in range(4):
                ref = np.sum(GP * psi[r] * cpsi)
                ref_m = np.sum(GP * psi[r])
                assert abs(got[r] - ref) < 5e-6 * max(1.0, abs(ref)), (X, a, b, r, got[r], ref)
                assert abs(got_m[r] - ref_m) < 5e-6 * max(1.0, abs(ref_m)), (X, a, b, r)


@pytest.mark.parametrize("prim", PRIMS)
def test_P2_micro_slope_round_trip_and_finite_difference(prim):
    rng = np.random.default_rng(7)
    prim = np.array(prim)
    for _ in range(5):
        c = rng.uniform(-1, 1, 4)
        s = prim[0] * ob.moment_T(prim, "Mu", c, 0, 0)          # rho <psi (c.psi)>
        c2 = ob.micro_slope(prim, s)
        assert np.allclose(c2, c, rtol=0, atol=1e-11 * max(1.0, np.max(np.abs(c)))), (c, c2)
        # d/d eps of M[prim(W + eps s)] = (c.psi) M  at a few velocity points
        W = ob.W_of_prim(prim)
        eps = 1e-6
        pp, pm = ob.prim_of_W(W + eps * s), ob.prim_of_W(W - eps * s)
        for (u, v) in [(0.0, 0.0), (0.7, -1.1), (-1.9, 0.4), (prim[1], prim[2])]:
            fd = (ob.maxwellian(pp, u, v) - ob.maxwellian(pm, u, v)) / (2 * eps)
            an = (c[0] + c[1] * u + c[2] * v + 0.5 * c[3] * (u * u + v * v)) * ob.maxwellian(prim, u, v)
            assert abs(fd - an) < 1e-7 * max(1e-3, abs(an)) + 1e-9, (u, v, fd, an)


def test_P3_time_coefficients_vs_quadrature_limits_and_continuity():
    integrands = [
        lambda t, tau: 1 - math.exp(-t / tau),
        lambda t, tau: -tau + tau * math.exp(-t / tau) + t * math.exp(-t / tau),
        lambda t, tau: t - tau + tau * math.exp(-t / tau),
        lambda t, tau: math.exp(-t / tau),
        lambda t, tau: t * math.exp(-t / tau),
    ]
    dt = 0.01
    for x in [5e-2, 1e-2, 0.3, 1.0, 7.0, 200.0]:
        tau = dt / x
        Mt = ob.time_coeffs(dt, tau)
        for k, fn in enumerate(integrands):
            if k in (1, 2) and x < 0.2:
                continue          # the naive integrand cancels catastrophically here; series checked below
            ref = integrate.quad(fn, 0, dt, args=(tau,), epsabs=1e-20, epsrel=1e-13)[0]
            assert abs(Mt[k] - ref) <= 1e-11 * max(abs(ref), dt * dt * min(1.0, x)), (x, k, Mt[k], ref)
    # exact algebraic identities of the five integrals (hold for all x)
    for x in [1e-6, 1e-4, 9.9e-4, 1e-3, 2e-3, 0.1, 3.0]:
        tau = dt / x
        Mt = ob.time_coeffs(dt, tau)
        assert abs(Mt[0] + Mt[3] - dt) < 1e-15 * dt                       # Mt1 + Mt4 = dt
        assert abs(Mt[2] - (0.5 * dt * dt - tau * Mt[0])) <= 2e-16 * dt * dt * max(1, 1 / x) * 4
    # small-x branch against the exact Taylor series of the five integrals (14 terms, rational
    # coefficients derived in DESIGN.md "O5"):  Mt4 = dt sum (-x)^k/(k+1)!,  Mt5 = dt^2 sum (k+1)(-x)^k/(k+2)!,
    # Mt1 = dt - Mt4,  Mt3 = -dt^2 sum_{k>=1} (-x)^k/(k+2)!,  Mt2 = dt^2 sum_{k>=1} k (-x)^k/(k+2)!
    f = math.factorial
    for x in [1e-8, 1e-5, 5e-4, 9.99e-4, 2e-3, 1e-2]:        # both branches
        tau = dt / x
        Mt = ob.time_coeffs(dt, tau)
        m4 = dt * sum((-x) ** k / f(k + 1) for k in range(14))
        m5 = dt * dt * sum((k + 1) * (-x) ** k / f(k + 2) for k in range(14))
        m1 = -dt * sum((-x) ** k / f(k + 1) for k in range(1, 14))
        m3 = -dt * dt * sum((-x) ** k / f(k + 2) for k in range(1, 14))
        m2 = dt * dt * sum(k * (-x) ** k / f(k + 2) for k in range(1, 14))
        rel = 1e-15 if x < 1e-3 else 1e-15 / x    # closed form: Mt1 = dt - Mt4 loses ~eps/x by cancellation,
        rel2 = 1e-15 if x < 1e-3 else 1e-15 / x ** 2   # Mt2, Mt3 = O(dt^2 x) differences of O(dt^2) terms lose ~eps/x^2
        assert abs(Mt[3] - m4) < 4e-16 * dt
        assert abs(Mt[4] - m5) < max(4e-16, rel) * dt * dt
        assert abs(Mt[0] - m1) < max(2e-14, rel) * abs(m1) + 1e-19 * dt   # 5-term series: x^4/360 truncation
        assert abs(Mt[2] - m3) < max(2e-14, rel2) * abs(m3), (x, Mt[2], m3)
        assert abs(Mt[1] - m2) < max(2e-14, rel2) * abs(m2), (x, Mt[1], m2)
    # continuity across the branch point x = 1e-3
    lo = ob.time_coeffs(dt, dt / (1e-3 * (1 - 1e-12)))
    hi = ob.time_coeffs(dt, dt / (1e-3 * (1 + 1e-12)))
    scale = np.array([dt * 1e-3, dt * dt * 1e-3, dt * dt * 1e-3, dt, dt * dt])
    tol = np.array([2e-11, 1e-9, 1e-9, 2e-11, 2e-11])     # Mt2, Mt3: eps/x^2 cancellation on the closed-form side
    assert np.all(np.abs(lo - hi) < tol * scale), (lo - hi) / scale
    # limits: collisionless (x -> 0) and continuum (x -> inf)
    Mt = ob.time_coeffs(dt, 1e30)
    assert Mt[3] == dt and abs(Mt[4] - 0.5 * dt * dt) < 1e-18 and max(abs(Mt[0]), abs(Mt[1]), abs(Mt[2])) < 1e-30
    tau = 1e-9
    Mt = ob.time_coeffs(dt, tau)
    assert abs(Mt[0] - (dt - tau)) < 1e-18 and abs(Mt[3] - tau) < 1e-24 and abs(Mt[2] - (0.5 * dt * dt - tau * (dt - tau))) < 1e-18


def test_P4_compatibility_condition_of_A():
    """O6: rho <psi (a n + b t + A)> = 0 with the half-range split, for random slopes."""
    rng = np.random.default_rng(11)
    for prim in PRIMS:
        aL, aR, b = rng.uniform(-1, 1, 4), rng.uniform(-1, 1, 4), rng.uniform(-1, 1, 4)
        rhs = ob.moment_T(prim, "ML", aL, 1, 0) + ob.moment_T(prim, "MR", aR, 1, 0) + ob.moment_T(prim, "Mu", b, 0, 1)
        A = ob.micro_slope(prim, -prim[0] * rhs)
        tot = ob.moment_T(prim, "Mu", A, 0, 0) + rhs
        assert np.max(np.abs(tot)) < 1e-12 * max(1.0, np.max(np.abs(rhs)))


def test_P5_discrete_maxwellian_moments_on_config_grids():
    """north_star: discrete moments of a Maxwellian match the closed forms to quadrature error.
    Expected truncation levels (erfc(a sqrt(lam)) and h-convergence of the trapezoid rule):"""
    expect = {"C1": (2e-7, 3e-6), "C2": (3e-11, 5e-10), "C4": (1e-14, 3e-14), "C5": (1e-14, 1e-14)}
    for name, (tol_rho, tol_E) in expect.items():
        p = workloads.channel_config(name, I=2, J=2)
        prim = np.array([1.0, 0.0, 0.0, 1.0])
        w = p.wv[:, None] * p.wu[None, :]
        U, V = np.meshgrid(p.u, p.v)
        g = np.array([[ob.maxwellian(prim, U[m, k], V[m, k]) for k in range(p.Nu)] for m in range(p.Nv)])
        Wd = np.array([np.sum(w * g), np.sum(w * U * g), np.sum(w * V * g), np.sum(w * 0.5 * (U * U + V * V) * g)])
        Wc = ob.W_of_prim(prim)
        assert abs(Wd[0] - Wc[0]) / Wc[0] < tol_rho, (name, Wd, Wc)
        assert abs(Wd[3] - Wc[3]) / Wc[3] < tol_E, (name, Wd, Wc)
        assert abs(Wd[1]) < 1e-15 and abs(Wd[2]) < 1e-15
        # and it is genuinely a quadrature error: it must not vanish on the coarse grid
        if name == "C1":
            assert abs(Wd[0] - Wc[0]) / Wc[0] > 1e-9
    # shifted, hot Maxwellian on the wide grid: all four moments
    p = workloads.channel_config("C5", I=2, J=2)
    prim = np.array([0.7, 1.5, -2.5, 0.4])
    U, V = np.meshgrid(p.u, p.v)
    w = p.wv[:, None] * p.wu[None, :]
    g = np.vectorize(lambda a, b: ob.maxwellian(prim, a, b))(U, V)
    Wd = np.array([np.sum(w * g), np.sum(w * U * g), np.sum(w * V * g), np.sum(w * 0.5 * (U * U + V * V) * g)])
    assert np.allclose(Wd, ob.W_of_prim(prim), rtol=1e-13, atol=0)


def test_small_formulas_van_leer_tau_mu_ref_prim_roundtrip():
    assert ob.van_leer(1.0, 3.0) == 1.5 and ob.van_leer(-1.0, -3.0) == -1.5
    assert ob.van_leer(1.0, -3.0) == 0.0 and ob.van_leer(0.0, 3.0) == 0.0 and ob.van_leer(2.0, 2.0) == 2.0
    assert ob.van_leer(1e-200, 1e-200) == 0.0          # AMB-4: product underflow -> 0
    # harmonic-mean property 1/VL = (1/a + 1/b)/2
    a, b = 0.37, 2.9
    assert abs(1 / ob.van_leer(a, b) - 0.5 * (1 / a + 1 / b)) < 1e-15
    # AMB-7: mu_ref = 0.7310334 Kn at omega = 0.81; hard spheres 5 sqrt(pi)/16 Kn
    assert abs(ob.mu_ref_from_kn(1.0, 0.81) - 0.7310334) < 5e-8
    assert abs(ob.mu_ref_from_kn(0.3, 0.5) - 5 * math.sqrt(math.pi) / 16 * 0.3) < 1e-16
    # tau = mu/p with mu = mu_ref T^omega, p = rho T / 2  (T = 1/lam)
    rho, T, mu_ref, om = 0.7, 1.9, 0.05, 0.81
    assert abs(ob.tau(mu_ref, om, rho, 1 / T) - mu_ref * T ** om / (rho * T / 2)) < 1e-16
    for prim in PRIMS:
        assert np.allclose(ob.prim_of_W(ob.W_of_prim(prim)), prim, rtol=1e-14)
    # gamma = 2 (K_int = 0): p = rho/(2 lam) = (gamma-1)(rhoE - rho|U|^2/2)
    W = ob.W_of_prim((1.3, 0.2, -0.4, 0.8))
    assert abs((W[3] - 0.5 * 1.3 * (0.04 + 0.16)) - 1.3 / (2 * 0.8)) < 1e-15


def test_golden_paper_dof_count_matches_state_layout():
    """dof = cells * (K*M + 4): one f value per velocity point + 4 macroscopic variables."""
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_dof.txt")
    rows = [list(map(int, l.split())) for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 2
    for I, J, K, M, dof in rows:
        p = workloads.periodic_box(I, J, K, M)
        W, f, _ = workloads.initial_state(p)
        assert W.size + f.size == dof
