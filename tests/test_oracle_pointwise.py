"""Pins for the oracle's per-point routines (run with -m "not gpu").

Each test checks the oracle against something OTHER than itself: constants the paper prints
(Eqs. 11, 14, 16, 17, 18, 19), exactness on polynomials, the 5-point Lagrange interpolant, split-flux
identities, finite-difference flux Jacobians, textbook values.  P:L<n> = /root/reference/PAPER.md line.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

rng = np.random.default_rng(7)


def random_state(n=1):
    rho = rng.uniform(0.3, 2.0, n)
    u, v, w = (rng.uniform(-1.5, 1.5, n) for _ in range(3))
    p = rng.uniform(0.2, 2.0, n)
    e = p / 0.4 + 0.5 * rho * (u * u + v * v + w * w)
    return np.stack([rho, rho * u, rho * v, rho * w, e], axis=1)


# ------------------------------------------------------------------------------------------------
# 6th-order central difference
# ------------------------------------------------------------------------------------------------
def test_d6_exact_up_to_degree_6(po):
    x = np.arange(-3, 4, dtype=float)
    for deg in range(0, 7):
        assert po.d6(x ** deg) == pytest.approx(1.0 if deg == 1 else 0.0, abs=1e-12)
    # degree 7 is NOT exact: leading error term -(1/140) f^(7) => d6(x^7) = 36
    assert po.d6(x ** 7) == pytest.approx(36.0, rel=1e-12)


def test_d6_antisymmetric_and_order(po):
    a = rng.normal(size=7)
    assert po.d6(a) == pytest.approx(-po.d6(a[::-1]), rel=1e-14)
    errs = []
    for h in (0.2, 0.1):
        x = 0.3 + h * np.arange(-3, 4)
        errs.append(abs(po.d6(np.sin(x)) / h - np.cos(0.3)))
    assert np.log2(errs[0] / errs[1]) == pytest.approx(6.0, abs=0.15)


# ------------------------------------------------------------------------------------------------
# Printed constants: Eq. 19 must follow from Eqs. 9, 11 and 18
# ------------------------------------------------------------------------------------------------
def test_eq19_constants_follow_from_eq11_and_eq18():
    # Eq. 18 at i+1/2 on points i-2..i+3, Eq. 11 coefficients
    fxx = [Fr(c, 48) for c in (-5, 39, -34, -34, 39, -5)]
    fxxxx = [Fr(c, 2) for c in (1, -3, 2, 2, -3, 1)]
    corr = [Fr(-1, 24) * a + Fr(7, 5760) * b for a, b in zip(fxx, fxxxx)]  # correction at i+1/2, points i-2..i+3
    # correction(i+1/2) - correction(i-1/2) expressed on points i-3..i+3
    tot = [Fr(0)] * 7
    for m, c in enumerate(corr):
        tot[m + 1] += c   # i+1/2 stencil starts at i-2 -> slot 1
        tot[m] -= c       # i-1/2 stencil starts at i-3 -> slot 0
    assert tot[3] == 0
    assert tot[4] == Fr(17, 256) and tot[2] == -Fr(17, 256)
    assert tot[5] == -Fr(13, 320) and tot[1] == Fr(13, 320)
    assert tot[6] == Fr(19, 3840) and tot[0] == -Fr(19, 3840)


def test_eq19_in_the_oracle_uniform_state_varying_metric(po):
    """With a uniform state along the line, U^L = U^R = Q, F+ + F- = F(Q, k_{i+1/2}) which is LINEAR in k.
    Then Eq. 19 acts on the metric alone and (reading U5) must collapse to the 6th-order central difference
    of k: D_i = F(Q, d6(k)_i) to round-off — for ANY sequence k, and equal to F(Q, k'(i)) for polynomials
    of degree <= 5.  Pins Eq. 19's constants, khat_half, the split-flux sum and the line indexing."""
    n = 9
    Q = random_state()[0]
    Ql = np.repeat(Q[:, None], n + 12, axis=1)
    # (a) random positive-ish metric sequence
    kl = rng.normal(size=(3, n + 12)) * 0.05 + np.array([[1.0], [0.3], [-0.2]])
    D = po.inviscid_line(Ql, kl)
    for i in range(n):
        dk = np.array([po.d6(kl[c, 6 + i - 3:6 + i + 4]) for c in range(3)])
        # F(Q, dk) computed as a difference of two oracle point fluxes (linear in k)
        ref = po.point_flux(Q, kl[:, 6 + i] + dk) - po.point_flux(Q, kl[:, 6 + i])
        assert np.allclose(D[:, i], ref, rtol=0, atol=2e-13)
    # (b) degree-5 polynomial metric: exact derivative
    s = np.arange(-6, n + 6, dtype=float)
    poly = np.polynomial.Polynomial([1.0, 0.02, -0.003, 0.0004, 0.00002, -0.000001])
    kl = np.stack([poly(s), 0.5 * poly(s) + 0.1, 0.0 * s + 0.2])
    D = po.inviscid_line(Ql, kl)
    for i in range(n):
        dk = np.array([poly.deriv()(float(i)), 0.5 * poly.deriv()(float(i)), 0.0])
        ref = po.point_flux(Q, kl[:, 6 + i] + dk) - po.point_flux(Q, kl[:, 6 + i])
        assert np.allclose(D[:, i], ref, rtol=0, atol=5e-13)


def test_khat_half_is_6point_lagrange(po):
    # exact for degree <= 5 at the half point between slots 2 and 3
    x = np.arange(-2, 4, dtype=float)
    for deg in range(6):
        assert po.khat_half(x ** deg) == pytest.approx(0.5 ** deg, abs=1e-12)
    assert abs(po.khat_half(x ** 6) - 0.5 ** 6) > 1e-3
    # symmetric
    a = rng.normal(size=6)
    assert po.khat_half(a) == pytest.approx(po.khat_half(a[::-1]), rel=1e-15)


# ------------------------------------------------------------------------------------------------
# WENO interpolation (Eqs. 13–17, reading U1)
# ------------------------------------------------------------------------------------------------
def test_beta_equals_printed_eq17(po):
    """Eq. 17 exactly as printed vs the oracle's Jiang–Shu form."""
    for _ in range(50):
        um2, um1, u0, up1, up2 = s = rng.normal(size=5)
        b1 = (4 * um2 ** 2 - 19 * um2 * um1 + 25 * um1 ** 2 + 11 * um2 * u0 - 31 * um1 * u0 + 10 * u0 ** 2) / 3
        b2 = (4 * um1 ** 2 - 13 * um1 * u0 + 13 * u0 ** 2 + 5 * um1 * up1 - 13 * u0 * up1 + 4 * up1 ** 2) / 3
        b3 = (10 * u0 ** 2 - 31 * u0 * up1 + 25 * up1 ** 2 + 11 * u0 * up2 - 19 * up1 * up2 + 4 * up2 ** 2) / 3
        assert np.allclose(po.weno5_beta(s), [b1, b2, b3], rtol=1e-11, atol=1e-13)


def test_weno_linear_weights_give_5point_lagrange(po):
    """With eps huge the weights are the linear ones (Eq. 16); the combination of the Eq. 14 interpolants
    must then be the 5-point Lagrange interpolant (3,-20,90,60,-5)/128 — true only if interpolants and
    weights are paired BY STENCIL (reading U1)."""
    cL = np.array([3, -20, 90, 60, -5]) / 128.0
    for _ in range(20):
        s = rng.normal(size=5)
        vL, vR = po.weno5(s, eps=1e40)
        assert vL == pytest.approx(cL @ s, abs=1e-13)
        assert vR == pytest.approx(cL[::-1] @ s, abs=1e-13)


def test_weno_exact_for_quadratics_any_weights(po):
    for _ in range(20):
        a, b, c = rng.normal(size=3)
        f = lambda x: a + b * x + c * x * x
        s = f(np.arange(-2, 3, dtype=float))
        vL, vR = po.weno5(s, eps=1e-6)
        assert vL == pytest.approx(f(0.5), abs=1e-12)
        assert vR == pytest.approx(f(-0.5), abs=1e-12)


def test_weno_fifth_order_on_smooth_data(po):
    errs = []
    for h in (0.1, 0.05, 0.025):
        x = 0.4 + h * np.arange(-2, 3)
        vL, vR = po.weno5(np.sin(x) + 2.0, eps=1e-6)
        errs.append(max(abs(vL - np.sin(0.4 + h / 2) - 2.0), abs(vR - np.sin(0.4 - h / 2) - 2.0)))
    assert np.log2(errs[0] / errs[1]) > 4.6 and np.log2(errs[1] / errs[2]) > 4.8


def test_weno_is_essentially_non_oscillatory(po):
    # step between i and i+1: left state at i+1/2 must come from the smooth stencil {i-2,i-1,i}
    vL, vR = po.weno5(np.array([1.0, 1.0, 1.0, 0.0, 0.0]))
    assert vL == pytest.approx(1.0, abs=1e-9)
    # step between i-1 and i: right state at i-1/2 must come from {i,i+1,i+2}
    vL, vR = po.weno5(np.array([0.0, 0.0, 1.0, 1.0, 1.0]))
    assert vR == pytest.approx(1.0, abs=1e-9)
    # mirror symmetry of the pair
    s = rng.normal(size=5)
    vL, vR = po.weno5(s)
    vL2, vR2 = po.weno5(s[::-1].copy())
    assert vL == pytest.approx(vR2, rel=1e-13) and vR == pytest.approx(vL2, rel=1e-13)


# ------------------------------------------------------------------------------------------------
# Fluxes and eigenvectors (Eq. 4, readings U3, U4)
# ------------------------------------------------------------------------------------------------
def test_point_flux_textbook_value(po):
    # rho=1, u=(1,0,0), p=1, gamma=1.4: e = 1/0.4 + 0.5 = 3; F_x = (rho u, rho u^2 + p, 0, 0, (e+p)u) = (1,2,0,0,4)
    F = po.point_flux([1.0, 1.0, 0.0, 0.0, 3.0], [1.0, 0.0, 0.0])
    assert np.allclose(F, [1.0, 2.0, 0.0, 0.0, 4.0], atol=1e-15)
    # a scaled, rotated metric: F(k) = kx Fx + ky Fy + kz Fz, with v = w = 0: Fy = (0,0,p,0,0), Fz = (0,0,0,p,0)
    F = po.point_flux([1.0, 1.0, 0.0, 0.0, 3.0], [2.0, 3.0, -1.0])
    assert np.allclose(F, [2.0, 4.0, 3.0, -1.0, 8.0], atol=1e-14)


def test_sw_split_sums_to_eq4_flux(po):
    for Q in random_state(100):
        k = rng.normal(size=3) * rng.uniform(0.01, 30)
        Fp, Fm, F = po.sw_flux(Q, k, +1), po.sw_flux(Q, k, -1), po.point_flux(Q, k)
        scale = np.abs(F).max() + np.linalg.norm(k) * np.abs(Q).max()
        assert np.abs(Fp + Fm - F).max() <= 1e-14 * scale


def test_sw_upwinding(po):
    # supersonic along +k: every eigenvalue positive -> F- = 0, F+ = F; and the reverse
    Q = np.array([1.0, 3.0, 0.1, -0.2, 1.0 / 0.4 / 1.4 + 0.5 * (9 + 0.01 + 0.04)])
    k = np.array([0.7, 0.0, 0.0])
    assert np.allclose(po.sw_flux(Q, k, -1), 0.0, atol=1e-16)
    assert np.allclose(po.sw_flux(Q, k, +1), po.point_flux(Q, k), rtol=1e-14)
    assert np.allclose(po.sw_flux(Q, -k, +1), 0.0, atol=1e-16)
    # at rest: F+ carries +c|k| wave only, mass flux = rho c |k| / (2 gamma)
    Q = np.array([1.0, 0, 0, 0, 1.0 / 1.4 / 0.4])
    Fp = po.sw_flux(Q, [2.0, 0, 0], +1)
    assert Fp[0] == pytest.approx(1.0 * 1.0 * 2.0 / 2.8, rel=1e-14)


def test_eigenvectors_diagonalise_the_flux_jacobian(po):
    """L R = I, L A R = diag(th, th, th, th+c, th-c) with A = d F(Q, n)/dQ by central differences of the
    oracle's Eq.-4 flux; and F+- = |k| R Lambda+- L Q (homogeneity of the Euler flux)."""
    for Q in random_state(40):
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        L, R = po.eig(Q, n)
        assert np.abs(L @ R - np.eye(5)).max() < 5e-14
        A = np.zeros((5, 5))
        for m in range(5):
            dq = np.zeros(5)
            dq[m] = 1e-6 * max(1.0, abs(Q[m]))
            A[:, m] = (po.point_flux(Q + dq, n) - po.point_flux(Q - dq, n)) / (2 * dq[m])
        rho, u = Q[0], Q[1:4] / Q[0]
        p = 0.4 * (Q[4] - 0.5 * rho * u @ u)
        c = np.sqrt(1.4 * p / rho)
        th = n @ u
        lam = np.array([th, th, th, th + c, th - c])
        assert np.abs(L @ A @ R - np.diag(lam)).max() < 2e-7
        kmag = rng.uniform(0.1, 10)
        for sgn in (+1, -1):
            ls = 0.5 * (lam + sgn * np.abs(lam))
            ref = kmag * (R @ (ls * (L @ Q)))
            assert np.allclose(po.sw_flux(Q, kmag * n, sgn), ref, rtol=0, atol=2e-12 * kmag * np.abs(Q).max() * 5)


# ------------------------------------------------------------------------------------------------
# Inviscid line operator (Fig. 11): consistency, order, upwinding
# ------------------------------------------------------------------------------------------------
def _line_state(x):
    rho = 1.0 + 0.2 * np.sin(x)
    u = 0.4 + 0.1 * np.cos(2 * x)
    v = 0.1 * np.sin(x + 0.3)
    w = -0.2 + 0.05 * np.cos(x)
    p = 1 / 1.4 + 0.1 * np.sin(2 * x + 1.0)
    return np.stack([rho, rho * u, rho * v, rho * w, p / 0.4 + 0.5 * rho * (u * u + v * v + w * w)])


@pytest.mark.parametrize("scheme", [0, 1])
def test_inviscid_line_fifth_order(po, scheme):
    """D_i / h -> dF/dx at 5th order on a smooth 1-D state (constant Cartesian metric k = (1,0,0)).
    Reference derivative: 6th-order central difference of the oracle's Eq.-4 flux on a 16x finer spacing."""
    errs = []
    for n in (32, 64, 128):
        h = 2 * np.pi / n
        x = h * np.arange(-6, n + 6)
        kl = np.zeros((3, n + 12))
        kl[0] = 1.0
        D = po.inviscid_line(_line_state(x), kl, scheme=scheme) / h
        d = h / 16
        ref = np.zeros((5, n))
        for i in range(n):
            xs = x[6 + i] + d * np.arange(-3, 4)
            Fs = np.array([po.point_flux(q, [1.0, 0, 0]) for q in _line_state(xs).T])  # (7,5)
            ref[:, i] = [po.d6(Fs[:, m].copy()) / d for m in range(5)]
        errs.append(np.abs(D - ref).max())
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    assert o1 > 4.5 and o2 > 4.8, (errs, o1, o2)


def test_inviscid_line_supersonic_uses_left_states_only(po):
    """Upwinding (reading U2): with every eigenvalue > 0 the numerical flux f_{i+1/2} may depend only on
    the left-biased stencil i-2..i+2, so D_i must not change when Q_{i+3} is perturbed in the WENO part.
    (Q_{i+3} still enters Eq. 19's central correction through F_{i+3}; compare against that part alone.)"""
    n = 8
    x = 0.3 * np.arange(-6, n + 6)
    Ql = _line_state(x)
    Ql[1] += 2.5 * Ql[0]  # add u = 2.5 -> supersonic along +x
    Ql[4] = Ql[4] + 0.5 * (Ql[1] ** 2 - (Ql[1] - 2.5 * Ql[0]) ** 2) / Ql[0]
    kl = np.zeros((3, n + 12))
    kl[0] = 1.0
    D0 = po.inviscid_line(Ql, kl)
    i = 3
    Qp = Ql.copy()
    Qp[:, 6 + i + 3] *= 1.01
    D1 = po.inviscid_line(Qp, kl)
    dF = po.point_flux(Qp[:, 6 + i + 3], [1.0, 0, 0]) - po.point_flux(Ql[:, 6 + i + 3], [1.0, 0, 0])
    assert np.allclose(D1[:, i] - D0[:, i], 19.0 / 3840.0 * dF, rtol=0, atol=1e-13)
    # and perturbing Q_{i-3} (which is inside the left-biased stencil of f_{i-1/2}) does change it beyond Eq. 19's term
    Qm = Ql.copy()
    Qm[:, 6 + i - 3] *= 1.01
    D2 = po.inviscid_line(Qm, kl)
    dFm = po.point_flux(Qm[:, 6 + i - 3], [1.0, 0, 0]) - po.point_flux(Ql[:, 6 + i - 3], [1.0, 0, 0])
    assert np.abs(D2[:, i] - D0[:, i] + 19.0 / 3840.0 * dFm).max() > 1e-6


# ------------------------------------------------------------------------------------------------
# Viscous point routines (Eqs. 5, 6, 21)
# ------------------------------------------------------------------------------------------------
def test_grad_point_chain_rule(po):
    # Cartesian stretched grid: khat^d_c = delta_dc * (product of the other two spacings), J = 1/(hx hy hz)
    hx, hy, hz = 0.5, 0.25, 2.0
    kh = np.diag([hy * hz, hx * hz, hx * hy])
    J = 1.0 / (hx * hy * hz)
    dphi = rng.normal(size=(3, 4))  # d phi / d xi^d
    g = po.grad_point(dphi, kh, J)
    assert np.allclose(g, dphi / np.array([[hx], [hy], [hz]]), rtol=1e-14)


def test_visc_flux_pure_shear_and_dilatation(po):
    mu, kappa = 0.01, 0.05
    # pure shear du/dy = s: tau_xy = mu s ; flux along y: (0, tau_xy, 0, 0, u tau_xy)
    g = np.zeros((3, 4))
    g[1, 0] = 2.0
    Fv = po.visc_flux_point([3.0, 0, 0], g, [0, 1.0, 0], mu, kappa)
    assert np.allclose(Fv, [0, mu * 2.0, 0, 0, 3.0 * mu * 2.0], atol=1e-16)
    # pure dilatation du/dx = a: tau_xx = (2 - 2/3) mu a, tau_yy = tau_zz = -2/3 mu a ; heat flux along x
    g = np.zeros((3, 4))
    g[0, 0] = 1.5
    g[0, 3] = -4.0
    Fv = po.visc_flux_point([0.0, 0, 0], g, [1.0, 0, 0], mu, kappa)
    assert np.allclose(Fv, [0, 4.0 / 3.0 * mu * 1.5, 0, 0, kappa * -4.0], atol=1e-16)
    Fv = po.visc_flux_point([0.0, 0, 0], g, [0, 0, 1.0], mu, kappa)
    assert np.allclose(Fv, [0, 0, 0, -2.0 / 3.0 * mu * 1.5, 0.0], atol=1e-16)
    # trace of tau vanishes (Stokes hypothesis, lambda = -2/3 mu): probe with three unit directions
    g = np.zeros((3, 4))
    g[:, :3] = rng.normal(size=(3, 3))
    tr = sum(po.visc_flux_point([0, 0, 0], g, np.eye(3)[c], mu, kappa)[1 + c] for c in range(3))
    assert abs(tr) < 1e-16


def test_sutherland_law_closed_forms(po):
    """mu(T) = T^(3/2) (1 + S)/(T + S) in the reference scales (U11): mu(1) = 1 for every S, hand values,
    the classical dimensional ratio for air, and S <= 0 switches it off (constant mu = 1)."""
    for S in (0.1, 0.4, 110.4 / 288.15, 2.0):
        assert abs(po.sutherland_mu(1.0, S) - 1.0) < 1e-15
    assert abs(po.sutherland_mu(2.0, 0.4) - 2.0 ** 1.5 * 1.4 / 2.4) < 1e-15
    assert abs(po.sutherland_mu(0.25, 0.5) - 0.125 * 1.5 / 0.75) < 1e-15
    # air, T_inf = 273.15 K, S = 110.4 K: mu(373.15 K)/mu(273.15 K) = (373.15/273.15)^1.5 (273.15 + 110.4)/(373.15 + 110.4)
    S = 110.4 / 273.15
    want = (373.15 / 273.15) ** 1.5 * (273.15 + 110.4) / (373.15 + 110.4)
    assert abs(po.sutherland_mu(373.15 / 273.15, S) / want - 1) < 1e-14
    for T in (0.3, 1.0, 4.0):
        assert po.sutherland_mu(T, 0.0) == 1.0 and po.sutherland_mu(T, -1.0) == 1.0
    # monotone in T
    Ts = np.linspace(0.2, 5.0, 50)
    mus = np.array([po.sutherland_mu(t, 0.4) for t in Ts])
    assert (np.diff(mus) > 0).all()
