"""Pins for the oracle's gradient of E = v.q (the one-electron term (grad* c^T) q of Eq. 14, Eq. 22).
The analytic derivative integrals (raised / lowered Obara-Saika brackets) are checked against something else:
central differences of the oracle's own *undifferentiated* integrals (already pinned by quadrature and closed forms in
test_oracle_integrals.py), the closed-form s-s derivative with scipy's incomplete gamma function, translation
invariance and the point-charge / far-field limits."""
import copy

import numpy as np
import pytest
from scipy.special import gammainc, gamma

import oracle
import synth


def boys_scipy(n, T):
    return gamma(n + 0.5) * gammainc(n + 0.5, T) / (2 * T ** (n + 0.5))


def richardson(f, h):
    """fourth-order central difference of f at 0 with steps h and h/2"""
    d1 = (f(h) - f(-h)) / (2 * h)
    d2 = (f(h / 2) - f(-h / 2)) / h
    return (4 * d2 - d1) / 3


A = np.array([0.0, 0.0, 0.0]); B = np.array([0.5, -0.3, 0.8]); Cp = np.array([1.0, 0.7, -0.4])


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (2, 1), (1, 2), (2, 2)])
def test_primitive_derivatives_vs_finite_differences(la, lb):
    alpha, beta, zeta = 0.9, 0.6, 1.3
    dA, dB = oracle.prim_deriv(la, alpha, A, lb, beta, B, zeta, Cp)
    for x in range(3):
        e = np.zeros(3); e[x] = 1.0
        fa = richardson(lambda h: oracle.prim_block(la, alpha, A + h * e, lb, beta, B, zeta, Cp), 2e-3)
        fb = richardson(lambda h: oracle.prim_block(la, alpha, A, lb, beta, B + h * e, zeta, Cp), 2e-3)
        fc = richardson(lambda h: oracle.prim_block(la, alpha, A, lb, beta, B, zeta, Cp + h * e), 2e-3)
        np.testing.assert_allclose(dA[x], fa, rtol=0, atol=2e-10)
        np.testing.assert_allclose(dB[x], fb, rtol=0, atol=2e-10)
        np.testing.assert_allclose(-(dA[x] + dB[x]), fc, rtol=0, atol=2e-10)   # the point's derivative


def test_ss_derivative_closed_form():
    # [s|J|s] = (2 pi/p) K w F_0(rho |P-C|^2), w = zeta/sqrt(p+zeta^2); dF_0/dT = -F_1 (independent Boys via scipy)
    alpha, beta, zeta = 0.9, 0.6, 1.3
    p = alpha + beta
    Pc = (alpha * A + beta * B) / p
    K = np.exp(-alpha * beta / p * np.sum((A - B) ** 2))
    rho = p * zeta ** 2 / (p + zeta ** 2)
    T = rho * np.sum((Pc - Cp) ** 2)
    pref = 2 * np.pi / p * K * zeta / np.sqrt(p + zeta ** 2)
    dC = pref * (-boys_scipy(1, T)) * rho * 2 * (Cp - Pc)
    dA, dB = oracle.prim_deriv(0, alpha, A, 0, beta, B, zeta, Cp)
    np.testing.assert_allclose(-(dA + dB)[:, 0, 0], dC, rtol=1e-12)
    # d/dA = (alpha/p) d/dP + dK/dA:  dK/dA = -2 mu (A-B) K
    dAx = pref * (-boys_scipy(1, T)) * rho * 2 * (Pc - Cp) * alpha / p + (-2 * alpha * beta / p * (A - B)) * pref * boys_scipy(0, T)
    np.testing.assert_allclose(dA[:, 0, 0], dAx, rtol=1e-12)


@pytest.fixture(scope="module")
def small():
    w = synth.make_workload(0, with_d=True, n_atoms=5)
    return w


def energy(w, basis=None, surface=None):
    b = basis if basis is not None else w.basis
    s = surface if surface is not None else w.surface
    return float(oracle.potential(b, s, w.P) @ w.q)


def test_contracted_gradient_vs_finite_differences_of_the_energy(small):
    w = small
    gs, gp = oracle.gradient(w.basis, w.surface, w.P, w.q)
    # every angular momentum: first s, first p, first d shell, and the last shell
    ls = list(w.basis.shell_l)
    picks = sorted({ls.index(0), ls.index(1), ls.index(2), len(ls) - 1})
    for S in picks:
        for x in range(3):
            def f(h):
                b = copy.deepcopy(w.basis)
                b.shell_xyz = b.shell_xyz.copy()
                b.shell_xyz[S, x] += h
                return energy(w, basis=b)
            assert gs[S, x] == pytest.approx(richardson(f, 4e-4), rel=2e-8, abs=2e-10)
    for k in (0, w.surface.M // 2, w.surface.M - 1):
        for x in range(3):
            def f(h):
                s = copy.deepcopy(w.surface)
                s.xyz = s.xyz.copy()
                s.xyz[k, x] += h
                return energy(w, surface=s)
            assert gp[k, x] == pytest.approx(richardson(f, 4e-4), rel=2e-8, abs=2e-10)
    # translation invariance of the whole system: the gradients sum to zero
    np.testing.assert_allclose(gs.sum(0) + gp.sum(0), 0.0, atol=1e-11)
    # selections return the same rows
    gs2, gp2 = oracle.gradient(w.basis, w.surface, w.P, w.q, shells=[3, 1], points=[7, 2, 5])
    np.testing.assert_array_equal(gs2, gs[[3, 1]])
    np.testing.assert_array_equal(gp2, gp[[7, 2, 5]])


def test_gradient_is_linear_in_P_and_q(small):
    w = small
    pts = [1, 4]
    sh = [0, 2]
    g1 = oracle.gradient(w.basis, w.surface, w.P, w.q, shells=sh, points=pts)
    P2 = np.diag(np.linspace(0.1, 1.0, w.P.shape[0]))
    g2 = oracle.gradient(w.basis, w.surface, P2, w.q, shells=sh, points=pts)
    g3 = oracle.gradient(w.basis, w.surface, 2 * w.P - P2, 3 * w.q, shells=sh, points=pts)
    for a, b, c in zip(g1, g2, g3):
        np.testing.assert_allclose(c, 3 * (2 * a - b), rtol=1e-11, atol=1e-13)


def test_far_point_feels_a_point_charge(small):
    # a point far from the molecule: E -> q tr(P S)/R, so dE/dr_k -> -q N_e (r_k - R_c)/R^3 with N_e = sum P.S
    w = small
    far = synth.Surface(xyz=np.array([[400.0, 0.0, 0.0]]), zeta=np.array([4.0]), switch=np.ones(1), atom=np.zeros(1, np.int32))
    q = np.array([0.7])
    _, gp = oracle.gradient(w.basis, far, w.P, q, shells=[])
    v = oracle.potential(w.basis, far, w.P)[0]          # = N_e / R to first order
    assert gp[0, 0] == pytest.approx(-q[0] * v / 400.0, rel=2e-2)
    assert abs(gp[0, 1]) < abs(gp[0, 0]) * 0.05 and abs(gp[0, 2]) < abs(gp[0, 0]) * 0.05
