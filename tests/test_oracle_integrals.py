"""Pins for the oracle's primitive smeared-charge integrals (oracle/pcm_oracle.c: os_tables,
orc_prim_integral, orc_prim_block) -- Eq. 6 / Eq. 12 of PAPER.md (lines 41-44, 72-77).

The paper gives only the definition  [chi_a| erf(zeta|r-C|)/|r-C| |chi_b]; SURVEY.md 8(c2) fixes the
Obara-Saika reading.  Every pin below reaches the same number by a route that shares nothing with
the oracle's recursion:
  * closed-form s-s with libm erf,
  * brute-force 3-D Gauss-Hermite quadrature of the defining integral,
  * an independent McMurchie-Davidson evaluation written here with scipy's incomplete gamma function,
  * the zeta -> infinity (point charge) and far-field (1/R) limits,
  * finite-difference derivative relations of the closed-form s-s integral,
  * a 1-D radial quadrature for the same-centre case,
  * bra/ket exchange symmetry, recursion-path independence, and the stored worked example.
"""
import itertools
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_checkvalues.json")))

CART = {0: [(0, 0, 0)], 1: [(1, 0, 0), (0, 1, 0), (0, 0, 1)],
        2: [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]}


# ----------------------------------------------------------------------------- independent routes
def ss_closed_form(alpha, A, beta, B, zeta, C):
    """(2 pi/p) K_AB zeta/sqrt(p+zeta^2) F_0(T), F_0 through libm erf."""
    A, B, C = map(np.asarray, (A, B, C))
    p = alpha + beta
    P = (alpha * A + beta * B) / p
    K = math.exp(-alpha * beta / p * float(np.dot(A - B, A - B)))
    rho = p * zeta * zeta / (p + zeta * zeta) if math.isfinite(zeta) else p
    T = rho * float(np.dot(P - C, P - C))
    F0 = 1.0 if T < 1e-300 else 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))
    w = zeta / math.sqrt(p + zeta * zeta) if math.isfinite(zeta) else 1.0
    return 2.0 * math.pi / p * K * w * F0


def quadrature(a, alpha, A, b, beta, B, zeta, C, n=80):
    """3-D Gauss-Hermite product rule centred at P with weight exp(-p r_P^2): the defining integral."""
    A, B, C = map(lambda v: np.asarray(v, float), (A, B, C))
    p = alpha + beta
    P = (alpha * A + beta * B) / p
    K = math.exp(-alpha * beta / p * float(np.dot(A - B, A - B)))
    x, w = np.polynomial.hermite.hermgauss(n)
    s = 1.0 / math.sqrt(p)
    X, Y, Z = np.meshgrid(P[0] + s * x, P[1] + s * x, P[2] + s * x, indexing="ij")
    W = w[:, None, None] * w[None, :, None] * w[None, None, :] * s ** 3
    r = np.sqrt((X - C[0]) ** 2 + (Y - C[1]) ** 2 + (Z - C[2]) ** 2)
    with np.errstate(divide="ignore", invalid="ignore"):
        op = np.where(r > 1e-14, special.erf(zeta * r) / r, 2.0 * zeta / math.sqrt(math.pi))
    poly = ((X - A[0]) ** a[0] * (Y - A[1]) ** a[1] * (Z - A[2]) ** a[2] *
            (X - B[0]) ** b[0] * (Y - B[1]) ** b[1] * (Z - B[2]) ** b[2])
    return K * float(np.sum(W * poly * op))


def boys_gamma(n, T):
    if T < 1e-13:
        return 1.0 / (2 * n + 1) - T / (2 * n + 3)
    return special.gamma(n + 0.5) * special.gammainc(n + 0.5, T) / (2.0 * T ** (n + 0.5))


def md_reference(a, alpha, A, b, beta, B, zeta, C):
    """McMurchie-Davidson: (2 pi/p) sqrt(rho/p) sum_tuv E_tuv R_tuv, rho inside R only;
    E by the standard two-index recursion, R by the standard auxiliary recursion, Boys by scipy."""
    A, B, C = map(lambda v: np.asarray(v, float), (A, B, C))
    p = alpha + beta
    P = (alpha * A + beta * B) / p
    mu = alpha * beta / p
    rho = p * zeta * zeta / (p + zeta * zeta) if math.isfinite(zeta) else p
    PC = P - C
    T = rho * float(np.dot(PC, PC))

    def E(i, j, t, Qx, PAx, PBx):
        if t < 0 or t > i + j:
            return 0.0
        if i == j == t == 0:
            return math.exp(-mu * Qx * Qx)
        if j == 0:
            return E(i - 1, j, t - 1, Qx, PAx, PBx) / (2 * p) + PAx * E(i - 1, j, t, Qx, PAx, PBx) + \
                (t + 1) * E(i - 1, j, t + 1, Qx, PAx, PBx)
        return E(i, j - 1, t - 1, Qx, PAx, PBx) / (2 * p) + PBx * E(i, j - 1, t, Qx, PAx, PBx) + \
            (t + 1) * E(i, j - 1, t + 1, Qx, PAx, PBx)

    def R(t, u, v, n):
        if t < 0 or u < 0 or v < 0:
            return 0.0
        if t == u == v == 0:
            return (-2.0 * rho) ** n * boys_gamma(n, T)
        if t > 0:
            return (t - 1) * R(t - 2, u, v, n + 1) + PC[0] * R(t - 1, u, v, n + 1)
        if u > 0:
            return (u - 1) * R(t, u - 2, v, n + 1) + PC[1] * R(t, u - 1, v, n + 1)
        return (v - 1) * R(t, u, v - 2, n + 1) + PC[2] * R(t, u, v - 1, n + 1)

    tot = 0.0
    for t in range(a[0] + b[0] + 1):
        Ex = E(a[0], b[0], t, A[0] - B[0], P[0] - A[0], P[0] - B[0])
        for u in range(a[1] + b[1] + 1):
            Ey = E(a[1], b[1], u, A[1] - B[1], P[1] - A[1], P[1] - B[1])
            for v in range(a[2] + b[2] + 1):
                Ez = E(a[2], b[2], v, A[2] - B[2], P[2] - A[2], P[2] - B[2])
                tot += Ex * Ey * Ez * R(t, u, v, 0)
    return 2.0 * math.pi / p * math.sqrt(rho / p) * tot


def random_case(rng, spread=1.0):
    A = rng.normal(0, spread, 3)
    B = A + rng.normal(0, 0.6, 3)
    C = A + rng.normal(0, 1.5 * spread, 3)
    alpha, beta = np.exp(rng.uniform(math.log(0.3), math.log(4.0), 2))
    zeta = math.exp(rng.uniform(math.log(0.4), math.log(1.2)))
    return A, B, C, float(alpha), float(beta), zeta


# ----------------------------------------------------------------------------- tests
def test_ss_closed_form(orc):
    rng = np.random.default_rng(11)
    for _ in range(200):
        A, B, C, al, be, ze = random_case(rng, 2.0)
        ze *= rng.choice([0.2, 1.0, 5.0, 40.0])
        got = orc.prim_integral((0, 0, 0), al, A, (0, 0, 0), be, B, ze, C)
        assert got == pytest.approx(ss_closed_form(al, A, be, B, ze, C), rel=3e-15, abs=1e-300)


def test_ss_at_T_zero(orc):
    """C = P: (2 pi/p) K_AB zeta/sqrt(p+zeta^2)"""
    A, B = np.array([0.1, -0.2, 0.3]), np.array([0.7, 0.4, -0.5])
    al, be, ze = 1.1, 0.7, 2.3
    p = al + be
    P = (al * A + be * B) / p
    K = math.exp(-al * be / p * np.dot(A - B, A - B))
    got = orc.prim_integral((0, 0, 0), al, A, (0, 0, 0), be, B, ze, P)
    assert got == pytest.approx(2 * math.pi / p * K * ze / math.sqrt(p + ze * ze), rel=1e-15)


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (0, 2), (2, 1), (1, 2), (2, 2)])
def test_brute_force_quadrature(orc, la, lb):
    """the defining 3-D integral, all Cartesian components of the class; zeta^2 <~ 2p so 80 nodes suffice"""
    rng = np.random.default_rng(100 + 10 * la + lb)
    for _ in range(2):
        A, B, C, al, be, ze = random_case(rng)
        ze = min(ze, math.sqrt(1.5 * (al + be)))
        blk = orc.prim_block(la, al, A, lb, be, B, ze, C)
        for ia, a in enumerate(CART[la]):
            for ib, b in enumerate(CART[lb]):
                ref = quadrature(a, al, A, b, be, B, ze, C)
                assert blk[ia, ib] == pytest.approx(ref, rel=2e-12, abs=2e-14), (a, b)


def test_against_independent_mcmurchie_davidson(orc):
    """all (a,b) up to d,d on random geometries, including tight charges (large zeta) and large T"""
    rng = np.random.default_rng(5)
    for trial in range(40):
        A, B, C, al, be, ze = random_case(rng, 1.5)
        ze *= [1.0, 6.0, 0.3, 25.0][trial % 4]
        if trial % 5 == 0:
            C = C + np.array([9.0, -7.0, 5.0])  # large T: exercises the T >= 35 Boys branch
        for la, lb in itertools.product(range(3), range(3)):
            blk = orc.prim_block(la, al, A, lb, be, B, ze, C)
            scale = abs(orc.prim_integral((0, 0, 0), al, A, (0, 0, 0), be, B, ze, C))
            for ia, a in enumerate(CART[la]):
                for ib, b in enumerate(CART[lb]):
                    ref = md_reference(a, al, A, b, be, B, ze, C)
                    assert blk[ia, ib] == pytest.approx(ref, rel=2e-12, abs=3e-14 * scale), (trial, a, b)


def test_zeta_to_infinity_is_point_charge(orc):
    """zeta -> infinity: rho -> p, sqrt(rho/p) -> 1: the textbook nuclear-attraction integral"""
    rng = np.random.default_rng(7)
    for _ in range(10):
        A, B, C, al, be, _ = random_case(rng)
        for la, lb in [(0, 0), (1, 0), (1, 1), (2, 1), (2, 2)]:
            a, b = CART[la][-1], CART[lb][0]
            pc = md_reference(a, al, A, b, be, B, math.inf, C)
            prev = None
            for ze in (1e2, 1e4, 1e6):
                got = orc.prim_integral(a, al, A, b, be, B, ze, C)
                err = abs(got - pc)
                if prev is not None:
                    assert err <= prev + 1e-13 * abs(pc) + 1e-15  # monotone approach
                prev = err
            assert got == pytest.approx(pc, rel=1e-10, abs=1e-13)


def test_zeta_to_infinity_stored_sequence(orc):
    e = GOLD["worked_example"]
    for row in GOLD["zeta_to_infinity_ss"]:
        if row["zeta"] == "point_charge":
            ref = ss_closed_form(e["alpha"], e["A"], e["beta"], e["B"], math.inf, e["C"])
            assert ref == pytest.approx(row["value"], rel=2e-12)
        else:
            got = orc.prim_integral((0, 0, 0), e["alpha"], np.array(e["A"]), (0, 0, 0), e["beta"], np.array(e["B"]),
                                    row["zeta"], np.array(e["C"]))
            assert got == pytest.approx(row["value"], rel=2e-12)


def test_far_field_is_overlap_over_distance(orc):
    """T >~ 50: erf = 1, ss -> (pi/p)^{3/2} K_AB / |P - C|; px s -> S_ps/R + S_ss * d/dAx-type dipole term
    is checked through the general multipole identity for the s-s case only (the p, d cases are covered by
    the independent MD route at large T)."""
    A, B = np.array([0.0, 0.1, -0.2]), np.array([0.4, -0.3, 0.5])
    al, be, ze = 0.8, 1.3, 3.0
    p = al + be
    P = (al * A + be * B) / p
    K = math.exp(-al * be / p * np.dot(A - B, A - B))
    for R in (6.0, 15.0, 80.0):
        C = P + R * np.array([2.0, -1.0, 2.0]) / 3.0
        got = orc.prim_integral((0, 0, 0), al, A, (0, 0, 0), be, B, ze, C)
        assert got == pytest.approx((math.pi / p) ** 1.5 * K / R, rel=1e-14)


def test_derivative_relation_by_finite_differences(orc):
    """[p_x s|J] = (1/2 alpha) d/dA_x [s s|J]  and  [s p_y|J] = (1/2 beta) d/dB_y [s s|J]  (coarse, ~1e-8)"""
    A, B, C = np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), np.array([0.9, 0.8, -0.7])
    al, be, ze = 0.9, 1.4, 1.7
    h = 1e-3

    def d(which, axis):
        def f(s):
            A2, B2 = A.copy(), B.copy()
            (A2 if which == 0 else B2)[axis] += s
            return ss_closed_form(al, A2, be, B2, ze, C)
        d1 = (f(h) - f(-h)) / (2 * h)
        d2 = (f(2 * h) - f(-2 * h)) / (4 * h)
        return (4 * d1 - d2) / 3  # Richardson

    for ax in range(3):
        a = [0, 0, 0]
        a[ax] = 1
        got = orc.prim_integral(tuple(a), al, A, (0, 0, 0), be, B, ze, C)
        assert got == pytest.approx(d(0, ax) / (2 * al), rel=1e-8)
        got = orc.prim_integral((0, 0, 0), al, A, tuple(a), be, B, ze, C)
        assert got == pytest.approx(d(1, ax) / (2 * be), rel=1e-8)


def test_same_centre_radial_quadrature(orc):
    """A = B = C: [a|J|b] = angular constant x int_0^inf r^{L+1} exp(-p r^2) erf(zeta r) dr  (scipy quad)"""
    O = np.zeros(3)
    al, be, ze = 0.7, 1.9, 1.3
    p = al + be

    def radial(k):  # int r^k e^{-p r^2} erf(zeta r) dr
        return integrate.quad(lambda r: r ** k * math.exp(-p * r * r) * math.erf(ze * r), 0, np.inf,
                              epsabs=0, epsrel=1e-13)[0]
    # <x^2i y^2j z^2k> over the unit sphere = 4 pi (2i-1)!!(2j-1)!!(2k-1)!!/(2n+1)!!, n = i+j+k
    assert orc.prim_integral((0, 0, 0), al, O, (0, 0, 0), be, O, ze, O) == pytest.approx(4 * math.pi * radial(1), rel=1e-12)
    assert orc.prim_integral((1, 0, 0), al, O, (1, 0, 0), be, O, ze, O) == pytest.approx(4 * math.pi / 3 * radial(3), rel=1e-12)
    assert orc.prim_integral((2, 0, 0), al, O, (0, 0, 0), be, O, ze, O) == pytest.approx(4 * math.pi / 3 * radial(3), rel=1e-12)
    assert orc.prim_integral((2, 0, 0), al, O, (2, 0, 0), be, O, ze, O) == pytest.approx(4 * math.pi * 3 / 15 * radial(5), rel=1e-12)
    assert orc.prim_integral((2, 0, 0), al, O, (0, 2, 0), be, O, ze, O) == pytest.approx(4 * math.pi / 15 * radial(5), rel=1e-12)
    assert orc.prim_integral((1, 1, 0), al, O, (1, 1, 0), be, O, ze, O) == pytest.approx(4 * math.pi / 15 * radial(5), rel=1e-12)
    # odd integrands vanish
    assert abs(orc.prim_integral((1, 0, 0), al, O, (0, 0, 0), be, O, ze, O)) < 1e-16
    assert abs(orc.prim_integral((1, 1, 0), al, O, (0, 1, 0), be, O, ze, O)) < 1e-16


def test_bra_ket_exchange_symmetry(orc):
    rng = np.random.default_rng(3)
    for _ in range(20):
        A, B, C, al, be, ze = random_case(rng)
        for la, lb in itertools.product(range(3), range(3)):
            ab = orc.prim_block(la, al, A, lb, be, B, ze, C)
            ba = orc.prim_block(lb, be, B, la, al, A, ze, C)
            np.testing.assert_allclose(ab, ba.T, rtol=1e-12, atol=1e-15)


def test_recursion_path_independence(orc):
    """lowering the first or the last non-zero Cartesian power in the vertical/horizontal steps"""
    rng = np.random.default_rng(4)
    for _ in range(20):
        A, B, C, al, be, ze = random_case(rng)
        for la, lb in itertools.product(range(3), range(3)):
            np.testing.assert_allclose(orc.prim_block(la, al, A, lb, be, B, ze, C, path=0),
                                       orc.prim_block(la, al, A, lb, be, B, ze, C, path=1), rtol=1e-12, atol=1e-15)


def test_worked_example_stored_values(orc):
    e = GOLD["worked_example"]
    for row in e["integrals"]:
        got = orc.prim_integral(tuple(row["a"]), e["alpha"], np.array(e["A"]), tuple(row["b"]), e["beta"],
                                np.array(e["B"]), e["zeta"], np.array(e["C"]))
        assert got == pytest.approx(row["value"], rel=2e-12), row
        # and the same number by quadrature (the stored values are a convenience, this is the authority)
        ref = quadrature(row["a"], e["alpha"], e["A"], row["b"], e["beta"], e["B"], e["zeta"], e["C"], n=90)
        assert got == pytest.approx(ref, rel=1e-12, abs=1e-14), row


def test_prim_block_matches_prim_integral(orc):
    rng = np.random.default_rng(8)
    A, B, C, al, be, ze = random_case(rng)
    for la, lb in itertools.product(range(3), range(3)):
        blk = orc.prim_block(la, al, A, lb, be, B, ze, C)
        for ia, a in enumerate(CART[la]):
            for ib, b in enumerate(CART[lb]):
                assert blk[ia, ib] == orc.prim_integral(a, al, A, b, be, B, ze, C)
