"""Pins for the oracle's A matrix, A.q, randomized block-Jacobi and PCG
(oracle/pcm_oracle.c: orc_a_entry, orc_amatrix, orc_amatvec, orc_pivot_order, orc_rbj_build, orc_pcg)
-- Eq. 2, 3, 8 and section 4b, readings R1 and R5.

Pins: numpy/scipy re-evaluation of Eq. 2 with scipy.special.erf, the 1/r and Boys-F_0 forms, the
Gaussian self-energy by 1-D quadrature (decides the sqrt(2/pi) reading of the garbled Eq. 3), symmetry,
positive definiteness, dense LAPACK solves, block size 1 == Jacobi, block size M == one
step, RBJ needs fewer steps than Jacobi for M >~ 1000.
"""
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_checkvalues.json")))


@pytest.fixture(scope="module")
def surf600():
    w = synth.make_workload(1, n_atoms=12, with_density=False, seed=5)
    return w.surface


@pytest.fixture(scope="module")
def surf2k():
    s, q, qt = synth.make_solver_points(2500, seed=1004)
    return s, q, qt


def numpy_A(s):
    d = s.xyz[:, None, :] - s.xyz[None, :, :]
    r = np.sqrt((d * d).sum(-1))
    zp = s.zeta[:, None] * s.zeta[None, :] / np.sqrt(s.zeta[:, None] ** 2 + s.zeta[None, :] ** 2)
    with np.errstate(divide="ignore", invalid="ignore"):
        A = special.erf(zp * r) / r
    A[np.diag_indices(s.M)] = s.zeta * math.sqrt(2 / math.pi) / s.switch
    return A


def test_amatrix_is_eq2_eq3(orc, surf600):
    A = orc.amatrix(surf600)
    np.testing.assert_allclose(A, numpy_A(surf600), rtol=4e-16, atol=0)
    np.testing.assert_array_equal(A, A.T)
    i, j = 5, 77
    assert orc.a_entry(surf600, i, j) == A[i, j]


def test_diagonal_is_gaussian_self_energy(orc):
    """Eq. 3 as printed (zeta/sqrt(2 pi)) is garbled: the Coulomb self-energy of a unit Gaussian charge
    (zeta^2/pi)^{3/2} exp(-zeta^2 r^2), i.e. the r -> 0 limit of Eq. 2 with zeta_k = zeta_l, is
    zeta sqrt(2/pi).  Quadrature: E = int_0^inf rho(r) phi(r) 4 pi r^2 dr, phi = erf(zeta r)/r."""
    z = GOLD["a_diagonal"]["zeta"]
    E = integrate.quad(lambda r: (z * z / math.pi) ** 1.5 * math.exp(-z * z * r * r) * math.erf(z * r) / r * 4 * math.pi * r * r,
                       0, np.inf, epsabs=0, epsrel=1e-13)[0]
    s = synth.Surface(np.zeros((1, 3)), np.array([z]), np.array([1.0]), np.zeros(1, np.int32))
    assert orc.a_entry(s, 0, 0) == pytest.approx(E, rel=1e-12)
    assert orc.a_entry(s, 0, 0) == pytest.approx(GOLD["a_diagonal"]["sqrt_2_over_pi"], rel=1e-7)
    # r -> 0 limit of the off-diagonal formula with equal exponents
    s2 = synth.Surface(np.array([[0, 0, 0], [1e-9, 0, 0]]), np.array([z, z]), np.ones(2), np.zeros(2, np.int32))
    assert orc.a_entry(s2, 0, 1) == pytest.approx(E, rel=1e-9)
    # switching function divides the diagonal only
    s3 = synth.Surface(np.zeros((1, 3)), np.array([z]), np.array([0.25]), np.zeros(1, np.int32))
    assert orc.a_entry(s3, 0, 0) == pytest.approx(4 * E, rel=1e-12)


def test_offdiagonal_limits(orc):
    """far: erf = 1 -> 1/r for zeta' r > 6;  general: (2 zeta'/sqrt pi) F_0(zeta'^2 r^2);  coincident: 2 zeta'/sqrt pi"""
    zi, zj = 4.1, 5.6
    zp = zi * zj / math.hypot(zi, zj)
    for r in (0.05, 0.4, 1.0, 2.0, 7.5, 40.0):
        s = synth.Surface(np.array([[0.3, 0.2, 0.1], [0.3 + r, 0.2, 0.1]]), np.array([zi, zj]), np.ones(2), np.zeros(2, np.int32))
        a = orc.a_entry(s, 0, 1)
        T = (zp * r) ** 2
        F0 = special.gamma(0.5) * special.gammainc(0.5, T) / (2 * math.sqrt(T))
        assert a == pytest.approx(2 * zp / math.sqrt(math.pi) * F0, rel=1e-14)
        if zp * r > 6:
            assert a == pytest.approx(1 / r, rel=1e-16)
        assert a == orc.a_entry(s, 1, 0)
    s = synth.Surface(np.zeros((2, 3)), np.array([zi, zj]), np.ones(2), np.zeros(2, np.int32))
    assert orc.a_entry(s, 0, 1) == pytest.approx(2 * zp / math.sqrt(math.pi), rel=1e-15)


def test_A_positive_definite(orc, surf2k):
    s = surf2k[0]
    A = orc.amatrix(s)
    np.linalg.cholesky(A)  # raises if not SPD
    assert np.linalg.eigvalsh(A)[0] > 0


def test_amatvec_is_dense_product(orc, surf2k):
    s, q, _ = surf2k
    A = numpy_A(s)
    y = orc.amatvec(s, q)
    ref = np.array([math.fsum(A[i] * q) for i in range(s.M)])
    np.testing.assert_allclose(y, ref, rtol=1e-13, atol=1e-15)
    rows = np.array([7, 0, s.M - 1, 1234])
    np.testing.assert_array_equal(orc.amatvec(s, q, rows), y[rows])


# ----------------------------------------------------------------------------- RBJ
def test_pivot_order_is_a_seeded_permutation(orc):
    p = orc.pivot_order(42, 1000)
    assert sorted(p.tolist()) == list(range(1000))
    np.testing.assert_array_equal(p, orc.pivot_order(42, 1000))
    assert (p != orc.pivot_order(43, 1000)).any()
    # splitmix64 finaliser restated: key_i = mix(seed + (i+1) * golden)
    mask = (1 << 64) - 1

    def mix(z):
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
        return z ^ (z >> 31)
    keys = [mix((42 + (i + 1) * 0x9E3779B97F4A7C15) & mask) for i in range(1000)]
    assert p.tolist() == sorted(range(1000), key=lambda i: (keys[i], i))


@pytest.mark.parametrize("l", [1, 7, 64])
def test_rbj_blocks(orc, surf600, l):
    s = surf600
    M = s.M
    piv = orc.pivot_order(9, M)
    order, bstart, inv = orc.rbj_build(s, l, piv)
    assert sorted(order.tolist()) == list(range(M))              # blocks partition {0..M-1}
    sizes = np.diff(bstart)
    assert (sizes[:-1] == l).all() and 0 < sizes[-1] <= l         # all but the last have size l
    A = numpy_A(s)
    assigned = np.zeros(M, bool)
    pos = 0
    ioff = 0
    for b in range(len(sizes)):
        idx = order[bstart[b]:bstart[b + 1]]
        while assigned[piv[pos]]:
            pos += 1
        k = piv[pos]
        assert idx[0] == k                                        # pivot = first unassigned in the pivot order
        # the block is the pivot plus the l-1 unassigned indices with the largest A_kj
        rest = np.flatnonzero(~assigned)
        rest = rest[rest != k]
        chosen = idx[1:]
        if len(chosen) and len(rest) > len(chosen):
            excluded = np.setdiff1d(rest, chosen)
            assert A[k, chosen].min() >= A[k, excluded].max()
        assert (np.diff(A[k, chosen]) <= 0).all()                 # stored by descending magnitude
        assigned[idx] = True
        n = len(idx)
        Minv = inv[ioff:ioff + n * n].reshape(n, n)
        np.testing.assert_allclose(Minv @ A[np.ix_(idx, idx)], np.eye(n), atol=1e-10)
        ioff += n * n


# ----------------------------------------------------------------------------- PCG
def test_pcg_matches_lapack(orc, surf2k):
    s, _, q_true = surf2k
    A = numpy_A(s)
    b = A @ q_true
    x_ref = np.linalg.solve(A, b)
    piv = orc.pivot_order(1, s.M)
    rbj = orc.rbj_build(s, 64, piv)
    res = {}
    for name, kw in (("none", dict(precond=0)), ("jacobi", dict(precond=1)), ("rbj", dict(precond=2, rbj=rbj))):
        x, it, rr, rt = orc.pcg(s, b, 1e-10, 2000, A=A, **kw)
        assert rr <= 1e-10 and rt <= 5e-10
        np.testing.assert_allclose(x, x_ref, rtol=0, atol=1e-8)
        np.testing.assert_allclose(x, q_true, rtol=0, atol=1e-8)
        res[name] = it
    # RBJ needs fewer CG steps than Jacobi for M >~ 1000
    assert res["rbj"] < res["jacobi"]
    # on-the-fly A gives the same iteration count and solution as stored A
    x2, it2, _, _ = orc.pcg(s, b, 1e-10, 2000, precond=2, rbj=rbj)
    assert abs(it2 - res["rbj"]) <= 1
    np.testing.assert_allclose(x2, x_ref, rtol=0, atol=1e-8)


def test_block_size_one_is_jacobi(orc, surf600):
    s = surf600
    b = np.random.default_rng(0).uniform(-1, 1, s.M)
    rbj1 = orc.rbj_build(s, 1, orc.pivot_order(3, s.M))
    xj, itj, _, _, hj = orc.pcg(s, b, 1e-9, 500, precond=1, history=True)
    x1, it1, _, _, h1 = orc.pcg(s, b, 1e-9, 500, precond=2, rbj=rbj1, history=True)
    assert abs(it1 - itj) <= 1
    # identical arithmetic up to division-vs-reciprocal rounding, which CG amplifies step by step
    np.testing.assert_allclose(h1[:8], hj[:8], rtol=1e-9)
    np.testing.assert_allclose(x1, xj, rtol=0, atol=1e-8)


def test_block_size_M_converges_in_one_step(orc, surf600):
    """'when the block size is equal to the dimension of A ... CG converges in 1 step'"""
    s = surf600
    b = np.random.default_rng(1).uniform(-1, 1, s.M)
    rbjM = orc.rbj_build(s, s.M, orc.pivot_order(3, s.M))
    x, it, rr, rt = orc.pcg(s, b, 1e-8, 50, precond=2, rbj=rbjM)
    assert it == 1 and rt < 1e-8


def test_pcg_warm_start_and_history(orc, surf600):
    s = surf600
    A = numpy_A(s)
    rng = np.random.default_rng(2)
    xt = rng.uniform(-0.05, 0.05, s.M)
    b = A @ xt
    x, it, rr, rt, h = orc.pcg(s, b, 1e-8, 500, precond=1, history=True)
    assert h[0] == pytest.approx(np.linalg.norm(b), rel=1e-14)   # x0 = 0: r0 = b
    assert h[-1] == rr <= 1e-8 < h[-2]                            # stops at the first ||r|| <= tol
    x2, it2, _, _ = orc.pcg(s, b, 1e-8, 500, precond=1, x0=x)    # already converged start: zero steps
    assert it2 == 0
    x3, it3, _, _ = orc.pcg(s, b, 1e-8, 500, precond=1, x0=xt + 1e-6 * rng.normal(size=s.M))
    assert 0 < it3 < it
    # max_iter is respected and reported through the residual
    x4, it4, rr4, _ = orc.pcg(s, b, 1e-8, 3, precond=1)
    assert it4 == 3 and rr4 > 1e-8
