"""Pins for the oracle's ISWIG switching function (Eq. 9) and the surface terms of the gradient (Eq. 14: z^T (grad B^T) q
and q^T (grad A) q / 2f, including A_kk through S_k).  Checked against scipy's erf on hand-built geometry, limits, and
central differences of the oracle's own (already pinned) energies B z . q and q . A q when single points and single
atoms are displaced."""
import copy

import numpy as np
import pytest
from scipy.special import erf

import oracle
import synth


def richardson(f, h):
    d1 = (f(h) - f(-h)) / (2 * h)
    d2 = (f(h / 2) - f(-h / 2)) / h
    return (4 * d2 - d1) / 3


def test_switching_two_atoms_closed_form_and_limits():
    # one point owned by atom 0, one other atom of radius R at distance d: S = 1 - [erf(z (R - d)) + erf(z (R + d))]/2
    zeta, R = 2.5, 3.0
    for d in (0.5, 2.9, 3.0, 3.4, 8.0):
        s = synth.Surface(xyz=np.array([[d, 0.0, 0.0]]), zeta=np.array([zeta]), switch=np.ones(1), atom=np.zeros(1, np.int32))
        atoms = np.array([[50.0, 0, 0], [0.0, 0, 0]])
        S = oracle.switching(s, atoms, np.array([1.0, R]))[0]
        assert S == pytest.approx(1 - 0.5 * (erf(zeta * (R - d)) + erf(zeta * (R + d))), rel=1e-14, abs=1e-300)
    assert S == pytest.approx(1.0, abs=1e-15)                       # far outside every other sphere
    s = synth.Surface(xyz=np.array([[0.5, 0.0, 0.0]]), zeta=np.array([zeta]), switch=np.ones(1), atom=np.zeros(1, np.int32))
    assert oracle.switching(s, atoms, np.array([1.0, R]))[0] < 1e-8   # deep inside: below the paper's 1e-8 screening
    s = synth.Surface(xyz=np.array([[3.0, 0.0, 0.0]]), zeta=np.array([40.0]), switch=np.ones(1), atom=np.zeros(1, np.int32))
    assert oracle.switching(s, atoms, np.array([1.0, R]))[0] == pytest.approx(0.5, rel=1e-12)   # on the sphere: 1/2
    # the owner is skipped, the others multiply
    s = synth.Surface(xyz=np.array([[3.2, 0.1, 0.0]]), zeta=np.array([1.1]), switch=np.ones(1), atom=np.array([2], np.int32))
    atoms = np.array([[0.0, 0, 0], [5.0, 1.0, 0], [3.0, 0.0, 0.5]])
    rad = np.array([3.0, 2.5, 2.0])
    d = np.linalg.norm(s.xyz[0] - atoms, axis=1)
    sw = 1 - 0.5 * (erf(1.1 * (rad - d)) + erf(1.1 * (rad + d)))
    assert oracle.switching(s, atoms, rad)[0] == pytest.approx(sw[0] * sw[1], rel=1e-14)


@pytest.fixture(scope="module")
def small():
    w = synth.make_workload(0, n_atoms=6, n_pts=14)
    rad = synth.cavity_radii(w.elements)
    z = synth.nuclear_charges(w.elements)
    return w, rad, z


def surface_energy(surface, atom_xyz, rad, z, q, f):
    s = copy.copy(surface)
    s.switch = oracle.switching(surface, atom_xyz, rad)
    u = oracle.nuclear_potential(s, atom_xyz, z)
    return float(u @ q + q @ oracle.amatvec(s, q) / (2 * f))


def test_surface_gradient_vs_finite_differences(small):
    w, rad, z = small
    s, f = w.surface, (78.39 - 1) / 78.39
    q = w.q * 10
    gp, ga = oracle.surface_gradient(s, w.atom_xyz, rad, z, q, f)
    for k in (0, s.M // 2, s.M - 1):
        for x in range(3):
            def e(h):
                s2 = copy.copy(s)
                s2.xyz = s.xyz.copy()
                s2.xyz[k, x] += h
                return surface_energy(s2, w.atom_xyz, rad, z, q, f)
            assert gp[k, x] == pytest.approx(richardson(e, 2e-3), rel=1e-8, abs=1e-10)
    for J in (0, len(z) - 1):
        for x in range(3):
            def e(h):
                a = w.atom_xyz.copy()
                a[J, x] += h
                return surface_energy(s, a, rad, z, q, f)
            assert ga[J, x] == pytest.approx(richardson(e, 2e-3), rel=1e-8, abs=1e-10)
    # translating everything changes nothing
    np.testing.assert_allclose(gp.sum(0) + ga.sum(0), 0.0, atol=1e-10)


def test_surface_gradient_two_body_closed_forms():
    # one nucleus and one point: dE/dr = z q d/dr[erf(zeta r)/r]; two points: (1/f) q1 q2 d/dr[erf(z' r)/r]
    zeta, r, zq, qq = 1.7, 1.3, 3.0, 0.4
    s = synth.Surface(xyz=np.array([[r, 0.0, 0.0]]), zeta=np.array([zeta]), switch=np.ones(1), atom=np.zeros(1, np.int32))
    gp, ga = oracle.surface_gradient(s, np.zeros((1, 3)), np.array([2.0]), np.array([zq]), np.array([qq]), 1.0)
    g = 2 * zeta / np.sqrt(np.pi) * np.exp(-(zeta * r) ** 2) / r - erf(zeta * r) / r ** 2
    assert gp[0, 0] == pytest.approx(zq * qq * g, rel=1e-13) and ga[0, 0] == pytest.approx(-zq * qq * g, rel=1e-13)
    s = synth.Surface(xyz=np.array([[0.0, 0, 0], [0.0, r, 0.0]]), zeta=np.array([zeta, 2.9]), switch=np.ones(2), atom=np.zeros(2, np.int32))
    gp, ga = oracle.surface_gradient(s, np.array([[99.0, 0, 0]]), np.array([1.0]), np.array([0.0]), np.array([qq, -0.7]), 0.8)
    zp = zeta * 2.9 / np.hypot(zeta, 2.9)
    g = 2 * zp / np.sqrt(np.pi) * np.exp(-(zp * r) ** 2) / r - erf(zp * r) / r ** 2
    assert gp[1, 1] == pytest.approx(qq * -0.7 / 0.8 * g, rel=1e-12) and gp[0, 1] == pytest.approx(-gp[1, 1], rel=1e-12)
