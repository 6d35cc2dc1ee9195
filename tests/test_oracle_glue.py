"""Pins for the oracle's C-PCM glue: B z (Eq. 4), the right-hand side of Eq. 1, the energy of
Eq. 13 and the dynamic CG threshold of Eq. 21.  Each check is something other than the oracle's own formula:
limits, a library special function on hand-built geometry, the stationarity identity of Eq. 13, and Eq. 21 inverted."""
import numpy as np
import pytest
from scipy.special import erf

import oracle
import synth


@pytest.fixture(scope="module")
def w0():
    return synth.make_workload(0)


def test_bz_single_nucleus_and_point_charge_limit():
    # one nucleus of charge 3 at the origin, points on the x axis: u = 3 erf(zeta d)/d (Eq. 4), -> 3/d for zeta d >> 1
    d = np.array([0.5, 1.0, 2.0, 4.0])
    xyz = np.stack([d, 0 * d, 0 * d], axis=1)
    for zeta in (0.7, 2.5, 40.0):
        s = synth.Surface(xyz=xyz, zeta=np.full(4, zeta), switch=np.ones(4), atom=np.zeros(4, np.int32))
        u = oracle.nuclear_potential(s, np.zeros((1, 3)), np.array([3.0]))
        np.testing.assert_allclose(u, 3.0 * erf(zeta * d) / d, rtol=1e-15)
    np.testing.assert_allclose(u, 3.0 / d, rtol=1e-15)            # zeta = 40: erf = 1 to fp64
    # a nucleus on a surface point: the r -> 0 limit 2 zeta/sqrt(pi), approached continuously
    s = synth.Surface(xyz=np.array([[0.0, 0, 0], [1e-7, 0, 0]]), zeta=np.array([1.3, 1.3]), switch=np.ones(2),
                      atom=np.zeros(2, np.int64))
    u = oracle.nuclear_potential(s, np.zeros((1, 3)), np.array([1.0]))
    assert u[0] == pytest.approx(2 * 1.3 / np.sqrt(np.pi), rel=1e-15)
    assert u[1] == pytest.approx(u[0], rel=1e-12)


def test_bz_is_linear_and_matches_numpy(w0):
    z = synth.nuclear_charges(w0.elements)
    u = oracle.nuclear_potential(w0.surface, w0.atom_xyz, z)
    r = np.linalg.norm(w0.surface.xyz[:, None, :] - w0.atom_xyz[None, :, :], axis=2)
    np.testing.assert_allclose(u, (erf(w0.surface.zeta[:, None] * r) / r) @ z, rtol=1e-13)
    z2 = np.linspace(-1, 2, len(z))
    u2 = oracle.nuclear_potential(w0.surface, w0.atom_xyz, z2)
    u12 = oracle.nuclear_potential(w0.surface, w0.atom_xyz, 2 * z - 3 * z2)
    np.testing.assert_allclose(u12, 2 * u - 3 * u2, rtol=0, atol=1e-12)
    # translation invariance, and B z of a distant molecule is (sum z)/R
    sh = np.array([0.3, -1.1, 2.0])
    s2 = synth.Surface(xyz=w0.surface.xyz + sh, zeta=w0.surface.zeta, switch=w0.surface.switch,
                       atom=w0.surface.atom)
    np.testing.assert_allclose(oracle.nuclear_potential(s2, w0.atom_xyz + sh, z), u, rtol=1e-12)
    far = synth.Surface(xyz=np.array([[1e6, 0.0, 0.0]]), zeta=np.array([3.0]), switch=np.ones(1), atom=np.zeros(1, np.int32))
    assert oracle.nuclear_potential(far, w0.atom_xyz, z)[0] == pytest.approx(z.sum() / 1e6, rel=1e-5)


def test_rhs_and_energy_identities(w0):
    # with q the exact solution of A q = -f (B z + c), Eq. 13 collapses to (B z + c).q / 2 (stationarity);
    # a conductor (f = 1) with the sign reading R2 (c = -v)
    s = w0.surface
    z = synth.nuclear_charges(w0.elements)
    u = oracle.nuclear_potential(s, w0.atom_xyz, z)
    v = oracle.potential(w0.basis, s, w0.P)
    A = oracle.amatrix(s)
    for f in (1.0, (78.39 - 1) / 78.39):
        b = oracle.rhs(u, v, f)
        np.testing.assert_array_equal(b, -f * (u - v))
        q = np.linalg.solve(A, b)
        e = oracle.energy(u, v, q, A @ q, f)
        assert e[3] == pytest.approx(e[0] + e[1] + e[2], rel=1e-15)
        assert e[0] == pytest.approx(u @ q, rel=1e-13)
        assert e[1] == pytest.approx(-(v @ q), rel=1e-13)
        assert e[3] == pytest.approx(0.5 * (u - v) @ q, rel=1e-10)
        # the energy is stationary at q: a perturbation changes it only at second order
        dq = 1e-4 * np.cos(np.arange(s.M))
        e2 = oracle.energy(u, v, q + dq, A @ (q + dq), f)
        assert abs(e2[3] - e[3]) == pytest.approx(dq @ A @ dq / (2 * f), rel=1e-5)


def test_dynamic_threshold_inverts_eq21():
    # Err(delta) = 0.01 delta^1.07 must equal 1e-3 x the previous DIIS error
    for d in (1e-1, 1e-2, 3e-4, 1e-6):
        delta = oracle.cg_threshold(d, 1e-12)
        assert 0.01 * delta ** 1.07 == pytest.approx(1e-3 * d, rel=1e-12)
    assert oracle.cg_threshold(0.0) == 1.0 and oracle.cg_threshold(-1.0) == 1.0       # first SCF iteration: delta = 1
    assert oracle.cg_threshold(1e4) == 1.0                                            # never looser than 1
    assert oracle.cg_threshold(1e-9, 1e-6) == 1e-6                                    # never tighter than delta_min
    ds = [oracle.cg_threshold(d, 1e-12) for d in np.logspace(-8, 0, 30)]
    assert all(a < b for a, b in zip(ds, ds[1:]))                                     # monotone in the DIIS error
