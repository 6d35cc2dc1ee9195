"""Pins for the oracle's ISWIG cavity construction (oracle.build_cavity: Eq. 7, Eq. 9 and the switching-function screening of
PAPER.md:106).  The unit-sphere quadrature is an input (the paper's Lebedev grids are not available offline; the tests use the
Fibonacci lattice of synth/ and a small hand-made weighted grid).  Checked against closed forms for one sphere, scipy's erf on
a hand-built two-atom geometry, the analytic area of a sphere cut by another sphere, the hard inside-test of the synthetic
generator on atoms whose spheres overlap at most pairwise, and invariance under atom reordering and rigid motion."""
import math

import numpy as np
import pytest
from scipy.special import erf

import oracle
import synth

ZETA_TAB = 4.9


def fibonacci(n):
    k = np.arange(n)
    z = 1.0 - (2.0 * k + 1.0) / n
    phi = k * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1), np.full(n, 4.0 * math.pi / n)


def test_single_sphere_closed_forms():
    # one atom: nothing switches anything off -- every node is kept, S = 1, the points lie on the sphere, zeta follows Eq. 7
    u, w = fibonacci(50)
    R, c = 3.1, np.array([[0.3, -1.2, 2.0]])
    xyz, zeta, S, own, node = oracle.build_cavity(c, [R], u, w, ZETA_TAB)
    assert len(zeta) == 50 and np.all(S == 1.0) and np.all(own == 0) and np.array_equal(node, np.arange(50))
    assert np.allclose(np.linalg.norm(xyz - c, axis=1), R, rtol=1e-15)
    assert np.allclose(zeta, ZETA_TAB / (R * math.sqrt(4 * math.pi / 50)), rtol=1e-15)
    assert np.allclose(xyz, c + R * u, rtol=0, atol=1e-15)
    # Eq. 7 with unequal weights: zeta_k sqrt(w_k) R_I = zeta for every node (an octahedron plus cube corners, 6 + 8 nodes)
    oct6 = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], float)
    cube8 = np.array([[a, b, c2] for a in (-1, 1) for b in (-1, 1) for c2 in (-1, 1)], float) / math.sqrt(3)
    u2 = np.concatenate([oct6, cube8])
    w2 = 4 * math.pi * np.concatenate([np.full(6, 1 / 15), np.full(8, 3 / 40)])      # the 14-point rule of degree 5
    assert w2.sum() == pytest.approx(4 * math.pi, rel=1e-15)
    _, zeta2, _, _, _ = oracle.build_cavity(c, [R], u2, w2, ZETA_TAB)
    assert np.allclose(zeta2 * np.sqrt(w2) * R, ZETA_TAB, rtol=1e-15)
    assert zeta2[0] / zeta2[6] == pytest.approx(math.sqrt((3 / 40) / (1 / 15)), rel=1e-14)


def test_two_atoms_against_scipy_erf_and_threshold():
    # atom 0 at the origin (radius 2), atom 1 on the x axis (radius 3): S of node g of atom 0 depends on one distance only
    u, w = fibonacci(200)
    atoms = np.array([[0.0, 0, 0], [3.5, 0, 0]])
    rad = np.array([2.0, 3.0])
    xyz, zeta, S, own, node = oracle.build_cavity(atoms, rad, u, w, ZETA_TAB, s_min=0.0)      # keep everything
    assert len(S) == 400 and np.array_equal(own, np.repeat([0, 1], 200)) and np.array_equal(node, np.tile(np.arange(200), 2))
    for I, J in ((0, 1), (1, 0)):
        p = atoms[I] + rad[I] * u
        z = ZETA_TAB / (rad[I] * np.sqrt(w))
        d = np.linalg.norm(p - atoms[J], axis=1)
        ref = 1.0 - 0.5 * (erf(z * (rad[J] - d)) + erf(z * (rad[J] + d)))
        assert np.allclose(S[own == I], ref, rtol=1e-13, atol=1e-300)
        assert np.allclose(zeta[own == I], z, rtol=1e-15)
    # the screening keeps exactly the points with S >= s_min, in the same order
    for s_min in (1e-8, 1e-3, 0.5, 0.999):
        x2, z2, S2, o2, n2 = oracle.build_cavity(atoms, rad, u, w, ZETA_TAB, s_min=s_min)
        keep = S >= s_min
        assert np.array_equal(S2, S[keep]) and np.array_equal(o2, own[keep]) and np.array_equal(n2, node[keep])
        assert np.array_equal(x2, xyz[keep]) and np.array_equal(z2, zeta[keep])
    assert 0 < (S >= 1e-8).sum() < 400         # some points are switched off at the paper's threshold, not all


def test_exposed_area_of_two_intersecting_spheres():
    # sum_k w_k S_k R_I^2 is the quadrature of the switched surface: for a fine grid it tends to the area of sphere I outside
    # sphere J, 2 pi R_I^2 (1 + cos theta), cos theta = (d^2 + R_I^2 - R_J^2)/(2 d R_I)  (spherical cap cut off by J)
    n = 20000
    u, w = fibonacci(n)
    R1, R2, d = 2.0, 2.6, 3.1
    atoms = np.array([[0.0, 0, 0], [0.0, d, 0]])
    _, _, S, own, node = oracle.build_cavity(atoms, [R1, R2], u, w, ZETA_TAB, s_min=0.0)
    for I, (Ri, Rj) in enumerate(((R1, R2), (R2, R1))):
        cos_t = (d * d + Ri * Ri - Rj * Rj) / (2 * d * Ri)
        frac = 0.5 * (1 + cos_t)
        assert float((w * S[own == I]).sum() / (4 * math.pi)) == pytest.approx(frac, abs=2e-3)
    # the points the paper's 1e-8 threshold removes all lie inside the other sphere, deeper than erfc^-1(2e-8)/zeta = 3.97/zeta
    xyz, zeta, S8, own8, _ = oracle.build_cavity(atoms, [R1, R2], u, w, ZETA_TAB, s_min=1e-8)
    xa, za, Sa, oa, _ = oracle.build_cavity(atoms, [R1, R2], u, w, ZETA_TAB, s_min=0.0)
    gone = Sa < 1e-8
    depth = np.where(oa == 0, R2 - np.linalg.norm(xa - atoms[1], axis=1), R1 - np.linalg.norm(xa - atoms[0], axis=1))
    assert gone.any() and np.all(depth[gone] * za[gone] > 3.9) and np.all(depth[~gone] * za[~gone] < 4.0)


def test_hard_inside_test_of_the_generator_when_spheres_overlap_pairwise():
    # S_wf = 1/2 exactly on the other sphere (the second erf is 1 to fp64), so s_min = 1/2 keeps a point iff it is not strictly
    # inside the one sphere it can reach: the hard test of synth.make_surface.  A zig-zag chain whose second neighbours are out
    # of reach (no point sees two spheres at once).
    el = ["C", "N", "O", "H", "C", "H"]
    rad = synth.cavity_radii(el)
    xyz = np.array([[0.0, 0, 0], [5.6, 0.8, 0], [11.2, 0.0, 0.5], [16.4, 1.0, 0.0], [21.9, -0.5, 0.3], [27.0, 0.6, 0.0]])
    dist = np.linalg.norm(xyz[:, None] - xyz[None], axis=2)
    for i in range(6):
        for j in range(6):
            if abs(i - j) >= 2:
                assert dist[i, j] > rad[i] + rad[j] + 1.0
    rng = np.random.Generator(np.random.PCG64(5))
    s = synth.make_surface(rng, el, xyz, 110)
    u, w = fibonacci(110)
    p, zeta, S, own, node = oracle.build_cavity(xyz, rad, u, w, 4.9, s_min=0.5)
    assert len(zeta) == s.M and np.array_equal(own, s.atom)
    assert np.allclose(p, s.xyz, rtol=0, atol=1e-12) and np.allclose(zeta, s.zeta, rtol=1e-14)
    assert 0 < s.M < 6 * 110


def test_reordering_and_rigid_motion():
    w0 = synth.make_workload(0, n_atoms=7, n_pts=14)
    atoms, rad = w0.atom_xyz, synth.cavity_radii(w0.elements)
    u, w = fibonacci(40)
    xyz, zeta, S, own, node = oracle.build_cavity(atoms, rad, u, w, ZETA_TAB)
    assert 0 < len(S) < 7 * 40 and np.all(S >= 1e-8) and np.all(S <= 1.0)
    # S agrees with the (separately pinned) switching function evaluated on the produced points
    surf = synth.Surface(xyz=xyz, zeta=zeta, switch=np.ones(len(S)), atom=own.astype(np.int32))
    assert np.allclose(S, oracle.switching(surf, atoms, rad), rtol=1e-15)
    # reordering the atoms reorders the blocks of points and nothing else
    perm = np.array([3, 0, 6, 1, 5, 2, 4])
    x2, z2, S2, o2, n2 = oracle.build_cavity(atoms[perm], rad[perm], u, w, ZETA_TAB)
    key = lambda o, n: np.lexsort((n, o))
    a, b = key(own, node), key(perm[o2], n2)
    assert np.array_equal(own[a], perm[o2][b]) and np.array_equal(node[a], n2[b])
    assert np.allclose(xyz[a], x2[b], rtol=0, atol=1e-14) and np.allclose(S[a], S2[b], rtol=1e-12) and np.array_equal(zeta[a], z2[b])
    # rotating atoms and grid together and translating: same zeta, same S, rotated points
    th = 0.7
    Rm = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1]]) @ \
        np.array([[1, 0, 0], [0, math.cos(0.4), -math.sin(0.4)], [0, math.sin(0.4), math.cos(0.4)]])
    t = np.array([1.5, -2.0, 0.3])
    x3, z3, S3, o3, n3 = oracle.build_cavity(atoms @ Rm.T + t, rad, u @ Rm.T, w, ZETA_TAB)
    assert np.array_equal(o3, own) and np.array_equal(n3, node) and np.allclose(z3, zeta, rtol=1e-15)
    assert np.allclose(S3, S, rtol=1e-10) and np.allclose(x3, xyz @ Rm.T + t, rtol=0, atol=1e-12)


def test_degenerate_sizes():
    u, w = fibonacci(10)
    for atoms, rad in ((np.zeros((0, 3)), np.zeros(0)),):
        xyz, zeta, S, own, node = oracle.build_cavity(atoms, rad, u, w, ZETA_TAB)
        assert len(zeta) == 0 and xyz.shape == (0, 3)
    xyz, zeta, S, own, node = oracle.build_cavity(np.zeros((1, 3)), [1.0], np.zeros((0, 3)), np.zeros(0), ZETA_TAB)
    assert len(zeta) == 0
    # an atom swallowed by a larger sphere loses all its points
    xyz, zeta, S, own, node = oracle.build_cavity(np.array([[0.0, 0, 0], [0.2, 0, 0]]), [4.0, 1.0], u, w, ZETA_TAB)
    assert np.all(own == 0) and len(own) == 10
