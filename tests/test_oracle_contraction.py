"""Pins for the oracle's contracted quantities (oracle/pcm_oracle.c: shell_block, orc_potential,
orc_fock_blocks) -- Eq. 5, Eq. 10, Eq. 11-12 of PAPER.md (lines 39, 66, 72-77) with the readings
R2-R4 of the oracle header (signs, raw-primitive coefficients, pure-d order, no Eq. 15 screening).

Pins: a Python re-assembly of the contraction from single primitive integrals (which are themselves
pinned in test_oracle_integrals.py), the pure-d combinations checked against an explicit real-solid-
harmonic quadrature, rotation invariance of the d-shell trace, F = F^T, the adjoint identity
v.q = tr(P F), translation invariance, linearity, and independence from the 1e-20 cutoff.
"""
import json
import math
import os

import numpy as np
import pytest

import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_checkvalues.json")))

CART = {0: [(0, 0, 0)], 1: [(1, 0, 0), (0, 1, 0), (0, 0, 1)],
        2: [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]}
S3 = math.sqrt(3.0)
# pure d components as polynomials {cartesian power: coefficient}  (include/pcm.h, reading R3)
PURE_D = [{(1, 1, 0): S3}, {(0, 1, 1): S3}, {(0, 0, 2): 1.0, (2, 0, 0): -0.5, (0, 2, 0): -0.5}, {(1, 0, 1): S3},
          {(2, 0, 0): 0.5 * S3, (0, 2, 0): -0.5 * S3}]


def components(l, d_pure):
    if l < 2 or not d_pure:
        return [{c: 1.0} for c in CART[l]]
    return PURE_D


def tiny_workload(with_d=True, d_pure=True, n_atoms=4, n_pts=6, seed=77):
    return synth.make_workload(0, n_atoms=n_atoms, n_pts=n_pts, with_d=with_d, d_pure=d_pure, seed=seed)


def python_shell_block(orc, basis, I, J, zeta, Cpt):
    """sum_ij c_i c_j [chi_i|J|chi_j] assembled from single primitive integrals, component by component"""
    po = basis.prim_offset
    ca, cb = components(int(basis.shell_l[I]), basis.d_pure), components(int(basis.shell_l[J]), basis.d_pure)
    out = np.zeros((len(ca), len(cb)))
    for i in range(po[I], po[I + 1]):
        for j in range(po[J], po[J + 1]):
            cc = basis.prim_coef[i] * basis.prim_coef[j]
            for m, pa in enumerate(ca):
                for n, pb in enumerate(cb):
                    for a, wa in pa.items():
                        for b, wb in pb.items():
                            out[m, n] += cc * wa * wb * orc.prim_integral(a, basis.prim_exp[i], basis.shell_xyz[I], b,
                                                                          basis.prim_exp[j], basis.shell_xyz[J], zeta, Cpt)
    return out


@pytest.mark.parametrize("d_pure", [True, False])
def test_shell_block_is_the_contraction_of_primitives(orc, d_pure):
    w = tiny_workload(d_pure=d_pure)
    b = w.basis
    rng = np.random.default_rng(1)
    shells_by_l = {l: np.flatnonzero(b.shell_l == l) for l in range(3)}
    for la in range(3):
        for lb in range(3):
            I = int(rng.choice(shells_by_l[la]))
            J = int(rng.choice(shells_by_l[lb]))
            k = int(rng.integers(w.surface.M))
            got = orc.shell_block(b, I, J, w.surface.zeta[k], w.surface.xyz[k])
            ref = python_shell_block(orc, b, I, J, w.surface.zeta[k], w.surface.xyz[k])
            np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-14)


def test_pure_d_components_by_quadrature(orc):
    """(d_m s|J) for a single primitive d shell against 3-D Gauss-Hermite quadrature of the explicit
    real solid harmonics sqrt3 xy, sqrt3 yz, zz-(xx+yy)/2, sqrt3 xz, (sqrt3/2)(xx-yy)."""
    A, B, C = np.array([0.1, -0.2, 0.15]), np.array([0.5, 0.3, -0.4]), np.array([1.1, 0.6, 0.9])
    al, be, ze = 0.8, 1.1, 1.2
    basis = synth.Basis(np.array([2, 0], np.int32), np.stack([A, B]), np.array([1, 1], np.int32), np.array([al, be]),
                        np.array([1.0, 1.0]), np.array([0, 1], np.int32), True)
    got = orc.shell_block(basis, 0, 1, ze, C)[:, 0]
    p = al + be
    P = (al * A + be * B) / p
    K = math.exp(-al * be / p * np.dot(A - B, A - B))
    x, wq = np.polynomial.hermite.hermgauss(70)
    s = 1 / math.sqrt(p)
    X, Y, Z = np.meshgrid(P[0] + s * x, P[1] + s * x, P[2] + s * x, indexing="ij")
    W = wq[:, None, None] * wq[None, :, None] * wq[None, None, :] * s ** 3
    from scipy import special
    r = np.sqrt((X - C[0]) ** 2 + (Y - C[1]) ** 2 + (Z - C[2]) ** 2)
    op = special.erf(ze * r) / r
    xa, ya, za = X - A[0], Y - A[1], Z - A[2]
    harm = [S3 * xa * ya, S3 * ya * za, za * za - 0.5 * (xa * xa + ya * ya), S3 * xa * za, 0.5 * S3 * (xa * xa - ya * ya)]
    ref = np.array([K * np.sum(W * h * op) for h in harm])
    np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-14)


def test_d_shell_trace_is_rotation_invariant(orc):
    """sum_m (d_m|J|d_m) for a same-centre d shell does not depend on the direction of the point
    (SURVEY.md 8(c3)); also pinned to the stored survey value."""
    g = GOLD["d_shell_rotation_invariant_sum"]
    O = np.zeros(3)
    basis = synth.Basis(np.array([2, 2], np.int32), np.stack([O, O]), np.array([1, 1], np.int32),
                        np.array([g["alpha"], g["beta"]]), np.array([1.0, 1.0]), np.array([0, 0], np.int32), True)
    vals = []
    rng = np.random.default_rng(2)
    dirs = [np.array([1.0, 0, 0]), np.array([1.0, 2.0, -2.0]) / 3.0] + [v / np.linalg.norm(v) for v in rng.normal(size=(5, 3))]
    for d in dirs:
        vals.append(np.trace(orc.shell_block(basis, 0, 1, g["zeta"], g["distance"] * d)))
    np.testing.assert_allclose(vals, vals[0], rtol=1e-13)
    assert vals[0] == pytest.approx(g["value"], rel=1e-12)


def test_potential_and_fock_are_the_definition(orc):
    """v_k = sum_{mu nu} P (mu|J_k|nu) and F = sum_k q_k (mu|J_k|nu) re-assembled in numpy from shell blocks"""
    w = tiny_workload()
    b, s = w.basis, w.surface
    off = b.bf_offset
    V = np.zeros((s.M, b.nbf, b.nbf))
    for k in range(s.M):
        for I in range(b.nshell):
            for J in range(b.nshell):
                V[k, off[I]:off[I + 1], off[J]:off[J + 1]] = orc.shell_block(b, I, J, s.zeta[k], s.xyz[k])
    v_ref = np.einsum("kmn,mn->k", V, w.P)
    F_ref = np.einsum("k,kmn->mn", w.q, V)
    np.testing.assert_allclose(orc.potential(b, s, w.P, cutoff=0.0), v_ref, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(orc.fock(b, s, w.q, cutoff=0.0), F_ref, rtol=1e-12, atol=1e-14)
    # a non-symmetric P is summed over the full square too (not symmetrised)
    Pn = np.random.default_rng(0).normal(size=w.P.shape)
    np.testing.assert_allclose(orc.potential(b, s, Pn, cutoff=0.0), np.einsum("kmn,mn->k", V, Pn), rtol=1e-11, atol=1e-13)
    # point selection
    sel = np.array([3, 0, s.M - 1])
    np.testing.assert_allclose(orc.potential(b, s, w.P, points=sel), v_ref[sel], rtol=1e-12, atol=1e-14)


@pytest.fixture(scope="module")
def small(orc):
    w = synth.make_workload(0, n_atoms=6, n_pts=12, with_d=True, seed=31)
    return w, orc.potential(w.basis, w.surface, w.P), orc.fock(w.basis, w.surface, w.q)


def test_fock_symmetric(small):
    _, _, F = small
    np.testing.assert_allclose(F, F.T, rtol=1e-12, atol=1e-14)
    assert np.abs(F).max() > 1e-3


def test_adjoint_identity(small):
    """v . q = tr(P F)  (ties the two contractions together)"""
    w, v, F = small
    assert float(v @ w.q) == pytest.approx(float(np.sum(w.P * F)), rel=1e-12)


def test_translation_invariance(orc, small):
    w, v, F = small
    t = np.array([3.7, -1.9, 2.2])
    b2 = synth.Basis(w.basis.shell_l, w.basis.shell_xyz + t, w.basis.shell_nprim, w.basis.prim_exp, w.basis.prim_coef,
                     w.basis.shell_atom, w.basis.d_pure)
    s2 = synth.Surface(w.surface.xyz + t, w.surface.zeta, w.surface.switch, w.surface.atom)
    np.testing.assert_allclose(orc.potential(b2, s2, w.P), v, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(orc.fock(b2, s2, w.q), F, rtol=1e-11, atol=1e-13)


def test_linearity(orc, small):
    w, v, F = small
    rng = np.random.default_rng(9)
    P2 = rng.normal(size=w.P.shape)
    P2 = P2 + P2.T
    q2 = rng.normal(size=w.q.shape)
    np.testing.assert_allclose(orc.potential(w.basis, w.surface, 2.0 * w.P - 0.5 * P2),
                               2.0 * v - 0.5 * orc.potential(w.basis, w.surface, P2), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(orc.fock(w.basis, w.surface, 3.0 * w.q + q2),
                               3.0 * F + orc.fock(w.basis, w.surface, q2), rtol=1e-10, atol=1e-12)


def test_cutoff_changes_nothing_visible(orc, small):
    """reading R4: skipping primitive pairs with |c_i c_j| K_AB < 1e-20 is invisible at 1e-16"""
    w, v, F = small
    np.testing.assert_allclose(orc.potential(w.basis, w.surface, w.P, cutoff=0.0), v, rtol=0, atol=1e-15)
    np.testing.assert_allclose(orc.fock(w.basis, w.surface, w.q, cutoff=0.0), F, rtol=0, atol=1e-16)


def test_fock_blocks_ordered_pairs(orc, small):
    w, _, F = small
    off = w.basis.bf_offset
    pairs = [(0, 3), (3, 0), (5, 5), (2, 7)]
    for (i, j), blk in zip(pairs, orc.fock_blocks(w.basis, w.surface, w.q, pairs)):
        np.testing.assert_array_equal(blk, F[off[i]:off[i + 1], off[j]:off[j + 1]])


def test_threads_do_not_change_results(orc, small):
    w, v, F = small
    n = orc.num_threads()
    try:
        orc.set_num_threads(1)
        np.testing.assert_array_equal(orc.potential(w.basis, w.surface, w.P), v)
        np.testing.assert_array_equal(orc.fock(w.basis, w.surface, w.q), F)
    finally:
        orc.set_num_threads(n)
