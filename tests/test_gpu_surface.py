"""GPU parity of the ISWIG switching function (Eq. 9) and of the surface terms of the gradient (Eq. 14: grad B, grad A
including A_kk through S_k) against the oracle, element by element at |gpu - oracle| <= 1e-10 |oracle| + 1e-12."""
import copy

import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def pcm():
    import paper_1505_07851_b200 as m
    m.lib(build=True)   # compiles the library first if it is missing or stale (nvcc is in the image)
    return m


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def close(got, ref, atol=1e-12):
    return np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref) + atol)


def term_magnitudes(s, atoms, rad, z, q, f):
    """Per element of g_point and g_atom: the sum of the ABSOLUTE values of the terms Eq. 14's surface gradient adds up (the B
    term per nucleus, the off-diagonal A term per point pair, the A_kk term per other sphere), with scipy's erf.  A sum of n
    rounded terms is off by at most n eps sum|terms|; the element-wise floor of the comparison is 8 eps times this."""
    from scipy.special import erf
    M, N = s.M, len(rad)
    pt, zk = s.xyz, s.zeta
    g = lambda zp, r: np.abs(2 * zp / np.sqrt(np.pi) * np.exp(-(zp * r) ** 2) / r) + np.abs(erf(zp * r) / r ** 2)
    mp, ma = np.zeros((M, 3)), np.zeros((N, 3))
    akk = zk * np.sqrt(2 / np.pi) / s.switch
    for J in range(N):
        e = pt - atoms[J]
        d = np.linalg.norm(e, axis=1)
        ok = d > 0
        w = np.zeros(M)
        w[ok] = np.abs(z[J] * q[ok]) * g(zk[ok], d[ok])
        other = ok & (s.atom != J)
        a_, b_ = zk * (rad[J] - d), zk * (rad[J] + d)
        swf = 1 - 0.5 * (erf(a_) + erf(b_))
        dswf = zk / np.sqrt(np.pi) * (np.exp(-a_ * a_) + np.exp(-b_ * b_))
        w[other] += 0.5 / abs(f) * q[other] ** 2 * akk[other] * dswf[other] / swf[other]
        t = np.where(ok[:, None], w[:, None] * np.abs(e) / np.where(ok, d, 1.0)[:, None], 0.0)
        mp += t
        ma[J] = t.sum(0)
    for k in range(M):
        e = pt[k] - pt
        r = np.linalg.norm(e, axis=1)
        ok = r > 0
        zp = zk[k] * zk / np.sqrt(zk[k] ** 2 + zk ** 2)
        w = np.zeros(M)
        w[ok] = np.abs(q[k] * q[ok] / f) * g(zp[ok], r[ok])
        mp[k] += (w[:, None] * np.abs(e) / np.where(ok, r, 1.0)[:, None]).sum(0)
    return mp, ma


def points_ctx(pcm, s):
    e = np.zeros(0)
    return pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), e, e, s.xyz, s.zeta, s.switch)


@pytest.mark.parametrize("config,n_atoms", [(0, None), (1, 80), (3, 40)])
def test_switching_parity(pcm, orc, config, n_atoms):
    w = synth.make_workload(config, n_atoms=n_atoms, with_density=False)
    rad = synth.cavity_radii(w.elements)
    S = pcm.pcm_switching(w.surface.xyz, w.surface.zeta, w.surface.atom, w.atom_xyz, rad)
    ref = orc.switching(w.surface, w.atom_xyz, rad)
    assert close(S, ref, atol=1e-15), np.abs(S - ref).max()
    assert (S > 0).all() and (S <= 1).all() and S.min() < 0.9        # exposed points only, some of them near a neighbour
    # points deep inside a neighbour are switched off (the paper ignores S_k < 1e-8)
    inside = copy.copy(w.surface)
    inside.xyz = w.atom_xyz[w.surface.atom] * 0.0 + w.atom_xyz[(w.surface.atom + 1) % len(rad)] + 0.05
    Si = pcm.pcm_switching(inside.xyz, inside.zeta, inside.atom, w.atom_xyz, rad)
    assert close(Si, orc.switching(inside, w.atom_xyz, rad), atol=1e-15) and Si.max() < 1e-8
    assert len(pcm.pcm_switching(np.zeros((0, 3)), np.zeros(0), np.zeros(0, np.int32), w.atom_xyz, rad)) == 0


@pytest.mark.parametrize("config,n_atoms", [(0, None), (1, 60)])
def test_surface_gradient_parity(pcm, orc, torch_cuda, config, n_atoms):
    w = synth.make_workload(config, n_atoms=n_atoms, with_density=False)
    rad = synth.cavity_radii(w.elements)
    z = synth.nuclear_charges(w.elements)
    s = copy.copy(w.surface)
    s.switch = orc.switching(s, w.atom_xyz, rad)                      # A_kk from Eq. 9, as the oracle's gradient assumes
    f = (78.39 - 1.0) / 78.39
    q = w.q
    ctx = points_ctx(pcm, s)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_surface_gradient(ctx, dev(torch_cuda, q), f)           # before pcm_set_nuclei / pcm_set_cavity
    pcm.pcm_set_nuclei(ctx, w.atom_xyz, z)
    pcm.pcm_set_cavity(ctx, rad, s.atom)
    gp, ga = pcm.pcm_surface_gradient(ctx, dev(torch_cuda, q), f)
    gp, ga = gp.cpu().numpy(), ga.cpu().numpy()
    rp, ra = orc.surface_gradient(s, w.atom_xyz, rad, z, q, f)
    assert close(gp, rp), np.abs(gp - rp).max()
    assert close(ga, ra, atol=1e-12 + 64 * np.finfo(float).eps * np.abs(q).sum() * z.max()), np.abs(ga - ra).max()
    assert np.abs(gp.sum(0) + ga.sum(0)).max() < 1e-9                 # translation invariance of the whole
    gp2, ga2 = pcm.pcm_surface_gradient(ctx, dev(torch_cuda, q), f)
    assert np.array_equal(gp2.cpu().numpy(), gp) and np.array_equal(ga2.cpu().numpy(), ga)   # fixed-order sums
    pcm.pcm_destroy(ctx)


def test_surface_gradient_small_exponents_and_coincidences(pcm, orc, torch_cuda):
    # small zeta (erf branch everywhere), a nucleus on a point, two coincident points: finite and equal to the oracle
    rng = np.random.default_rng(9)
    M, N = 300, 5
    xyz = rng.normal(size=(M, 3)) * 2.5
    xyz[11] = xyz[4]
    atoms = rng.normal(size=(N, 3)) * 2.0
    atoms[2] = xyz[20]
    rad = rng.uniform(0.8, 1.6, N)
    own = rng.integers(0, N, M).astype(np.int32)
    s = synth.Surface(xyz=xyz, zeta=rng.uniform(0.4, 5.0, M), switch=np.ones(M), atom=own)
    s.switch = np.maximum(orc.switching(s, atoms, rad), 1e-3)
    # the oracle derives A_kk from Eq. 9 itself: keep only points whose S_k was not clipped
    keep = orc.switching(s, atoms, rad) >= 1e-3
    s = s.subset(np.flatnonzero(keep))
    s.switch = orc.switching(s, atoms, rad)
    q = rng.uniform(-0.5, 0.5, s.M)
    z = rng.uniform(1, 8, N)
    ctx = points_ctx(pcm, s)
    pcm.pcm_set_nuclei(ctx, atoms, z)
    pcm.pcm_set_cavity(ctx, rad, s.atom)
    gp, ga = pcm.pcm_surface_gradient(ctx, dev(torch_cuda, q), 0.9)
    gp, ga = gp.cpu().numpy(), ga.cpu().numpy()
    assert np.isfinite(gp).all() and np.isfinite(ga).all()
    rp, ra = orc.surface_gradient(s, atoms, rad, z, q, 0.9)
    # element-wise: 1e-10 |ref| + 1e-12 + 8 eps x (sum of the absolute terms of that element) -- the terms reach 1e3 here (small
    # exponents, charges up to 0.5, a nucleus 1e-3 from a point) and largely cancel, so eps x their magnitude is the rounding
    # floor of any summation order
    mp, ma = term_magnitudes(s, atoms, rad, z, q, 0.9)
    eps8 = 8 * np.finfo(float).eps
    assert np.all(np.abs(gp - rp) <= 1e-10 * np.abs(rp) + 1e-12 + eps8 * mp), np.abs(gp - rp).max()
    assert np.all(np.abs(ga - ra) <= 1e-10 * np.abs(ra) + 1e-12 + eps8 * ma), np.abs(ga - ra).max()
    pcm.pcm_destroy(ctx)
