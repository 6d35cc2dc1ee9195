"""GPU parity of the ISWIG cavity construction (pcm_build_cavity / pcm_setup_cavity) against
oracle.build_cavity (Eq. 7, Eq. 9, the S_k >= 1e-8 screening of PAPER.md:106).

The kept set is integer work: the (atom, node) lists must be equal.  S is computed on both sides as Eq. 9 prints it,
1 - [erf + erf]/2, which for a point deep inside another sphere loses digits (absolute error ~ 1 ulp of 1, so a relative error
of ~ 2e-16 / S); the decision S >= s_min is taken in fp64 on both sides and can differ only for a point whose S lies within that
absolute error of the threshold: such a point is allowed to differ and checked to lie in the band.  Values: |gpu - oracle| <=
1e-10 |oracle| + 1e-12 per element for xyz, zeta and S.
"""
import math

import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu
RTOL, ATOL = 1e-10, 1e-12
ZETA_TAB = 4.9


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def pcm():
    import paper_1505_07851_b200 as m
    m.lib(build=True)
    return m


def fibonacci(n):
    k = np.arange(n)
    z = 1.0 - (2.0 * k + 1.0) / n
    phi = k * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1), np.full(n, 4.0 * math.pi / n)


def close(a, b, atol=ATOL):
    return np.all(np.abs(np.asarray(a) - np.asarray(b)) <= RTOL * np.abs(b) + atol)


def compare_cavity(pcm, orc, atoms, rad, u, w, s_min):
    cav = pcm.pcm_build_cavity(atoms, rad, u, w, ZETA_TAB, s_min)
    gx, gz, gS, ga, gn = pcm.pcm_cavity_get(cav)
    ox, oz, oS, oa, on = orc.build_cavity(atoms, rad, u, w, ZETA_TAB, s_min)
    G = len(w)
    gid, oid = ga.astype(np.int64) * G + gn, oa * G + on
    assert np.all(np.diff(gid) > 0) and np.all(np.diff(oid) > 0)            # (atom, node) order on both sides
    common, gi, oi = np.intersect1d(gid, oid, return_indices=True)
    # a point kept by one side only must have S within the rounding error of the printed formula of the threshold
    for only, S in ((np.setdiff1d(np.arange(len(gid)), gi), gS), (np.setdiff1d(np.arange(len(oid)), oi), oS)):
        assert np.all(np.abs(S[only] - s_min) <= 4 * np.finfo(float).eps), "kept sets differ outside the rounding band"
    assert len(common) >= max(len(oid) - 2, 0)
    assert close(gx[gi], ox[oi]) and close(gz[gi], oz[oi]) and close(gS[gi], oS[oi])
    assert cav.npoint == len(gid)
    return cav, (gx, gz, gS, ga, gn), (ox, oz, oS, oa, on), len(common) == len(oid) == len(gid)


def test_cavity_configs0_and_degenerate(pcm, orc):
    w0 = synth.make_workload(0)
    rad = synth.cavity_radii(w0.elements)
    u, w = fibonacci(50)
    for s_min in (1e-8, 0.0, 0.5):
        cav, g, o, same = compare_cavity(pcm, orc, w0.atom_xyz, rad, u, w, s_min)
        assert 0 < cav.npoint <= 12 * 50
        if s_min == 0.0:
            assert cav.npoint == 12 * 50
    # unequal weights (octahedron + cube corners), one atom, no atom, no grid
    oct6 = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], float)
    cube8 = np.array([[a, b, c] for a in (-1, 1) for b in (-1, 1) for c in (-1, 1)], float) / math.sqrt(3)
    u2, w2 = np.concatenate([oct6, cube8]), 4 * math.pi * np.concatenate([np.full(6, 1 / 15), np.full(8, 3 / 40)])
    compare_cavity(pcm, orc, w0.atom_xyz, rad, u2, w2, 1e-8)
    cav, g, o, _ = compare_cavity(pcm, orc, w0.atom_xyz[:1], rad[:1], u, w, 1e-8)
    assert cav.npoint == 50 and np.all(g[2] == 1.0)
    assert pcm.pcm_build_cavity(np.zeros((0, 3)), np.zeros(0), u, w, ZETA_TAB).npoint == 0
    assert pcm.pcm_build_cavity(w0.atom_xyz, rad, np.zeros((0, 3)), np.zeros(0), ZETA_TAB).npoint == 0
    with pytest.raises(pcm.PcmError):
        pcm.pcm_build_cavity(w0.atom_xyz, -rad, u, w, ZETA_TAB)


def test_cavity_configs1_sixty_atoms_and_compaction_across_blocks(pcm, orc):
    # 60 atoms of the configs[1] recipe x 110 nodes = 6 600 candidates: several compaction blocks, a ragged last one
    w1 = synth.make_workload(1, n_atoms=60)
    rad = synth.cavity_radii(w1.elements)
    u, w = fibonacci(110)
    cav, g, o, same = compare_cavity(pcm, orc, w1.atom_xyz, rad, u, w, 1e-8)
    assert 1000 < cav.npoint < 60 * 110
    # more points than the generator's hard inside-test keeps: the switching region reaches ~ 4/zeta into the other spheres
    assert cav.npoint > w1.surface.M
    # the device arrays are what pcm_cavity_get copied
    import torch
    ptrs = pcm.pcm_cavity_device(cav)
    assert all(p for p in ptrs)
    pcm.pcm_cavity_destroy(cav)


def test_setup_cavity_feeds_the_hot_path(pcm, orc, torch_cuda):
    # configs[0] with d shells: context straight from the cavity; v, A q against the oracle on the ORACLE's cavity
    torch = torch_cuda
    w0 = synth.make_workload(0, with_d=True)
    rad = synth.cavity_radii(w0.elements)
    u, w = fibonacci(50)
    cav, g, o, same = compare_cavity(pcm, orc, w0.atom_xyz, rad, u, w, 1e-8)
    assert same
    b = w0.basis
    ctx = pcm.pcm_setup_cavity(b.shell_l, b.shell_xyz, b.shell_nprim, b.prim_exp, b.prim_coef, cav, d_pure=bool(b.d_pure))
    assert ctx.M == cav.npoint
    surf = synth.Surface(xyz=o[0], zeta=o[1], switch=o[2], atom=o[3].astype(np.int32))
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")
    v = pcm.pcm_potential(ctx, dev(w0.P)).cpu().numpy()
    assert close(v, orc.potential(b, surf, w0.P))
    rng = np.random.default_rng(3)
    q = rng.uniform(-0.05, 0.05, surf.M)
    F = pcm.pcm_fock(ctx, dev(q)).cpu().numpy()
    assert close(F, orc.fock(b, surf, q))
    # A q: A_kk = zeta sqrt(2/pi)/S_k inherits the relative rounding error of S_k, eps/S_k (docstring) -- it enters the floor
    y = pcm.pcm_amatvec(ctx, dev(q)).cpu().numpy()
    akk = surf.zeta * math.sqrt(2 / math.pi) / surf.switch
    floor = ATOL + 4 * np.finfo(float).eps / surf.switch * akk * np.abs(q)
    ref = orc.amatvec(surf, q)
    assert np.all(np.abs(y - ref) <= RTOL * np.abs(ref) + floor)
    big = surf.switch >= 1e-3
    assert np.all(np.abs(y - ref)[big] <= RTOL * np.abs(ref)[big] + ATOL)
    # the same context through pcm_setup with the arrays copied back by the caller: bit-identical results
    gx, gz, gS, ga, gn = g
    ctx2 = pcm.pcm_setup(b.shell_l, b.shell_xyz, b.shell_nprim, b.prim_exp, b.prim_coef, gx, gz, gS, d_pure=bool(b.d_pure))
    assert np.array_equal(pcm.pcm_potential(ctx2, dev(w0.P)).cpu().numpy(), v)
    assert np.array_equal(pcm.pcm_amatvec(ctx2, dev(q)).cpu().numpy(), y)
    pcm.pcm_destroy(ctx2)
    pcm.pcm_destroy(ctx)


def test_surface_gradient_on_a_library_built_cavity(pcm, orc, torch_cuda):
    # s_min = 1e-3 here: the A_kk term of the gradient carries 1/S_k, whose rounding error (eps/S_k^2 relative to S_k ~ 1) would
    # otherwise swamp the 1e-12 floor; the kept-set logic at 1e-8 is covered above
    torch = torch_cuda
    w0 = synth.make_workload(0, n_atoms=8, n_pts=30)
    rad = synth.cavity_radii(w0.elements)
    z = synth.nuclear_charges(w0.elements)
    u, w = fibonacci(30)
    cav, g, o, same = compare_cavity(pcm, orc, w0.atom_xyz, rad, u, w, 1e-3)
    assert same
    ctx = pcm.pcm_setup_cavity(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0), cav)
    surf = synth.Surface(xyz=o[0], zeta=o[1], switch=o[2], atom=o[3].astype(np.int32))
    q = np.random.default_rng(4).uniform(-0.05, 0.05, surf.M)
    qd = torch.as_tensor(q, dtype=torch.float64, device="cuda")
    with pytest.raises(pcm.PcmError):
        pcm.pcm_surface_gradient(ctx, qd, 0.9)             # the nuclei are still missing
    pcm.pcm_set_nuclei(ctx, w0.atom_xyz, z)                 # registers the cavity's radii and owners as well
    gp, ga = pcm.pcm_surface_gradient(ctx, qd, 0.9)
    rp, ra = orc.surface_gradient(surf, w0.atom_xyz, rad, z, q, 0.9)
    floor = ATOL + 64 * np.finfo(float).eps * np.abs(q).sum() * z.max()     # sums over all points that largely cancel
    assert close(gp.cpu().numpy(), rp, atol=floor) and close(ga.cpu().numpy(), ra, atol=floor)
    pcm.pcm_destroy(ctx)
