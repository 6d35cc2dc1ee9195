"""GPU parity of pcm_gradient (the one-electron PCM gradient term of Eq. 14 / Eq. 22) against the
oracle's raised/lowered Obara-Saika brackets: per shell centre and per surface point, element by element."""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-10, 1e-12   # the north_star tolerance, applied to every gradient component


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


def check(got, ref, what):
    err = np.abs(got - ref)
    bound = RTOL * np.abs(ref) + ATOL
    assert np.all(err <= bound), f"{what}: max err {err.max():.3e} at {np.unravel_index(np.argmax(err - bound), err.shape)}, ref there {ref.flat[np.argmax(err - bound)]:.6e}"


@pytest.mark.parametrize("d_pure", [True, False])
def test_gradient_all_classes_full(pcm, orc, torch_cuda, d_pure):
    w = synth.make_workload(0, with_d=True, d_pure=d_pure)
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=True)
    gs, gp = pcm.pcm_gradient(ctx, dev(torch_cuda, w.P), dev(torch_cuda, w.q))
    gs, gp = gs.cpu().numpy(), gp.cpu().numpy()
    rs, rp = orc.gradient(w.basis, w.surface, w.P, w.q)
    check(gs, rs, "g_shell")
    check(gp, rp, "g_point")
    # the whole system is translation invariant
    assert np.abs(gs.sum(0) + gp.sum(0)).max() < 1e-10
    # bit-reproducible, and the energy calls still work on a gradient-enabled context
    gs2, gp2 = pcm.pcm_gradient(ctx, dev(torch_cuda, w.P), dev(torch_cuda, w.q))
    assert np.array_equal(gs2.cpu().numpy(), gs) and np.array_equal(gp2.cpu().numpy(), gp)
    v = pcm.pcm_potential(ctx, dev(torch_cuda, w.P)).cpu().numpy()
    ref = orc.potential(w.basis, w.surface, w.P)
    assert np.all(np.abs(v - ref) <= 1e-10 * np.abs(ref) + 1e-12)
    pcm.pcm_destroy(ctx)


def test_gradient_unmerged_products_and_disabled(pcm, orc, torch_cuda):
    w = synth.make_workload(0, with_d=False)
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=True, merge_products=False)
    gs, gp = pcm.pcm_gradient(ctx, dev(torch_cuda, w.P), dev(torch_cuda, w.q))
    rs, rp = orc.gradient(w.basis, w.surface, w.P, w.q)
    check(gs.cpu().numpy(), rs, "g_shell")
    check(gp.cpu().numpy(), rp, "g_point")
    pcm.pcm_destroy(ctx)
    ctx = pcm.setup_from_workload(w.basis, w.surface)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_gradient(ctx, dev(torch_cuda, w.P), dev(torch_cuda, w.q))
    pcm.pcm_destroy(ctx)


def test_gradient_medium_sampled(pcm, orc, torch_cuda):
    # a 60-atom chain with d shells (several tiles, far and near patches): sampled shells and points against the oracle,
    # translation invariance on the full output
    w = synth.make_workload(3, n_atoms=60)
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=True)
    gs, gp = pcm.pcm_gradient(ctx, dev(torch_cuda, w.P), dev(torch_cuda, w.q))
    gs, gp = gs.cpu().numpy(), gp.cpu().numpy()
    rng = np.random.default_rng(11)
    ls = np.asarray(w.basis.shell_l)
    shells = sorted({int(np.flatnonzero(ls == l)[i]) for l in (0, 1, 2) for i in (0, -1)})
    points = sorted(rng.choice(w.surface.M, 24, replace=False).tolist())
    rs, rp = orc.gradient(w.basis, w.surface, w.P, w.q, shells=shells, points=points)
    check(gs[shells], rs, "g_shell")
    check(gp[points], rp, "g_point")
    assert np.abs(gs.sum(0) + gp.sum(0)).max() < 1e-9
    pcm.pcm_destroy(ctx)


def test_gradient_degenerate_sizes(pcm, orc, torch_cuda):
    """no points / no shells / one primitive and one point: zeros of the right shape, and the closed form through the oracle"""
    torch = torch_cuda
    w = synth.make_workload(0, with_d=False)
    b, s = w.basis, w.surface
    ctx = pcm.pcm_setup(b.shell_l, b.shell_xyz, b.shell_nprim, b.prim_exp, b.prim_coef, np.zeros((0, 3)), np.zeros(0), gradient=True)
    gs, gp = pcm.pcm_gradient(ctx, dev(torch, w.P), torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert gs.shape == (b.nshell, 3) and gp.shape == (0, 3) and (gs == 0).all()
    pcm.pcm_destroy(ctx)
    ctx = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0), s.xyz, s.zeta, gradient=True)
    gs, gp = pcm.pcm_gradient(ctx, torch.zeros((0, 0), dtype=torch.float64, device="cuda"), dev(torch, w.q))
    assert gs.shape == (0, 3) and gp.shape == (s.M, 3) and (gp == 0).all()
    pcm.pcm_destroy(ctx)
    one = synth.Basis(np.array([1], np.int32), np.array([[0.1, 0.2, 0.3]]), np.array([1], np.int32), np.array([0.9]),
                      np.array([1.3]), np.array([0], np.int32), True)
    s1 = synth.Surface(np.array([[1.0, -0.5, 0.7]]), np.array([2.2]), np.ones(1), np.zeros(1, np.int32))
    P = np.array([[1.0, 0.2, -0.3], [0.2, 0.5, 0.1], [-0.3, 0.1, 2.0]])
    ctx = pcm.setup_from_workload(one, s1, gradient=True)
    gs, gp = pcm.pcm_gradient(ctx, dev(torch, P), dev(torch, [0.7]))
    rs, rp = orc.gradient(one, s1, P, np.array([0.7]))
    check(gs.cpu().numpy(), rs, "one p shell, one point: g_shell")
    check(gp.cpu().numpy(), rp, "one p shell, one point: g_point")
    assert np.abs(gs.cpu().numpy() + gp.cpu().numpy()).max() < 1e-14      # two bodies: equal and opposite
    pcm.pcm_destroy(ctx)
