"""GPU parity of the C-PCM glue around the hot path: u = B z (Eq. 4), b = -f (u - v) (Eq. 1),
Delta G_els (Eq. 13) against the oracle, element by element at |gpu - oracle| <= 1e-10 |oracle| + 1e-12, and one full
C-PCM step  v -> b -> q (PCG) -> energy  whose energy must equal the oracle's (dense LAPACK solve) to the CG tolerance."""
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


def close(got, ref):
    return np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref) + 1e-12)


@pytest.mark.parametrize("config,n_atoms", [(0, None), (1, 60)])
def test_nuclear_potential_rhs_energy_parity(pcm, orc, torch_cuda, config, n_atoms):
    w = synth.make_workload(config, n_atoms=n_atoms)
    s = w.surface
    z = synth.nuclear_charges(w.elements)
    ctx = pcm.setup_from_workload(w.basis, s)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_nuclear_potential(ctx)                       # before pcm_set_nuclei
    pcm.pcm_set_nuclei(ctx, w.atom_xyz, z)
    u = pcm.pcm_nuclear_potential(ctx).cpu().numpy()
    u_ref = orc.nuclear_potential(s, w.atom_xyz, z)
    assert close(u, u_ref), np.abs(u - u_ref).max()
    v = pcm.pcm_potential(ctx, dev(torch_cuda, w.P))
    v_ref = orc.potential(w.basis, s, w.P)
    f = (78.39 - 1.0) / 78.39
    b = pcm.pcm_rhs(ctx, dev(torch_cuda, u_ref), dev(torch_cuda, v_ref), f).cpu().numpy()
    assert close(b, orc.rhs(u_ref, v_ref, f))
    q = w.q
    e = pcm.pcm_energy(ctx, dev(torch_cuda, u_ref), dev(torch_cuda, v_ref), dev(torch_cuda, q), f)
    e_ref = orc.energy(u_ref, v_ref, q, orc.amatvec(s, q), f)
    assert close(e, e_ref), (e, e_ref)
    e2 = pcm.pcm_energy(ctx, dev(torch_cuda, u_ref), dev(torch_cuda, v_ref), dev(torch_cuda, q), f)
    assert np.array_equal(e, e2)                              # fixed-order sums
    # one whole step on the device: v -> b -> q -> energy; at the solution Eq. 13 equals (u - v).q / 2
    bd = pcm.pcm_rhs(ctx, pcm.pcm_nuclear_potential(ctx), v, f)
    pcm.pcm_rbj_build(ctx, 64, seed=3)
    qd, it, rr, rt, ok = pcm.pcm_cg_solve(ctx, bd, tol=1e-11, max_iter=2000, precond=2)
    assert ok
    eg = pcm.pcm_energy(ctx, dev(torch_cuda, u), v, qd, f)
    q_ref = np.linalg.solve(orc.amatrix(s), orc.rhs(u_ref, v_ref, f))
    eo = orc.energy(u_ref, v_ref, q_ref, orc.amatvec(s, q_ref), f)
    assert eg[3] == pytest.approx(eo[3], rel=1e-8, abs=1e-10)
    assert eg[3] == pytest.approx(0.5 * float((u - v.cpu().numpy()) @ qd.cpu().numpy()), rel=1e-8, abs=1e-10)
    pcm.pcm_destroy(ctx)


def test_nuclear_potential_near_field_and_edge_cases(pcm, orc, torch_cuda):
    # small exponents and nuclei close to (and on) surface points: the erf branch and the r = 0 limit
    rng = np.random.default_rng(5)
    M, N = 333, 7
    xyz = rng.normal(size=(M, 3)) * 2.0
    zeta = rng.uniform(0.3, 6.0, M)
    atoms = rng.normal(size=(N, 3)) * 1.5
    atoms[0] = xyz[10]                                        # a nucleus exactly on a surface point
    atoms[1] = xyz[20] + 1e-9
    z = rng.uniform(-3, 8, N)
    s = synth.Surface(xyz=xyz, zeta=zeta, switch=np.ones(M), atom=np.zeros(M, np.int32))
    e = np.zeros(0)
    ctx = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), e, e, xyz, zeta, s.switch)
    pcm.pcm_set_nuclei(ctx, atoms, z)
    u = pcm.pcm_nuclear_potential(ctx).cpu().numpy()
    assert np.isfinite(u).all()
    assert close(u, orc.nuclear_potential(s, atoms, z))
    pcm.pcm_set_nuclei(ctx, np.zeros((0, 3)), np.zeros(0))    # no nuclei: u = 0
    assert (pcm.pcm_nuclear_potential(ctx).cpu().numpy() == 0).all()
    pcm.pcm_set_nuclei(ctx, atoms[:3], z[:3])                 # replaced by a smaller set
    assert close(pcm.pcm_nuclear_potential(ctx).cpu().numpy(), orc.nuclear_potential(s, atoms[:3], z[:3]))
    pcm.pcm_destroy(ctx)
