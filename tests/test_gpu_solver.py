"""GPU checks of the randomized block-Jacobi build and pcm_cg_solve against the
oracle.  The 1e-10 parity bar applies to v, F and A q entries; the iterative solve is pinned by its residual, by
dense LAPACK on small M, by the oracle's iteration count (+-2) and by the paper's qualitative statements
(block size 1 = Jacobi, block size M = one step, RBJ beats Jacobi for M >~ 1000).

Block selection decides integers from floating point (the l-1 largest A_kj): both sides evaluate A_kj in fp64 but
not bit-identically (libm erf vs tabulated Boys), so near-ties may legitimately be ordered differently.  The test
therefore checks what is unique (partition, sizes, pivots) and that every chosen set is valid with respect to the
oracle's A to a relative 1e-12, and compares the block sets exactly where no near-tie exists.
"""
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


def points_ctx(pcm, s, **kw):
    z = np.zeros(0)
    return pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), z, z, s.xyz, s.zeta, s.switch, **kw)


@pytest.fixture(scope="module")
def sys2500(pcm, orc):
    s, q, q_true = synth.make_solver_points(2500, seed=1004)
    A = orc.amatrix(s)
    return s, A, q_true, points_ctx(pcm, s)


@pytest.mark.parametrize("l", [1, 7, 64, 100])
def test_rbj_blocks_valid(pcm, orc, sys2500, l):
    s, A, _, ctx = sys2500
    M = s.M
    piv = pcm.pcm_pivot_order(77, M)
    pcm.pcm_rbj_build(ctx, l, seed=77)
    order, bstart, inv = pcm.pcm_rbj_get(ctx)
    info = pcm.pcm_get_info(ctx)
    assert info.rbj_block == l and info.rbj_nblocks == (M + l - 1) // l == len(bstart) - 1
    assert sorted(order.tolist()) == list(range(M))
    sizes = np.diff(bstart)
    assert (sizes[:-1] == l).all() and 0 < sizes[-1] <= l
    o_order, o_bstart, _ = orc.rbj_build(s, l, piv)
    np.testing.assert_array_equal(bstart, o_bstart)
    assigned = np.zeros(M, bool)
    pos = 0
    same_sets = 0
    for b in range(len(sizes)):
        idx = order[bstart[b]:bstart[b + 1]]
        while assigned[piv[pos]]:
            pos += 1
        k = piv[pos]
        assert idx[0] == k
        rest = np.flatnonzero(~assigned)
        rest = rest[rest != k]
        chosen = idx[1:]
        assert not assigned[chosen].any()
        if len(chosen) and len(rest) > len(chosen):
            excluded = np.setdiff1d(rest, chosen)
            assert A[k, chosen].min() >= A[k, excluded].max() * (1 - 1e-12)
        assert (np.diff(A[k, chosen]) <= 1e-12 * A[k, chosen][1:]).all()
        assigned[idx] = True
        same_sets += set(idx.tolist()) == set(o_order[bstart[b]:bstart[b + 1]].tolist())
        n = len(idx)
        np.testing.assert_allclose(inv[b] @ A[np.ix_(idx, idx)], np.eye(n), atol=1e-9)
        np.testing.assert_array_equal(inv[b], inv[b].T)
    assert same_sets == len(sizes)  # no near-ties in this geometry: the partition equals the oracle's


def test_rbj_given_pivot_order_and_bad_input(pcm, sys2500):
    s, _, _, ctx = sys2500
    perm = np.random.default_rng(1).permutation(s.M)
    pcm.pcm_rbj_build(ctx, 32, pivot_order=perm)
    order, bstart, _ = pcm.pcm_rbj_get(ctx)
    assert order[0] == perm[0]
    bad = perm.copy()
    bad[0] = bad[1]
    with pytest.raises(pcm.PcmError):
        pcm.pcm_rbj_build(ctx, 32, pivot_order=bad)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_rbj_build(ctx, 0)


def test_cg_matches_lapack_and_oracle(pcm, orc, sys2500, torch_cuda):
    s, A, q_true, ctx = sys2500
    b = A @ q_true
    x_ref = np.linalg.solve(A, b)
    piv = pcm.pcm_pivot_order(5, s.M)
    pcm.pcm_rbj_build(ctx, 64, seed=5)
    o_rbj = orc.rbj_build(s, 64, piv)
    iters = {}
    for name, precond, okw in (("none", 0, {}), ("jacobi", 1, {}), ("rbj", 2, dict(rbj=o_rbj))):
        x, it, rr, rt, ok = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-8, max_iter=2000, precond=precond)
        assert ok and rr <= 1e-8 and rt <= 2e-8
        np.testing.assert_allclose(x.cpu().numpy(), x_ref, rtol=0, atol=2e-7)
        _, o_it, _, _ = orc.pcg(s, b, 1e-8, 2000, precond=precond, A=A, **okw)
        assert abs(it - o_it) <= 2, (name, it, o_it)
        iters[name] = it
        xh, ith, _, _, okh = pcm.pcm_cg_solve_host(ctx, b, tol=1e-8, max_iter=2000, precond=precond)
        assert okh and ith == it
        np.testing.assert_array_equal(xh, x.cpu().numpy())
    assert iters["rbj"] < iters["jacobi"]


def test_cg_block_one_is_jacobi_and_block_M_is_one_step(pcm, orc, torch_cuda):
    w = synth.make_workload(1, n_atoms=12, with_density=False, seed=5)
    s = w.surface
    ctx = points_ctx(pcm, s)
    b = np.random.default_rng(0).uniform(-1, 1, s.M)
    xj, itj, *_ = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-9, precond=1)
    pcm.pcm_rbj_build(ctx, 1, seed=3)
    x1, it1, *_ = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-9, precond=2)
    assert abs(it1 - itj) <= 1
    np.testing.assert_allclose(x1.cpu().numpy(), xj.cpu().numpy(), rtol=0, atol=1e-8)
    pcm.pcm_rbj_build(ctx, s.M, seed=3)       # block size = dimension of A -> CG converges in 1 step
    xM, itM, rr, rt, ok = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-8, precond=2)
    assert ok and itM == 1 and rt < 1e-8


def test_cg_warm_start_max_iter_and_errors(pcm, orc, sys2500, torch_cuda):
    s, A, q_true, ctx = sys2500
    b = A @ q_true
    x, it, rr, rt, ok = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-8, precond=1)
    x2, it2, _, _, ok2 = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), x=x.clone(), tol=1e-8, precond=1, use_x0=True)
    assert ok2 and it2 == 0
    x3, it3, rr3, _, ok3 = pcm.pcm_cg_solve(ctx, dev(torch_cuda, b), tol=1e-8, max_iter=3, precond=1)
    assert not ok3 and it3 == 3 and rr3 > 1e-8
    fresh = points_ctx(pcm, s)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_cg_solve(fresh, dev(torch_cuda, b), precond=2)   # RBJ before pcm_rbj_build
    with pytest.raises(pcm.PcmError):
        pcm.pcm_cg_solve(fresh, dev(torch_cuda, b), precond=9)


def test_rbj_build_async_equals_sync(pcm, orc, sys2500, torch_cuda):
    """pcm_rbj_build_async on a side stream: same blocks and inverses as the synchronous build, completed by pcm_cg_solve
    (or pcm_rbj_get); the seeded pivot order is reused from the previous build with the same seed."""
    torch = torch_cuda
    s, A, q_true, ctx = sys2500
    pcm.pcm_rbj_build(ctx, 64, seed=5)
    o1, b1, i1 = pcm.pcm_rbj_get(ctx)
    side = torch.cuda.Stream()
    pcm.pcm_rbj_build_async(ctx, 32, seed=9, stream=side)      # something else in between
    pcm.pcm_rbj_build_async(ctx, 64, seed=5, stream=side)      # waits for the pending one first
    b = dev(torch, A @ q_true)
    x, it, rr, rt, ok = pcm.pcm_cg_solve(ctx, b, tol=1e-10, max_iter=500, precond=2)
    assert ok and np.abs(x.cpu().numpy() - q_true).max() < 1e-8
    o2, b2, i2 = pcm.pcm_rbj_get(ctx)
    assert np.array_equal(o1, o2) and np.array_equal(b1, b2) and all(np.array_equal(a, c) for a, c in zip(i1, i2))
    pcm.pcm_rbj_build(ctx, 64, seed=5)
    x2, it2, *_ = pcm.pcm_cg_solve(ctx, b, tol=1e-10, max_iter=500, precond=2)
    assert it2 == it and torch.equal(x, x2)
    pcm.pcm_rbj_build_async(ctx, 64, seed=5, stream=side)
    o3, _, _ = pcm.pcm_rbj_get(ctx)                            # pcm_rbj_get completes a pending build too
    assert np.array_equal(o1, o3)
    with pytest.raises(pcm.PcmError):
        pcm.pcm_rbj_build_async(ctx, 0, seed=1, stream=side)


def test_fused_cg_and_neighbourhood_selection_are_exact_rewrites(pcm, orc, sys2500, torch_cuda):
    """DESIGN.md claims that (i) the one-CTA neighbourhood block selection finds the blocks of the global row scan and
    (ii) the fused cooperative CG update kernel of the separate-launch path reproduces the separate kernels bit for bit.
    Both have a switch in pcm_options (cg_path = 1 / 3, rbj_global_scan)."""
    torch = torch_cuda
    s, A, q_true, _ = sys2500
    c_fused, c_sep, c_glob = points_ctx(pcm, s, cg_path=1), points_ctx(pcm, s, cg_path=3), points_ctx(pcm, s, cg_path=1, rbj_global_scan=True)
    b = dev(torch, A @ q_true)
    for c in (c_fused, c_sep, c_glob):
        pcm.pcm_rbj_build(c, 48, seed=11)
    o_local, b_local, inv_local = pcm.pcm_rbj_get(c_fused)
    x_fused, it_fused, rr_fused, _, ok = pcm.pcm_cg_solve(c_fused, b, tol=1e-10, max_iter=500, precond=2)
    assert ok
    x_sep, it_sep, rr_sep, _, ok = pcm.pcm_cg_solve(c_sep, b, tol=1e-10, max_iter=500, precond=2)
    assert ok and it_sep == it_fused and rr_sep == rr_fused and torch.equal(x_sep, x_fused)
    o_glob, b_glob, inv_glob = pcm.pcm_rbj_get(c_glob)
    assert np.array_equal(o_local, o_glob) and np.array_equal(b_local, b_glob)
    assert all(np.array_equal(a, c) for a, c in zip(inv_local, inv_glob))
    for c in (c_fused, c_sep, c_glob):
        pcm.pcm_destroy(c)


@pytest.mark.parametrize("M", [300, 2500, 9000, 23000])
def test_persistent_solve_equals_the_separate_launch_path(pcm, orc, torch_cuda, M):
    """Below 26k points pcm_cg_solve runs every iteration inside one persistent cooperative kernel and pcm_amatvec is one
    launch (pcm_cgp.cu); pcm_options.cg_path = 1 keeps the separate launches.  Same recurrences, another (fixed) order of the
    A q partial sums: A q agrees to rounding, the iteration counts are equal (up to one, when the residual of an iteration sits
    at the tolerance) and the solutions agree to 1e-11 where the counts are equal."""
    torch = torch_cuda
    s, q, q_true = synth.make_solver_points(M, seed=1004)
    cp, cr = points_ctx(pcm, s), points_ctx(pcm, s, cg_path=1)
    assert pcm.pcm_get_info(cp).amat_persistent == 1 and pcm.pcm_get_info(cr).amat_persistent == 0
    qd = dev(torch, q)
    yp, yr = pcm.pcm_amatvec(cp, qd).cpu().numpy(), pcm.pcm_amatvec(cr, qd).cpu().numpy()
    assert np.all(np.abs(yp - yr) <= 1e-13 * np.abs(yr) + 1e-15)
    assert np.array_equal(pcm.pcm_amatvec(cp, qd).cpu().numpy(), yp)                 # fixed order: bit-reproducible
    rows = np.arange(M) if M <= 2500 else np.random.default_rng(M).choice(M, 64, replace=False)
    ref = orc.amatvec(s, q, rows=rows)
    assert np.all(np.abs(yp[rows] - ref) <= 1e-10 * np.abs(ref) + 1e-12)
    b = pcm.pcm_amatvec(cr, dev(torch, q_true))
    for c in (cp, cr):
        pcm.pcm_rbj_build(c, 64, seed=7)
    for precond in (0, 1, 2):
        xp, itp, rrp, rtp, okp = pcm.pcm_cg_solve(cp, b, tol=1e-9, max_iter=3000, precond=precond)
        xr, itr, rrr, rtr, okr = pcm.pcm_cg_solve(cr, b, tol=1e-9, max_iter=3000, precond=precond)
        assert okp and okr and abs(itp - itr) <= 1, (precond, itp, itr)
        assert rtp <= 2e-9 and float((xp - xr).abs().max()) <= (1e-11 if itp == itr else 1e-9)
        xp2, itp2, rrp2, _, _ = pcm.pcm_cg_solve(cp, b, tol=1e-9, max_iter=3000, precond=precond)
        assert itp2 == itp and rrp2 == rrp and torch.equal(xp, xp2)                  # bit-reproducible run to run
    assert float((xp - dev(torch, q_true)).abs().max()) < 1e-7
    # max_iter and warm start behave as on the reference path
    x3, it3, rr3, _, ok3 = pcm.pcm_cg_solve(cp, b, tol=1e-9, max_iter=3, precond=2)
    assert not ok3 and it3 == 3
    x4, it4, _, _, ok4 = pcm.pcm_cg_solve(cp, b, x=xp.clone(), tol=1e-8, precond=2, use_x0=True)
    assert ok4 and it4 == 0
    for c in (cp, cr):
        pcm.pcm_destroy(c)


def test_cg_non_finite_right_hand_side_is_an_error(pcm, torch_cuda):
    s, q, _ = synth.make_solver_points(300, seed=1004)
    for path in (0, 1):
        c = points_ctx(pcm, s, cg_path=path)
        b = dev(torch_cuda, q)
        b[5] = float("nan")
        with pytest.raises(pcm.PcmError):
            pcm.pcm_cg_solve(c, b, tol=1e-8, precond=1)
        pcm.pcm_destroy(c)


@pytest.mark.parametrize("M", [700, 3000])
def test_stored_far_field_equals_the_on_the_fly_sweep(pcm, orc, torch_cuda, M):
    """SURVEY.md 8(f) rank 3 ('A is explicitly stored'): pcm_options.store_far keeps the far-field 1/r values the
    sweep would evaluate (on top of the stored near patches), and the sweep reads them back in the same order -- A q and the
    solve are bit-identical to the on-the-fly path, and equal to the oracle.  The default stores when everything fits in L2."""
    torch = torch_cuda
    s, q, q_true = synth.make_solver_points(M, seed=1004)
    c_store, c_fly, c_auto = points_ctx(pcm, s, store_far=1), points_ctx(pcm, s, store_far=-1), points_ctx(pcm, s)
    i_store, i_fly, i_auto = (pcm.pcm_get_info(c) for c in (c_store, c_fly, c_auto))
    assert i_store.amat_persistent == 1 and i_fly.amat_persistent == 1
    assert i_fly.amat_far_stored_bytes == 0 and i_store.amat_far_stored_bytes > 0
    assert i_auto.amat_far_stored_bytes == i_store.amat_far_stored_bytes          # a few MB: resident in L2, the rule stores
    assert i_store.amat_far_stored_bytes + i_store.amat_stored_bytes >= 8 * (M * (M - 1) // 2)   # every pair is stored once at least
    qd = dev(torch, q)
    ys, yf = pcm.pcm_amatvec(c_store, qd).cpu().numpy(), pcm.pcm_amatvec(c_fly, qd).cpu().numpy()
    assert np.array_equal(ys, yf)
    ref = orc.amatvec(s, q)
    assert np.all(np.abs(ys - ref) <= 1e-10 * np.abs(ref) + 1e-12)
    e = np.zeros(M)
    e[M // 3] = 1.0
    col = pcm.pcm_amatvec(c_store, dev(torch, e)).cpu().numpy()
    refc = np.array([orc.a_entry(s, i, M // 3) for i in range(M)])
    assert np.all(np.abs(col - refc) <= 1e-10 * np.abs(refc) + 1e-12)            # single stored entries
    b = dev(torch, orc.amatvec(s, q_true))
    for c in (c_store, c_fly):
        pcm.pcm_rbj_build(c, 64, seed=7)
    for precond in (1, 2):
        xs, its, rrs, _, oks = pcm.pcm_cg_solve(c_store, b, tol=1e-9, precond=precond)
        xf, itf, rrf, _, okf = pcm.pcm_cg_solve(c_fly, b, tol=1e-9, precond=precond)
        assert oks and okf and its == itf and rrs == rrf and torch.equal(xs, xf)
    assert float((xs - dev(torch, q_true)).abs().max()) < 1e-7
    for c in (c_store, c_fly, c_auto):
        pcm.pcm_destroy(c)


def test_store_far_rule_leaves_large_cavities_on_the_fly(pcm):
    s, _, _ = synth.make_solver_points(9000, seed=1004)
    c = points_ctx(pcm, s)
    info = pcm.pcm_get_info(c)
    assert info.amat_persistent == 1 and info.amat_far_stored_bytes == 0      # 4 M^2 = 324 MB does not stay in L2
    pcm.pcm_destroy(c)
    s, _, _ = synth.make_solver_points(30000, seed=1004)
    c = points_ctx(pcm, s)
    assert pcm.pcm_get_info(c).amat_persistent == 0                            # 20k points and more: separate launches
    pcm.pcm_destroy(c)


def test_rbj_neighbourhood_radius_is_bisected_when_candidates_overflow(pcm, torch_cuda):
    """A sparse shell of points around a dense ball of 6 000: when a pivot of the shell has used up its sparse neighbours, the next
    growth step of its search radius takes in the whole ball -- more candidates than the one-CTA selection stores.  The radius is
    then bisected between the last one that was too small and the one that overflowed; the selection stays with the one-CTA
    form (rbj_selection = 1) and finds the blocks of the global row scan."""
    rng = np.random.default_rng(5)
    nb, ns = 6000, 1500
    d = rng.normal(size=(nb, 3))
    ball = d / np.linalg.norm(d, axis=1)[:, None] * 1.5 * rng.uniform(0, 1, (nb, 1)) ** (1 / 3)
    d = rng.normal(size=(ns, 3))
    shell = d / np.linalg.norm(d, axis=1)[:, None] * rng.uniform(6.0, 40.0, (ns, 1))
    xyz = np.concatenate([shell, ball])
    M = nb + ns
    s = synth.Surface(xyz=xyz, zeta=rng.uniform(4.0, 6.0, M), switch=rng.uniform(0.2, 1.0, M), atom=np.zeros(M, np.int32))
    po = np.arange(M, dtype=np.int64)               # the shell's points are the first pivots
    c_loc, c_scan = points_ctx(pcm, s), points_ctx(pcm, s, rbj_global_scan=True)
    pcm.pcm_rbj_build(c_loc, 64, pivot_order=po)
    pcm.pcm_rbj_build(c_scan, 64, pivot_order=po)
    assert pcm.pcm_get_info(c_loc).rbj_selection == 1 and pcm.pcm_get_info(c_scan).rbj_selection == 2
    o1, b1, i1 = pcm.pcm_rbj_get(c_loc)
    o2, b2, i2 = pcm.pcm_rbj_get(c_scan)
    assert sorted(o1.tolist()) == list(range(M))
    assert np.array_equal(o1, o2) and np.array_equal(b1, b2)
    assert all(np.array_equal(a, b) for a, b in zip(i1, i2))
    for c in (c_loc, c_scan):
        pcm.pcm_destroy(c)


def test_rbj_capacity_fallback_sync_and_async(pcm, orc, torch_cuda):
    """One point at the centre of a sphere that carries 4 999 others, the centre first in the pivot order: every radius of the
    one-CTA neighbourhood selection holds either no candidate or 4 999 of them, more than its store takes, and bisecting the
    radius cannot separate points that are equally far -- it reports 'capacity' and the build repeats with the global row
    scan (pcm_info.rbj_selection = 3).  Synchronous build, asynchronous build (completed by pcm_rbj_get) and a build forced
    onto the scan give the same blocks; the blocks are valid against the oracle's A, and the preconditioned solve converges."""
    torch = torch_cuda
    rng = np.random.default_rng(23)
    M = 5000
    d = rng.normal(size=(M, 3))
    xyz = d / np.linalg.norm(d, axis=1)[:, None] * 2.0
    xyz[0] = 0.0
    s = synth.Surface(xyz=xyz, zeta=rng.uniform(4.0, 6.0, M), switch=rng.uniform(0.2, 1.0, M), atom=np.zeros(M, np.int32))
    po = np.arange(M, dtype=np.int64)
    c_sync, c_async, c_scan = points_ctx(pcm, s), points_ctx(pcm, s), points_ctx(pcm, s, rbj_global_scan=True)
    pcm.pcm_rbj_build(c_sync, 64, pivot_order=po)
    side = torch.cuda.Stream()
    pcm.pcm_rbj_build_async(c_async, 64, pivot_order=po, stream=side)
    pcm.pcm_rbj_build(c_scan, 64, pivot_order=po)
    o1, b1, i1 = pcm.pcm_rbj_get(c_sync)
    o2, b2, i2 = pcm.pcm_rbj_get(c_async)          # completes the pending build (and its fallback)
    o3, b3, i3 = pcm.pcm_rbj_get(c_scan)
    assert [pcm.pcm_get_info(c).rbj_selection for c in (c_sync, c_async, c_scan)] == [3, 3, 2]
    assert o1[0] == 0
    assert sorted(o1.tolist()) == list(range(M))
    assert np.array_equal(o1, o2) and np.array_equal(o1, o3) and np.array_equal(b1, b3)
    assert all(np.array_equal(a, b) and np.array_equal(a, c) for a, b, c in zip(i1, i2, i3))
    A = orc.amatrix(s)
    blk = o1[b1[0]:b1[1]]
    np.testing.assert_allclose(i1[0] @ A[np.ix_(blk, blk)], np.eye(len(blk)), atol=1e-7)
    q_true = rng.uniform(-0.05, 0.05, M)
    b = dev(torch, A @ q_true)
    x, it, rr, rt, ok = pcm.pcm_cg_solve(c_async, b, tol=1e-8, max_iter=5000, precond=2)
    assert ok and rt < 2e-8
    for c in (c_sync, c_async, c_scan):
        pcm.pcm_destroy(c)
