"""Parity of the solve on an adaptive oct-tree of 8^3 sub-grids (octo_fmm_tree_*, reading R9) against
oracle.solve_tree, through the C ABI (-m gpu).

Bar: the pair set bit-exact (ordered pairs per kind: multipole, leaf-leaf, across a refinement boundary); phi within 1e-12
cell by cell at every leaf of every level (the potential of positive masses never vanishes), g within 1e-12 of the
largest |g| of the tree (it passes through zero)."""
import numpy as np
import pytest

import fmm_inputs as fi
import oracle

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    assert torch.cuda.is_available()
    return p, torch


def _run(env, tree, theta, correction, counts=True, box=None):
    """tree: fmm_inputs.Tree on whole lattices, or (n0, h0, kind, mass) with box given."""
    p, torch = env
    if box is None:
        n0, h0, kind, masses = tree.n0, tree.h0, tree.kind, tree.mass
    else:
        n0, h0, kind, masses = tree
    t = p.OctoFMMTree(n0, h0, theta, kind, correction, box=box)
    mass = [torch.from_numpy(m).cuda() for m in masses]
    if counts:
        cnt, out = t.interaction_counts(mass)
    else:
        cnt, out = None, t.solve(mass)
    torch.cuda.synchronize()
    assert t.status() == p.OK
    res = [o.cpu().numpy() for o in out]
    t.close()
    return res, cnt


def _compare(tree, got, ref):
    gmax = max(np.abs(r[1:]).max() for r in ref)
    worst_phi = worst_g = 0.0
    for l in range(tree.depth):
        leaf = tree.kind[l] == fi.TREE_LEAF
        assert np.all(got[l][:, ~leaf] == 0.0)
        if not leaf.any():
            continue
        worst_phi = max(worst_phi, float((np.abs(got[l][0] - ref[l][0])[leaf] / np.abs(ref[l][0])[leaf]).max()))
        worst_g = max(worst_g, float(np.abs(got[l][1:] - ref[l][1:])[:, leaf].max() / gmax))
    return worst_phi, worst_g


@pytest.mark.parametrize("seed,theta,correction", [(1, 0.5, True), (2, 0.35, True), (3, 0.7, True), (4, 0.5, False)])
def test_seeded_trees(env, seed, theta, correction):
    """Seeded random trees of depth 3 on a 16^3 base (leaves on two levels, refinement boundaries everywhere)."""
    tree = fi.seeded_tree(seed)
    assert fi.tree_is_properly_nested(tree)
    ref, cref = oracle.solve_tree(tree.n0, tree.h0, theta, tree.kind, tree.mass, correction)
    got, cnt = _run(env, tree, theta, correction)
    assert cnt == {k: cref[k] for k in ("m2l", "p2p", "cross")}
    e_phi, e_g = _compare(tree, got, ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)


def test_deep_tree_and_the_paper_like_refinement_pattern(env):
    """Four levels (leaves on three of them), and the two-star field refined around the stars (density-based refinement,
    Eq. 34-35), dynamic range 1e-10."""
    for tree, theta in ((fi.seeded_tree(1, depth=4, frac=0.3), 0.5), (fi.star_tree(16, 3), 0.5)):
        assert fi.tree_is_properly_nested(tree)
        ref, cref = oracle.solve_tree(tree.n0, tree.h0, theta, tree.kind, tree.mass, True)
        got, cnt = _run(env, tree, theta, True)
        assert cnt == {k: cref[k] for k in ("m2l", "p2p", "cross")}
        e_phi, e_g = _compare(tree, got, ref)
        assert e_phi < TOL and e_g < TOL, (e_phi, e_g)


def test_fully_refined_tree_equals_the_uniform_solver(env):
    """No refinement boundary: the tree path must reproduce the uniform solve (oracle) and agree with the uniform GPU
    solver to round-off; a single-level tree (everything a leaf on level 0) as well."""
    p, torch = env
    n, h = 32, 1.0 / 32
    m = np.random.default_rng(3).uniform(0.5, 1.5, (n, n, n)) * h ** 3
    kind = [np.full((8,) * 3, 2, np.uint8), np.full((16,) * 3, 2, np.uint8), np.full((32,) * 3, 1, np.uint8)]
    mass = [np.zeros((8,) * 3), np.zeros((16,) * 3), m]
    tree = fi.Tree(8, 1.0 / 8, kind, mass)
    ref = oracle.solve(n, h, 0.5, m, True)
    got, cnt = _run(env, tree, 0.5, True)
    assert cnt["cross"] == 0
    assert (np.abs(got[2][0] - ref[0]) / np.abs(ref[0])).max() < TOL
    assert np.abs(got[2][1:] - ref[1:]).max() / np.abs(ref[1:]).max() < TOL
    s = p.OctoFMMSolver(n, h, 0.5, True)
    uni = s.solve(torch.from_numpy(m).cuda()).cpu().numpy()
    s.close()
    assert np.abs(got[2] - uni).max() / np.abs(uni).max() < 1e-13
    one = fi.Tree(32, h, [np.full((32,) * 3, 1, np.uint8)], [m])
    got1, _ = _run(env, one, 0.5, True)
    assert (np.abs(got1[0][0] - ref[0]) / np.abs(ref[0])).max() < TOL


def test_conservation_on_the_gpu_result(env):
    """Newton's third law over the leaves of all levels and, with the correction, the torque balance (L125, L127)."""
    tree = fi.seeded_tree(2)
    pos, ms, lv, idx = tree.leaf_points()
    for corr in (True, False):
        got, _ = _run(env, tree, 0.5, corr, counts=False)
        res = np.concatenate([got[l][:, tree.kind[l] == fi.TREE_LEAF].T for l in range(tree.depth)])
        F = ms[:, None] * res[:, 1:4]
        T = np.cross(pos, F)
        assert np.abs(F.sum(0)).max() / np.abs(F).sum() < 1e-14
        t = np.abs(T.sum(0)).max() / np.abs(T).sum()
        assert (t < 1e-13) if corr else (t > 1e-8)


def test_bad_topologies_are_refused(env):
    p, torch = env
    tree = fi.seeded_tree(1)
    bad = [k.copy() for k in tree.kind]
    bad[2][0, 0, 0] = 2 if bad[2][0, 0, 0] != 2 else 1            # not constant over a sub-grid
    with pytest.raises(p.OctoFmmError):
        p.OctoFMMTree(tree.n0, tree.h0, 0.5, bad)
    bad = [k.copy() for k in tree.kind]
    bad[1][:8, :8, :8] = 1                                          # children of a leaf exist (level 2 was built for it)
    if (tree.kind[1][:8, :8, :8] == 2).all():
        with pytest.raises(p.OctoFmmError):
            p.OctoFMMTree(tree.n0, tree.h0, 0.5, bad)
    with pytest.raises(ValueError):
        p.OctoFMMTree(tree.n0, tree.h0, 0.5, [k[:4] for k in tree.kind])


def _compare_lists(kind, got, ref):
    gmax = max(np.abs(r[1:]).max() for r in ref)
    worst_phi = worst_g = 0.0
    for l in range(len(kind)):
        leaf = kind[l] == fi.TREE_LEAF
        assert np.all(got[l][:, ~leaf] == 0.0)
        if leaf.any():
            worst_phi = max(worst_phi, float((np.abs(got[l][0] - ref[l][0])[leaf] / np.abs(ref[l][0])[leaf]).max()))
            worst_g = max(worst_g, float(np.abs(got[l][1:] - ref[l][1:])[:, leaf].max() / gmax))
    return worst_phi, worst_g


@pytest.mark.parametrize("which", ["star", "seeded"])
def test_levels_stored_as_boxes(env, which):
    """The same trees with every level stored as the bounding box of its cells (boxes that shrink and move from level to
    level): pair counts and numbers against the oracle, and bit-identical to the whole-lattice run of the library."""
    tree = fi.star_tree(32, 4) if which == "star" else fi.seeded_tree(3, depth=4, frac=0.25)
    boxes = fi.tree_boxes(tree)
    kind, mass = fi.crop_tree(tree, boxes)
    ref, cref = oracle.solve_tree(tree.n0, tree.h0, 0.5, kind, mass, True, box=boxes)
    got, cnt = _run(env, (tree.n0, tree.h0, kind, mass), 0.5, True, box=boxes)
    assert cnt == {k: cref[k] for k in ("m2l", "p2p", "cross")}
    e_phi, e_g = _compare_lists(kind, got, ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)
    whole, _ = _run(env, tree, 0.5, True, counts=False)
    for l, b in enumerate(boxes):
        assert np.array_equal(whole[l][:, b[2]:b[2] + b[5], b[1]:b[1] + b[4], b[0]:b[0] + b[3]], got[l])


def test_nine_level_tree(env):
    """The paper's production depth (9 levels, L684): 16^3 base cells, a 4096^3 lattice at the bottom, every level a box of
    at most 64 cells per axis around the star -- 1.2 million leaves on eight levels, against the oracle."""
    boxes, kind, mass = fi.nested_tree(16, 9)
    ref, cref = oracle.solve_tree(16, 1.0 / 16, 0.5, kind, mass, True, box=boxes)
    got, cnt = _run(env, (16, 1.0 / 16, kind, mass), 0.5, True, box=boxes)
    assert cnt == {k: cref[k] for k in ("m2l", "p2p", "cross")}
    e_phi, e_g = _compare_lists(kind, got, ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)


def test_bad_boxes_are_refused(env):
    p, torch = env
    tree = fi.star_tree(32, 3)
    boxes = fi.tree_boxes(tree)
    kind, mass = fi.crop_tree(tree, boxes)
    bad = [list(b) for b in boxes]
    bad[1][0] += 4                                             # not aligned to the sub-grids
    with pytest.raises(p.OctoFmmError):
        p.OctoFMMTree(tree.n0, tree.h0, 0.5, kind, box=bad)
    bad = [list(b) for b in boxes]
    bad[2][0] += 8                                             # shifted: the children of a refined sub-grid fall outside / kinds disagree
    with pytest.raises(p.OctoFmmError):
        p.OctoFMMTree(tree.n0, tree.h0, 0.5, kind, box=bad)
    bad = [list(b) for b in boxes]
    bad[0][3] = 16                                             # level 0 must be the whole lattice
    with pytest.raises((p.OctoFmmError, ValueError)):
        p.OctoFMMTree(tree.n0, tree.h0, 0.5, [kind[0][:, :, :16].copy()] + kind[1:], box=bad)


@pytest.mark.parametrize("theta,correction", [(0.35, True), (0.7, False)])
def test_boxes_at_other_opening_angles(env, theta, correction):
    """Boxes + the widest (reach 5) and the narrowest lists, correction on and off."""
    tree = fi.star_tree(32, 3)
    boxes = fi.tree_boxes(tree)
    kind, mass = fi.crop_tree(tree, boxes)
    ref, cref = oracle.solve_tree(tree.n0, tree.h0, theta, kind, mass, correction, box=boxes)
    got, cnt = _run(env, (tree.n0, tree.h0, kind, mass), theta, correction, box=boxes)
    assert cnt == {k: cref[k] for k in ("m2l", "p2p", "cross")}
    e_phi, e_g = _compare_lists(kind, got, ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)


def test_repeated_and_concurrent_solves_are_deterministic(env):
    """The levels of a solve run side by side on streams of the library's own; two trees are driven from two caller
    streams at the same time, several solves each without host synchronisation in between: every solve of a tree gives
    bit-identical results, equal to a solve run alone."""
    p, torch = env
    trees = [fi.seeded_tree(1), fi.seeded_tree(2, depth=4, frac=0.3)]
    alone = []
    for tr in trees:
        got, _ = _run(env, tr, 0.5, True, counts=False)
        alone.append(got)
    streams = [torch.cuda.Stream() for _ in trees]
    handles, masses, outs = [], [], []
    for tr, st in zip(trees, streams):
        h = p.OctoFMMTree(tr.n0, tr.h0, 0.5, tr.kind, True, stream=st)
        with torch.cuda.stream(st):
            masses.append([torch.from_numpy(m).cuda() for m in tr.mass])
        outs.append([h.empty_out() for _ in range(3)])
        handles.append(h)
    torch.cuda.synchronize()
    for rnd in range(3):
        for i in (0, 1):
            handles[i].solve(masses[i], outs[i][rnd])
    torch.cuda.synchronize()
    for i, tr in enumerate(trees):
        assert handles[i].status() == p.OK
        for rnd in range(3):
            for l in range(tr.depth):
                assert np.array_equal(outs[i][rnd][l].cpu().numpy(), alone[i][l])
        handles[i].close()


def test_tree_solve_host_entry_point(env):
    """octo_fmm_tree_solve_host (copies in on the leaf streams, solve, copies out level by level as the finishes end)
    gives the device-pointer route's numbers bit for bit -- on two calls in a row with different masses (the second call
    meets the first call's contents in the scratch), and a device-pointer solve afterwards is unchanged."""
    p, torch = env
    dense = fi.star_tree(32, 3)
    boxes = fi.tree_boxes(dense)
    kinds, masses = fi.crop_tree(dense, boxes)
    t = p.OctoFMMTree(32, dense.h0, 0.5, kinds, True, box=boxes)
    nb = p.octo_fmm_tree_host_scratch_bytes(t.handle)
    scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
    depth = len(kinds)
    for scale in (1.0, 0.37):
        ms = [m * (scale if l % 2 == 0 else 1.0) for l, m in enumerate(masses)]
        dev = [o.cpu().numpy() for o in t.solve([torch.from_numpy(m).cuda() for m in ms])]
        m_h = [torch.from_numpy(np.ascontiguousarray(m)).pin_memory() for m in ms]
        o_h = [torch.full((4,) + t.shape[l], float("nan"), dtype=torch.float64).pin_memory() for l in range(depth)]
        p.octo_fmm_tree_solve_host(t.handle, m_h, o_h, scratch, nb)
        for l in range(depth):
            assert np.array_equal(o_h[l].numpy(), dev[l]), (scale, l)
        again = [o.cpu().numpy() for o in t.solve([torch.from_numpy(m).cuda() for m in ms])]
        for l in range(depth):
            assert np.array_equal(again[l], dev[l])
    assert t.status() == p.OK
    with pytest.raises(p.OctoFmmError):
        p.octo_fmm_tree_solve_host(t.handle, m_h, o_h, scratch, nb - 1)
    t.close()


@pytest.mark.parametrize("boxed", [False, True])
def test_second_right_hand_side_on_the_tree(env, boxed):
    """octo_fmm_tree_solve_rhs2 (L81-83 on the adaptive mesh): d(phi)/dt of signed sources on the tree and centres of the
    density's solve, against oracle.solve_tree_rhs2 at 1e-12 of the largest value; the density's solve is unchanged by it
    (bit-identical before and after); ESTATE before the first solve."""
    p, torch = env
    tree = fi.star_tree(32, 3) if boxed else fi.seeded_tree(2)
    rng = np.random.default_rng(8)
    dm = [rng.normal(size=m.shape) * m for m in tree.mass]
    if boxed:
        boxes = fi.tree_boxes(tree)
        kind, mass = fi.crop_tree(tree, boxes)
        dm = [np.ascontiguousarray(x[b[2]:b[2] + b[5], b[1]:b[1] + b[4], b[0]:b[0] + b[3]]) for x, b in zip(dm, boxes)]
    else:
        boxes, kind, mass = None, tree.kind, tree.mass
    ref = oracle.solve_tree_rhs2(tree.n0, tree.h0, 0.5, kind, mass, dm, box=boxes)
    t = p.OctoFMMTree(tree.n0, tree.h0, 0.5, kind, True, box=boxes)
    m_d = [torch.from_numpy(m).cuda() for m in mass]
    d_d = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in dm]
    with pytest.raises(p.OctoFmmError):
        t.solve_rhs2(d_d)
    before = [o.clone() for o in t.solve(m_d)]
    got = t.solve_rhs2(d_d)
    after = t.solve(m_d)
    torch.cuda.synchronize()
    assert t.status() == p.OK
    scale = max(np.abs(r[0]).max() for r in ref)
    for l in range(tree.depth):
        leaf = kind[l] == fi.TREE_LEAF
        g = got[l].cpu().numpy()
        assert np.all(g[~leaf] == 0.0)
        if leaf.any():
            assert np.abs(g - ref[l][0])[leaf].max() < TOL * scale
        assert torch.equal(before[l], after[l])
    t.close()
