"""Parity of the complete uniform-grid solve (octo_fmm_solver_*, NEXT f1) against the oracle's, through the C ABI.

Bar: leaf list bit-exact, interaction count exact, phi within 1e-12 CELL BY CELL (the potential of positive masses never
vanishes) and g within 1e-12 of the grid's largest |g| (cell-wise normalisation is meaningless where g passes through
zero at a star's centre)."""
import os

import numpy as np
import pytest

import fmm_inputs as fi
import oracle
from helpers import load_golden

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


def _errors(got, ref):
    return ((np.abs(got[0] - ref[0]) / np.abs(ref[0])).max(), np.abs(got[1:] - ref[1:]).max() / np.abs(ref[1:]).max())


def _oracle_count(n, theta):
    total = 0
    m = n // 2
    while m >= 2:
        total += oracle.interaction_count((m, m, m), theta)
        m //= 2
    return total


@pytest.mark.parametrize("theta", [0.5, 0.35, 0.7])
def test_leaf_list_bit_exact(env, theta):
    p, torch = env
    s = p.OctoFMMSolver(16, 1.0 / 16, theta)
    for par in range(8):
        assert np.array_equal(s.leaf_stencil(par), oracle.stencil_leaf(theta, par))
    s.close()


@pytest.mark.parametrize("theta,correction", [(0.5, True), (0.5, False), (0.35, True), (0.7, True)])
def test_random_masses_32(env, theta, correction):
    """32^3 random masses: levels 32 (leaves), 16, 8 (staged kernel), 4, 2 (direct kernel)."""
    p, torch = env
    n, h = 32, 1.0 / 32
    mass = np.random.default_rng(11).uniform(0.5, 1.5, (n, n, n)) * h ** 3
    s = p.OctoFMMSolver(n, h, theta, correction)
    out = s.solve(torch.from_numpy(mass).cuda())
    torch.cuda.synchronize()
    assert s.status() == p.OK
    ref = oracle.solve(n, h, theta, mass, correction)
    leaf_cnt = oracle.interact_monopole_leaf((n, n, n), h, theta, mass)[1]
    assert s.interaction_count() == leaf_cnt + _oracle_count(n, theta)
    assert s.leaf_interaction_count() == leaf_cnt
    assert s.num_levels() == (4, 18)       # the tensor-core leaf kernel evaluates the parent expansion itself
    e_phi, e_g = _errors(out.cpu().numpy(), ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)
    s.close()


def test_binary_field_64_and_conservation(env):
    """64^3 two-polytrope field (cfg-4 masses, dynamic range 1e-10): parity, then the paper's invariants on the GPU
    result -- linear momentum to machine precision (L125) and, with the correction, angular momentum (L127)."""
    p, torch = env
    w = fi.config4(ncell=64)
    n, h, mass = 64, w.h, np.ascontiguousarray(w.moments[0])
    s = p.OctoFMMSolver(n, h, 0.5, True)
    out = s.solve(torch.from_numpy(mass).cuda()).cpu().numpy()
    assert s.status() == p.OK
    ref = oracle.solve(n, h, 0.5, mass, True)
    e_phi, e_g = _errors(out, ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)
    x = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    F = mass[None] * out[1:]
    T = np.cross(np.stack([X, Y, Z]), F, axis=0)
    assert np.abs(F.sum(axis=(1, 2, 3))).max() / np.abs(F).sum() < 1e-14
    assert np.abs(T.sum(axis=(1, 2, 3))).max() / np.abs(T).sum() < 1e-13
    s.close()


@pytest.mark.parametrize("n,theta", [(128, 0.5), (256, 0.5), (512, 0.5), (128, 0.35), (256, 0.35)])
def test_uniform_sphere_residuals_table1(env, n, theta):
    """Section 3.4 on the GPU at the grids of Table 1 (tests/golden/table1_sphere.txt): residuals against the
    analytic potential within a factor 3 of the printed max and mean (the paper does not state its rasterisation nor
    how a cell's own mass enters), the maximum outside the sphere (L456)."""
    p, torch = env
    golden = load_golden(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "table1_sphere.txt"))
    rows = {(int(a), float(b)): (float(c), float(d)) for a, b, c, d in golden["_multi"]["sphere"]}
    pmax, pmean = rows[(n, theta)]
    h = 1.0 / n
    x = (np.arange(n) + 0.5) * h - 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r = np.sqrt(X * X + Y * Y + Z * Z)
    rho = np.where(r < 0.25, 1.0, 1e-10)
    mass = rho / rho.sum()
    phi = np.where(r < 0.25, -(3 * 0.0625 - r * r) / (2 * 0.25 ** 3), -1.0 / r)
    s = p.OctoFMMSolver(n, h, theta, True)
    out = s.solve(torch.from_numpy(mass).cuda())
    torch.cuda.synchronize()
    assert s.status() == p.OK
    eps = np.abs(out[0].cpu().numpy() - phi) / np.abs(phi)
    assert pmax / 3 < eps.max() < pmax * 3 and pmean / 3 < eps.mean() < pmean * 3, (eps.max(), eps.mean())
    assert r[np.unravel_index(np.argmax(eps), eps.shape)] > 0.25
    s.close()
    del out
    torch.cuda.empty_cache()


def test_solver_rejects_bad_configurations(env):
    p, torch = env
    for n, theta in ((24, 0.5), (8, 0.5), (32, 0.3), (32, 1.0)):
        assert p.octo_fmm_solver_workspace_bytes(p.make_solver_config(n, 1.0 / n, theta)) == 0
        with pytest.raises(p.OctoFmmError):
            p.octo_fmm_solver_create(p.make_solver_config(n, 1.0 / n, theta))
    with pytest.raises(p.OctoFmmError):          # no workspace
        p.octo_fmm_solver_create(p.make_solver_config(32, 1.0 / 32, 0.5))


def test_solve_host_entry_point(env):
    """octo_fmm_solver_solve_host (H2D + solve + D2H) gives the device-pointer route's numbers bit for bit."""
    p, torch = env
    n = 32
    h, mass, _, _ = fi.uniform_sphere(n)
    s = p.OctoFMMSolver(n, h, 0.5, True)
    dev_out = s.solve(torch.from_numpy(mass).cuda()).cpu().numpy()
    nb = p.octo_fmm_solver_host_scratch_bytes(s.cfg)
    scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
    m_h = torch.from_numpy(mass).pin_memory()
    o_h = torch.full((4, n, n, n), float("nan"), dtype=torch.float64).pin_memory()
    p.octo_fmm_solver_solve_host(s.handle, m_h, o_h, scratch, nb)
    assert np.array_equal(o_h.numpy(), dev_out)
    with pytest.raises(p.OctoFmmError):
        p.octo_fmm_solver_solve_host(s.handle, m_h, o_h, scratch, nb - 1)
    s.close()


@pytest.mark.parametrize("theta", [0.5, 0.35])
def test_second_right_hand_side_32(env, theta):
    """f2 (L81-83): d(phi)/dt from d(mass)/dt on the tree and the expansion centres of the density's solve, no
    correction, against the oracle's solve_rhs2; signed sources with zero net change.  The leaf sum of this pass is
    the potential-only tensor-core kernel (rows = the 8 children of a parent)."""
    p, torch = env
    n, h = 32, 1.0 / 32
    rng = np.random.default_rng(12)
    mass = rng.uniform(0.5, 1.5, (n, n, n)) * h ** 3
    dm = rng.uniform(-1.0, 1.0, (n, n, n)) * h ** 3
    dm -= dm.mean()
    s = p.OctoFMMSolver(n, h, theta, True)
    with pytest.raises(p.OctoFmmError):                       # no centres before the first solve
        s.solve_rhs2(torch.from_numpy(dm).cuda())
    out = s.solve(torch.from_numpy(mass).cuda()).clone()
    out2 = s.solve_rhs2(torch.from_numpy(dm).cuda())
    torch.cuda.synchronize()
    assert s.status() == p.OK
    ref2 = oracle.solve_rhs2(n, h, theta, mass, dm)[0]
    e_phi = np.abs(out2.cpu().numpy() - ref2).max() / np.abs(ref2).max()
    assert e_phi < TOL, e_phi
    # the density's solve is unchanged by the second right-hand side having run on the same handles
    again = s.solve(torch.from_numpy(mass).cuda())
    torch.cuda.synchronize()
    assert torch.equal(again, out)
    ref = oracle.solve(n, h, theta, mass, True)
    e_phi, e_g = _errors(out.cpu().numpy(), ref)
    assert e_phi < TOL and e_g < TOL, (e_phi, e_g)
    s.close()


@pytest.mark.parametrize("theta,n", [(0.5, 32), (0.35, 32), (0.5, 64)])
def test_both_right_hand_sides_in_one_call(env, theta, n):
    """octo_fmm_solver_solve2 (f2: L81-83, Alg. 1): (phi, g) of the density AND d(phi)/dt of its time derivative from
    ONE call -- against oracle.solve and oracle.solve_rhs2 at 1e-12, with the fused kernel on the one-warp-per-cell levels
    only (default) and on every level ("f2_fused" = 1), and against the two separate calls."""
    p, torch = env
    h = 1.0 / n
    rng = np.random.default_rng(12 + n)
    mass = rng.uniform(0.5, 1.5, (n, n, n)) * h ** 3
    dm = rng.uniform(-1.0, 1.0, (n, n, n)) * h ** 3
    dm -= dm.mean()
    ref = oracle.solve(n, h, theta, mass, True)
    ref2 = oracle.solve_rhs2(n, h, theta, mass, dm)[0]
    s = p.OctoFMMSolver(n, h, theta, True, two_rhs=True)
    m_d, dm_d = torch.from_numpy(mass).cuda(), torch.from_numpy(dm).cuda()
    sep = s.solve(m_d).clone()
    sep2 = s.solve_rhs2(dm_d).clone()
    for fused in (0, 1):
        s.set_option("f2_fused", fused)
        out, dphi = s.solve2(m_d, dm_d)
        torch.cuda.synchronize()
        assert s.status() == p.OK
        e_phi, e_g = _errors(out.cpu().numpy(), ref)
        e2 = np.abs(dphi.cpu().numpy() - ref2).max() / np.abs(ref2).max()
        assert e_phi < TOL and e_g < TOL and e2 < TOL, (fused, e_phi, e_g, e2)
        assert float((out - sep).abs().max() / sep.abs().max()) < 1e-13
        assert float((dphi - sep2).abs().max() / sep2.abs().max()) < 1e-13
    s.close()
    plain = p.OctoFMMSolver(n, h, theta, True)
    with pytest.raises(p.OctoFmmError):                      # needs the second set of buffers
        plain.solve2(m_d, dm_d)
    plain.close()
