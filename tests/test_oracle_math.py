"""Pins of the oracle's pair arithmetic (SURVEY 8(c) W1, P6, P7, P9, P10 and a convergence-order pin).

The expected values come from (i) the worked example W1, (ii) sympy differentiating -1/r,
(iii) the exact potential of point masses: the truncated expansion
    L^(n) = sum_{m <= 3-n} ((-1)^m/m!) M^(m) . D^(n+m)
is the Taylor series of the exact derivative in the source offsets, so with sources of extent
eps its error must scale like eps^(4-n).  A wrong sign, factorial, multiplicity or index in the
(n, m) term leaves an O(eps^m) error with m <= 3-n and breaks the observed order.
"""
import os

import numpy as np
import pytest

import oracle
from helpers import (IDX3, exact_local_expansion, full3, green_tensor, load_golden, moments_of_points,
                     unique2, unique3)

W1 = load_golden(os.path.join(os.path.dirname(__file__), "golden", "w1_pair.txt"))


def test_worked_example_w1():
    L, dL1 = oracle.pair(W1["R"], W1["MB"], float(W1["MA0"][0]), W1["MA3"], correction=True)
    np.testing.assert_allclose(L[0], W1["L0"][0], rtol=2e-15)
    np.testing.assert_allclose(L[1:4], W1["L1"], rtol=5e-15)
    np.testing.assert_allclose(L[4:10], W1["L2"], rtol=2e-14)
    np.testing.assert_allclose(L[10:20], W1["L3"], rtol=2e-14)
    np.testing.assert_allclose(dL1, W1["dL1"], rtol=1e-13)
    D = oracle.green(W1["R"])
    np.testing.assert_allclose(D[4][0, 0, 0, 0], W1["D4_xxxx"][0], rtol=1e-14)
    np.testing.assert_allclose(D[4][0, 0, 1, 2], W1["D4_xxyz"][0], rtol=1e-14)
    np.testing.assert_allclose(D[4][1, 1, 2, 2], W1["D4_yyzz"][0], rtol=1e-13)


def test_w1_monopole_pair():
    """W1's monopole line through the monopole entry point: a 2-cell grid with h chosen so that
    the only in-domain partner sits at R = (3,1,2) is not possible on a lattice with the stencil,
    so use the point-mass special case of the pair function: L0 = phi, L1 = -g."""
    MB = np.zeros(20)
    MB[0] = W1["mono_m"][0]
    L, _ = oracle.pair(W1["R"], MB)
    np.testing.assert_allclose(L[0], W1["mono_phi"][0], rtol=2e-15)
    np.testing.assert_allclose(-L[1:4], W1["mono_g"], rtol=5e-15)


@pytest.mark.parametrize("seed", range(4))
def test_green_tensors_against_symbolic_derivatives(seed):
    """P9: the closed forms equal the symbolic derivatives of -1/r; traces vanish; parity."""
    rng = np.random.default_rng(seed)
    R = rng.uniform(-3, 3, 3) + np.array([0.0, 0.0, 4.0])
    D = oracle.green(R)
    for n in range(5):
        ref = green_tensor(R, n)
        np.testing.assert_allclose(D[n], ref, rtol=0, atol=2e-15 * np.abs(ref).max())
    assert abs(np.trace(D[2])) < 1e-15 * np.abs(D[2]).max()
    assert np.abs(np.einsum("iik->k", D[3])).max() < 1e-15 * np.abs(D[3]).max()
    assert np.abs(np.einsum("iikl->kl", D[4])).max() < 2e-15 * np.abs(D[4]).max()
    Dm = oracle.green(-R)
    for n in range(5):
        np.testing.assert_allclose(Dm[n], (-1) ** n * np.asarray(D[n]), rtol=0, atol=1e-18)


def _random_cluster(rng, npts=7):
    m = rng.uniform(0.5, 1.5, npts)
    b = rng.uniform(-1, 1, (npts, 3))
    return m, b


@pytest.mark.parametrize("seed", range(3))
def test_truncation_order_of_every_coefficient(seed):
    """err(L^(n)) ~ eps^(4-n).  The expansion centre is deliberately NOT the centre of mass, so
    the dipole terms are exercised too."""
    rng = np.random.default_rng(100 + seed)
    m, b = _random_cluster(rng)
    zB = np.array([0.1, -0.2, 0.05])
    zA = zB + np.array([1.3, -0.7, 0.9])
    errs = []
    for eps in (0.08, 0.04):
        y = zB + eps * b
        MB = moments_of_points(m, y, zB)
        L, _ = oracle.pair(zA - zB, MB)
        ex = exact_local_expansion(m, y, zA)
        errs.append([np.abs(L[sl] - ex[sl]).max() for sl in (slice(0, 1), slice(1, 4), slice(4, 10), slice(10, 20))])
    errs = np.array(errs)
    for n in range(4):
        ratio = errs[0, n] / errs[1, n]
        assert 0.72 * 2 ** (4 - n) < ratio < 1.4 * 2 ** (4 - n), (n, ratio, errs)
    # and the absolute size: leading neglected term ~ eps^(4-n) |D^(4)| * sum m |b|^(4-n) / (4-n)!
    D4max = np.abs(green_tensor(zA - zB, 4)).max()
    for n in range(4):
        assert errs[1, n] < 30 * D4max * (0.04 ** (4 - n)) * m.sum()


@pytest.mark.parametrize("seed", range(3))
def test_correction_is_the_next_order_term_of_L1(seed):
    """With a target whose own third moment vanishes, dL1 = -1/6 M3_B : D4 is exactly the (n=1, m=3)
    term that the n + m <= 3 truncation drops, so L1 + dL1 must converge like eps^4 (L1 alone eps^3).
    Pins the sign, the 1/6, the D4 contraction and its multiplicities."""
    rng = np.random.default_rng(200 + seed)
    m, b = _random_cluster(rng)
    zB = np.zeros(3)
    zA = np.array([-1.1, 0.8, 1.2])
    e3, e4 = [], []
    for eps in (0.08, 0.04):
        y = zB + eps * b
        MB = moments_of_points(m, y, zB)
        L, dL1 = oracle.pair(zA - zB, MB, MA0=1.0, MA3=np.zeros(10), correction=True)
        ex = exact_local_expansion(m, y, zA)
        e3.append(np.abs(L[1:4] - ex[1:4]).max())
        e4.append(np.abs(L[1:4] + dL1 - ex[1:4]).max())
    assert 0.72 * 8 < e3[0] / e3[1] < 1.4 * 8
    assert 0.72 * 16 < e4[0] / e4[1] < 1.4 * 16
    assert e4[1] < 0.2 * e3[1]


def test_correction_pair_antisymmetry():
    """M_A dL1_A + M_B dL1_B = 0 for any pair: the correction preserves linear momentum (L127)."""
    rng = np.random.default_rng(7)
    MA, MB = rng.uniform(-1, 1, 20), rng.uniform(-1, 1, 20)
    MA[0], MB[0] = 1.7, 0.6
    R = np.array([0.9, -2.1, 1.4])
    _, dA = oracle.pair(R, MB, MA[0], MA[10:20], True)
    _, dB = oracle.pair(-R, MA, MB[0], MB[10:20], True)
    assert np.abs(MA[0] * dA + MB[0] * dB).max() < 1e-16 * max(np.abs(MA[0] * dA).max(), 1e-300) * 10
    # and it is literally -1/6 n3 : D4 with n3 = M3_B - (M_B/M_A) M3_A, D4 from sympy
    n3 = full3(MB[10:20] - MB[0] / MA[0] * MA[10:20])
    ref = -np.einsum("jkl,ijkl->i", n3, green_tensor(R, 4)) / 6.0
    np.testing.assert_allclose(dA, ref, rtol=1e-12)


def test_point_mass_and_uniform_sphere():
    """P6: a pure monopole source gives L^(n) = M D^(n)(R).  P7: a uniform sphere of radius a
    (M2 = M a^2/5 delta_ij, M3 = 0) gives the same coefficients (shell theorem: all traces of
    D^(n) vanish)."""
    R = np.array([2.2, -1.4, 0.6])
    M, a = 1.3, 0.45
    MB = np.zeros(20)
    MB[0] = M
    L, _ = oracle.pair(R, MB)
    ref = np.concatenate([[M * green_tensor(R, 0)], M * green_tensor(R, 1), M * unique2(green_tensor(R, 2)),
                          M * unique3(green_tensor(R, 3))])
    np.testing.assert_allclose(L, ref, rtol=0, atol=3e-16 * np.abs(ref).max())
    MS = MB.copy()
    MS[[4, 7, 9]] = M * a * a / 5.0
    Ls, _ = oracle.pair(R, MS)
    np.testing.assert_allclose(Ls, L, rtol=0, atol=3e-16 * np.abs(L).max())


def test_linearity_and_component_order():
    """P10: L is linear in the source moments; each unique slot feeds the documented tensor entry."""
    rng = np.random.default_rng(3)
    R = np.array([1.5, 2.5, -0.5])
    MB = rng.uniform(-1, 1, 20)
    L1, _ = oracle.pair(R, MB)
    L2, _ = oracle.pair(R, 2.0 * MB)
    np.testing.assert_allclose(L2, 2.0 * L1, rtol=1e-15)
    # slot t of M3 alone contributes -1/6 * multiplicity * D3[idx] to L0
    D3 = green_tensor(R, 3)
    mult = [1, 3, 3, 3, 6, 3, 1, 3, 3, 1]
    for t, idx in enumerate(IDX3):
        e = np.zeros(20)
        e[10 + t] = 1.0
        L, _ = oracle.pair(R, e)
        np.testing.assert_allclose(L[0], -mult[t] * D3[idx] / 6.0, rtol=1e-13)
        assert np.all(L[1:] == 0.0)


def test_device_invariant_helper_matches_the_numpy_one():
    """helpers.invariants_on_device (torch, used on 256^3 GPU results) against helpers.cell_forces_and_torques (numpy)
    on a small random level: same force and torque sums."""
    import torch
    from helpers import cell_forces_and_torques, invariants_on_device
    rng = np.random.default_rng(5)
    n, h = 6, 0.37
    mom = rng.normal(size=(20, n, n, n))
    com = rng.normal(size=(3, n, n, n)) * 0.1 * h
    L = rng.normal(size=(20, n, n, n))
    F, T = cell_forces_and_torques(mom, com, L, h)
    eF = np.abs(F.sum(axis=(1, 2, 3))).max() / np.abs(F).sum()
    eT = np.abs(T.sum(axis=(1, 2, 3))).max() / np.abs(T).sum()
    gF, gT = invariants_on_device(torch, torch.from_numpy(mom), torch.from_numpy(com), torch.from_numpy(L), h)
    assert abs(gF - eF) < 1e-12 * max(eF, 1.0) and abs(gT - eT) < 1e-12 * max(eT, 1.0)
    assert eF > 1e-3 and eT > 1e-3          # random L: nothing cancels, so the comparison is not 0 == 0
