"""Pins of the oracle's mixed level (one level of an adaptive mesh whose sub-grids are leaves or
refined, oracle.interact_multipole_mixed; reading R8).  The paper does not describe the gravity side of a
refinement boundary, so the pins are what the mathematics fixes: the two uniform limits reduce to routines that are
pinned on their own, the pair set is the stated rule enumerated independently, and a symmetric pair set keeps the
conservation laws of L125 / L127."""
import itertools

import numpy as np
import pytest

import fmm_inputs as fi
import oracle
from helpers import cell_forces_and_torques


def _level(seed=5, n=16, frac=0.5):
    w = fi.config1(seed=seed, ncell=n)
    sub = np.random.default_rng(seed).random((n // 8,) * 3) < frac
    leaf = np.repeat(np.repeat(np.repeat(sub, 8, 0), 8, 1), 8, 2).astype(np.uint8)
    mom, com = w.moments.copy(), w.com_off.copy()
    mom[1:, leaf == 1] = 0.0                       # leaves are point masses at their cell centres
    com[:, leaf == 1] = 0.0
    return w, mom, com, leaf


def test_no_leaves_is_the_plain_step_and_all_leaves_is_the_leaf_monopole_sum():
    w, _, _, _ = _level()
    zero = np.zeros(w.n[::-1], np.uint8)
    a = oracle.interact_multipole(w.n, w.h, 0.5, w.moments, w.com_off, None, None, True)
    b = oracle.interact_multipole_mixed(w.n, w.h, 0.5, w.moments, w.com_off, zero, None, None, True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[2] == b[2]
    mono = w.moments.copy()
    mono[1:] = 0.0
    c = oracle.interact_multipole_mixed(w.n, w.h, 0.5, mono, np.zeros_like(w.com_off), np.ones_like(zero), None, None, False)
    d, cnt = oracle.interact_monopole_leaf(w.n, w.h, 0.5, mono[0])
    assert c[2] == cnt
    assert np.abs(c[0][0] - d[0]).max() / np.abs(d[0]).max() < 1e-15          # L0 = phi
    assert np.abs(c[0][1:4] + d[1:4]).max() / np.abs(d[1:4]).max() < 1e-15     # L1 = -g


@pytest.mark.parametrize("theta", [0.5, 0.35, 0.7])
def test_pair_set_is_the_rule_enumerated_independently(theta):
    """Partners of A = well-separated cells whose parents are not (Eq. 15) + not-well-separated cells whose parents are
    not well separated either, if A or B is a leaf -- counted here with plain Python over global indices."""
    n = 16
    w, mom, com, leaf = _level(seed=9, n=n)
    _, _, cnt = oracle.interact_multipole_mixed(w.n, w.h, theta, mom, com, leaf, None, None, False)
    ws = lambda d2: float(d2) * theta * theta > 1.0
    total = 0
    rng = range(-7, 8)
    offs = [(dx, dy, dz) for dz in rng for dy in rng for dx in rng if (dx, dy, dz) != (0, 0, 0)]
    for k, j, i in itertools.product(range(n), repeat=3):
        for dx, dy, dz in offs:
            bi, bj, bk = i + dx, j + dy, k + dz
            if not (0 <= bi < n and 0 <= bj < n and 0 <= bk < n):
                continue
            D2 = ((bi >> 1) - (i >> 1)) ** 2 + ((bj >> 1) - (j >> 1)) ** 2 + ((bk >> 1) - (k >> 1)) ** 2
            if D2 > 0 and ws(D2):
                continue                                            # the parents took it
            if ws(dx * dx + dy * dy + dz * dz) or leaf[k, j, i] or leaf[bk, bj, bi]:
                total += 1
    assert cnt == total


@pytest.mark.parametrize("theta", [0.5, 0.35])
def test_mixed_level_conserves_momentum_and_angular_momentum(theta):
    """The pair set is symmetric (A or B a leaf), so pair forces still cancel (L125) and, with the correction, so do
    the torques (L127) -- near-field pairs included."""
    w, mom, com, leaf = _level(seed=11, n=16)
    L, Lc, _ = oracle.interact_multipole_mixed(w.n, w.h, theta, mom, com, leaf, None, None, True)
    F, T = cell_forces_and_torques(mom, com, L, w.h)
    assert np.abs(F.sum(axis=(1, 2, 3))).max() / np.abs(F).sum() < 2e-15
    x = np.stack(np.meshgrid(*[np.arange(16) * w.h] * 3, indexing="ij"))
    scale = np.abs(np.cross(x, F, axis=0)).sum()
    on = np.abs(T.sum(axis=(1, 2, 3))).max() / scale
    L0, _, _ = oracle.interact_multipole_mixed(w.n, w.h, theta, mom, com, leaf, None, None, False)
    _, T0 = cell_forces_and_torques(mom, com, L0, w.h)
    off = np.abs(T0.sum(axis=(1, 2, 3))).max() / scale
    assert on < 5e-15 and off > 1e3 * on, (on, off)


def test_near_field_pairs_change_only_cells_next_to_leaves():
    """A refined cell all of whose near-field neighbours are refined gets exactly the plain step's coefficients."""
    w, mom, com, leaf = _level(seed=13, n=24, frac=0.3)
    a, _, _ = oracle.interact_multipole(w.n, w.h, 0.5, mom, com, None, None, True)
    b, _, _ = oracle.interact_multipole_mixed(w.n, w.h, 0.5, mom, com, leaf, None, None, True)
    changed = np.abs(a - b).max(axis=0) > 0
    near = [d for d in oracle.stencil_leaf(0.5, 0) if tuple(d) not in {tuple(v) for v in oracle.stencil(0.5, 0)}]
    reach = max(abs(int(c)) for d in near for c in d)
    # dilate the leaf mask by the near-field reach: nothing outside it may change
    pad = np.pad(leaf, reach)
    dil = np.zeros_like(leaf)
    for dz, dy, dx in itertools.product(range(-reach, reach + 1), repeat=3):
        dil |= pad[reach + dz:reach + dz + 24, reach + dy:reach + dy + 24, reach + dx:reach + dx + 24]
    assert changed.any() and not (changed & (dil == 0)).any()
