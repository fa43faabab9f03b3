"""Pins of the oracle's interaction list -- CPU only.

What fixes the expected values:
  * Eq. 15: partners = cells well separated whose parents are not.  The
    parents-not-well-separated set is {Delta_I : |Delta_I|^2 <= 1/theta^2}, each parent has 8
    children, and the not-well-separated cells are {Delta : |Delta|^2 <= 1/theta^2}, all of
    which lie inside the first set; hence  |S_p| = 8 N - N = 7 N  with N the number of integer
    lattice points in the closed ball of radius 1/theta (a closed form, counted here directly).
  * theta_min = 0.34 for 8x8x8 sub-grids (L137): reach <= 5 cells for theta >= 0.34 and a jump
    at theta = 1/3.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from helpers import load_golden

GOLD = load_golden(os.path.join(os.path.dirname(__file__), "golden", "counts.txt"))


def lattice_ball(theta):
    r2max = 1.0 / (theta * theta)
    m = int(np.floor(np.sqrt(r2max))) + 1
    return sum(1 for v in itertools.product(range(-m, m + 1), repeat=3) if (v[0] ** 2 + v[1] ** 2 + v[2] ** 2) * theta * theta <= 1.0)


@pytest.mark.parametrize("row", GOLD["_multi"]["stencil"])
def test_stencil_counts(row):
    theta, per, union, inter, reach, near = float(row[0]), *[int(v) for v in row[1:]]
    lists = [oracle.stencil(theta, p) for p in range(8)]
    sets = [set(map(tuple, s.tolist())) for s in lists]
    assert [len(s) for s in lists] == [per] * 8
    assert all(len(sets[p]) == per for p in range(8))          # no duplicates
    assert len(set.union(*sets)) == union
    assert len(set.intersection(*sets)) == inter
    assert max(int(np.abs(s).max()) for s in lists) == reach
    # closed form 7 N and near-field count N - 1
    N = lattice_ball(theta)
    assert per == 7 * N
    assert near == N - 1
    for s in sets:
        assert (0, 0, 0) not in s


def test_theta_min():
    """L137: theta_min = 0.34 for 8^3 sub-grids <=> the halo reach stays at 5 down to 0.34."""
    row = GOLD["_multi"]["stencil_below_min"][0]
    lists = [oracle.stencil(float(row[0]), p) for p in range(8)]
    assert [len(s) for s in lists] == [int(row[1])] * 8
    assert max(int(np.abs(s).max()) for s in lists) == int(row[2])
    for theta in (0.34, 0.35, 0.4, 0.45, 0.5):
        assert max(int(np.abs(oracle.stencil(theta, p)).max()) for p in range(8)) == 5


@pytest.mark.parametrize("theta", [0.5, 0.35, 0.7])
def test_stencil_symmetry_and_definition(theta):
    """P2: B in list(A) <=> A in list(B); and every listed pair satisfies Eq. 15 literally
    (distance test in floating point on cell/parent centres, not on integer norms)."""
    lists = {p: set(map(tuple, oracle.stencil(theta, p).tolist())) for p in range(8)}
    for p in range(8):
        pa = np.array([p & 1, (p >> 1) & 1, (p >> 2) & 1])
        for d in lists[p]:
            d = np.array(d)
            pb = (pa + d) & 1
            q = int(pb[0] + 2 * pb[1] + 4 * pb[2])
            assert tuple((-d).tolist()) in lists[q]
            # Eq. 15 on geometric centres: cell width 1, parent width 2
            xa, xb = pa + 0.5, pa + d + 0.5
            assert 1.0 / np.linalg.norm(xa - xb) < theta
            Xa, Xb = 2.0 * np.floor(pa / 2) + 1.0, 2.0 * np.floor((pa + d) / 2) + 1.0
            dist = np.linalg.norm(Xa - Xb)
            assert dist == 0.0 or not (2.0 / dist < theta)
    # completeness: nothing within a generous box is missed
    S = 9
    for p in (0, 5, 7):
        pa = np.array([p & 1, (p >> 1) & 1, (p >> 2) & 1])
        for d in itertools.product(range(-S, S + 1), repeat=3):
            if d == (0, 0, 0):
                continue
            d = np.array(d)
            cell_ws = float(d @ d) * theta * theta > 1.0
            dI = np.floor((pa + d) / 2) - np.floor(pa / 2)
            par_ws = (dI @ dI) > 0 and float(dI @ dI) * theta * theta > 1.0
            assert (tuple(d.tolist()) in lists[p]) == (cell_ws and not par_ws)


def test_stencil_order_is_lexicographic():
    s = oracle.stencil(0.5, 3).astype(int)
    keys = [(d[2], d[1], d[0]) for d in s]
    assert keys == sorted(keys)


def _count_from_lists(n, lo, hi, theta):
    """Ordered in-domain pairs, per axis closed form from the partner lists."""
    total = 0
    for p in range(8):
        par = (p & 1, (p >> 1) & 1, (p >> 2) & 1)
        for d in oracle.stencil(theta, p).astype(int):
            c = 1
            for a in range(3):
                idx = np.arange(lo, hi)
                idx = idx[(idx & 1) == par[a]]
                c *= int(((idx + d[a] >= 0) & (idx + d[a] < n)).sum())
            total += c
    return total


@pytest.mark.parametrize("row", GOLD["_multi"]["interactions"])
def test_interaction_counts(row):
    name, n, lo, hi, theta, expect = row[0], int(row[1]), int(row[2]), int(row[3]), float(row[4]), int(row[5])
    assert _count_from_lists(n, lo, hi, theta) == expect
    if n <= 128:  # brute-force enumeration on the index grid by the oracle itself
        assert oracle.interaction_count((n, n, n), theta, (lo,) * 3, (hi,) * 3) == expect
