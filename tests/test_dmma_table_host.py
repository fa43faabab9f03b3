"""Host logic of the tensor-core monopole kernels (no GPU): the operand tables octo_fmm_create builds, seen through the
host-only octo_fmm_dmma_table, against the oracle's lists and weights written out here with numpy.

Checked: every offset of every row's list appears exactly once, in the row that owns it, with the weight of that offset
(-1/|R|, -R/|R|^3, R = -Delta h) bit for bit; every other entry of the table is zero; all four slots of a chunk and all
eight rows name the same source position; the chunks follow the bank rule the kernel's shared-memory loads rely on; the
number of chunks is within a few of |U| / 4."""
import itertools

import numpy as np
import pytest

import oracle


@pytest.fixture(scope="module")
def pkg():
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    return p


def _positions():
    """tile offset -> source position (sx, sy, sz), positions -5 .. 6 per axis (header of octo_fmm_dmma_table)."""
    m = {}
    for sz, sy, sx in itertools.product(range(-5, 7), repeat=3):
        m[(sz * 26 + sy) * 28 + ((sx + 5) & 1) * 14 + ((sx + 5) >> 1)] = (sx, sy, sz)
    assert len(m) == 12 ** 3
    return m


def _weight(delta, h, comp):
    R = -np.asarray(delta, dtype=np.float64) * h
    r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2]
    r = np.sqrt(r2)
    return -1.0 / r if comp == 0 else R[comp - 1] * (-1.0 / (r2 * r))


@pytest.mark.parametrize("theta", [0.5, 0.35, 0.7])
@pytest.mark.parametrize("leaf", [0, 1])
@pytest.mark.parametrize("which", [0, 1, 2, 3, 4])
def test_table_holds_each_list_entry_once_with_its_weight(pkg, theta, leaf, which):
    h = 1.0 / 64
    a, off = pkg.octo_fmm_dmma_table(theta, h, leaf, which)
    pos = _positions()
    lists = [oracle.stencil_leaf(theta, p) if leaf else oracle.stencil(theta, p) for p in range(8)]
    # row i: (parity class of its list, shift of its target from the base target, weight component)
    if which < 4:
        py, pz = which & 1, which >> 1
        rows = [((i >> 2) + 2 * py + 4 * pz, (i >> 2, 0, 0), i & 3) for i in range(8)]
    else:
        rows = [(v, (v & 1, (v >> 1) & 1, v >> 2), 0) for v in range(8)]
    assert (off == off[:, :1, :]).all()                       # the eight rows of a slot name the same position
    union = set()
    for i, (cls, shift, comp) in enumerate(rows):
        want = {tuple(int(c) for c in d) for d in lists[cls]}
        union |= {tuple(d[c] + shift[c] for c in range(3)) for d in want}
        seen = set()
        for c, k in itertools.product(range(a.shape[0]), range(4)):
            if a[c, i, k] == 0.0:
                continue
            s = pos[int(off[c, i, k])]
            d = tuple(s[c2] - shift[c2] for c2 in range(3))
            assert d in want and d not in seen, (i, d)
            seen.add(d)
            assert a[c, i, k] == _weight(d, h, comp), (i, d)
        # offsets whose weight component is exactly zero (e.g. g_x at dx = 0) cannot be told from padding: they must
        # be the only ones missing
        for d in want - seen:
            assert comp > 0 and d[comp - 1] == 0, (i, d)
    # every position of the union is there, once
    slots = [pos[int(o)] for c in range(a.shape[0]) for k, o in enumerate(off[c, 0]) if (a[c, :, k] != 0.0).any()]
    assert len(slots) == len(set(slots)) and set(slots) == union
    assert a.shape[0] <= int(np.ceil(len(union) / 4)) + max(2, len(union) // 100)     # greedy grouping: a few slots stay empty


@pytest.mark.parametrize("theta,leaf,which", [(0.5, 0, 0), (0.5, 1, 3), (0.35, 1, 4), (0.7, 0, 2), (0.5, 1, 4)])
def test_chunks_follow_the_bank_rule(pkg, theta, leaf, which):
    """The B-fragment load of a half-warp reads off_k + j, j = 0..3, for the four slots k: two slots may share a bank
    (8-byte banks, 16 per wavefront) only where they read the same address."""
    _, off = pkg.octo_fmm_dmma_table(theta, 1.0, leaf, which)
    for c in range(off.shape[0]):
        addr = {}
        for k in range(4):
            for j in range(4):
                ad = int(off[c, 0, k]) + j
                assert addr.setdefault(ad % 16, ad) == ad, (c, off[c, 0])


def test_rejects_bad_arguments(pkg):
    for theta, h, which in ((0.2, 1.0, 0), (0.5, 0.0, 0), (0.5, 1.0, 5), (0.5, 1.0, -1)):
        with pytest.raises(pkg.OctoFmmError):
            pkg.octo_fmm_dmma_table(theta, h, 0, which)
