"""Seeded synthetic inputs for the FMM cell-to-cell interaction step.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2101_08226_b200/``).  It holds none of the method's arithmetic
(no Green's-function tensors, no stencil, no M2L): it only manufactures the
per-cell multipole moments that the interaction step takes as *input*.

What the inputs stand in for
----------------------------
The paper measures on stationary n=3/2 polytropes (§3.5;
scaling runs §5: 128^3 = 4096 sub-grids, 256^3 = 32768 sub-grids of
8x8x8 cells) and on a q<1 binary (§4).  Its input decks (Zenodo, L1144-1146)
are not available, so seeded synthetic fields of the same shape are used:
Lane-Emden n=1.5 density profiles on the unit cube with the 1e-10 ambient
floor of Eq. 36 (L325-327).

Cell model
----------
"The multipoles of each cell are composed of the multipoles of its child
cells" (L125).  Every cell is 8 child point masses at
x_cell + (+-h/4, +-h/4, +-h/4); the cell's raw Cartesian moments about its
centre of mass,  M^(n) = sum_p m_p (y_p - z)^{(x) n},  n = 0..3, are the 20
unique components in lexicographic order
  [0] [x y z] [xx xy xz yy yz zz] [xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz]
with no factorials or multiplicities folded in.  The expansion centre is
handed over as the OFFSET  delta = z - x_cell  (3 doubles per cell).

Array layout (both outputs): component-major SoA, C order, x fastest:
  moments[20][nz][ny][nx],  com_off[3][nz][ny][nx].

Random numbers: SplitMix64 counter stream, u = (x >> 11) * 2^-53.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

DEFAULT_SEED = 20210108

# unique-component index tables (lexicographic), exported for tests/harness
IDX2 = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
IDX3 = [(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 1, 2), (0, 2, 2),
        (1, 1, 1), (1, 1, 2), (1, 2, 2), (2, 2, 2)]

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_MIX1 = np.uint64(0xBF58476D1CE4E5B9)
_MIX2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, count: int, offset: int = 0) -> np.ndarray:
    """``count`` SplitMix64 outputs, draws number offset+1 .. offset+count of the stream."""
    with np.errstate(over="ignore"):
        idx = np.arange(offset + 1, offset + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + idx * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _MIX1
        z = (z ^ (z >> np.uint64(27))) * _MIX2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, count: int, offset: int = 0) -> np.ndarray:
    """Doubles in [0,1): (x >> 11) * 2^-53."""
    return (splitmix64(seed, count, offset) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


# --------------------------------------------------------------------------------------
# Lane-Emden n = 1.5 profile (Eq. 43 / §3.5: polytropic index n = 3/2)
# --------------------------------------------------------------------------------------
_LE_CACHE = {}


def lane_emden(n: float = 1.5, dxi: float = 1.0e-4):
    """Integrate theta'' + 2 theta'/xi + theta^n = 0 by RK4.

    Returns (xi_grid, theta_grid, xi1) with theta(xi1) = 0 the first zero
    (xi1 = 3.65375... for n = 1.5)."""
    key = (n, dxi)
    if key in _LE_CACHE:
        return _LE_CACHE[key]

    def rhs(xi, th, ph):
        return ph, -(max(th, 0.0) ** n) - 2.0 * ph / xi

    xi = dxi
    th = 1.0 - xi * xi / 6.0 + n * xi ** 4 / 120.0
    ph = -xi / 3.0 + n * xi ** 3 / 30.0
    xs, ths = [0.0, xi], [1.0, th]
    xi1 = None
    while True:
        k1t, k1p = rhs(xi, th, ph)
        k2t, k2p = rhs(xi + 0.5 * dxi, th + 0.5 * dxi * k1t, ph + 0.5 * dxi * k1p)
        k3t, k3p = rhs(xi + 0.5 * dxi, th + 0.5 * dxi * k2t, ph + 0.5 * dxi * k2p)
        k4t, k4p = rhs(xi + dxi, th + dxi * k3t, ph + dxi * k3p)
        th_new = th + dxi * (k1t + 2 * k2t + 2 * k3t + k4t) / 6.0
        ph_new = ph + dxi * (k1p + 2 * k2p + 2 * k3p + k4p) / 6.0
        xi_new = xi + dxi
        if th_new <= 0.0:
            xi1 = xi + dxi * th / (th - th_new)
            xs.append(xi_new)
            ths.append(0.0)
            break
        xi, th, ph = xi_new, th_new, ph_new
        xs.append(xi)
        ths.append(th)
    out = (np.asarray(xs), np.asarray(ths), float(xi1))
    _LE_CACHE[key] = out
    return out


def polytrope_density(r: np.ndarray, radius: float, rho_c: float) -> np.ndarray:
    """rho(r) = rho_c * theta_LE(xi1 r / radius)^1.5 inside the star, 0 outside."""
    xs, ths, xi1 = lane_emden()
    xi = np.asarray(r) * (xi1 / radius)
    th = np.interp(xi, xs, ths, right=0.0)
    th = np.where(xi < xi1, np.maximum(th, 0.0), 0.0)
    return rho_c * th ** 1.5


# --------------------------------------------------------------------------------------
# fields
# --------------------------------------------------------------------------------------
@dataclass
class Star:
    centre: tuple
    radius: float
    rho_c: float


FLOOR = 1.0e-10  # ambient density floor, PAPER.md L325-327 (Eq. 36)

SINGLE_STAR = [Star((0.5, 0.5, 0.5), 0.4, 1.0)]
# M ~ rho_c R^3 for a fixed polytropic index, so M2/M1 = 0.7 needs rho_c2 = 0.7 (0.15/0.12)^3
BINARY = [Star((0.3, 0.5, 0.5), 0.15, 1.0), Star((0.7, 0.5, 0.5), 0.12, 0.7 * (0.15 / 0.12) ** 3)]


def field_density(stars, x, y, z):
    rho = np.zeros(np.broadcast(x, y, z).shape)
    for s in stars:
        r = np.sqrt((x - s.centre[0]) ** 2 + (y - s.centre[1]) ** 2 + (z - s.centre[2]) ** 2)
        rho = rho + polytrope_density(r, s.radius, s.rho_c)
    return np.maximum(rho, FLOOR)


# --------------------------------------------------------------------------------------
# cells from 8 child point masses
# --------------------------------------------------------------------------------------
# child c = bx + 2 by + 4 bz, sign s = 2 b - 1
CHILD_SIGNS = np.array([[2 * ((c >> a) & 1) - 1 for a in range(3)] for c in range(8)], dtype=np.float64)


def cells_from_children(child_mass: np.ndarray, h: float):
    """P2M of the 8-child cell model.

    child_mass: [8][...cells...] masses of the children at +-h/4 offsets.
    Returns (moments[20][...], com_off[3][...])."""
    shape = child_mass.shape[1:]
    q = 0.25 * h
    m0 = child_mass.sum(axis=0)
    com = np.zeros((3,) + shape)
    for c in range(8):
        for a in range(3):
            com[a] += child_mass[c] * (CHILD_SIGNS[c, a] * q)
    com /= m0
    mom = np.zeros((20,) + shape)
    mom[0] = m0
    for c in range(8):
        d = [CHILD_SIGNS[c, a] * q - com[a] for a in range(3)]
        m = child_mass[c]
        for a in range(3):
            mom[1 + a] += m * d[a]
        for t, (a, b) in enumerate(IDX2):
            mom[4 + t] += m * d[a] * d[b]
        for t, (a, b, e) in enumerate(IDX3):
            mom[10 + t] += m * d[a] * d[b] * d[e]
    return mom, com


@dataclass
class Workload:
    name: str
    n: tuple            # (nx, ny, nz) cells
    h: float
    theta: float
    kind: str           # "multipole" | "monopole"
    am_correction: bool
    out_lo: tuple       # target region, cells (x, y, z)
    out_hi: tuple
    moments: np.ndarray             # [20][nz][ny][nx]  (monopole: [1][nz][ny][nx])
    com_off: Optional[np.ndarray]   # [3][nz][ny][nx]   (monopole: None)
    child_mass: Optional[np.ndarray] = None  # [8][nz][ny][nx], kept only on request (brute force)
    meta: dict = field(default_factory=dict)

    @property
    def out_shape(self):
        return tuple(self.out_hi[a] - self.out_lo[a] for a in range(3))


def _cell_axis(n, h):
    return (np.arange(n, dtype=np.float64) + 0.5) * h


def _star_children(stars, n, h, kslice, factor=None):
    """Child masses [8][kz][ny][nx] for z-layers kslice, sampled on the 2n lattice."""
    nx, ny, nz = n
    xc = _cell_axis(nx, h)[None, None, :]
    yc = _cell_axis(ny, h)[None, :, None]
    zc = _cell_axis(nz, h)[kslice][:, None, None]
    q = 0.25 * h
    cm = np.empty((8, zc.shape[0], ny, nx))
    vol = (0.5 * h) ** 3
    for c in range(8):
        sx, sy, sz = CHILD_SIGNS[c]
        cm[c] = field_density(stars, xc + sx * q, yc + sy * q, zc + sz * q) * vol
    if factor is not None:
        cm *= factor[None]
    return cm


def _uniform_field(name, stars, ncell, theta, seed, perturb, keep_children=False, kind="multipole",
                   dtype_out=np.float64):
    n = (ncell, ncell, ncell)
    h = 1.0 / ncell
    ncells = ncell ** 3
    factor = None
    if perturb is not None:
        lo, hi = perturb
        factor = (lo + (hi - lo) * uniform01(seed, ncells)).reshape(ncell, ncell, ncell)
    if kind == "monopole":
        xc = _cell_axis(ncell, h)
        mass = np.empty((1, ncell, ncell, ncell))
        chunk = max(1, min(ncell, (1 << 22) // (ncell * ncell)))
        for k0 in range(0, ncell, chunk):
            ks = slice(k0, min(ncell, k0 + chunk))
            rho = field_density(stars, xc[None, None, :], xc[None, :, None], xc[ks][:, None, None])
            mass[0, ks] = rho * h ** 3
        if factor is not None:
            mass[0] *= factor
        return Workload(name, n, h, theta, "monopole", False, (0, 0, 0), n, mass, None,
                        meta={"seed": seed, "stars": len(stars)})
    mom = np.empty((20, ncell, ncell, ncell))
    com = np.empty((3, ncell, ncell, ncell))
    children = np.empty((8, ncell, ncell, ncell)) if keep_children else None
    chunk = max(1, min(ncell, (1 << 21) // (ncell * ncell)))
    for k0 in range(0, ncell, chunk):
        ks = slice(k0, min(ncell, k0 + chunk))
        cm = _star_children(stars, n, h, ks, None if factor is None else factor[ks])
        m, c = cells_from_children(cm, h)
        mom[:, ks] = m
        com[:, ks] = c
        if keep_children:
            children[:, ks] = cm
    return Workload(name, n, h, theta, "multipole", True, (0, 0, 0), n, mom, com, children,
                    meta={"seed": seed, "stars": len(stars)})


def config1(seed: int = DEFAULT_SEED, theta: float = 0.5, ncell: int = 24, keep_children: bool = True,
            out_lo=None, out_hi=None) -> Workload:
    """cfg 1: one 8^3 sub-grid + its 26 neighbours (24^3 cells, h = 1/24), random cells.

    rho ~ U(0.5,1.5), m = rho h^3; alpha ~ U(-0.4,0.4)^3; child masses
    (m/8) prod_c (1 + alpha_c s_c)  =>  COM offset = alpha h/4 ~ U(-0.1h, 0.1h)."""
    h = 1.0 / ncell
    ncells = ncell ** 3
    u = uniform01(seed, 4 * ncells).reshape(ncell, ncell, ncell, 4)
    m = (0.5 + u[..., 0]) * h ** 3
    alpha = -0.4 + 0.8 * u[..., 1:4]
    cm = np.empty((8, ncell, ncell, ncell))
    for c in range(8):
        w = np.ones((ncell, ncell, ncell))
        for a in range(3):
            w = w * (1.0 + alpha[..., a] * CHILD_SIGNS[c, a])
        cm[c] = (m / 8.0) * w
    mom, com = cells_from_children(cm, h)
    n = (ncell,) * 3
    if out_lo is None:
        out_lo, out_hi = ((8, 8, 8), (16, 16, 16)) if ncell == 24 else ((0, 0, 0), n)
    return Workload("cfg1_random_%d" % ncell, n, h, theta, "multipole", True, tuple(out_lo), tuple(out_hi),
                    mom, com, cm if keep_children else None, meta={"seed": seed})


def config2(seed: int = DEFAULT_SEED, theta: float = 0.5, ncell: int = 32, keep_children: bool = False) -> Workload:
    """cfg 2: single n=1.5 polytrope (R = 0.4, centred), ncell^3 cells on the unit cube."""
    return _uniform_field("cfg2_polytrope_%d" % ncell, SINGLE_STAR, ncell, theta, seed, None, keep_children)


def config3(seed: int = DEFAULT_SEED, theta: float = 0.5, ncell: int = 128, keep_children: bool = False) -> Workload:
    """cfg 3: two-polytrope binary, per-cell factor ~U(0.99,1.01), ncell^3 cells (paper: 128^3, L1004)."""
    return _uniform_field("cfg3_binary_%d" % ncell, BINARY, ncell, theta, seed, (0.99, 1.01), keep_children)


def config4(seed: int = DEFAULT_SEED, theta: float = 0.5, ncell: int = 128) -> Workload:
    """cfg 4: monopole (leaf) variant on the cfg-3 field: m = h^3 rho(x_cell) * factor."""
    return _uniform_field("cfg4_monopole_%d" % ncell, BINARY, ncell, theta, seed, (0.99, 1.01), kind="monopole")


def config5(seed: int = DEFAULT_SEED, theta: float = 0.5, ncell: int = 256, keep_children: bool = False) -> Workload:
    """cfg 5: binary with 1e-8 density noise, ncell^3 cells (paper: 256^3 = 32768 sub-grids, L986)."""
    return _uniform_field("cfg5_binary_%d" % ncell, BINARY, ncell, theta, seed,
                          (1.0 - 1.0e-8, 1.0 + 1.0e-8), keep_children)


CONFIGS = {"cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4, "cfg5": config5}


def uniform_sphere(ncell: int = 64, radius: float = 0.25, total_mass: float = 1.0, ambient: float = 1.0e-10):
    """Paper section 3.4 (L448-456): a uniform sphere of radius 0.25 and mass 1 at the centre of the unit box, ambient
    density 1e-10 of the sphere's, uniform grid.  The paper does not say how the sphere is rasterised: cells are
    sampled at their centres and the masses scaled to the total mass.  Returns (h, mass[n][n][n], phi_analytic, r):
    phi_analytic = -M (3 R^2 - r^2) / (2 R^3) inside, -M / r outside (the potential Eq. 42 compares with)."""
    h = 1.0 / ncell
    x = (np.arange(ncell) + 0.5) * h - 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r = np.sqrt(X * X + Y * Y + Z * Z)
    rho = np.where(r < radius, 1.0, ambient)
    mass = rho * (total_mass / rho.sum())
    phi = np.where(r < radius, -total_mass * (3.0 * radius ** 2 - r * r) / (2.0 * radius ** 3), -total_mass / r)
    return h, mass, phi, r


# ---------------------------------------------------------------------------------------------
# Adaptive oct-trees of 8^3 sub-grids.  Inputs only: topology and leaf masses.
# ---------------------------------------------------------------------------------------------
TREE_ABSENT, TREE_LEAF, TREE_REFINED = 0, 1, 2


class Tree:
    """An oct-tree of 8^3 sub-grids over a cube of width n0 * h0.  Level l is a dense
    [n_l][n_l][n_l] lattice, n_l = n0 2^l, h_l = h0 / 2^l, with kind[l] (uint8: 0 absent, 1 leaf, 2 refined; constant
    over every aligned 8^3 sub-grid) and mass[l] (float64; the point mass of every leaf cell, 0 elsewhere).
    "A node is either fully refined with eight child nodes (an interior node) or not refined at all (a leaf node)"
    (L287): a cell exists on level l+1 iff its parent cell is refined; the tree is properly nested (2:1 over the 26
    neighbours of a sub-grid), so a refinement boundary involves exactly two levels (L287-291)."""

    def __init__(self, n0, h0, kind, mass):
        self.n0, self.h0, self.kind, self.mass = int(n0), float(h0), kind, mass

    @property
    def depth(self):
        return len(self.kind)

    def n(self, l):
        return self.n0 << l

    def h(self, l):
        return self.h0 / (1 << l)

    def leaf_points(self):
        """(pos[np][3], mass[np], level[np], index[np][3]) of all leaf cells, levels in order, C order inside a level."""
        pos, ms, lv, idx = [], [], [], []
        for l in range(self.depth):
            k, j, i = np.nonzero(self.kind[l] == TREE_LEAF)
            h = self.h(l)
            pos.append(np.stack([(i + 0.5) * h, (j + 0.5) * h, (k + 0.5) * h], axis=1))
            ms.append(self.mass[l][k, j, i])
            lv.append(np.full(len(i), l))
            idx.append(np.stack([i, j, k], axis=1))
        return np.concatenate(pos), np.concatenate(ms), np.concatenate(lv), np.concatenate(idx)


def tree_boxes(tree, margin: int = 0):
    """Per level the bounding box (lo_x, lo_y, lo_z, n_x, n_y, n_z), aligned to the 8^3 sub-grids and grown by `margin`
    sub-grids, of the cells that exist on that level of a tree given on whole lattices; level 0: the whole lattice."""
    out = []
    for l in range(tree.depth):
        n = tree.n(l)
        if l == 0 or not (tree.kind[l] != TREE_ABSENT).any():
            out.append((0, 0, 0, n, n, n) if l == 0 else (0, 0, 0, 8, 8, 8))
            continue
        k, j, i = np.nonzero(tree.kind[l] != TREE_ABSENT)
        b = []
        for v in (i, j, k):
            lo = max((int(v.min()) // 8 - margin) * 8, 0)
            hi = min((int(v.max()) // 8 + 1 + margin) * 8, n)
            b.append((lo, hi - lo))
        out.append((b[0][0], b[1][0], b[2][0], b[0][1], b[1][1], b[2][1]))
    return out


def crop_tree(tree, boxes):
    """(kind, mass) lists of the tree's levels restricted to the boxes (contiguous copies)."""
    kind, mass = [], []
    for l, b in enumerate(boxes):
        sl = (slice(b[2], b[2] + b[5]), slice(b[1], b[1] + b[4]), slice(b[0], b[0] + b[3]))
        kind.append(np.ascontiguousarray(tree.kind[l][sl]))
        mass.append(np.ascontiguousarray(tree.mass[l][sl]))
    return kind, mass


def _expand8(a):
    return np.repeat(np.repeat(np.repeat(a, 8, 0), 8, 1), 8, 2)


def _dilate26(a):
    """True where a sub-grid or any of its 26 neighbours is True (sub-grid lattice, isolated domain)."""
    p = np.pad(a, 1)
    out = np.zeros_like(a)
    s = a.shape[0]
    for dz in range(3):
        for dy in range(3):
            for dx in range(3):
                out |= p[dz:dz + s, dy:dy + s, dx:dx + s]
    return out


def make_tree(n0, depth, want_refined, density, box=1.0):
    """Build a properly nested tree.  n0: cells per axis of level 0 (a multiple of 8, every cell exists); depth: number
    of levels; want_refined(l, cx, cy, cz) -> bool array over the sub-grid lattice of level l (centres of the sub-grids
    as arrays): the sub-grids the caller wants refined on level l < depth - 1; density(x, y, z) -> rho at leaf centres
    (mass = rho h_l^3).  Proper nesting is enforced bottom-up: a sub-grid is refined as well if any of the 26 neighbours
    of one of its child sub-grids is refined (then no leaf touches a leaf two levels finer)."""
    assert n0 % 8 == 0 and depth >= 1
    h0 = box / n0
    ref = []                                   # refined flags over the sub-grid lattice of each level
    exists = [np.ones((n0 // 8,) * 3, dtype=bool)]
    for l in range(depth - 1):
        s = (n0 // 8) << l
        c = (np.arange(s) + 0.5) * (box / s)
        CZ, CY, CX = np.meshgrid(c, c, c, indexing="ij")
        r = np.asarray(want_refined(l, CX, CY, CZ), dtype=bool) & exists[l]
        ref.append(r)
        exists.append(np.repeat(np.repeat(np.repeat(r, 2, 0), 2, 1), 2, 2))
    ref.append(np.zeros_like(exists[-1]))
    # 2:1 over the 26 neighbours, bottom-up: the parent of every neighbour of a refined sub-grid must be refined
    for l in range(depth - 2, 0, -1):
        need = _dilate26(ref[l])                       # sub-grids of level l that must EXIST
        s = need.shape[0] // 2
        need_parent = need.reshape(s, 2, s, 2, s, 2).any(axis=(1, 3, 5))
        ref[l - 1] |= need_parent
    # top-down again: existence follows the (grown) refinement
    exists = [np.ones((n0 // 8,) * 3, dtype=bool)]
    for l in range(depth - 1):
        ref[l] &= exists[l]
        exists.append(np.repeat(np.repeat(np.repeat(ref[l], 2, 0), 2, 1), 2, 2))
    ref[depth - 1] &= False
    kind, mass = [], []
    for l in range(depth):
        k = np.where(exists[l], np.where(ref[l], TREE_REFINED, TREE_LEAF), TREE_ABSENT).astype(np.uint8)
        k = _expand8(k)
        n = n0 << l
        h = h0 / (1 << l)
        x = (np.arange(n) + 0.5) * h
        Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
        m = np.where(k == TREE_LEAF, np.asarray(density(X, Y, Z), dtype=np.float64) * h ** 3, 0.0)
        kind.append(np.ascontiguousarray(k))
        mass.append(np.ascontiguousarray(m))
    return Tree(n0, h0, kind, mass)


def tree_is_properly_nested(tree) -> bool:
    """Every refined cell's children exist; no leaf sub-grid has a neighbour (26) two levels finer."""
    for l in range(tree.depth - 1):
        k, kf = tree.kind[l], tree.kind[l + 1]
        par = np.repeat(np.repeat(np.repeat(k, 2, 0), 2, 1), 2, 2)
        if ((kf != TREE_ABSENT) != (par == TREE_REFINED)).any():
            return False
        # sub-grid lattice of level l+1: refined sub-grids need all 26 neighbours to exist (inside the domain)
        sub = kf[::8, ::8, ::8]
        need = _dilate26(sub == TREE_REFINED)
        if (need & (sub == TREE_ABSENT)).any():
            return False
    return not (tree.kind[-1] == TREE_REFINED).any()


def seeded_tree(seed: int, n0: int = 16, depth: int = 3, frac: float = 0.4):
    """A seeded random tree for the pins and the parity tests: level 0 is refined everywhere, on every deeper level each
    existing sub-grid is refined with probability `frac` (proper nesting then refines some more); leaf densities
    ~ U(0.5, 1.5) (SplitMix64 stream per level, C order)."""
    def want(l, cx, cy, cz):
        u = uniform01(seed + 1000 * (l + 1), cx.size).reshape(cx.shape)
        return (u < frac) | (l == 0)

    def rho(X, Y, Z):
        return 0.5 + uniform01(seed + 77 + X.shape[0], X.size).reshape(X.shape)
    return make_tree(n0, depth, want, rho)


def star_tree(n0: int = 16, depth: int = 3, stars=None, radius_factor: float = 1.3):
    """The paper's refinement pattern in miniature (density-based refinement, Eq. 34-35: finer where the
    density is higher): level l refines the sub-grids within radius_factor * R_star / 2^l... of a star centre; density
    = the n = 1.5 polytropes of `stars` (default: the two-star binary of cfg 3) over the 1e-10 floor."""
    stars = BINARY if stars is None else stars

    def want(l, cx, cy, cz):
        w = np.zeros(cx.shape, dtype=bool)
        for s in stars:
            rr = np.sqrt((cx - s.centre[0]) ** 2 + (cy - s.centre[1]) ** 2 + (cz - s.centre[2]) ** 2)
            w |= rr < radius_factor * s.radius / (1.5 ** l)
        return w
    return make_tree(n0, depth, want, lambda X, Y, Z: field_density(stars, X, Y, Z))


def nested_tree(n0: int = 16, depth: int = 9, centre=(0.37, 0.52, 0.61), reach: float = 1.6, star_radius: float = 0.05,
                box: float = 1.0):
    """A DEEP tree built directly in boxes (the paper's production runs use 9 levels, L684; a 2048^3 lattice cannot be
    held whole): on every level the sub-grids whose centre lies within `reach` sub-grid widths of `centre` are refined, so
    that each level is a window of a few sub-grids around the same point; proper nesting over the 26 neighbours is
    enforced bottom-up on the sparse sets of sub-grids.  Density: one n = 1.5 polytrope of radius `star_radius` at
    `centre` over the 1e-10 floor.  Returns (boxes, kind, mass) with kind[l], mass[l] of shape [n_z][n_y][n_x] of box l."""
    assert n0 % 8 == 0 and depth >= 1
    refined = []                                   # per level: set of refined sub-grids (lattice coordinates)
    for l in range(depth - 1):
        s = (n0 // 8) << l                         # sub-grids per axis
        w = box / s
        c = [centre[a] / w for a in range(3)]      # centre in sub-grid units
        r = set()
        lo = [max(int(c[a] - reach - 1), 0) for a in range(3)]
        hi = [min(int(c[a] + reach + 2), s) for a in range(3)]
        for K in range(lo[2], hi[2]):
            for J in range(lo[1], hi[1]):
                for I in range(lo[0], hi[0]):
                    if (I + 0.5 - c[0]) ** 2 + (J + 0.5 - c[1]) ** 2 + (K + 0.5 - c[2]) ** 2 < reach * reach:
                        r.add((I, J, K))
        refined.append(r)
    refined.append(set())
    if depth > 1:
        refined[0] = {(I, J, K) for K in range(n0 // 8) for J in range(n0 // 8) for I in range(n0 // 8)} if n0 <= 16 else refined[0]
    # bottom-up: every 26-neighbour of a refined sub-grid must exist, i.e. its parent must be refined
    for l in range(depth - 2, 0, -1):
        s = (n0 // 8) << l
        for (I, J, K) in list(refined[l]):
            for dz in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dx in (-1, 0, 1):
                        q = (I + dx, J + dy, K + dz)
                        if 0 <= q[0] < s and 0 <= q[1] < s and 0 <= q[2] < s:
                            refined[l - 1].add((q[0] // 2, q[1] // 2, q[2] // 2))
    # top-down: a sub-grid exists iff its parent is refined; refined sub-grids must exist
    exists = [{(I, J, K) for K in range(n0 // 8) for J in range(n0 // 8) for I in range(n0 // 8)}]
    for l in range(depth - 1):
        refined[l] &= exists[l]
        exists.append({(2 * I + a, 2 * J + b, 2 * K + c) for (I, J, K) in refined[l] for a in (0, 1) for b in (0, 1) for c in (0, 1)})
    star = [Star(tuple(centre), star_radius, 1.0)]
    boxes, kind, mass = [], [], []
    for l in range(depth):
        n = n0 << l
        h = box / n
        if not exists[l]:
            boxes.append((0, 0, 0, 8, 8, 8)); kind.append(np.zeros((8, 8, 8), np.uint8)); mass.append(np.zeros((8, 8, 8)))
            continue
        lo = [min(q[a] for q in exists[l]) for a in range(3)]
        hi = [max(q[a] for q in exists[l]) + 1 for a in range(3)]
        b = (8 * lo[0], 8 * lo[1], 8 * lo[2], 8 * (hi[0] - lo[0]), 8 * (hi[1] - lo[1]), 8 * (hi[2] - lo[2]))
        sub = np.zeros((hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]), np.uint8)
        for (I, J, K) in exists[l]:
            sub[K - lo[2], J - lo[1], I - lo[0]] = TREE_REFINED if (I, J, K) in refined[l] else TREE_LEAF
        k = _expand8(sub)
        x = [(np.arange(b[3 + a]) + b[a] + 0.5) * h for a in range(3)]
        Z, Y, X = np.meshgrid(x[2], x[1], x[0], indexing="ij")
        m = np.where(k == TREE_LEAF, field_density(star, X, Y, Z) * h ** 3, 0.0)
        boxes.append(b); kind.append(np.ascontiguousarray(k)); mass.append(np.ascontiguousarray(m))
    return boxes, kind, mass
