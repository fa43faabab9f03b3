"""Independent mathematics used to pin the oracle and to post-process results.

Nothing here calls the oracle or the CUDA path.  The derivative tensors of -1/r are obtained
by letting sympy differentiate the potential (not by retyping closed forms), and the direct
sums are plain numpy over point masses.
"""
from __future__ import annotations

import functools
import itertools

import numpy as np

IDX2 = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
IDX3 = [(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 1, 2), (0, 2, 2),
        (1, 1, 1), (1, 1, 2), (1, 2, 2), (2, 2, 2)]


@functools.lru_cache(maxsize=None)
def _sym_derivatives(max_order=4):
    """Lambdified d^n(-1/r)/dx_i.. for every sorted multi-index, by symbolic differentiation."""
    import sympy as sp
    x, y, z = sp.symbols("x y z", real=True)
    v = (x, y, z)
    g = -1 / sp.sqrt(x * x + y * y + z * z)
    table = {(): sp.lambdify(v, g, "numpy")}
    exprs = {(): g}
    for n in range(1, max_order + 1):
        for idx in itertools.combinations_with_replacement(range(3), n):
            e = sp.diff(exprs[idx[:-1]], v[idx[-1]])
            exprs[idx] = e
            table[idx] = sp.lambdify(v, sp.simplify(e), "numpy")
    return table


def green_tensor(R, n):
    """Full rank-n derivative tensor of -1/|R| at R (numpy array of shape (3,)*n)."""
    tab = _sym_derivatives(4)
    out = np.zeros((3,) * n)
    for idx in itertools.product(range(3), repeat=n):
        out[idx] = tab[tuple(sorted(idx))](float(R[0]), float(R[1]), float(R[2]))
    return out if n else float(out)


def full2(u):
    T = np.zeros((3, 3) + np.shape(u)[1:])
    for t, (a, b) in enumerate(IDX2):
        T[a, b] = u[t]
        T[b, a] = u[t]
    return T


def full3(u):
    T = np.zeros((3, 3, 3) + np.shape(u)[1:])
    for t, idx in enumerate(IDX3):
        for p in set(itertools.permutations(idx)):
            T[p] = u[t]
    return T


def unique2(T):
    return np.array([T[a, b] for a, b in IDX2])


def unique3(T):
    return np.array([T[a, b, c] for a, b, c in IDX3])


def moments_of_points(m, y, centre):
    """Raw Cartesian moments (20 unique) of point masses m[p] at y[p] about `centre`."""
    d = np.asarray(y) - np.asarray(centre)[None, :]
    out = np.zeros(20)
    out[0] = m.sum()
    for a in range(3):
        out[1 + a] = (m * d[:, a]).sum()
    for t, (a, b) in enumerate(IDX2):
        out[4 + t] = (m * d[:, a] * d[:, b]).sum()
    for t, (a, b, c) in enumerate(IDX3):
        out[10 + t] = (m * d[:, a] * d[:, b] * d[:, c]).sum()
    return out


def exact_local_expansion(m, y, zA):
    """Exact derivatives (orders 0..3, 20 unique) at zA of phi = -sum m_p/|x - y_p|."""
    out = np.zeros(20)
    for mp, yp in zip(m, y):
        R = np.asarray(zA) - np.asarray(yp)
        out[0] += mp * green_tensor(R, 0)
        out[1:4] += mp * green_tensor(R, 1)
        out[4:10] += mp * unique2(green_tensor(R, 2))
        out[10:20] += mp * unique3(green_tensor(R, 3))
    return out


def cell_forces_and_torques(moments, com_off, L, h, lo=(0, 0, 0)):
    """Force and torque on every cell from its local expansion.

    F_A,i = -[M_A L1_i + M1_A,j L2_ij + 1/2 M2_A,jk L3_ijk]
    T_A   = z_A x F_A - eps_abc [M1_b L1_c + M2_bj L2_cj + 1/2 M3_bjk L3_cjk]
    moments [20][nz][ny][nx], com_off [3][...], L [20][...] on the same cells.
    z_A = (index + 1/2) h + delta.  Returns F[3][...], T[3][...]."""
    M0, M1, M2, M3 = moments[0], moments[1:4], full2(moments[4:10]), full3(moments[10:20])
    L1, L2, L3 = L[1:4], full2(L[4:10]), full3(L[10:20])
    gradphi = M0[None] * L1 + np.einsum("j...,ij...->i...", M1, L2) + 0.5 * np.einsum("jk...,ijk...->i...", M2, L3)
    F = -gradphi
    nz, ny, nx = M0.shape
    zx = ((np.arange(nx) + lo[0] + 0.5) * h)[None, None, :] + com_off[0]
    zy = ((np.arange(ny) + lo[1] + 0.5) * h)[None, :, None] + com_off[1]
    zz = ((np.arange(nz) + lo[2] + 0.5) * h)[:, None, None] + com_off[2]
    zc = np.stack([zx, zy, zz])
    T = np.cross(zc, F, axis=0)
    inner = (np.einsum("b...,c...->bc...", M1, L1) + np.einsum("bj...,cj...->bc...", M2, L2)
             + 0.5 * np.einsum("bjk...,cjk...->bc...", M3, L3))
    # eps_abc inner_bc
    T[0] -= inner[1, 2] - inner[2, 1]
    T[1] -= inner[2, 0] - inner[0, 2]
    T[2] -= inner[0, 1] - inner[1, 0]
    return F, T


def invariants_on_device(torch, mom, com, L, h):
    """Sum of the forces and of the torques over a whole closed level (the formulas of
    helpers.cell_forces_and_torques, component by component on device tensors so that 256^3 cells fit and take
    seconds).  Returns (max_i |sum F_i| / sum |F|, max_i |sum T_i| / sum |T|)."""
    i2 = {}
    for t, (a, b) in enumerate([(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]):
        i2[(a, b)] = i2[(b, a)] = 4 + t
    i3 = {}
    import itertools
    for t, idx in enumerate([(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 1, 2), (0, 2, 2), (1, 1, 1), (1, 1, 2), (1, 2, 2), (2, 2, 2)]):
        for q in set(itertools.permutations(idx)):
            i3[q] = 10 + t
    nz, ny, nx = mom.shape[1:]
    F = []
    for i in range(3):
        g = mom[0] * L[1 + i]
        for j in range(3):
            g = g + mom[1 + j] * L[i2[(i, j)]]
            for k in range(3):
                g = g + 0.5 * mom[i2[(j, k)]] * L[i3[(i, j, k)]]
        F.append(-g)
    ar = lambda m: (torch.arange(m, dtype=torch.float64, device=mom.device) + 0.5) * h
    z = [ar(nx)[None, None, :] + com[0], ar(ny)[None, :, None] + com[1], ar(nz)[:, None, None] + com[2]]
    inner = {}
    for b in range(3):
        for c in range(3):
            if b == c:
                continue
            v = mom[1 + b] * L[1 + c]
            for j in range(3):
                v = v + mom[i2[(b, j)]] * L[i2[(c, j)]]
                for k in range(3):
                    v = v + 0.5 * mom[i3[(b, j, k)]] * L[i3[(c, j, k)]]
            inner[(b, c)] = v
    T = []
    for a in range(3):
        b, c = (a + 1) % 3, (a + 2) % 3
        T.append(z[b] * F[c] - z[c] * F[b] - (inner[(b, c)] - inner[(c, b)]))

    def ratio(V):
        # plane sums on the device, the few hundred plane values summed exactly on the host
        import math
        tot = max(abs(math.fsum(v.sum(dim=(1, 2)).cpu().tolist())) for v in V)
        den = math.fsum(sum(v.abs().sum(dim=(1, 2)) for v in V).cpu().tolist())
        return tot / den
    return ratio(F), ratio(T)


def parity_error(got, ref):
    """north_star metric: per-cell max-norm error normalised by the cell's largest |coefficient|.

    got, ref: [ncoef][...cells...].  Returns the maximum over cells."""
    scale = np.abs(ref).max(axis=0)
    err = np.abs(got - ref).max(axis=0)
    scale = np.where(scale > 0, scale, 1.0)
    return float((err / scale).max())


def per_order_error(got, ref):
    """Max-norm error of each expansion order, normalised by that order's max |coefficient| per cell."""
    out = []
    for sl in (slice(0, 1), slice(1, 4), slice(4, 10), slice(10, 20)):
        out.append(parity_error(got[sl], ref[sl]))
    return out


def conditioned_order_error(got, gotc, ref, refc, labs):
    """Condition-aware per-order error: for each expansion order, and for the correction alone, the
    largest |got - ref| of the order's coefficients in a cell divided by the largest sum_B |term| of that order in the
    cell (labs [23][...] from oracle.interact_multipole_cond).  A correct kernel stays at a few n eps whatever the
    cancellation between partners; gotc/refc None skips the correction.  Returns [e0, e1, e2, e3, ecorr]."""
    out = []
    for sl in (slice(0, 1), slice(1, 4), slice(4, 10), slice(10, 20)):
        den = labs[sl].max(axis=0)
        den = np.where(den > 0, den, 1.0)
        out.append(float((np.abs(got[sl] - ref[sl]).max(axis=0) / den).max()))
    if gotc is not None and refc is not None:
        den = labs[20:23].max(axis=0)
        den = np.where(den > 0, den, 1.0)
        out.append(float((np.abs(gotc - refc).max(axis=0) / den).max()))
    else:
        out.append(0.0)
    return out


def load_golden(path):
    vals = {}
    multi = {}
    with open(path) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = line.split()
            multi.setdefault(parts[0], []).append(parts[1:])
            vals[parts[0]] = np.array([float(v) for v in parts[1:]]) if _all_float(parts[1:]) else parts[1:]
    vals["_multi"] = multi
    return vals


def _all_float(parts):
    try:
        [float(p) for p in parts]
        return True
    except ValueError:
        return False
