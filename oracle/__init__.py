"""ctypes binding of the CPU oracle (oracle/fmm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It never
imports the CUDA path (paper_2101_08226_b200) and shares no code with it.

The C source is compiled on first use with the host gcc:
    gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC fmm_oracle.c -o libfmm_oracle.so -lm
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fmm_oracle.c")
_LIB = os.path.join(_HERE, "libfmm_oracle.so")
_lib = None

OK, EINVAL, EMASS = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle if the shared object is missing or older than its source."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99",
               _SRC, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        ullp = ctypes.POINTER(ctypes.c_ulonglong)
        L.fmm_oracle_stencil.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int, ip,
                                         ctypes.POINTER(ctypes.c_byte)]
        L.fmm_oracle_green.argtypes = [dp, dp]
        L.fmm_oracle_pair.argtypes = [dp, dp, ctypes.c_double, dp, ctypes.c_int, dp, dp]
        L.fmm_oracle_interact_multipole.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                                    dp, dp, dp, dp, ullp]
        L.fmm_oracle_interact_multipole_cond.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                                         dp, dp, dp, dp, dp, ullp]
        L.fmm_oracle_interact_monopole.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, dp, dp, ullp]
        L.fmm_oracle_interact_multipole_mixed.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                                          dp, dp, ctypes.POINTER(ctypes.c_ubyte), dp, dp, ullp]
        L.fmm_oracle_interaction_count.argtypes = [ip, ip, ip, ctypes.c_double, ullp]
        L.fmm_oracle_stencil_leaf.argtypes = L.fmm_oracle_stencil.argtypes
        L.fmm_oracle_interact_monopole_leaf.argtypes = L.fmm_oracle_interact_monopole.argtypes
        L.fmm_oracle_m2m.argtypes = [ip, ctypes.c_double, dp, dp, dp, dp]
        L.fmm_oracle_m2m_about.argtypes = [ip, ctypes.c_double, dp, dp, dp, dp]
        L.fmm_oracle_l2l.argtypes = [ip, ctypes.c_double, dp, dp, dp, dp, dp, dp]
        L.fmm_oracle_direct_sum.argtypes = [ip, ctypes.c_double, dp, dp]
        ubp = ctypes.POINTER(ctypes.c_ubyte)
        L.fmm_oracle_tree_interact_multipole.argtypes = [ip, ctypes.c_double, ctypes.c_double, ctypes.c_int, dp, dp, ubp,
                                                         dp, dp, ullp]
        L.fmm_oracle_tree_leaf_p2p.argtypes = [ip, ctypes.c_double, ctypes.c_double, ubp, dp, dp, ullp]
        L.fmm_oracle_tree_cross_level.argtypes = [ip, ctypes.c_double, ctypes.c_double, ubp, dp, ubp, dp, dp, dp, ullp]
        L.fmm_oracle_direct_sum_points.argtypes = [ctypes.c_long, dp, dp, dp]
        L.fmm_oracle_num_threads.restype = ctypes.c_int
        L.fmm_oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i3(v):
    return (ctypes.c_int * 3)(*[int(x) for x in v])


def _check(rc, what):
    if rc != OK:
        raise RuntimeError("%s failed with status %d" % (what, rc))


def stencil(theta: float, parity: int) -> np.ndarray:
    """Partner offsets (dx,dy,dz) of parity class px+2py+4pz, int8 [count][3], (dz,dy,dx)-lexicographic."""
    L = lib()
    cnt = ctypes.c_int(0)
    _check(L.fmm_oracle_stencil(theta, parity, 0, ctypes.byref(cnt), None), "stencil")
    out = np.zeros((cnt.value, 3), dtype=np.int8)
    _check(L.fmm_oracle_stencil(theta, parity, cnt.value, ctypes.byref(cnt),
                                out.ctypes.data_as(ctypes.POINTER(ctypes.c_byte))), "stencil")
    return out


def green(R) -> tuple:
    """Full derivative tensors (D0, D1[3], D2[3,3], D3[3,3,3], D4[3,3,3,3]) of -1/|R|."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    out = np.zeros(121)
    _check(lib().fmm_oracle_green(_dp(R), _dp(out)), "green")
    return (out[0], out[1:4].copy(), out[4:13].reshape(3, 3).copy(), out[13:40].reshape(3, 3, 3).copy(),
            out[40:121].reshape(3, 3, 3, 3).copy())


def pair(R, MB, MA0=1.0, MA3=None, correction=False):
    """One ordered pair A<-B: returns (L[20] without correction, dL1[3])."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    MB = np.ascontiguousarray(MB, dtype=np.float64)
    MA3 = np.zeros(10) if MA3 is None else np.ascontiguousarray(MA3, dtype=np.float64)
    Lo, dL = np.zeros(20), np.zeros(3)
    _check(lib().fmm_oracle_pair(_dp(R), _dp(MB), float(MA0), _dp(MA3), int(bool(correction)), _dp(Lo), _dp(dL)),
           "pair")
    return Lo, dL


def interact_multipole(n, h, theta, moments, com_off, out_lo=None, out_hi=None, am_correction=True, threads=None):
    """Returns (L[20][oz][oy][ox], Lcorr[3][oz][oy][ox], n_interactions)."""
    L = lib()
    if threads:
        L.fmm_oracle_set_num_threads(int(threads))
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    nx, ny, nz = n
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    Lout = np.zeros((20, o[2], o[1], o[0]))
    Lc = np.zeros((3, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    rc = L.fmm_oracle_interact_multipole(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta),
                                         int(bool(am_correction)), _dp(moments), _dp(com_off), _dp(Lout), _dp(Lc),
                                         ctypes.byref(cnt))
    _check(rc, "interact_multipole")
    return Lout, Lc, cnt.value


def interact_multipole_cond(n, h, theta, moments, com_off, out_lo=None, out_hi=None, am_correction=True):
    """interact_multipole plus the condition of every sum: returns (L, Lcorr, Labs[23][oz][oy][ox], n_interactions),
    Labs = sum over the partners of |term| for the 20 coefficients and the 3 components of the correction."""
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    nx, ny, nz = n
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    Lout = np.zeros((20, o[2], o[1], o[0]))
    Lc = np.zeros((3, o[2], o[1], o[0]))
    La = np.zeros((23, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    rc = lib().fmm_oracle_interact_multipole_cond(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta),
                                                  int(bool(am_correction)), _dp(moments), _dp(com_off), _dp(Lout), _dp(Lc),
                                                  _dp(La), ctypes.byref(cnt))
    _check(rc, "interact_multipole_cond")
    return Lout, Lc, La, cnt.value


def interact_multipole_mixed(n, h, theta, moments, com_off, leaf, out_lo=None, out_hi=None, am_correction=True):
    """One level of an adaptive mesh: leaf[nz][ny][nx] = 1 where the cell belongs to a leaf sub-grid.
    Partners of A = the Eq. 15 list + the near-field cells B with leaf[A] or leaf[B].  Returns (L, Lcorr, n_interactions)."""
    L = lib()
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    leaf = np.ascontiguousarray(leaf, dtype=np.uint8)
    nx, ny, nz = n
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx) and leaf.shape == (nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    Lout = np.zeros((20, o[2], o[1], o[0]))
    Lc = np.zeros((3, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    rc = L.fmm_oracle_interact_multipole_mixed(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta),
                                               int(bool(am_correction)), _dp(moments), _dp(com_off),
                                               leaf.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)), _dp(Lout), _dp(Lc),
                                               ctypes.byref(cnt))
    _check(rc, "interact_multipole_mixed")
    return Lout, Lc, cnt.value


def interact_monopole(n, h, theta, mass, out_lo=None, out_hi=None, threads=None):
    """Returns (out[4][oz][oy][ox] = phi,gx,gy,gz ; n_interactions)."""
    L = lib()
    if threads:
        L.fmm_oracle_set_num_threads(int(threads))
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    nx, ny, nz = n
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    out = np.zeros((4, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    _check(L.fmm_oracle_interact_monopole(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta), _dp(mass),
                                          _dp(out), ctypes.byref(cnt)), "interact_monopole")
    return out, cnt.value


def interaction_count(n, theta, out_lo=None, out_hi=None) -> int:
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_interaction_count(_i3(n), _i3(out_lo), _i3(out_hi), float(theta), ctypes.byref(cnt)),
           "interaction_count")
    return cnt.value


def num_threads() -> int:
    return int(lib().fmm_oracle_num_threads())


# ---- NEXT f1: the other passes of a complete uniform-grid solve ------------------------------------
def stencil_leaf(theta: float, parity: int) -> np.ndarray:
    """Leaf-level list of the complete solve: the Eq. 15 list plus the near field (every Delta != 0 whose
    parents are not well separated), int8 [count][3], (dz,dy,dx)-lexicographic."""
    L = lib()
    cnt = ctypes.c_int(0)
    _check(L.fmm_oracle_stencil_leaf(theta, parity, 0, ctypes.byref(cnt), None), "stencil_leaf")
    out = np.zeros((cnt.value, 3), dtype=np.int8)
    _check(L.fmm_oracle_stencil_leaf(theta, parity, cnt.value, ctypes.byref(cnt),
                                     out.ctypes.data_as(ctypes.POINTER(ctypes.c_byte))), "stencil_leaf")
    return out


def interact_monopole_leaf(n, h, theta, mass):
    """Monopole sum over the leaf-level list (Eq. 15 list + near field), whole grid.  Returns (out[4], count)."""
    nx, ny, nz = n
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(nz, ny, nx)
    out = np.zeros((4, nz, ny, nx))
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_interact_monopole_leaf(_i3(n), _i3((0, 0, 0)), _i3(n), float(h), float(theta), _dp(mass),
                                                   _dp(out), ctypes.byref(cnt)), "interact_monopole_leaf")
    return out, cnt.value


def m2m(n_child, h_child, moments, com_off):
    """Parent multipoles [20][n/2] and centre-of-mass offsets [3][n/2] from the children's (L125)."""
    nx, ny, nz = n_child
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx)
    pm = np.zeros((20, nz // 2, ny // 2, nx // 2))
    po = np.zeros((3, nz // 2, ny // 2, nx // 2))
    _check(lib().fmm_oracle_m2m(_i3(n_child), float(h_child), _dp(moments), _dp(com_off), _dp(pm), _dp(po)), "m2m")
    return pm, po


def m2m_about(n_child, h_child, moments, com_off, parent_off):
    """Parent multipoles [20][n/2] about PRESCRIBED parent centres parent_off [3][n/2] (second right-hand side, L81-83)."""
    nx, ny, nz = n_child
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    parent_off = np.ascontiguousarray(parent_off, dtype=np.float64)
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx)
    assert parent_off.shape == (3, nz // 2, ny // 2, nx // 2)
    pm = np.zeros((20, nz // 2, ny // 2, nx // 2))
    _check(lib().fmm_oracle_m2m_about(_i3(n_child), float(h_child), _dp(moments), _dp(com_off), _dp(parent_off), _dp(pm)),
           "m2m_about")
    return pm


def l2l(n_child, h_child, parent_L, parent_corr, parent_off, child_off, child_L, child_corr):
    """child_L += parent_L shifted to the child centres, child_corr += parent_corr (in place; L125)."""
    for a in (parent_L, parent_corr, parent_off, child_off, child_L, child_corr):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    _check(lib().fmm_oracle_l2l(_i3(n_child), float(h_child), _dp(parent_L), _dp(parent_corr), _dp(parent_off),
                                _dp(child_off), _dp(child_L), _dp(child_corr)), "l2l")


def direct_sum(n, h, mass):
    """Exact point-mass sum on the cell centres, out[4][nz][ny][nx] = (phi, g).  O(N^2)."""
    nx, ny, nz = n
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(nz, ny, nx)
    out = np.zeros((4, nz, ny, nx))
    _check(lib().fmm_oracle_direct_sum(_i3(n), float(h), _dp(mass), _dp(out)), "direct_sum")
    return out


def solve_rhs2(n, h, theta, mass, dmass, coarsest=2):
    """Second right-hand side (Alg. 1: "Compute g, phi, and d(phi)/dt using the FMM ... with
    the numerically computed value of d(rho)/dt as the source term"): the same tree, lists and EXPANSION CENTRES as
    solve(n, h, theta, mass) -- the centres of mass of `mass` -- but the sources are the signed point sources
    `dmass` at the leaf centres, and no angular-momentum correction (it belongs to the force, L127).
    Returns out[4][n][n][n] = (d(phi)/dt, -grad of it)."""
    n = int(n)
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(n, n, n)
    dmass = np.ascontiguousarray(dmass, dtype=np.float64).reshape(n, n, n)
    # ---- centres: upward pass of the density ----
    lev_n, lev_h = [n], [float(h)]
    mom = np.zeros((20, n, n, n)); mom[0] = mass
    mom2 = np.zeros((20, n, n, n)); mom2[0] = dmass
    lev_m, lev_o, lev_m2 = [mom], [np.zeros((3, n, n, n))], [mom2]
    while lev_n[-1] > coarsest:
        nc, hc = lev_n[-1], lev_h[-1]
        pm, po = m2m((nc, nc, nc), hc, lev_m[-1], lev_o[-1])
        pm2 = m2m_about((nc, nc, nc), hc, lev_m2[-1], lev_o[-1], po)
        lev_n.append(nc // 2); lev_h.append(2.0 * hc); lev_m.append(pm); lev_o.append(po); lev_m2.append(pm2)
    # ---- downward pass of the second right-hand side ----
    L_par = None
    for lv in range(len(lev_n) - 1, 0, -1):
        nl, hl = lev_n[lv], lev_h[lv]
        L, Lc, _ = interact_multipole((nl, nl, nl), hl, theta, lev_m2[lv], lev_o[lv], None, None, False)
        L = L.copy()
        zero_c = np.zeros_like(Lc)
        if L_par is not None:
            l2l((nl, nl, nl), hl, L_par, np.zeros((3,) + L_par.shape[1:]), lev_o[lv + 1], lev_o[lv], L, zero_c)
        L_par = L
    out, _ = interact_monopole_leaf((n, n, n), h, theta, dmass)
    if L_par is not None:
        Ll = np.zeros((20, n, n, n)); cl = np.zeros((3, n, n, n))
        l2l((n, n, n), h, L_par, np.zeros((3,) + L_par.shape[1:]), lev_o[1], lev_o[0], Ll, cl)
        out[0] += Ll[0]
        out[1:4] -= Ll[1:4]
    return out


def solve(n, h, theta, mass, am_correction=True, coarsest=2):
    """Complete uniform-grid solve on an isolated cubic grid of n = 2^k leaf cells per axis (2^3-cell level is the
    coarsest that can hold interacting cells: siblings interact there when 3 theta^2 > 1):
    leaves are point masses at their cell centres; upward pass (M2M) to the level of `coarsest`^3 cells; at every
    multipole level the same-level interaction step (the hot path, Eq. 15 list, correction optional) plus the
    parent's expansion (L2L); at the leaves the expansion of the parent evaluated at the cell centre plus the
    monopole sum over the leaf-level list (Eq. 15 list + near field).  Returns out[4][n][n][n] = (phi, g_x, g_y, g_z),
    g = -(L1 + correction) + direct part.  A cell's own mass contributes nothing (point-mass model)."""
    n = int(n)
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(n, n, n)
    # ---- upward pass ----
    lev_n, lev_h = [n], [float(h)]
    mom = np.zeros((20, n, n, n))
    mom[0] = mass
    lev_m, lev_o = [mom], [np.zeros((3, n, n, n))]
    while lev_n[-1] > coarsest:
        nc, hc = lev_n[-1], lev_h[-1]
        assert nc % 2 == 0
        pm, po = m2m((nc, nc, nc), hc, lev_m[-1], lev_o[-1])
        lev_n.append(nc // 2); lev_h.append(2.0 * hc); lev_m.append(pm); lev_o.append(po)
    # ---- downward pass over the multipole levels (coarsest first) ----
    L_par = corr_par = None
    for lv in range(len(lev_n) - 1, 0, -1):
        nl, hl = lev_n[lv], lev_h[lv]
        Lf, Lc, _ = interact_multipole((nl, nl, nl), hl, theta, lev_m[lv], lev_o[lv], None, None, am_correction)
        L = Lf.copy()
        L[1:4] -= Lc                       # the expansion proper; the correction is carried beside it
        corr = Lc.copy()
        if L_par is not None:
            l2l((nl, nl, nl), hl, L_par, corr_par, lev_o[lv + 1], lev_o[lv], L, corr)
        L_par, corr_par = L, corr
    # ---- leaves ----
    out, _ = interact_monopole_leaf((n, n, n), h, theta, mass)
    if L_par is not None:
        Ll = np.zeros((20, n, n, n)); cl = np.zeros((3, n, n, n))
        l2l((n, n, n), h, L_par, corr_par, lev_o[1], lev_o[0], Ll, cl)
        out[0] += Ll[0]
        out[1:4] -= Ll[1:4] + cl
    return out


# ---- adaptive oct-tree of 8^3 sub-grids (reading R9) ------------------------------------
def _ub(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte))


def _n3(n):
    """(nx, ny, nz) from an int (cubic) or a 3-tuple."""
    return (int(n),) * 3 if np.isscalar(n) else tuple(int(v) for v in n)


def tree_interact_multipole(n, h, theta, moments, com_off, kind, am_correction=True):
    """Same-level multipole step on one level of a tree (kind: 0 absent, 1 leaf, 2 refined): every existing cell takes
    the existing cells of its Eq. 15 list, except that two leaves do not meet here.  Returns (L, Lcorr, count)."""
    nx, ny, nz = _n3(n)
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx) and kind.shape == (nz, ny, nx)
    Lout, Lc = np.zeros((20, nz, ny, nx)), np.zeros((3, nz, ny, nx))
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_tree_interact_multipole(_i3((nx, ny, nz)), float(h), float(theta), int(bool(am_correction)),
                                                    _dp(moments), _dp(com_off), _ub(kind), _dp(Lout), _dp(Lc),
                                                    ctypes.byref(cnt)), "tree_interact_multipole")
    return Lout, Lc, cnt.value


def tree_leaf_p2p(n, h, theta, kind, mass):
    """Point-mass sum of the leaf cells of one level over the leaf-level list.  Returns (out[4][n][n][n], count)."""
    nx, ny, nz = _n3(n)
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    assert kind.shape == (nz, ny, nx) and mass.shape == (nz, ny, nx)
    out = np.zeros((4, nz, ny, nx))
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_tree_leaf_p2p(_i3((nx, ny, nz)), float(h), float(theta), _ub(kind), _dp(mass), _dp(out),
                                          ctypes.byref(cnt)), "tree_leaf_p2p")
    return out, cnt.value


def tree_cross_level(nc, hc, theta, kind_c, mass_c, kind_f, mass_f, out_c, out_f):
    """Point-mass pairs across a refinement boundary: a coarse leaf and the 8 children of every refined cell of its
    near field, both directions; ADDED to out_c [4][nc]^3 and out_f [4][2 nc]^3.  Returns the number of ordered pairs."""
    cx, cy, cz = _n3(nc)
    for a in (kind_c, kind_f):
        assert a.dtype == np.uint8 and a.flags["C_CONTIGUOUS"]
    for a in (mass_c, mass_f, out_c, out_f):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    assert kind_c.shape == (cz, cy, cx) and kind_f.shape == (2 * cz, 2 * cy, 2 * cx) and out_c.shape == (4, cz, cy, cx)
    assert out_f.shape == (4, 2 * cz, 2 * cy, 2 * cx) and mass_f.shape == kind_f.shape and mass_c.shape == kind_c.shape
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_tree_cross_level(_i3((cx, cy, cz)), float(hc), float(theta), _ub(kind_c), _dp(mass_c), _ub(kind_f),
                                             _dp(mass_f), _dp(out_c), _dp(out_f), ctypes.byref(cnt)), "tree_cross_level")
    return cnt.value


def direct_sum_points(pos, mass):
    """Exact (phi, g) of point masses at arbitrary positions; pos [np][3], returns out [np][4].  O(N^2)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    out = np.zeros((len(mass), 4))
    _check(lib().fmm_oracle_direct_sum_points(len(mass), _dp(pos), _dp(mass), _dp(out)), "direct_sum_points")
    return out


def _embed(arr, box, frame):
    """arr [..., nz, ny, nx] living on box = (lo_x, lo_y, lo_z, n_x, n_y, n_z) of a lattice, placed into zeros of the
    frame (same convention); the parts of the box outside the frame are dropped."""
    out = np.zeros(arr.shape[:-3] + (frame[5], frame[4], frame[3]), dtype=arr.dtype)
    src, dst = [], []
    for a in (2, 1, 0):                     # z, y, x
        lo = max(box[a], frame[a]); hi = min(box[a] + box[3 + a], frame[a] + frame[3 + a])
        if hi <= lo:
            return out
        src.append(slice(lo - box[a], hi - box[a])); dst.append(slice(lo - frame[a], hi - frame[a]))
    out[(Ellipsis,) + tuple(dst)] = arr[(Ellipsis,) + tuple(src)]
    return out


def _extract(arr, frame, box):
    """Inverse of _embed for a box that lies inside the frame."""
    sl = tuple(slice(box[a] - frame[a], box[a] - frame[a] + box[3 + a]) for a in (2, 1, 0))
    return np.ascontiguousarray(arr[(Ellipsis,) + sl])


def solve_tree(n0, h0, theta, kind, mass, am_correction=True, coarsest=2, box=None):
    """The gravity solve on an adaptive oct-tree of 8^3 sub-grids ("The FMM adapts naturally to an
    oct-tree based adaptive mesh refinement"; L287-291; reading R9).  Level l = 0 .. len(kind)-1 lives on the
    lattice of n_l = n0 2^l cells per axis, h_l = h0 / 2^l, with kind[l] (0 absent, 1 leaf, 2 refined) and mass[l] (leaf
    masses); above level 0 the uniform levels n0/2 .. `coarsest` as in solve().  box = None: every array is its whole
    lattice [n_l]^3; else box[l] = (lo_x, lo_y, lo_z, n_x, n_y, n_z): the arrays of level l cover that box only and cells
    outside it do not exist (level 0: the whole lattice).  Steps, in the paper's order (L125):
      upward    leaf = point mass at its geometric centre; refined cell = M2M of its 8 children (leaf or refined);
      downward  every existing cell: same-level step over its Eq. 15 list (two leaves excepted) + its parent's
                expansion (L2L), the correction carried beside it;
      leaves    phi = L0 + point-mass sums, g = -(L1 + correction) + point-mass sums, the sums being (a) the leaves of
                its own level on the leaf-level list, (b) the children of the refined cells of its near field, (c) the
                coarser leaves in the near field of its parent.
    The parent <-> child steps (M2M, L2L, cross-level pairs) are the dense ones applied to the child arrays embedded in
    the frame of the children of the parent's box (zeros outside the child's box: absent cells).
    Returns (out, counts): out[l] = [4] + shape of level l = (phi, g) at the leaf cells of level l (0 elsewhere);
    counts = {"m2l": .., "p2p": .., "cross": .., and per tree level "m2l_levels", "p2p_levels", "cross_levels"} ordered pairs
    ("m2l" includes the uniform levels above level 0)."""
    D = len(kind)
    n0 = int(n0)
    if box is None:
        box = [(0, 0, 0) + (n0 << l,) * 3 for l in range(D)]
    box = [tuple(int(v) for v in b) for b in box]
    assert box[0] == (0, 0, 0, n0, n0, n0)
    shp = [(b[5], b[4], b[3]) for b in box]
    kind = [np.ascontiguousarray(k, dtype=np.uint8) for k in kind]
    for l in range(D):
        assert kind[l].shape == shp[l] and np.shape(mass[l]) == shp[l]
    mass = [np.ascontiguousarray(np.where(k == 1, m, 0.0), dtype=np.float64) for k, m in zip(kind, mass)]
    hs = [float(h0) / (1 << l) for l in range(D)]
    # the frame of the children of level l's box, on the lattice of level l + 1
    cframe = [tuple(2 * v for v in b) for b in box]
    # ---- upward pass over the tree levels ----
    mom, off = [None] * D, [None] * D
    for l in range(D - 1, -1, -1):
        m = np.zeros((20,) + shp[l]); m[0] = mass[l]
        o = np.zeros((3,) + shp[l])
        if l < D - 1:
            f = cframe[l]
            pm, po = m2m((f[3], f[4], f[5]), hs[l + 1], _embed(mom[l + 1], box[l + 1], f), _embed(off[l + 1], box[l + 1], f))
            ref = kind[l] == 2
            m = np.where(ref[None], pm, m)
            o = np.where(ref[None], po, o)
        mom[l], off[l] = np.ascontiguousarray(m), np.ascontiguousarray(o)
    # ---- the uniform levels above level 0 ----
    up_n, up_h, up_m, up_o = [n0], [hs[0]], [mom[0]], [off[0]]
    while up_n[-1] > coarsest:
        nc, hc = up_n[-1], up_h[-1]
        pm, po = m2m((nc, nc, nc), hc, up_m[-1], up_o[-1])
        up_n.append(nc // 2); up_h.append(2.0 * hc); up_m.append(pm); up_o.append(po)
    counts = {"m2l": 0, "p2p": 0, "cross": 0, "m2l_levels": [], "p2p_levels": [], "cross_levels": []}
    L_par = corr_par = off_par = None
    for lv in range(len(up_n) - 1, 0, -1):
        nl, hl = up_n[lv], up_h[lv]
        Lf, Lc, c = interact_multipole((nl, nl, nl), hl, theta, up_m[lv], up_o[lv], None, None, am_correction)
        counts["m2l"] += c
        L = Lf.copy(); L[1:4] -= Lc
        corr = Lc.copy()
        if L_par is not None:
            l2l((nl, nl, nl), hl, L_par, corr_par, off_par, up_o[lv], L, corr)
        L_par, corr_par, off_par = L, corr, up_o[lv]
    # ---- downward pass over the tree levels, leaves evaluated on the way ----
    out, exp = [None] * D, [None] * D
    for l in range(D):
        n3, h = (box[l][3], box[l][4], box[l][5]), hs[l]
        Lf, Lc, c = tree_interact_multipole(n3, h, theta, mom[l], off[l], kind[l], am_correction)
        counts["m2l"] += c
        counts["m2l_levels"].append(c)
        L = Lf.copy(); L[1:4] -= Lc
        corr = Lc.copy()
        if L_par is not None:
            if l == 0:
                l2l(n3, h, L_par, corr_par, off_par, off[l], L, corr)
            else:
                f = cframe[l - 1]                  # the parent's arrays cover box[l-1]; this level embedded in its children's frame
                Le, ce = _embed(L, box[l], f), _embed(corr, box[l], f)
                l2l((f[3], f[4], f[5]), h, L_par, corr_par, off_par, _embed(off[l], box[l], f), Le, ce)
                L, corr = _extract(Le, f, box[l]), _extract(ce, f, box[l])
        o, c = tree_leaf_p2p(n3, h, theta, kind[l], mass[l])
        counts["p2p"] += c
        counts["p2p_levels"].append(c)
        out[l] = o
        L_par, corr_par, off_par = L, corr, off[l]
        exp[l] = (L, corr)
    for l in range(D - 1):
        f = cframe[l]
        of = _embed(out[l + 1], box[l + 1], f)
        c = tree_cross_level((box[l][3], box[l][4], box[l][5]), hs[l], theta, kind[l], mass[l], _embed(kind[l + 1], box[l + 1], f),
                             _embed(mass[l + 1], box[l + 1], f), out[l], of)
        out[l + 1] = _extract(of, f, box[l + 1])
        counts["cross"] += c
        counts["cross_levels"].append(c)
    for l in range(D):
        L, corr = exp[l]
        leaf = kind[l] == 1
        out[l][0] += np.where(leaf, L[0], 0.0)
        out[l][1:4] -= np.where(leaf[None], L[1:4] + corr, 0.0)
    return out, counts


# ---- the five calls of the boundary on host arrays: one harness drives the oracle and the library -------
class _OracleConfig(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int * 3), ("out_lo", ctypes.c_int * 3), ("out_hi", ctypes.c_int * 3), ("h", ctypes.c_double),
                ("theta", ctypes.c_double), ("kind", ctypes.c_int), ("am_correction", ctypes.c_int)]


class Oracle:
    """The oracle behind the call sequence of the library's boundary -- create / set_moments / interact / get_expansions /
    destroy (`fmm_oracle_*` in fmm_oracle.c) -- with the method names of paper_2101_08226_b200.OctoFMM, on numpy arrays."""
    MULTIPOLE, MONOPOLE = 0, 1

    def __init__(self, n, h, theta, kind=0, am_correction=True, out_lo=(0, 0, 0), out_hi=(0, 0, 0)):
        L = lib()
        L.fmm_oracle_create.argtypes = [ctypes.POINTER(_OracleConfig), ctypes.POINTER(ctypes.c_void_p)]
        dp = ctypes.POINTER(ctypes.c_double)
        L.fmm_oracle_set_moments.argtypes = [ctypes.c_void_p, dp, dp]
        L.fmm_oracle_interact.argtypes = [ctypes.c_void_p]
        L.fmm_oracle_get_expansions.argtypes = [ctypes.c_void_p, dp, dp]
        L.fmm_oracle_destroy.argtypes = [ctypes.c_void_p]
        L.fmm_oracle_handle_interaction_count.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_ulonglong)]
        c = _OracleConfig()
        for a in range(3):
            c.n[a], c.out_lo[a], c.out_hi[a] = int(n[a]), int(out_lo[a]), int(out_hi[a])
        c.h, c.theta, c.kind, c.am_correction = float(h), float(theta), int(kind), int(bool(am_correction))
        self.kind, self.n = int(kind), tuple(int(v) for v in n)
        whole = all(v == 0 for v in tuple(out_lo) + tuple(out_hi))
        lo, hi = ((0, 0, 0), self.n) if whole else (tuple(out_lo), tuple(out_hi))
        self.out_shape = (hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0])
        self.handle = ctypes.c_void_p()
        _check(L.fmm_oracle_create(ctypes.byref(c), ctypes.byref(self.handle)), "create")

    def set_moments(self, moments, com_off=None):
        moments = np.ascontiguousarray(moments, dtype=np.float64)
        com = None if com_off is None else np.ascontiguousarray(com_off, dtype=np.float64)
        _check(lib().fmm_oracle_set_moments(self.handle, _dp(moments), None if com is None else _dp(com)), "set_moments")

    def interact(self):
        _check(lib().fmm_oracle_interact(self.handle), "interact")

    def get_expansions(self):
        Lo = np.zeros(((20 if self.kind == 0 else 4),) + self.out_shape)
        Lc = np.zeros((3,) + self.out_shape) if self.kind == 0 else None
        _check(lib().fmm_oracle_get_expansions(self.handle, _dp(Lo), None if Lc is None else _dp(Lc)), "get_expansions")
        return Lo, Lc

    def interaction_count(self):
        n = ctypes.c_ulonglong(0)
        _check(lib().fmm_oracle_handle_interaction_count(self.handle, ctypes.byref(n)), "interaction_count")
        return int(n.value)

    def close(self):
        if self.handle:
            lib().fmm_oracle_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def solve_tree_rhs2(n0, h0, theta, kind, mass, dmass, coarsest=2, box=None):
    """Second right-hand side on the adaptive tree (Alg. 1: "Compute g, phi, and d(phi)/dt using
    the FMM"): the tree, lists and EXPANSION CENTRES of solve_tree(.., mass) -- the centres of mass of `mass` -- with the
    signed point sources dmass[l] at the leaf centres, no angular-momentum correction (readings R6, R7 of solve_rhs2, on
    the tree of R9).  Same arguments as solve_tree.  Returns out[l] = [4] + shape of level l = (d(phi)/dt, -grad of it)
    at the leaf cells."""
    D = len(kind)
    n0 = int(n0)
    if box is None:
        box = [(0, 0, 0) + (n0 << l,) * 3 for l in range(D)]
    box = [tuple(int(v) for v in b) for b in box]
    shp = [(b[5], b[4], b[3]) for b in box]
    kind = [np.ascontiguousarray(k, dtype=np.uint8) for k in kind]
    mass = [np.ascontiguousarray(np.where(k == 1, m, 0.0), dtype=np.float64) for k, m in zip(kind, mass)]
    dmass = [np.ascontiguousarray(np.where(k == 1, m, 0.0), dtype=np.float64) for k, m in zip(kind, dmass)]
    hs = [float(h0) / (1 << l) for l in range(D)]
    cframe = [tuple(2 * v for v in b) for b in box]
    # ---- upward: the density fixes the centres; d(rho)/dt is expanded about them ----
    mom, mom2, off = [None] * D, [None] * D, [None] * D
    for l in range(D - 1, -1, -1):
        m = np.zeros((20,) + shp[l]); m[0] = mass[l]
        m2 = np.zeros((20,) + shp[l]); m2[0] = dmass[l]
        o = np.zeros((3,) + shp[l])
        if l < D - 1:
            f = cframe[l]
            cm, co = _embed(mom[l + 1], box[l + 1], f), _embed(off[l + 1], box[l + 1], f)
            pm, po = m2m((f[3], f[4], f[5]), hs[l + 1], cm, co)
            ref = kind[l] == 2
            o = np.where(ref[None], po, o)
            pm2 = m2m_about((f[3], f[4], f[5]), hs[l + 1], _embed(mom2[l + 1], box[l + 1], f), co, np.ascontiguousarray(o))
            m = np.where(ref[None], pm, m)
            m2 = np.where(ref[None], pm2, m2)
        mom[l], mom2[l], off[l] = np.ascontiguousarray(m), np.ascontiguousarray(m2), np.ascontiguousarray(o)
    up_n, up_h, up_m, up_m2, up_o = [n0], [hs[0]], [mom[0]], [mom2[0]], [off[0]]
    while up_n[-1] > coarsest:
        nc, hc = up_n[-1], up_h[-1]
        pm, po = m2m((nc, nc, nc), hc, up_m[-1], up_o[-1])
        pm2 = m2m_about((nc, nc, nc), hc, up_m2[-1], up_o[-1], po)
        up_n.append(nc // 2); up_h.append(2.0 * hc); up_m.append(pm); up_m2.append(pm2); up_o.append(po)
    # ---- downward: the uniform levels, then the tree levels; no correction ----
    L_par = off_par = None
    for lv in range(len(up_n) - 1, 0, -1):
        nl, hl = up_n[lv], up_h[lv]
        L, Lc, _ = interact_multipole((nl, nl, nl), hl, theta, up_m2[lv], up_o[lv], None, None, False)
        L = L.copy()
        if L_par is not None:
            l2l((nl, nl, nl), hl, L_par, np.zeros((3,) + L_par.shape[1:]), off_par, up_o[lv], L, np.zeros_like(Lc))
        L_par, off_par = L, up_o[lv]
    out, exp = [None] * D, [None] * D
    for l in range(D):
        n3, h = (box[l][3], box[l][4], box[l][5]), hs[l]
        L, Lc, _ = tree_interact_multipole(n3, h, theta, mom2[l], off[l], kind[l], False)
        L = L.copy()
        if L_par is not None:
            zp = np.zeros((3,) + L_par.shape[1:])
            if l == 0:
                l2l(n3, h, L_par, zp, off_par, off[l], L, np.zeros_like(Lc))
            else:
                f = cframe[l - 1]
                Le = _embed(L, box[l], f)
                l2l((f[3], f[4], f[5]), h, L_par, zp, off_par, _embed(off[l], box[l], f), Le, np.zeros((3,) + Le.shape[1:]))
                L = _extract(Le, f, box[l])
        out[l], _ = tree_leaf_p2p(n3, h, theta, kind[l], dmass[l])
        L_par, off_par = L, off[l]
        exp[l] = L
    for l in range(D - 1):
        f = cframe[l]
        of = _embed(out[l + 1], box[l + 1], f)
        tree_cross_level((box[l][3], box[l][4], box[l][5]), hs[l], theta, kind[l], dmass[l], _embed(kind[l + 1], box[l + 1], f),
                         _embed(dmass[l + 1], box[l + 1], f), out[l], of)
        out[l + 1] = _extract(of, f, box[l + 1])
    for l in range(D):
        leaf = kind[l] == 1
        out[l][0] += np.where(leaf, exp[l][0], 0.0)
        out[l][1:4] -= np.where(leaf[None], exp[l][1:4], 0.0)
    return out
