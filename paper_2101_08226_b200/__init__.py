"""Python binding of the octo_fmm C ABI (include/octo_fmm.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libocto_fmm.so; PyTorch provides device
memory and the stream.  There is no CPU fallback: if the shared library is missing, the first
call into the library raises ImportError.  Build it with `python -m paper_2101_08226_b200.build` (or
`__graft_entry__.build()`).

The module-level functions carry the C names (octo_fmm_create, ...); `OctoFMM` is a small
convenience wrapper that owns the workspace tensor.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libocto_fmm.so")

OK, EINVAL, ESTATE, ENOMEM, ECUDA, EMASS, ESIZE = 0, 1, 2, 3, 4, 5, 6
MULTIPOLE, MONOPOLE = 0, 1
_STATUS = {0: "OK", 1: "EINVAL", 2: "ESTATE", 3: "ENOMEM", 4: "ECUDA", 5: "EMASS",
           6: "ESIZE: more cells than the static scratch of octo_fmm_interact_static holds"}


class OctoFmmError(RuntimeError):
    def __init__(self, call, status):
        super().__init__("%s failed: OCTO_FMM_%s (%d)" % (call, _STATUS.get(status, "?"), status))
        self.status = status


class octo_fmm_config(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int * 3), ("out_lo", ctypes.c_int * 3), ("out_hi", ctypes.c_int * 3),
                ("h", ctypes.c_double), ("origin", ctypes.c_double * 3), ("theta", ctypes.c_double),
                ("kind", ctypes.c_int), ("am_correction", ctypes.c_int), ("device", ctypes.c_int),
                ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t)]


class octo_fmm_peer(ctypes.Structure):
    _fields_ = [("sources", ctypes.c_void_p), ("flags", ctypes.c_void_p), ("nz", ctypes.c_int)]


class octo_fmm_tree_config(ctypes.Structure):
    _fields_ = [("n0", ctypes.c_int), ("depth", ctypes.c_int), ("h0", ctypes.c_double), ("theta", ctypes.c_double),
                ("am_correction", ctypes.c_int), ("device", ctypes.c_int), ("stream", ctypes.c_void_p),
                ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t)]


class octo_fmm_solver_config(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int), ("h", ctypes.c_double), ("theta", ctypes.c_double), ("am_correction", ctypes.c_int),
                ("device", ctypes.c_int), ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p),
                ("workspace_bytes", ctypes.c_size_t), ("two_rhs", ctypes.c_int)]


class _Library:
    """Loads libocto_fmm.so on first use and fails loudly when it is missing (no CPU fallback).

    Loading is deferred only so that `paper_2101_08226_b200.build` can be imported to produce it."""

    def __init__(self):
        self._cdll = None

    def _load(self):
        if not os.path.exists(_LIB_PATH):
            raise ImportError("paper_2101_08226_b200: %s is missing -- build it with "
                              "`python -m paper_2101_08226_b200.build`; there is no CPU fallback" % _LIB_PATH)
        lib = ctypes.CDLL(_LIB_PATH)
        vp, ip, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)
        cfgp = ctypes.POINTER(octo_fmm_config)
        lib.octo_fmm_workspace_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_workspace_bytes.argtypes = [cfgp]
        lib.octo_fmm_host_scratch_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_host_scratch_bytes.argtypes = [cfgp]
        lib.octo_fmm_create.argtypes = [cfgp, ctypes.POINTER(vp)]
        lib.octo_fmm_set_moments.argtypes = [vp, vp, vp]
        lib.octo_fmm_interact.argtypes = [vp]
        lib.octo_fmm_get_expansions.argtypes = [vp, vp, vp]
        lib.octo_fmm_destroy.argtypes = [vp]
        lib.octo_fmm_bind_outputs.argtypes = [vp, vp, vp]
        lib.octo_fmm_get_stencil.argtypes = [vp, ctypes.c_int, ip, vp]
        lib.octo_fmm_interact_mixed.argtypes = [vp, vp]
        lib.octo_fmm_mixed_interaction_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_dmma_table.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int, ip, vp, vp]
        lib.octo_fmm_interaction_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_status.argtypes = [vp]
        peerp = ctypes.POINTER(octo_fmm_peer)
        lib.octo_fmm_staged_sources.argtypes = [vp, peerp]
        lib.octo_fmm_set_neighbours.argtypes = [vp, peerp, peerp]
        lib.octo_fmm_ipc_export.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_ipc_import.argtypes = [ctypes.c_char_p, ctypes.c_ulonglong, ctypes.POINTER(vp), ctypes.POINTER(vp)]
        lib.octo_fmm_ipc_close.argtypes = [vp]
        lib.octo_fmm_run_host.argtypes = [vp, vp, vp, vp, vp, vp, ctypes.c_size_t]
        lib.octo_fmm_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
        lib.octo_fmm_launch_info.argtypes = [vp, ip, ip, ip, ip, ip]
        lib.octo_fmm_fp64_peak_probe.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, dp, ip, ip]
        lib.octo_fmm_fp64_issue_probe.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, ctypes.c_int, dp]
        lib.octo_fmm_flops_per_interaction.argtypes = [ctypes.c_int, ctypes.c_int, ip, ip]
        lib.octo_fmm_flops_per_interaction_path.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ip, ip]
        lib.octo_fmm_dipole_terms_used.argtypes = [vp, ip]
        lib.octo_fmm_version.restype = ctypes.c_char_p
        lib.octo_fmm_static_max_cells.argtypes = []
        lib.octo_fmm_interact_static.argtypes = [cfgp, vp, vp, vp, vp]
        lib.octo_fmm_static_status.argtypes = [ctypes.c_int]
        tcfgp = ctypes.POINTER(octo_fmm_tree_config)
        vpp = ctypes.POINTER(ctypes.c_void_p)
        lib.octo_fmm_tree_workspace_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_tree_workspace_bytes.argtypes = [tcfgp, vpp, ip]
        lib.octo_fmm_tree_create.argtypes = [tcfgp, vpp, ip, ctypes.POINTER(vp)]
        lib.octo_fmm_tree_solve.argtypes = [vp, vpp, vpp]
        lib.octo_fmm_tree_solve_rhs2.argtypes = [vp, vpp, vpp]
        lib.octo_fmm_tree_interaction_counts.argtypes = [vp, vpp, vpp, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_tree_host_scratch_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_tree_host_scratch_bytes.argtypes = [vp]
        lib.octo_fmm_tree_solve_host.argtypes = [vp, vpp, vpp, vp, ctypes.c_size_t]
        lib.octo_fmm_tree_status.argtypes = [vp]
        lib.octo_fmm_tree_launches.argtypes = [vp, ip]
        lib.octo_fmm_tree_destroy.argtypes = [vp]
        scfgp = ctypes.POINTER(octo_fmm_solver_config)
        lib.octo_fmm_solver_workspace_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_solver_workspace_bytes.argtypes = [scfgp]
        lib.octo_fmm_solver_create.argtypes = [scfgp, ctypes.POINTER(vp)]
        lib.octo_fmm_solver_solve.argtypes = [vp, vp, vp]
        lib.octo_fmm_solver_solve_rhs2.argtypes = [vp, vp, vp]
        lib.octo_fmm_solver_solve2.argtypes = [vp, vp, vp, vp, vp]
        lib.octo_fmm_solver_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
        lib.octo_fmm_solver_status.argtypes = [vp]
        lib.octo_fmm_solver_host_scratch_bytes.restype = ctypes.c_size_t
        lib.octo_fmm_solver_host_scratch_bytes.argtypes = [scfgp]
        lib.octo_fmm_solver_solve_host.argtypes = [vp, vp, vp, vp, ctypes.c_size_t]
        lib.octo_fmm_solver_destroy.argtypes = [vp]
        lib.octo_fmm_solver_interaction_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_solver_leaf_interaction_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
        lib.octo_fmm_solver_get_leaf_stencil.argtypes = [vp, ctypes.c_int, ip, vp]
        lib.octo_fmm_solver_num_levels.argtypes = [vp, ip, ip]
        self._cdll = lib

    def __getattr__(self, name):
        if self._cdll is None:
            self._load()
        return getattr(self._cdll, name)


_lib = _Library()
_vp = ctypes.c_void_p


def _ptr(t):
    """Device/host address of a torch tensor or numpy array (or None).  The C ABI takes plain pointers to dense
    arrays, so anything that is not contiguous is refused here instead of being read out of bounds there."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        if not t.is_contiguous():
            raise ValueError("octo_fmm: tensors must be contiguous")
        return t.data_ptr()
    if not t.flags["C_CONTIGUOUS"]:
        raise ValueError("octo_fmm: arrays must be C-contiguous")
    return t.ctypes.data


def _check_device_tensor(t, name, dtype, numel, device, stream=None):
    """Argument check of the convenience classes: a CUDA tensor of the handle's device, of the exact dtype and element
    count the C ABI will read or write.  `stream`: the handle's stream; a tensor allocated on another stream is tied to
    it (record_stream) so that the caching allocator does not hand its memory out while the library still uses it."""
    if t is None:
        return
    if not hasattr(t, "is_cuda") or not t.is_cuda:
        raise ValueError("octo_fmm: %s must be a CUDA tensor (there is no CPU path)" % name)
    if t.device != device:
        raise ValueError("octo_fmm: %s is on %s, the handle on %s" % (name, t.device, device))
    if t.dtype != dtype:
        raise ValueError("octo_fmm: %s must be %s, got %s" % (name, dtype, t.dtype))
    if not t.is_contiguous():
        raise ValueError("octo_fmm: %s must be contiguous" % name)
    if t.numel() != numel:
        raise ValueError("octo_fmm: %s has %d elements, expected %d" % (name, t.numel(), numel))
    if stream is not None:
        t.record_stream(stream)


def make_config(n, h, theta, kind=MULTIPOLE, am_correction=True, out_lo=(0, 0, 0), out_hi=(0, 0, 0),
                origin=(0.0, 0.0, 0.0), device=0, stream=0, workspace=0, workspace_bytes=0):
    c = octo_fmm_config()
    for a in range(3):
        c.n[a], c.out_lo[a], c.out_hi[a], c.origin[a] = int(n[a]), int(out_lo[a]), int(out_hi[a]), float(origin[a])
    c.h, c.theta, c.kind, c.am_correction = float(h), float(theta), int(kind), int(bool(am_correction))
    c.device, c.stream, c.workspace, c.workspace_bytes = int(device), stream or None, workspace or None, int(workspace_bytes)
    return c


# ---- the C ABI, same names ----------------------------------------------------------------
def octo_fmm_version():
    return _lib.octo_fmm_version().decode()


def octo_fmm_workspace_bytes(cfg):
    return int(_lib.octo_fmm_workspace_bytes(ctypes.byref(cfg)))


def octo_fmm_host_scratch_bytes(cfg):
    return int(_lib.octo_fmm_host_scratch_bytes(ctypes.byref(cfg)))


def octo_fmm_create(cfg):
    h = _vp()
    rc = _lib.octo_fmm_create(ctypes.byref(cfg), ctypes.byref(h))
    if rc != OK:
        raise OctoFmmError("octo_fmm_create", rc)
    return h


def octo_fmm_set_moments(h, moments, com_off=None):
    rc = _lib.octo_fmm_set_moments(h, _ptr(moments), _ptr(com_off))
    if rc != OK:
        raise OctoFmmError("octo_fmm_set_moments", rc)


def octo_fmm_interact(h):
    rc = _lib.octo_fmm_interact(h)
    if rc != OK:
        raise OctoFmmError("octo_fmm_interact", rc)


def octo_fmm_get_expansions(h, L, Lcorr=None):
    rc = _lib.octo_fmm_get_expansions(h, _ptr(L), _ptr(Lcorr))
    if rc != OK:
        raise OctoFmmError("octo_fmm_get_expansions", rc)


def octo_fmm_bind_outputs(h, L, Lcorr=None):
    rc = _lib.octo_fmm_bind_outputs(h, _ptr(L), _ptr(Lcorr))
    if rc != OK:
        raise OctoFmmError("octo_fmm_bind_outputs", rc)


def octo_fmm_destroy(h):
    rc = _lib.octo_fmm_destroy(h)
    if rc != OK:
        raise OctoFmmError("octo_fmm_destroy", rc)


def octo_fmm_status(h):
    return int(_lib.octo_fmm_status(h))


def octo_fmm_get_stencil(h, parity):
    import numpy as np
    cnt = ctypes.c_int(0)
    rc = _lib.octo_fmm_get_stencil(h, int(parity), ctypes.byref(cnt), None)
    if rc != OK:
        raise OctoFmmError("octo_fmm_get_stencil", rc)
    out = np.zeros((cnt.value, 3), dtype=np.int8)
    rc = _lib.octo_fmm_get_stencil(h, int(parity), ctypes.byref(cnt), out.ctypes.data)
    if rc != OK:
        raise OctoFmmError("octo_fmm_get_stencil", rc)
    return out


def octo_fmm_interact_mixed(h, leaf):
    rc = _lib.octo_fmm_interact_mixed(h, _ptr(leaf))
    if rc != OK:
        raise OctoFmmError("octo_fmm_interact_mixed", rc)


def octo_fmm_mixed_interaction_count(h):
    n = ctypes.c_ulonglong(0)
    rc = _lib.octo_fmm_mixed_interaction_count(h, ctypes.byref(n))
    if rc != OK:
        raise OctoFmmError("octo_fmm_mixed_interaction_count", rc)
    return int(n.value)


def octo_fmm_dmma_table(theta, h, leaf, which):
    """Host-only: (a[nchunk][8][4], off[nchunk][8][4]) of the operand table of the tensor-core monopole kernels."""
    import numpy as np
    n = ctypes.c_int(0)
    rc = _lib.octo_fmm_dmma_table(float(theta), float(h), int(leaf), int(which), 0, ctypes.byref(n), None, None)
    if rc != OK:
        raise OctoFmmError("octo_fmm_dmma_table", rc)
    a = np.zeros((n.value, 8, 4))
    off = np.zeros((n.value, 8, 4), dtype=np.int32)
    rc = _lib.octo_fmm_dmma_table(float(theta), float(h), int(leaf), int(which), n.value, ctypes.byref(n), a.ctypes.data,
                                  off.ctypes.data)
    if rc != OK:
        raise OctoFmmError("octo_fmm_dmma_table", rc)
    return a, off


def octo_fmm_interaction_count(h):
    n = ctypes.c_ulonglong(0)
    rc = _lib.octo_fmm_interaction_count(h, ctypes.byref(n))
    if rc != OK:
        raise OctoFmmError("octo_fmm_interaction_count", rc)
    return int(n.value)


def octo_fmm_staged_sources(h):
    """(sources pointer, flags pointer, nz) of the handle's staged array: what a z-neighbour needs."""
    me = octo_fmm_peer()
    rc = _lib.octo_fmm_staged_sources(h, ctypes.byref(me))
    if rc != OK:
        raise OctoFmmError("octo_fmm_staged_sources", rc)
    return int(me.sources), int(me.flags), int(me.nz)


def _peer(p):
    if p is None:
        return None
    return ctypes.byref(octo_fmm_peer(int(p[0]), int(p[1]), int(p[2])))


def octo_fmm_set_neighbours(h, below, above):
    """below / above: None (domain boundary) or (sources pointer, flags pointer, nz) valid in this process."""
    rc = _lib.octo_fmm_set_neighbours(h, _peer(below), _peer(above))
    if rc != OK:
        raise OctoFmmError("octo_fmm_set_neighbours", rc)


def octo_fmm_ipc_export(dev_ptr):
    """(64-byte handle of the allocation holding dev_ptr, offset of dev_ptr in it)."""
    buf = ctypes.create_string_buffer(64)
    off = ctypes.c_ulonglong(0)
    rc = _lib.octo_fmm_ipc_export(ctypes.c_void_p(int(dev_ptr)), buf, ctypes.byref(off))
    if rc != OK:
        raise OctoFmmError("octo_fmm_ipc_export", rc)
    return buf.raw, int(off.value)


def octo_fmm_ipc_import(handle, offset):
    """(base of the mapped allocation, pointer at the offset); close the base with octo_fmm_ipc_close."""
    if len(handle) != 64:
        raise ValueError("a CUDA IPC handle has 64 bytes")
    base, ptr = ctypes.c_void_p(0), ctypes.c_void_p(0)
    rc = _lib.octo_fmm_ipc_import(bytes(handle), int(offset), ctypes.byref(base), ctypes.byref(ptr))
    if rc != OK:
        raise OctoFmmError("octo_fmm_ipc_import", rc)
    return int(base.value), int(ptr.value)


def octo_fmm_ipc_close(base):
    rc = _lib.octo_fmm_ipc_close(ctypes.c_void_p(int(base)))
    if rc != OK:
        raise OctoFmmError("octo_fmm_ipc_close", rc)


def octo_fmm_static_max_cells():
    return int(_lib.octo_fmm_static_max_cells())


def octo_fmm_interact_static(cfg, moments, com_off, L, Lcorr=None):
    """The step without any allocation: scratch in the library's static device array (octo_fmm.h)."""
    rc = _lib.octo_fmm_interact_static(ctypes.byref(cfg), _ptr(moments), _ptr(com_off), _ptr(L), _ptr(Lcorr))
    if rc != OK:
        raise OctoFmmError("octo_fmm_interact_static", rc)


def octo_fmm_static_status(device=0):
    return int(_lib.octo_fmm_static_status(int(device)))


def octo_fmm_run_host(h, moments_host, com_off_host, L_host, Lcorr_host, scratch, scratch_bytes):
    rc = _lib.octo_fmm_run_host(h, _ptr(moments_host), _ptr(com_off_host), _ptr(L_host), _ptr(Lcorr_host),
                                _ptr(scratch), int(scratch_bytes))
    if rc != OK:
        raise OctoFmmError("octo_fmm_run_host", rc)


def octo_fmm_set_option(h, key, value):
    rc = _lib.octo_fmm_set_option(h, key.encode(), int(value))
    if rc != OK:
        raise OctoFmmError("octo_fmm_set_option", rc)


def octo_fmm_launch_info(h):
    v = [ctypes.c_int(0) for _ in range(5)]
    rc = _lib.octo_fmm_launch_info(h, *[ctypes.byref(x) for x in v])
    if rc != OK:
        raise OctoFmmError("octo_fmm_launch_info", rc)
    return dict(zip(("grid", "block", "smem_bytes", "regs", "launches_per_interact"), [x.value for x in v]))


def octo_fmm_fp64_peak_probe(device, stream, scratch, iters=20000):
    f, sm, clk = ctypes.c_double(0), ctypes.c_int(0), ctypes.c_int(0)
    rc = _lib.octo_fmm_fp64_peak_probe(int(device), stream or None, _ptr(scratch), int(iters), ctypes.byref(f),
                                       ctypes.byref(sm), ctypes.byref(clk))
    if rc != OK:
        raise OctoFmmError("octo_fmm_fp64_peak_probe", rc)
    return {"flops_per_s": f.value, "sm_count": sm.value, "clock_khz": clk.value}


def octo_fmm_fp64_issue_probe(device, stream, scratch, mode, iters=2000):
    r = ctypes.c_double(0)
    rc = _lib.octo_fmm_fp64_issue_probe(int(device), stream or None, _ptr(scratch), int(mode), int(iters), ctypes.byref(r))
    if rc != OK:
        raise OctoFmmError("octo_fmm_fp64_issue_probe", rc)
    return r.value


def octo_fmm_flops_per_interaction(kind, am_correction):
    f, i = ctypes.c_int(0), ctypes.c_int(0)
    rc = _lib.octo_fmm_flops_per_interaction(int(kind), int(bool(am_correction)), ctypes.byref(f), ctypes.byref(i))
    if rc != OK:
        raise OctoFmmError("octo_fmm_flops_per_interaction", rc)
    return f.value, i.value


def octo_fmm_flops_per_interaction_path(kind, am_correction, dipole_terms):
    f, i = ctypes.c_int(0), ctypes.c_int(0)
    rc = _lib.octo_fmm_flops_per_interaction_path(int(kind), int(bool(am_correction)), int(bool(dipole_terms)),
                                                  ctypes.byref(f), ctypes.byref(i))
    if rc != OK:
        raise OctoFmmError("octo_fmm_flops_per_interaction_path", rc)
    return f.value, i.value


def octo_fmm_dipole_terms_used(h):
    u = ctypes.c_int(0)
    rc = _lib.octo_fmm_dipole_terms_used(h, ctypes.byref(u))
    if rc != OK:
        raise OctoFmmError("octo_fmm_dipole_terms_used", rc)
    return bool(u.value)


# ---- complete uniform-grid solve (octo_fmm_solver_*) ------------------------------------------
def make_solver_config(n, h, theta, am_correction=True, device=0, stream=0, workspace=0, workspace_bytes=0, two_rhs=False):
    c = octo_fmm_solver_config()
    c.n, c.h, c.theta, c.am_correction = int(n), float(h), float(theta), int(bool(am_correction))
    c.device, c.stream, c.workspace, c.workspace_bytes = int(device), stream or None, workspace or None, int(workspace_bytes)
    c.two_rhs = int(bool(two_rhs))
    return c


def octo_fmm_solver_workspace_bytes(cfg):
    return int(_lib.octo_fmm_solver_workspace_bytes(ctypes.byref(cfg)))


def octo_fmm_solver_create(cfg):
    h = _vp()
    rc = _lib.octo_fmm_solver_create(ctypes.byref(cfg), ctypes.byref(h))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_create", rc)
    return h


def octo_fmm_solver_solve(s, mass, out):
    rc = _lib.octo_fmm_solver_solve(s, _ptr(mass), _ptr(out))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_solve", rc)


def octo_fmm_solver_solve_rhs2(s, dmass, out):
    rc = _lib.octo_fmm_solver_solve_rhs2(s, _ptr(dmass), _ptr(out))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_solve_rhs2", rc)


def octo_fmm_solver_solve2(s, mass, dmass, out, dphi_dt):
    rc = _lib.octo_fmm_solver_solve2(s, _ptr(mass), _ptr(dmass), _ptr(out), _ptr(dphi_dt))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_solve2", rc)


def octo_fmm_solver_set_option(s, key, value):
    rc = _lib.octo_fmm_solver_set_option(s, key.encode(), int(value))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_set_option", rc)


def octo_fmm_solver_host_scratch_bytes(cfg):
    return int(_lib.octo_fmm_solver_host_scratch_bytes(ctypes.byref(cfg)))


def octo_fmm_solver_solve_host(s, mass_host, out_host, scratch, scratch_bytes):
    rc = _lib.octo_fmm_solver_solve_host(s, _ptr(mass_host), _ptr(out_host), _ptr(scratch), int(scratch_bytes))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_solve_host", rc)


def octo_fmm_solver_status(s):
    return int(_lib.octo_fmm_solver_status(s))


def octo_fmm_solver_destroy(s):
    rc = _lib.octo_fmm_solver_destroy(s)
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_destroy", rc)


def octo_fmm_solver_interaction_count(s):
    n = ctypes.c_ulonglong(0)
    rc = _lib.octo_fmm_solver_interaction_count(s, ctypes.byref(n))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_interaction_count", rc)
    return int(n.value)


def octo_fmm_solver_leaf_interaction_count(s):
    n = ctypes.c_ulonglong(0)
    rc = _lib.octo_fmm_solver_leaf_interaction_count(s, ctypes.byref(n))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_leaf_interaction_count", rc)
    return int(n.value)


def octo_fmm_solver_get_leaf_stencil(s, parity):
    import numpy as np
    cnt = ctypes.c_int(0)
    rc = _lib.octo_fmm_solver_get_leaf_stencil(s, int(parity), ctypes.byref(cnt), None)
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_get_leaf_stencil", rc)
    out = np.zeros((cnt.value, 3), dtype=np.int8)
    rc = _lib.octo_fmm_solver_get_leaf_stencil(s, int(parity), ctypes.byref(cnt), out.ctypes.data)
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_get_leaf_stencil", rc)
    return out


def octo_fmm_solver_num_levels(s):
    a, b = ctypes.c_int(0), ctypes.c_int(0)
    rc = _lib.octo_fmm_solver_num_levels(s, ctypes.byref(a), ctypes.byref(b))
    if rc != OK:
        raise OctoFmmError("octo_fmm_solver_num_levels", rc)
    return a.value, b.value


class OctoFMMSolver:
    """Owns the workspace tensor and the handle of a complete uniform-grid solve."""

    def __init__(self, n, h, theta, am_correction=True, device=0, stream=None, two_rhs=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("octo_fmm needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.n = int(n)
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        cfg = make_solver_config(n, h, theta, am_correction, device=device, stream=self.stream.cuda_stream, two_rhs=two_rhs)
        nbytes = octo_fmm_solver_workspace_bytes(cfg)
        if nbytes == 0:
            raise OctoFmmError("octo_fmm_solver_workspace_bytes", EINVAL)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        cfg.workspace, cfg.workspace_bytes = self.workspace.data_ptr(), nbytes
        self.cfg = cfg
        self.handle = octo_fmm_solver_create(cfg)

    def _check(self, t, name, numel):
        _check_device_tensor(t, name, self.torch.float64, numel, self.device, self.stream)

    def solve(self, mass, out=None):
        if out is None:
            out = self.torch.empty((4, self.n, self.n, self.n), dtype=self.torch.float64, device=self.device)
        self._check(mass, "mass", self.n ** 3)
        self._check(out, "out", 4 * self.n ** 3)
        octo_fmm_solver_solve(self.handle, mass, out)
        return out

    def solve_rhs2(self, dmass, out=None):
        """d(phi)/dt [n][n][n] of the sources dmass on the tree and centres of the last solve()."""
        if out is None:
            out = self.torch.empty((self.n, self.n, self.n), dtype=self.torch.float64, device=self.device)
        self._check(dmass, "dmass", self.n ** 3)
        self._check(out, "out", self.n ** 3)
        octo_fmm_solver_solve_rhs2(self.handle, dmass, out)
        return out

    def solve2(self, mass, dmass, out=None, dphi_dt=None):
        """Both right-hand sides in one call (needs two_rhs=True): returns (out [4][n][n][n], dphi_dt [n][n][n])."""
        if out is None:
            out = self.torch.empty((4, self.n, self.n, self.n), dtype=self.torch.float64, device=self.device)
        if dphi_dt is None:
            dphi_dt = self.torch.empty((self.n, self.n, self.n), dtype=self.torch.float64, device=self.device)
        self._check(mass, "mass", self.n ** 3)
        self._check(dmass, "dmass", self.n ** 3)
        self._check(out, "out", 4 * self.n ** 3)
        self._check(dphi_dt, "dphi_dt", self.n ** 3)
        octo_fmm_solver_solve2(self.handle, mass, dmass, out, dphi_dt)
        return out, dphi_dt

    def set_option(self, key, value):
        octo_fmm_solver_set_option(self.handle, key, value)

    def status(self):
        return octo_fmm_solver_status(self.handle)

    def interaction_count(self):
        return octo_fmm_solver_interaction_count(self.handle)

    def leaf_interaction_count(self):
        return octo_fmm_solver_leaf_interaction_count(self.handle)

    def leaf_stencil(self, parity):
        return octo_fmm_solver_get_leaf_stencil(self.handle, parity)

    def num_levels(self):
        return octo_fmm_solver_num_levels(self.handle)

    def close(self):
        if getattr(self, "handle", None) is not None:
            octo_fmm_solver_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- the solve on an adaptive oct-tree of 8^3 sub-grids (octo_fmm_tree_*) ----------------------
def make_tree_config(n0, depth, h0, theta, am_correction=True, device=0, stream=0, workspace=0, workspace_bytes=0):
    c = octo_fmm_tree_config()
    c.n0, c.depth, c.h0, c.theta, c.am_correction = int(n0), int(depth), float(h0), float(theta), int(bool(am_correction))
    c.device, c.stream, c.workspace, c.workspace_bytes = int(device), stream or None, workspace or None, int(workspace_bytes)
    return c


def _ptr_array(items):
    """A C array of void* from tensors / arrays / raw addresses (the per-level pointer tables of the tree calls)."""
    arr = (ctypes.c_void_p * len(items))()
    for i, t in enumerate(items):
        arr[i] = t if isinstance(t, int) else _ptr(t)
    return arr


def _box_array(box, depth):
    """depth x 6 C ints (lo_x, lo_y, lo_z, n_x, n_y, n_z) or None (every level is its whole lattice)."""
    if box is None:
        return None
    flat = [int(v) for b in box for v in b]
    if len(flat) != 6 * depth:
        raise ValueError("octo_fmm: box needs 6 integers per level")
    return (ctypes.c_int * len(flat))(*flat)


def octo_fmm_tree_workspace_bytes(cfg, kind_host, box=None):
    return int(_lib.octo_fmm_tree_workspace_bytes(ctypes.byref(cfg), _ptr_array(kind_host), _box_array(box, cfg.depth)))


def octo_fmm_tree_create(cfg, kind_host, box=None):
    h = _vp()
    rc = _lib.octo_fmm_tree_create(ctypes.byref(cfg), _ptr_array(kind_host), _box_array(box, cfg.depth), ctypes.byref(h))
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_create", rc)
    return h


def octo_fmm_tree_solve(t, mass, out):
    rc = _lib.octo_fmm_tree_solve(t, _ptr_array(mass), _ptr_array(out))
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_solve", rc)


def octo_fmm_tree_solve_rhs2(t, dmass, dphi_dt):
    rc = _lib.octo_fmm_tree_solve_rhs2(t, _ptr_array(dmass), _ptr_array(dphi_dt))
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_solve_rhs2", rc)


def octo_fmm_tree_interaction_counts(t, mass, out):
    c = (ctypes.c_ulonglong * 3)()
    rc = _lib.octo_fmm_tree_interaction_counts(t, _ptr_array(mass), _ptr_array(out), c)
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_interaction_counts", rc)
    return {"m2l": int(c[0]), "p2p": int(c[1]), "cross": int(c[2])}


def octo_fmm_tree_host_scratch_bytes(t):
    return int(_lib.octo_fmm_tree_host_scratch_bytes(t))


def octo_fmm_tree_solve_host(t, mass_host, out_host, scratch, scratch_bytes):
    rc = _lib.octo_fmm_tree_solve_host(t, _ptr_array(mass_host), _ptr_array(out_host), _ptr(scratch), int(scratch_bytes))
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_solve_host", rc)


def octo_fmm_tree_status(t):
    return int(_lib.octo_fmm_tree_status(t))


def octo_fmm_tree_launches(t):
    n = ctypes.c_int(0)
    rc = _lib.octo_fmm_tree_launches(t, ctypes.byref(n))
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_launches", rc)
    return n.value


def octo_fmm_tree_destroy(t):
    rc = _lib.octo_fmm_tree_destroy(t)
    if rc != OK:
        raise OctoFmmError("octo_fmm_tree_destroy", rc)


class OctoFMMTree:
    """Owns the workspace tensor and the handle of a solve on an adaptive tree.  kind: list of numpy uint8 arrays
    (host; 0 absent, 1 leaf, 2 refined), one per level; box: None (kind[l] is the whole lattice [n_l]^3) or per level
    (lo_x, lo_y, lo_z, n_x, n_y, n_z) in cells, kind[l] then has shape [n_z][n_y][n_x]."""

    def __init__(self, n0, h0, theta, kind, am_correction=True, device=0, stream=None, box=None):
        import numpy as np
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("octo_fmm needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.n0, self.depth = int(n0), len(kind)
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.kind = [np.ascontiguousarray(k, dtype=np.uint8) for k in kind]
        self.box = None if box is None else [tuple(int(v) for v in b) for b in box]
        self.shape = [(self.n0 << l,) * 3 if self.box is None else (self.box[l][5], self.box[l][4], self.box[l][3])
                      for l in range(self.depth)]
        for l, k in enumerate(self.kind):
            if k.shape != self.shape[l]:
                raise ValueError("octo_fmm: kind[%d] must have shape %s" % (l, (self.shape[l],)))
        cfg = make_tree_config(n0, self.depth, h0, theta, am_correction, device=device, stream=self.stream.cuda_stream)
        nbytes = octo_fmm_tree_workspace_bytes(cfg, self.kind, self.box)
        if nbytes == 0:
            raise OctoFmmError("octo_fmm_tree_workspace_bytes", EINVAL)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        cfg.workspace, cfg.workspace_bytes = self.workspace.data_ptr(), nbytes
        self.cfg = cfg
        self.handle = octo_fmm_tree_create(cfg, self.kind, self.box)

    def cells(self, l):
        s = self.shape[l]
        return s[0] * s[1] * s[2]

    def _check(self, mass, out):
        if len(mass) != self.depth or len(out) != self.depth:
            raise ValueError("octo_fmm: one mass and one out tensor per level")
        for l in range(self.depth):
            _check_device_tensor(mass[l], "mass[%d]" % l, self.torch.float64, self.cells(l), self.device, self.stream)
            _check_device_tensor(out[l], "out[%d]" % l, self.torch.float64, 4 * self.cells(l), self.device, self.stream)

    def empty_out(self):
        return [self.torch.empty((4,) + self.shape[l], dtype=self.torch.float64, device=self.device) for l in range(self.depth)]

    def solve(self, mass, out=None):
        out = self.empty_out() if out is None else out
        self._check(mass, out)
        octo_fmm_tree_solve(self.handle, mass, out)
        return out

    def solve_rhs2(self, dmass, dphi_dt=None):
        """d(phi)/dt per level ([box shape]) of the sources dmass on the tree and centres of the last solve()."""
        if dphi_dt is None:
            dphi_dt = [self.torch.empty(self.shape[l], dtype=self.torch.float64, device=self.device) for l in range(self.depth)]
        if len(dmass) != self.depth or len(dphi_dt) != self.depth:
            raise ValueError("octo_fmm: one dmass and one dphi_dt tensor per level")
        for l in range(self.depth):
            _check_device_tensor(dmass[l], "dmass[%d]" % l, self.torch.float64, self.cells(l), self.device, self.stream)
            _check_device_tensor(dphi_dt[l], "dphi_dt[%d]" % l, self.torch.float64, self.cells(l), self.device, self.stream)
        octo_fmm_tree_solve_rhs2(self.handle, dmass, dphi_dt)
        return dphi_dt

    def interaction_counts(self, mass, out=None):
        out = self.empty_out() if out is None else out
        self._check(mass, out)
        return octo_fmm_tree_interaction_counts(self.handle, mass, out), out

    def status(self):
        return octo_fmm_tree_status(self.handle)

    def launches(self):
        return octo_fmm_tree_launches(self.handle)

    def close(self):
        if getattr(self, "handle", None) is not None:
            octo_fmm_tree_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- convenience wrapper ---------------------------------------------------------------------
class OctoFMM:
    """Owns a workspace tensor and a handle.  Tensors are torch CUDA float64, SoA as in octo_fmm.h."""

    def __init__(self, n, h, theta, kind=MULTIPOLE, am_correction=True, out_lo=(0, 0, 0), out_hi=(0, 0, 0),
                 device=0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("octo_fmm needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.kind = kind
        self.n = tuple(int(v) for v in n)
        whole = all(v == 0 for v in tuple(out_lo) + tuple(out_hi))
        self.out_lo = (0, 0, 0) if whole else tuple(out_lo)
        self.out_hi = self.n if whole else tuple(out_hi)
        cfg = make_config(n, h, theta, kind, am_correction, out_lo, out_hi, device=device,
                          stream=self.stream.cuda_stream)
        nbytes = octo_fmm_workspace_bytes(cfg)
        if nbytes == 0:
            raise OctoFmmError("octo_fmm_workspace_bytes", EINVAL)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        cfg.workspace, cfg.workspace_bytes = self.workspace.data_ptr(), nbytes
        self.cfg = cfg
        self.handle = octo_fmm_create(cfg)

    @property
    def out_shape(self):
        o = [self.out_hi[a] - self.out_lo[a] for a in range(3)]
        return (o[2], o[1], o[0])

    def _ncell(self):
        return self.n[0] * self.n[1] * self.n[2]

    def _ocell(self):
        o = self.out_shape
        return o[0] * o[1] * o[2]

    def _check(self, t, name, numel, dtype=None):
        _check_device_tensor(t, name, dtype or self.torch.float64, numel, self.device, self.stream)

    def set_moments(self, moments, com_off=None):
        self._check(moments, "moments", (20 if self.kind == MULTIPOLE else 1) * self._ncell())
        if self.kind == MULTIPOLE:
            self._check(com_off, "com_off", 3 * self._ncell())
        octo_fmm_set_moments(self.handle, moments, com_off)

    def interact(self):
        octo_fmm_interact(self.handle)

    def interact_mixed(self, leaf):
        """One level of an adaptive mesh: leaf = uint8 [nz][ny][nx] on the device, 1 where the cell is a leaf."""
        self._check(leaf, "leaf", self._ncell(), self.torch.uint8)
        octo_fmm_interact_mixed(self.handle, leaf)

    def mixed_interaction_count(self):
        return octo_fmm_mixed_interaction_count(self.handle)

    def get_expansions(self, L=None, Lcorr=None, want_corr=True):
        torch = self.torch
        ncoef = 20 if self.kind == MULTIPOLE else 4
        if L is None:
            L = torch.empty((ncoef,) + self.out_shape, dtype=torch.float64, device=self.device)
        if Lcorr is None and want_corr and self.kind == MULTIPOLE:
            Lcorr = torch.empty((3,) + self.out_shape, dtype=torch.float64, device=self.device)
        self._check(L, "L", ncoef * self._ocell())
        self._check(Lcorr, "Lcorr", 3 * self._ocell())
        octo_fmm_get_expansions(self.handle, L, Lcorr)
        return L, Lcorr

    def bind_outputs(self, L, Lcorr=None):
        """interact() then writes straight into L / Lcorr (kept alive here); None unbinds."""
        self._check(L, "L", (20 if self.kind == MULTIPOLE else 4) * self._ocell())
        self._check(Lcorr, "Lcorr", 3 * self._ocell())
        self._bound = (L, Lcorr)
        octo_fmm_bind_outputs(self.handle, L, Lcorr)

    def solve(self, moments, com_off=None):
        self.set_moments(moments, com_off)
        self.interact()
        return self.get_expansions()

    def status(self):
        return octo_fmm_status(self.handle)

    def stencil(self, parity):
        return octo_fmm_get_stencil(self.handle, parity)

    def interaction_count(self):
        return octo_fmm_interaction_count(self.handle)

    def staged_sources(self):
        return octo_fmm_staged_sources(self.handle)

    def set_neighbours(self, below=None, above=None):
        """z-neighbours whose staged layers interact() reads in place of a halo: None, another OctoFMM of this process
        (kept alive here), or (sources pointer, flags pointer, nz) as octo_fmm_ipc_import returned them."""
        self._neighbours = (below, above)
        as_peer = lambda p: p.staged_sources() if isinstance(p, OctoFMM) else p
        octo_fmm_set_neighbours(self.handle, as_peer(below), as_peer(above))

    def launch_info(self):
        return octo_fmm_launch_info(self.handle)

    def dipole_terms_used(self):
        return octo_fmm_dipole_terms_used(self.handle)

    def set_option(self, key, value):
        octo_fmm_set_option(self.handle, key, value)

    def close(self):
        if getattr(self, "handle", None) is not None:
            octo_fmm_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
