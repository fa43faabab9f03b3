"""octo_fmm_interact_static: the step with its scratch in the library's static device array (no allocation at all).

Collected LAST on purpose (the suite runs with pytest -x).  Compared with the existing path -- a handle over a
caller-lent workspace, set_moments + interact + get_expansions -- on two calls in a row that differ in size, inputs and
opening angle, so that the second call meets the first call's left-overs in the shared array."""
import numpy as np
import pytest

import fmm_inputs as fi
from helpers import parity_error

pytestmark = pytest.mark.gpu

TOL = 1e-12          # the bar of the parity tests


def _existing_path(p, torch, n, h, theta, mom, com):
    f = p.OctoFMM(n, h, theta, p.MULTIPOLE, True)
    L, C = f.solve(mom, com)
    torch.cuda.synchronize()
    assert f.status() == p.OK
    f.close()
    return L, C


def test_static_scratch_entry_point_matches_the_workspace_path_twice():
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    assert p.octo_fmm_static_max_cells() == 32768
    w = fi.config2(ncell=64)
    stream = torch.cuda.current_stream().cuda_stream
    # call 1: the maximum size, 32^3 cells (the slab-fed kernel); call 2: a smaller, non-cubic grid with other inputs
    # and another opening angle -- other lists, another layout of the same bytes; call 3: call 2's configuration again
    # with other values (the cached configuration: nothing is rebuilt)
    cases = [((32, 32, 32), 0.5, 1.0, (0, 0, 0)), ((16, 24, 32), 0.35, 2.5, (8, 16, 24)), ((16, 24, 32), 0.35, 0.75, (32, 8, 0))]
    free_before = None
    for it, (n, theta, scale, o) in enumerate(cases):
        sl = (slice(None), slice(o[2], o[2] + n[2]), slice(o[1], o[1] + n[1]), slice(o[0], o[0] + n[0]))
        hm = np.ascontiguousarray(w.moments[sl]) * scale
        hc = np.ascontiguousarray(w.com_off[sl])
        if it == 1:                                        # this call's sources carry dipoles, the one before had none
            hm[1:4] = 0.03 * w.h * hm[0] * np.random.default_rng(11).uniform(-1, 1, hm[1:4].shape)
        mom, com = torch.from_numpy(hm).cuda(), torch.from_numpy(hc).cuda()
        Lr, Cr = _existing_path(p, torch, n, w.h, theta, mom, com)
        L = torch.full((20, n[2], n[1], n[0]), float("nan"), dtype=torch.float64, device="cuda")
        C = torch.full((3, n[2], n[1], n[0]), float("nan"), dtype=torch.float64, device="cuda")
        cfg = p.make_config(n, w.h, theta, p.MULTIPOLE, True, device=0, stream=stream)
        torch.cuda.synchronize()
        if it == 2:
            free_before = torch.cuda.mem_get_info()[0]
        p.octo_fmm_interact_static(cfg, mom, com, L, C)
        torch.cuda.synchronize()
        if it == 2:                                        # nothing was allocated on the device by the call
            assert free_before - torch.cuda.mem_get_info()[0] < (1 << 20)
        assert p.octo_fmm_static_status(0) == p.OK
        Lh, Ch, Lrh, Crh = L.cpu().numpy(), C.cpu().numpy(), Lr.cpu().numpy(), Cr.cpu().numpy()
        assert np.isfinite(Lh).all() and np.isfinite(Ch).all()
        assert parity_error(Lh, Lrh) <= TOL, (it, parity_error(Lh, Lrh))
        assert np.abs(Ch - Crh).max() <= TOL * np.abs(Lrh[1:4]).max()
        assert torch.equal(L, Lr) and torch.equal(C, Cr)   # the same kernels on the same staged bytes
    # Lcorr is optional
    L2 = torch.empty_like(L)
    p.octo_fmm_interact_static(cfg, mom, com, L2, None)
    torch.cuda.synchronize()
    assert torch.equal(L2, L)


def test_static_scratch_entry_point_rejects_what_does_not_fit():
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    n = (40, 32, 32)                                       # 40 960 cells > 32 768
    mom = torch.zeros((20, n[2], n[1], n[0]), dtype=torch.float64, device="cuda")
    com = torch.zeros((3, n[2], n[1], n[0]), dtype=torch.float64, device="cuda")
    L = torch.full((20, n[2], n[1], n[0]), 7.0, dtype=torch.float64, device="cuda")
    cfg = p.make_config(n, 1.0, 0.5, p.MULTIPOLE, True, device=0, stream=torch.cuda.current_stream().cuda_stream)
    with pytest.raises(p.OctoFmmError) as e:
        p.octo_fmm_interact_static(cfg, mom, com, L, None)
    assert e.value.status == p.ESIZE and "ESIZE" in str(e.value)
    torch.cuda.synchronize()
    assert bool((L == 7.0).all())                          # nothing was launched
    mono = p.make_config((16, 16, 16), 1.0, 0.5, p.MONOPOLE, True, device=0)
    with pytest.raises(p.OctoFmmError) as e:
        p.octo_fmm_interact_static(mono, mom, None, L, None)
    assert e.value.status == p.EINVAL
