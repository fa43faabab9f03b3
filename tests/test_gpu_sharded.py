"""The sharded level on ONE GPU: the slabs of 2 and of 4 "ranks" are computed one after the other from the halos the
exchange would deliver (the exchange itself is covered by the gloo tests) and must (i) match the ORACLE on sampled regions
of every slab, (ii) reproduce the whole-grid GPU result bit for bit; the per-slab interaction counts add up to the whole
grid's."""
import numpy as np
import pytest

import fmm_inputs as fi
import oracle
from helpers import parity_error

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [1, 2, 4])
def test_slabs_match_the_oracle_and_the_whole_grid(world):
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200.sharded import HALO, ShardedLevel, slab_layout
    w = fi.config2(ncell=64)
    hm = np.ascontiguousarray(w.moments[:, :, :32, :32])                                  # 32 x 32 x 64 grid
    hc = np.ascontiguousarray(w.com_off[:, :, :32, :32])
    mom, com = torch.from_numpy(hm).cuda(), torch.from_numpy(hc).cuda()
    n = (32, 32, 64)
    whole = p.OctoFMM(n, w.h, 0.5, p.MULTIPOLE, True)
    whole.set_option("kernel", 0)
    Lw, Cw = whole.solve(mom, com)
    nzl = 64 // world
    total = 0
    for rank in range(world):
        lvl = ShardedLevel((32, 32, nzl), w.h, 0.5, True, rank=rank, world=world)
        lvl.fmm.set_option("kernel", 0)
        lo, hi, nz_ext = slab_layout(rank, world, nzl)
        assert lvl.moments_ext.shape[1] == nz_ext and lvl.moments.shape[1] == nzl
        # the owned layers go into the views, the neighbours' layers where the exchange would put them
        lvl.moments.copy_(mom[:, rank * nzl:(rank + 1) * nzl])
        lvl.com_off.copy_(com[:, rank * nzl:(rank + 1) * nzl])
        ext = slice(rank * nzl - lo, (rank + 1) * nzl + hi)
        lvl.moments_ext[:, :lo].copy_(mom[:, ext][:, :lo])
        lvl.com_ext[:, :lo].copy_(com[:, ext][:, :lo])
        if hi:
            lvl.moments_ext[:, -hi:].copy_(mom[:, ext][:, -hi:])
            lvl.com_ext[:, -hi:].copy_(com[:, ext][:, -hi:])
        L, C = lvl.step_extended(lvl.moments_ext, lvl.com_ext)
        torch.cuda.synchronize()
        own = slice(rank * nzl, (rank + 1) * nzl)
        assert torch.equal(L, Lw[:, own]) and torch.equal(C, Cw[:, own])
        # against the oracle: the slab's first and last 8 layers (the ones that depend on the halos) and a middle block
        Lh, Ch = L.cpu().numpy(), C.cpu().numpy()
        for z0 in sorted({0, nzl - 8, (nzl // 16) * 8}):
            glo, ghi = (8, 0, rank * nzl + z0), (24, 32, rank * nzl + z0 + 8)
            Lr, Lcr, _ = oracle.interact_multipole(n, w.h, 0.5, hm, hc, glo, ghi, True)
            sl = (slice(None), slice(z0, z0 + 8), slice(0, 32), slice(8, 24))
            assert parity_error(Lh[sl], Lr) < 1e-12 and np.abs(Ch[sl] - Lcr).max() <= 1e-12 * np.abs(Lr[1:4]).max()
        total += lvl.interaction_count()
        lvl.close()
    assert total == whole.interaction_count()
    whole.close()
    assert HALO == 8
