"""The sharded level on ONE GPU: the slabs of 2 and of 4 "ranks" are computed one after the other from the halos the
exchange would deliver (the exchange itself is covered by the gloo tests) and must reproduce the whole-grid result bit
for bit; the per-slab interaction counts add up to the whole grid's."""
import numpy as np
import pytest

import fmm_inputs as fi

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [1, 2, 4])
def test_slabs_reproduce_the_whole_grid(world):
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200.sharded import HALO, ShardedLevel, assemble, pack_boundary, slab_layout
    w = fi.config2(ncell=64)
    mom = torch.from_numpy(np.ascontiguousarray(w.moments[:, :, :32, :32])).cuda()       # 32 x 32 x 64 grid
    com = torch.from_numpy(np.ascontiguousarray(w.com_off[:, :, :32, :32])).cuda()
    whole = p.OctoFMM((32, 32, 64), w.h, 0.5, p.MULTIPOLE, True)
    whole.set_option("kernel", 0)
    Lw, Cw = whole.solve(mom, com)
    nzl = 64 // world
    total = 0
    for rank in range(world):
        own = slice(rank * nzl, (rank + 1) * nzl)
        m, c = mom[:, own].contiguous(), com[:, own].contiguous()
        below = pack_boundary(mom[:, (rank - 1) * nzl:rank * nzl], com[:, (rank - 1) * nzl:rank * nzl], top=True) if rank > 0 else None
        above = pack_boundary(mom[:, (rank + 1) * nzl:(rank + 2) * nzl], com[:, (rank + 1) * nzl:(rank + 2) * nzl], top=False) if rank < world - 1 else None
        mext, cext = assemble(m, c, below, above)
        lvl = ShardedLevel((32, 32, nzl), w.h, 0.5, True, rank=rank, world=world)
        lvl.fmm.set_option("kernel", 0)
        assert mext.shape[1] == slab_layout(rank, world, nzl)[2]
        L, C = lvl.step_extended(mext, cext)
        torch.cuda.synchronize()
        assert torch.equal(L, Lw[:, own]) and torch.equal(C, Cw[:, own])
        total += lvl.interaction_count()
        lvl.close()
    assert total == whole.interaction_count()
    whole.close()
    assert HALO == 8
