"""The sharded level on ONE GPU: the slabs of 2 and of 4 "ranks" are computed one after the other from the halos the
exchange would deliver (the exchange itself is covered by the gloo tests) and must (i) match the ORACLE on sampled regions
of every slab, (ii) reproduce the whole-grid GPU result bit for bit; the per-slab interaction counts add up to the whole
grid's."""
import os

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


@pytest.mark.parametrize("heights,theta", [((16, 16), 0.5), ((16, 16, 16, 16), 0.5), ((16, 16, 16), 0.35), ((8, 24, 16), 0.5)])
def test_peer_memory_halos_in_one_process(heights, theta):
    """octo_fmm_set_neighbours: every slab has a handle of its own that stages only its own layers; interact() fetches
    the neighbours' layers through their staged arrays.  Bit-identical to one handle over the whole grid; matches the
    ORACLE on the layers next to the cuts; counts add up; one slab WITHOUT dipole moments next to one WITH them takes
    the dipole terms (the neighbours' flag words are read)."""
    import torch
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    world = len(heights)                              # slabs of unequal height too: a neighbour's layer index differs from mine
    z0s = [sum(heights[:r]) for r in range(world)]
    nz = sum(heights)
    nzl = heights[0]
    w = fi.config2(ncell=64)
    hm = np.ascontiguousarray(w.moments[:, :nz, :32, :32])
    hc = np.ascontiguousarray(w.com_off[:, :nz, :32, :32])
    hm[1:4] = 0.0                                     # slab 0: expanded about the centre of mass; the others carry dipoles
    hm[1:4, nzl:] = 0.05 * w.h * hm[0, nzl:] * np.random.default_rng(5).uniform(-1, 1, (3, nz - nzl, 32, 32))
    mom, com = torch.from_numpy(hm).cuda(), torch.from_numpy(hc).cuda()
    n = (32, 32, nz)
    whole = p.OctoFMM(n, w.h, theta, p.MULTIPOLE, True)
    whole.set_option("kernel", 0)
    Lw, Cw = whole.solve(mom, com)
    slabs = [p.OctoFMM((32, 32, heights[r]), w.h, theta, p.MULTIPOLE, True) for r in range(world)]
    for r, s in enumerate(slabs):
        s.set_option("kernel", 0)
        s.set_neighbours(slabs[r - 1] if r > 0 else None, slabs[r + 1] if r < world - 1 else None)
        s.set_moments(mom[:, z0s[r]:z0s[r] + heights[r]].contiguous(), com[:, z0s[r]:z0s[r] + heights[r]].contiguous())
    torch.cuda.synchronize()
    total = 0
    for r, s in enumerate(slabs):
        s.interact()
        L, C = s.get_expansions()
        torch.cuda.synchronize()
        assert s.status() == p.OK
        assert s.dipole_terms_used()                 # slab 0 has none of its own: it takes the terms for its neighbour's
        own = slice(z0s[r], z0s[r] + heights[r])
        assert torch.equal(L, Lw[:, own]) and torch.equal(C, Cw[:, own])
        Lh, Ch = L.cpu().numpy(), C.cpu().numpy()
        for z0 in sorted({0, heights[r] - 8}):
            glo, ghi = (8, 8, z0s[r] + z0), (24, 24, z0s[r] + z0 + 8)
            Lr, Lcr, _ = oracle.interact_multipole(n, w.h, theta, hm, hc, glo, ghi, True)
            sl = (slice(None), slice(z0, z0 + 8), slice(8, 24), slice(8, 24))
            assert parity_error(Lh[sl], Lr) < 1e-12 and np.abs(Ch[sl] - Lcr).max() <= 1e-12 * np.abs(Lr[1:4]).max()
        total += s.interaction_count()
    assert total == whole.interaction_count()
    # neighbours removed again: the slab is an isolated grid of its own
    alone = p.OctoFMM((32, 32, nzl), w.h, theta, p.MULTIPOLE, True)
    alone.set_option("kernel", 0)
    La, Ca = alone.solve(mom[:, :nzl].contiguous(), com[:, :nzl].contiguous())
    slabs[0].set_neighbours(None, None)
    slabs[0].interact()
    L0, C0 = slabs[0].get_expansions()
    torch.cuda.synchronize()
    assert torch.equal(L0, La) and torch.equal(C0, Ca) and slabs[0].interaction_count() == alone.interaction_count()
    # argument checks
    with pytest.raises(p.OctoFmmError):
        slabs[0].set_neighbours((0, 0, nzl), None)
    with pytest.raises(p.OctoFmmError):
        slabs[0].set_neighbours((slabs[1].staged_sources()[0], slabs[1].staged_sources()[1], 2), None)
    mono = p.OctoFMM((32, 32, nzl), w.h, theta, p.MONOPOLE)
    with pytest.raises(p.OctoFmmError):
        mono.set_neighbours(None, None)
    for s in slabs + [whole, alone, mono]:
        s.close()


def _peer_rank(rank, world, port, nzl, theta, q):
    import os
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200.sharded import PeerShardedLevel
    try:
        dist.init_process_group("gloo", rank=rank, world_size=world)
        nz = nzl * world
        w = fi.config2(ncell=64)
        hm = np.ascontiguousarray(w.moments[:, :nz, :32, :32])
        hc = np.ascontiguousarray(w.com_off[:, :nz, :32, :32])
        mom, com = torch.from_numpy(hm).cuda(), torch.from_numpy(hc).cuda()
        whole = p.OctoFMM((32, 32, nz), w.h, theta, p.MULTIPOLE, True)
        whole.set_option("kernel", 0)
        Lw, Cw = whole.solve(mom, com)
        lvl = PeerShardedLevel((32, 32, nzl), w.h, theta, True, rank=rank, world=world)
        lvl.fmm.set_option("kernel", 0)
        own = slice(rank * nzl, (rank + 1) * nzl)
        ok = True
        for it in range(3):                                    # repeated steps: the barriers keep the slabs consistent
            scale = 1.0 + it
            L, C = lvl.step((mom[:, own] * scale).contiguous(), com[:, own].contiguous())
            torch.cuda.synchronize()
            Lref, Cref = whole.solve(mom * scale, com)
            torch.cuda.synchronize()
            ok = ok and bool(torch.equal(L, Lref[:, own])) and bool(torch.equal(C, Cref[:, own]))
        counts = [None] * world
        dist.all_gather_object(counts, lvl.interaction_count())
        ok = ok and sum(counts) == whole.interaction_count()
        lvl.close()
        whole.close()
        q.put((rank, ok, ""))
    except Exception as e:                                     # pragma: no cover
        q.put((rank, False, repr(e)))
    finally:
        if dist.is_initialized():
            dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_peer_memory_halos_across_processes(world):
    """One process per rank, all on this one GPU: the ranks trade CUDA IPC handles (gloo carries them) and read each
    other's staged layers through TMA.  No kernel waits on another rank's kernel -- the ranks meet at host barriers --
    so sharing the GPU is safe.  Each rank compares its slab bit for bit with the whole-grid result it computes itself."""
    import torch.multiprocessing as mp
    from paper_2101_08226_b200 import build
    build.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_peer_rank, args=(r, world, port, 16, 0.5, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    res = [q.get(timeout=600) for _ in procs]
    for pr in procs:
        pr.join(timeout=120)
    assert all(ok for _, ok, _ in res), res
