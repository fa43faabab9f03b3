"""Host logic of the multi-GPU path (paper_2101_08226_b200/sharded.py): the halo exchange over a world_size-2 and a
world_size-3 gloo group on CPU reproduces the slices of the global arrays (no kernels involved)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_slab_layout():
    from paper_2101_08226_b200.sharded import HALO, slab_layout
    assert HALO == 8
    assert slab_layout(0, 1, 32) == (0, 0, 32)
    assert slab_layout(0, 4, 32) == (0, 8, 40)
    assert slab_layout(2, 4, 32) == (8, 8, 48)
    assert slab_layout(3, 4, 32) == (8, 0, 40)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from paper_2101_08226_b200.sharded import exchange_halos, exchange_into, slab_layout
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nx, ny, nzl = 8, 16, 16
    rng = np.random.default_rng(5)                         # every rank builds the same global arrays
    gm = torch.from_numpy(rng.normal(size=(20, nzl * world, ny, nx)))
    gc = torch.from_numpy(rng.normal(size=(3, nzl * world, ny, nx)))
    mine = slice(rank * nzl, (rank + 1) * nzl)
    mext, cext = exchange_halos(gm[:, mine].contiguous(), gc[:, mine].contiguous(), rank, world)
    lo, hi, nz_ext = slab_layout(rank, world, nzl)
    ref = slice(rank * nzl - lo, (rank + 1) * nzl + hi)
    ok = bool(mext.shape[1] == nz_ext and torch.equal(mext, gm[:, ref]) and torch.equal(cext, gc[:, ref]))
    # the in-place route on persistent extended arrays: owned layers filled, outer layers poisoned, exchanged in place
    pm = torch.full((20, nz_ext, ny, nx), float("nan"), dtype=torch.float64)
    pc = torch.full((3, nz_ext, ny, nx), float("nan"), dtype=torch.float64)
    pm[:, lo:lo + nzl] = gm[:, mine]
    pc[:, lo:lo + nzl] = gc[:, mine]
    sent = exchange_into(pm, pc, rank, world)
    ok = ok and torch.equal(pm, gm[:, ref]) and torch.equal(pc, gc[:, ref])
    ok = ok and sent == ((lo > 0) + (hi > 0)) * 23 * 8 * ny * nx * 8
    out[rank] = ok
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_over_gloo(world):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    assert all(out[r] for r in range(world)) and len(out) == world
