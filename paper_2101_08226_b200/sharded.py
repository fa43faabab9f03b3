"""One uniform level sharded over several GPUs: z-slabs + one halo exchange.

The interaction step shards naturally: sub-grids are independent given the moments of their neighbours within the
stencil's reach (5 cells) -- the paper's "boundary data from sibling sub-grids" (L388).  Rank r of a
torch.distributed group owns the z-layers [r * nz_local, (r + 1) * nz_local) of a grid of nz_local * world layers.
Before the step it receives HALO = 8 layers of raw moments and centre-of-mass offsets from each z-neighbour (5 are
needed; 8 keeps the output region aligned to the 8^3 sub-grids) -- ONE exchange of point-to-point messages (NCCL over
NVLink on GPUs), no collective afterwards: outputs are disjoint.  Everything of the method still runs in the library's
kernels; this module only moves boundary layers and calls the C ABI on the extended slab with the owned layers as the
output region.  The lowest and highest rank see the isolated domain boundary (L321) on their outer side.
"""
from __future__ import annotations

HALO = 8


def slab_layout(rank: int, world: int, nz_local: int):
    """(layers received from below, layers received from above, z-extent of the extended slab)."""
    lo = HALO if rank > 0 else 0
    hi = HALO if rank < world - 1 else 0
    return lo, hi, lo + nz_local + hi


def pack_boundary(moments, com_off, top: bool):
    """The HALO outermost owned layers (top or bottom) of the 23 per-cell arrays as one contiguous buffer [23][HALO][ny][nx]."""
    import torch
    sl = slice(-HALO, None) if top else slice(0, HALO)
    return torch.cat([moments[:, sl], com_off[:, sl]], dim=0).contiguous()


def exchange_halos(moments, com_off, rank: int, world: int, group=None):
    """Returns (moments_ext [20][nz_ext][ny][nx], com_ext [3][nz_ext][ny][nx]): the rank's slab with the neighbours'
    boundary layers attached.  moments [20][nz_local][ny][nx], com_off [3][...] on the rank's device (CPU tensors with
    the gloo backend in the tests).  One batch of point-to-point operations; blocks until the layers have arrived."""
    import torch
    import torch.distributed as dist
    nz_local = moments.shape[1]
    if nz_local < HALO:
        raise ValueError("a slab must have at least %d layers" % HALO)
    lo, hi, nz_ext = slab_layout(rank, world, nz_local)
    shape = (23, HALO) + tuple(moments.shape[2:])
    ops, recv_lo, recv_hi, keep = [], None, None, []
    if lo:
        send = pack_boundary(moments, com_off, top=False)
        recv_lo = torch.empty(shape, dtype=moments.dtype, device=moments.device)
        keep.append(send)
        ops += [dist.P2POp(dist.isend, send, rank - 1, group), dist.P2POp(dist.irecv, recv_lo, rank - 1, group)]
    if hi:
        send = pack_boundary(moments, com_off, top=True)
        recv_hi = torch.empty(shape, dtype=moments.dtype, device=moments.device)
        keep.append(send)
        ops += [dist.P2POp(dist.isend, send, rank + 1, group), dist.P2POp(dist.irecv, recv_hi, rank + 1, group)]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return assemble(moments, com_off, recv_lo, recv_hi)


def assemble(moments, com_off, below=None, above=None):
    """Extended slab from the owned layers and the received boundary buffers ([23][HALO][ny][nx] or None)."""
    import torch
    mparts, cparts = [], []
    if below is not None:
        mparts.append(below[:20]); cparts.append(below[20:])
    mparts.append(moments); cparts.append(com_off)
    if above is not None:
        mparts.append(above[:20]); cparts.append(above[20:])
    return torch.cat(mparts, dim=1).contiguous(), torch.cat(cparts, dim=1).contiguous()


class ShardedLevel:
    """The interaction step of one rank's slab.  `step(moments, com_off)` = halo exchange + set_moments + interact on
    the extended slab with the owned layers as the output region; returns (L [20][nz_local][ny][nx], Lcorr [3][...])."""

    def __init__(self, n_local, h, theta, am_correction=True, rank=0, world=1, group=None, device=0, stream=None):
        from . import MULTIPOLE, OctoFMM
        nx, ny, nzl = (int(v) for v in n_local)
        if nzl % 8 or nzl < HALO:
            raise ValueError("nz_local must be a multiple of 8")
        self.rank, self.world, self.group = int(rank), int(world), group
        self.lo, self.hi, self.nz_ext = slab_layout(self.rank, self.world, nzl)
        self.n_local = (nx, ny, nzl)
        self.fmm = OctoFMM((nx, ny, self.nz_ext), h, theta, MULTIPOLE, am_correction, out_lo=(0, 0, self.lo),
                           out_hi=(nx, ny, self.lo + nzl), device=device, stream=stream)

    def step(self, moments, com_off, L=None, Lcorr=None):
        if self.world > 1:
            mext, cext = exchange_halos(moments, com_off, self.rank, self.world, self.group)
        else:
            mext, cext = moments, com_off
        return self.step_extended(mext, cext, L, Lcorr)

    def step_extended(self, moments_ext, com_ext, L=None, Lcorr=None):
        """The step on an already assembled extended slab ([..][nz_ext][ny][nx])."""
        assert moments_ext.shape[1] == self.nz_ext
        self.fmm.set_moments(moments_ext, com_ext)
        self.fmm.interact()
        return self.fmm.get_expansions(L, Lcorr)

    def interaction_count(self):
        return self.fmm.interaction_count()

    def close(self):
        self.fmm.close()
