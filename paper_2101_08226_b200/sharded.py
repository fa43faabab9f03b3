"""One uniform level sharded over several GPUs: z-slabs + one halo exchange.

The interaction step shards naturally: sub-grids are independent given the moments of their neighbours within the
stencil's reach (5 cells) -- the paper's "boundary data from sibling sub-grids" (L388).  Rank r of a
torch.distributed group owns the z-layers [r * nz_local, (r + 1) * nz_local) of a grid of nz_local * world layers.
Before the step it receives HALO = 8 layers of raw moments and centre-of-mass offsets from each z-neighbour (5 are
needed; 8 keeps the output region aligned to the 8^3 sub-grids) -- ONE batch of point-to-point messages (NCCL over
NVLink on GPUs), no collective afterwards: outputs are disjoint.  Everything of the method still runs in the library's
kernels; this module only moves boundary layers and calls the C ABI on the extended slab with the owned layers as the
output region.  The lowest and highest rank see the isolated domain boundary (L321) on their outer side.

Data movement: the rank keeps ONE persistent extended array per input, [20][nz_ext][ny][nx] and [3][nz_ext][ny][nx].
The owned layers are views into it (`ShardedLevel.moments`, `.com_off`: the producer of the moments writes there), the
neighbours' layers are received straight into its outer layers and sent straight out of its owned layers: for a fixed
component a z-range of layers is one contiguous block, so the exchange is 23 sends and 23 receives per neighbour in one
batch with no packing, no concatenation and no transient memory (97 MB per neighbour at 256^2 against a 3 GB slab).
"""
from __future__ import annotations

HALO = 8


def slab_layout(rank: int, world: int, nz_local: int):
    """(layers received from below, layers received from above, z-extent of the extended slab)."""
    lo = HALO if rank > 0 else 0
    hi = HALO if rank < world - 1 else 0
    return lo, hi, lo + nz_local + hi


def exchange_into(moments_ext, com_ext, rank: int, world: int, group=None):
    """Halo exchange IN PLACE on the extended arrays [20][nz_ext][ny][nx] / [3][nz_ext][ny][nx] whose owned layers
    [lo, lo + nz_local) are filled: sends the HALO outermost owned layers of every component to each z-neighbour and
    receives theirs into the outer layers.  One batch of point-to-point operations (works on CPU tensors with the gloo
    backend and on CUDA tensors with NCCL); blocks until the layers have arrived.  Returns the number of bytes sent."""
    import torch.distributed as dist
    nz_ext = moments_ext.shape[1]
    lo = HALO if rank > 0 else 0
    hi = HALO if rank < world - 1 else 0
    nzl = nz_ext - lo - hi
    if nzl < HALO:
        raise ValueError("a slab must have at least %d layers" % HALO)
    if com_ext.shape[1] != nz_ext or not moments_ext.is_contiguous() or not com_ext.is_contiguous():
        raise ValueError("extended arrays must be contiguous and of equal z-extent")
    ops, sent = [], 0
    for arr in (moments_ext, com_ext):
        for c in range(arr.shape[0]):
            if lo:
                ops.append(dist.P2POp(dist.isend, arr[c, lo:lo + HALO], rank - 1, group))
                ops.append(dist.P2POp(dist.irecv, arr[c, 0:lo], rank - 1, group))
                sent += arr[c, lo:lo + HALO].numel() * arr.element_size()
            if hi:
                ops.append(dist.P2POp(dist.isend, arr[c, lo + nzl - HALO:lo + nzl], rank + 1, group))
                ops.append(dist.P2POp(dist.irecv, arr[c, lo + nzl:nz_ext], rank + 1, group))
                sent += arr[c, lo + nzl - HALO:lo + nzl].numel() * arr.element_size()
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return sent


def pack_boundary(moments, com_off, top: bool):
    """The HALO outermost owned layers (top or bottom) of the 23 per-cell arrays as one buffer [23][HALO][ny][nx] (what a
    neighbour receives; used by the single-GPU geometry test to play the neighbour's part)."""
    import torch
    sl = slice(-HALO, None) if top else slice(0, HALO)
    return torch.cat([moments[:, sl], com_off[:, sl]], dim=0).contiguous()


def exchange_halos(moments, com_off, rank: int, world: int, group=None):
    """Convenience for callers that hold only their owned slab: allocates the extended arrays, copies the slab in and
    exchanges.  Returns (moments_ext, com_ext).  ShardedLevel does NOT use this (it owns persistent extended arrays)."""
    import torch
    nzl = moments.shape[1]
    lo, hi, nz_ext = slab_layout(rank, world, nzl)
    mext = torch.empty((20, nz_ext) + tuple(moments.shape[2:]), dtype=moments.dtype, device=moments.device)
    cext = torch.empty((3, nz_ext) + tuple(moments.shape[2:]), dtype=moments.dtype, device=moments.device)
    mext[:, lo:lo + nzl].copy_(moments)
    cext[:, lo:lo + nzl].copy_(com_off)
    exchange_into(mext, cext, rank, world, group)
    return mext, cext


class ShardedLevel:
    """The interaction step of one rank's slab.

    `moments` / `com_off` are the rank's OWNED layers as views into the persistent extended arrays: fill them (e.g.
    `lvl.moments.copy_(...)`, or let the producer write there) and call `step()` = halo exchange in place + set_moments
    + interact on the extended slab with the owned layers as the output region.
    Returns (L [20][nz_local][ny][nx], Lcorr [3][...])."""

    def __init__(self, n_local, h, theta, am_correction=True, rank=0, world=1, group=None, device=0, stream=None):
        import torch
        from . import MULTIPOLE, OctoFMM
        nx, ny, nzl = (int(v) for v in n_local)
        if nzl % 8 or nzl < HALO:
            raise ValueError("nz_local must be a multiple of 8")
        self.rank, self.world, self.group = int(rank), int(world), group
        self.lo, self.hi, self.nz_ext = slab_layout(self.rank, self.world, nzl)
        self.n_local = (nx, ny, nzl)
        self.fmm = OctoFMM((nx, ny, self.nz_ext), h, theta, MULTIPOLE, am_correction, out_lo=(0, 0, self.lo),
                           out_hi=(nx, ny, self.lo + nzl), device=device, stream=stream)
        dev = self.fmm.device
        self.moments_ext = torch.zeros((20, self.nz_ext, ny, nx), dtype=torch.float64, device=dev)
        self.com_ext = torch.zeros((3, self.nz_ext, ny, nx), dtype=torch.float64, device=dev)
        self.moments = self.moments_ext[:, self.lo:self.lo + nzl]
        self.com_off = self.com_ext[:, self.lo:self.lo + nzl]
        self.halo_bytes_sent = 0

    def step(self, moments=None, com_off=None, L=None, Lcorr=None):
        """moments / com_off given: copied into the owned views first (one device copy; callers on the hot path write
        into `self.moments` / `self.com_off` themselves and pass nothing)."""
        if moments is not None:
            self.moments.copy_(moments)
        if com_off is not None:
            self.com_off.copy_(com_off)
        if self.world > 1:
            self.halo_bytes_sent = exchange_into(self.moments_ext, self.com_ext, self.rank, self.world, self.group)
        return self.step_extended(self.moments_ext, self.com_ext, L, Lcorr)

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


class PeerShardedLevel:
    """The same step with NO exchange and no halo storage (octo_fmm.h, octo_fmm_set_neighbours): every rank stages only
    its own slab; at construction the ranks trade the CUDA IPC handles of their workspaces once, and from then on the
    slab-fed kernel's TMA loads fetch the neighbours' boundary layers straight from their staged arrays (over NVLink when
    they sit on other GPUs) while it computes.  Per step: set_moments, a barrier (every slab staged), interact.
    A second barrier at the start of the next step keeps a rank from staging over layers a neighbour is still reading.
    Results are bit-identical to ShardedLevel's and to one handle over the whole grid.

    One process per GPU; `group` may be a gloo or an NCCL group (it carries 100 bytes per rank once, then barriers)."""

    def __init__(self, n_local, h, theta, am_correction=True, rank=0, world=1, group=None, device=0, stream=None):
        from . import (MULTIPOLE, OctoFMM, octo_fmm_ipc_export, octo_fmm_ipc_import)
        nx, ny, nzl = (int(v) for v in n_local)
        if nzl % 8 or nzl < HALO:
            raise ValueError("nz_local must be a multiple of 8")
        self.rank, self.world, self.group = int(rank), int(world), group
        self.n_local = (nx, ny, nzl)
        self.fmm = OctoFMM((nx, ny, nzl), h, theta, MULTIPOLE, am_correction, device=device, stream=stream)
        self._bases = []
        self._dirty = False
        if self.world > 1:
            import torch.distributed as dist
            src, flg, nz = self.fmm.staged_sources()
            ws = self.fmm.workspace.data_ptr()
            handle, off = octo_fmm_ipc_export(ws)
            everyone = [None] * self.world
            dist.all_gather_object(everyone, (handle, off, src - ws, flg - ws, nz), group=group)
            peers = {}
            for r in (self.rank - 1, self.rank + 1):
                if 0 <= r < self.world:
                    hd, o, dsrc, dflg, pnz = everyone[r]
                    base, pws = octo_fmm_ipc_import(hd, o)
                    self._bases.append(base)
                    peers[r] = (pws + dsrc, pws + dflg, pnz)
            self.fmm.set_neighbours(peers.get(self.rank - 1), peers.get(self.rank + 1))

    def _barrier(self):
        if self.world > 1:
            import torch.distributed as dist
            self.fmm.stream.synchronize()
            dist.barrier(group=self.group)

    def step(self, moments, com_off, L=None, Lcorr=None):
        """moments [20][nz_local][ny][nx], com_off [3][...] of the OWNED slab.  Returns (L, Lcorr) of the owned slab."""
        if self._dirty:
            self._barrier()            # the neighbours have finished reading my previous sources
        self.fmm.set_moments(moments, com_off)
        self._barrier()                # every rank's slab is staged
        self.fmm.interact()
        self._dirty = True
        return self.fmm.get_expansions(L, Lcorr)

    def interaction_count(self):
        return self.fmm.interaction_count()

    def close(self):
        from . import octo_fmm_ipc_close
        if self._dirty:
            self._barrier()
            self._dirty = False
        self.fmm.close()
        for b in self._bases:
            octo_fmm_ipc_close(b)
        self._bases = []
