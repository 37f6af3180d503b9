"""Domain decomposition and halo exchange: plumbing around the C ABI.

The paper decomposes the domain into 3D blocks, one per device, and before every evaluation of L exchanges the
ghost ("halo") regions of the blocks with blocking sends and receives of packed 1-D buffers.  Here:

* a block is an ordinary state array ``q[eq, z, y, x]`` with ``ng = 3`` ghost layers; its context is created with
  ``MFC_BC_HALO`` on every side, so the library reads ghost cells and never writes them;
* ``fill_ghosts`` fills them dimension by dimension, x then y then z, each pass over the FULL padded extent of the other
  dimensions -- exactly the order of the single-block ghost fill (oracle ``orc_fill_ghosts``), so edges and corners come
  out the same: a side on the physical boundary is filled locally (zero-gradient copy, or wrap when the block spans the
  periodic dimension alone), every other side receives the 3 layers next to the neighbour's face;
* packing is a strided slice made contiguous (one device copy per slab), the transfer is
  ``torch.distributed.batch_isend_irecv`` -- NCCL send/recv over NVLink between GPUs, gloo between CPU processes in the
  tests -- and unpacking is a copy into the ghost slice.  Nothing of the method's arithmetic happens here.

No 8-GPU node was available to this build: the exchange is covered by world_size-2 gloo tests on CPU
(tests/test_halo_gloo.py) and by a one-GPU test in which a block is its own periodic neighbour.  The benchmark stays
"replicas only".
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

NG = 3
BC_PERIODIC, BC_EXTRAP, BC_HALO = 0, 1, 2


@dataclass(frozen=True)
class Decomposition:
    """Cartesian grid of ranks: ``dims[d]`` blocks along dimension d (x, y, z); rank = ix + dims[0] (iy + dims[1] iz)."""

    dims: Tuple[int, int, int]
    bc_lo: Tuple[int, int, int]      # boundary kind of the GLOBAL domain per dimension (periodic / extrapolation)
    bc_hi: Tuple[int, int, int]

    @property
    def world(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]

    def coords(self, rank: int) -> Tuple[int, int, int]:
        ix = rank % self.dims[0]
        iy = (rank // self.dims[0]) % self.dims[1]
        iz = rank // (self.dims[0] * self.dims[1])
        return ix, iy, iz

    def rank_of(self, c: Sequence[int]) -> int:
        return c[0] + self.dims[0] * (c[1] + self.dims[1] * c[2])

    def neighbour(self, rank: int, d: int, side: int) -> Optional[int]:
        """Rank owning the block beyond face (d, side) (side 0 = low, 1 = high); None on a non-periodic physical boundary.
        With periodic wrap a block can be its own neighbour."""
        c = list(self.coords(rank))
        c[d] += -1 if side == 0 else 1
        if c[d] < 0 or c[d] >= self.dims[d]:
            kind = self.bc_lo[d] if side == 0 else self.bc_hi[d]
            if kind != BC_PERIODIC:
                return None
            c[d] %= self.dims[d]
        return self.rank_of(c)

    def local_cells(self, rank: int, n_global: Sequence[int]) -> Tuple[Tuple[int, int], ...]:
        """Per dimension the [start, stop) range of global interior cells this rank owns (as even a split as possible)."""
        out = []
        for d in range(3):
            c = self.coords(rank)[d]
            base, rem = divmod(int(n_global[d]), self.dims[d])
            start = c * base + min(c, rem)
            out.append((start, start + base + (1 if c < rem else 0)))
        return tuple(out)


def _axis(ndim_total: int, d: int) -> int:
    """Tensor axis of spatial dimension d in q[eq, z, y, x]."""
    return ndim_total - 1 - d


def slab(q, d: int, side: int, ghost: bool, n_d: int):
    """View of the 3 layers of dimension d next to face ``side``: the ghost layers (``ghost=True``, what is received) or the
    interior layers adjacent to the face (what is sent).  Full padded extent in every other dimension."""
    ax = _axis(q.dim(), d)
    if ghost:
        start = 0 if side == 0 else NG + n_d
    else:
        start = NG if side == 0 else n_d
    return q.narrow(ax, start, NG)


def _interior_extent(q, d: int) -> int:
    return q.shape[_axis(q.dim(), d)] - 2 * NG


def fill_side_locally(q, d: int, side: int, nb: Optional[int], rank: int) -> bool:
    """The two kinds of ghost slab that need no other block -- shared by the P2P exchange and the in-process one.  Returns
    False when the slab belongs to another block (the caller then moves the neighbour's layers into it)."""
    n_d = _interior_extent(q, d)
    dst = slab(q, d, side, True, n_d)
    if nb is None:                                           # physical boundary, zero-gradient (PAPER.md:168 as read in B14)
        ax = _axis(q.dim(), d)
        edge = q.narrow(ax, NG if side == 0 else NG + n_d - 1, 1)
        dst.copy_(edge.expand_as(dst))
        return True
    if nb == rank:                                           # the block is its own periodic neighbour: local wrap
        dst.copy_(slab(q, d, 1 - side, False, n_d))
        return True
    return False


def fill_ghosts_in_process(blocks, ndim: int, decomp: Decomposition) -> None:
    """The same fill for ALL blocks of a decomposition held by one process (``blocks[rank]``, tensors on one device): the
    slab a rank would receive is copied straight out of the neighbour's array.  Same slabs, same order (dimension by
    dimension over the full padded extent of the others, every block finishing dimension d before any starts d + 1) as
    ``fill_ghosts``; only the wire is missing.  Used to check a decomposed run against the undivided one on a single GPU."""
    for d in range(ndim):
        for rank, q in enumerate(blocks):
            for side in (0, 1):
                nb = decomp.neighbour(rank, d, side)
                if not fill_side_locally(q, d, side, nb, rank):
                    src = blocks[nb]
                    slab(q, d, side, True, _interior_extent(q, d)).copy_(slab(src, d, 1 - side, False, _interior_extent(src, d)))


def fill_ghosts(q, ndim: int, decomp: Decomposition, rank: int, group=None) -> None:
    """Fills every ghost cell of the block ``q`` (torch tensor [eq, z, y, x], CPU or CUDA) in place."""
    import torch
    import torch.distributed as dist

    for d in range(ndim):
        n_d = _interior_extent(q, d)
        sends, recvs, landing = [], [], []
        for side in (0, 1):
            nb = decomp.neighbour(rank, d, side)
            dst = slab(q, d, side, True, n_d)
            if not fill_side_locally(q, d, side, nb, rank):
                # what I send through face `side` are my interior layers next to it; what lands in my ghost layers of that
                # side are the neighbour's layers next to ITS opposite face.  The tag names the sender's face (gloo matches
                # by tag); NCCL matches the operations between two ranks in posting order, so when one rank is the
                # neighbour on both sides (two blocks in a periodic dimension) the receives are posted high side first:
                # the peer's first send (its low face) is my high-side ghost.
                send = slab(q, d, side, False, n_d).contiguous()
                recv = torch.empty_like(dst, memory_format=torch.contiguous_format)
                sends.append(dist.P2POp(dist.isend, send, nb, group=group, tag=2 * d + side))
                recvs.insert(0, dist.P2POp(dist.irecv, recv, nb, group=group, tag=2 * d + (1 - side)))
                landing.append((dst, recv))
        if sends:
            for w in dist.batch_isend_irecv(sends + recvs):
                w.wait()
            for dst, recv in landing:
                dst.copy_(recv)


class _DevArray:
    """A device pointer owned by the library, exposed to torch through the CUDA array interface (no copy)."""

    def __init__(self, ptr: int, shape):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": "<f8", "data": (int(ptr), False), "version": 3}


class BlockSolver:
    """One block of a decomposed domain on the current CUDA device: halo exchange before every evaluation of L, one
    global CFL step.  ``prob`` describes the LOCAL block (its n, lo, hi / edges); the global boundary kinds live in
    ``decomp``.  With a 1 x 1 x 1 decomposition this reproduces the single-block solver (tested bit for bit)."""

    def __init__(self, prob, decomp: Decomposition, rank: int, group=None, **kw):
        import dataclasses

        import torch

        from . import binding as B

        self.B, self.torch = B, torch
        self.prob, self.decomp, self.rank, self.group = prob, decomp, rank, group
        halo = (BC_HALO,) * 3
        self.ctx = B.init_from_problem(dataclasses.replace(prob, bc_lo=halo, bc_hi=halo), **kw)
        shape = prob.shape()
        self.stage = [None] + [torch.as_tensor(_DevArray(B.mfc_stage_array(self.ctx, k), shape), device="cuda") for k in (1, 2)]

    def close(self):
        if self.ctx is not None:
            self.B.mfc_destroy(self.ctx)
            self.ctx = None

    def cfl_dt(self, q) -> float:
        """CFL step of the whole domain: the minimum over the blocks."""
        import torch.distributed as dist

        stream = self.torch.cuda.current_stream().cuda_stream
        dt = self.B.mfc_cfl_dt(self.ctx, q.data_ptr(), stream)
        if self.decomp.world > 1:
            t = self.torch.tensor([dt], dtype=self.torch.float64, device=q.device)
            dist.all_reduce(t, op=dist.ReduceOp.MIN, group=self.group)
            dt = float(t.item())
        return dt

    def rhs(self, q, out) -> None:
        fill_ghosts(q, self.prob.ndim, self.decomp, self.rank, self.group)
        self.B.mfc_rhs(self.ctx, q.data_ptr(), out.data_ptr(), self.torch.cuda.current_stream().cuda_stream)

    def rk3_step(self, q, dt: float) -> None:
        stream = self.torch.cuda.current_stream().cuda_stream
        for k, arr in enumerate((q, self.stage[1], self.stage[2])):
            fill_ghosts(arr, self.prob.ndim, self.decomp, self.rank, self.group)
            self.B.mfc_rk3_stage(self.ctx, k, q.data_ptr(), dt, stream)


def split_problem(prob, q_global, decomp: Decomposition, rank: int):
    """The local block of ``rank``: a Problem for its cells (with its slice of the edges / its part of [lo, hi]) and its
    padded array (interior copied from the global array, ghost cells zero).  Numpy in, numpy out."""
    import dataclasses

    import numpy as np

    rng = decomp.local_cells(rank, prob.n)
    n = tuple(rng[d][1] - rng[d][0] if d < prob.ndim else 1 for d in range(3))
    lo, hi, edges = list(prob.lo), list(prob.hi), [None, None, None]
    for d in range(prob.ndim):
        if prob.edges is not None and prob.edges[d] is not None:
            edges[d] = np.asarray(prob.edges[d])[rng[d][0]:rng[d][1] + 1].copy()
            lo[d], hi[d] = float(edges[d][0]), float(edges[d][-1])
        else:
            h = prob.dx[d]
            lo[d], hi[d] = prob.lo[d] + rng[d][0] * h, prob.lo[d] + rng[d][1] * h
    # the reciprocal width every block divides by is the GLOBAL n / (hi - lo), formed as mfc_init forms it (ADVICE r2:
    # recomputed from a block's own lo, hi it differs in the last bits from block to block)
    inv_dx = tuple(float(prob.n[d]) / (prob.hi[d] - prob.lo[d]) if d < prob.ndim and edges[d] is None else 0.0 for d in range(3))
    local = dataclasses.replace(prob, name=f"{prob.name}_r{rank}", n=n, lo=tuple(lo), hi=tuple(hi),
                                edges=tuple(edges) if any(e is not None for e in edges) else None, inv_dx=inv_dx)
    ql = np.zeros(local.shape())
    it = prob.interior()
    sl = [slice(None)]
    for ax, d in ((1, 2), (2, 1), (3, 0)):
        if d < prob.ndim:
            sl.append(slice(it[ax].start + rng[d][0], it[ax].start + rng[d][1]))
        else:
            sl.append(slice(0, 1))
    ql[local.interior()] = q_global[tuple(sl)]
    return local, ql


class LocalBlocks:
    """Every block of a decomposition in ONE process on the current device: one context per block, the in-process ghost
    fill between them, the global CFL minimum.  A decomposed run without the wire -- what a single GPU can check of
    PAPER.md:176-182: partitioning, slab geometry, the order of exchange and stages, the per-stage entry points."""

    def __init__(self, prob, q_global, decomp: Decomposition, **kw):
        import dataclasses

        import torch

        from . import binding as B

        self.B, self.torch, self.prob, self.decomp = B, torch, prob, decomp
        halo = (BC_HALO,) * 3
        self.local, self.ctx, self.q, self.stage = [], [], [], []
        for rank in range(decomp.world):
            lp, ql = split_problem(prob, q_global, decomp, rank)
            ctx = B.init_from_problem(dataclasses.replace(lp, bc_lo=halo, bc_hi=halo), **kw)
            self.local.append(lp)
            self.ctx.append(ctx)
            self.q.append(torch.from_numpy(ql).cuda())
            self.stage.append([None] + [torch.as_tensor(_DevArray(B.mfc_stage_array(ctx, k), lp.shape()), device="cuda") for k in (1, 2)])

    def close(self):
        for ctx in self.ctx:
            self.B.mfc_destroy(ctx)
        self.ctx = []

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def _stream(self) -> int:
        return self.torch.cuda.current_stream().cuda_stream

    def cfl_dt(self) -> float:
        return min(self.B.mfc_cfl_dt(ctx, q.data_ptr(), self._stream) for ctx, q in zip(self.ctx, self.q))

    def rhs(self):
        """-> one array per block: L of the decomposed state (ghost entries unspecified)"""
        fill_ghosts_in_process(self.q, self.prob.ndim, self.decomp)
        outs = [self.torch.full_like(q, float("nan")) for q in self.q]
        for ctx, q, o in zip(self.ctx, self.q, outs):
            self.B.mfc_rhs(ctx, q.data_ptr(), o.data_ptr(), self._stream)
        return outs

    def rk3_step(self, dt: float) -> None:
        for k in range(3):
            arrays = self.q if k == 0 else [st[k] for st in self.stage]
            fill_ghosts_in_process(arrays, self.prob.ndim, self.decomp)
            for ctx, q in zip(self.ctx, self.q):
                self.B.mfc_rk3_stage(ctx, k, q.data_ptr(), dt, self._stream)

    def gather(self, blocks=None):
        """Stitches the interiors of ``blocks`` (default: the state) into a global padded numpy array (ghost cells zero)."""
        import numpy as np

        blocks = self.q if blocks is None else blocks
        self.torch.cuda.synchronize()
        out = np.zeros(self.prob.shape())
        it = self.prob.interior()
        for rank, (lp, b) in enumerate(zip(self.local, blocks)):
            rng = self.decomp.local_cells(rank, self.prob.n)
            sl = [slice(None)]
            for ax, d in ((1, 2), (2, 1), (3, 0)):
                sl.append(slice(it[ax].start + rng[d][0], it[ax].start + rng[d][1]) if d < self.prob.ndim else slice(0, 1))
            out[tuple(sl)] = b.cpu().numpy()[lp.interior()]
        return out
