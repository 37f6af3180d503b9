"""Halo exchange of the block decomposition: the slab pack / unpack index maps
and the neighbour logic, with world_size 2 (and 4) on CPU over gloo.  The reference is the single-block ghost fill of
the GLOBAL array, numpy.pad (wrap / edge), restricted to each block: after fill_ghosts every block's padded array --
edges and corners included -- must equal its window of the globally padded array, bit for bit."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2305_09163_b200 import halo  # noqa: E402
from paper_2305_09163_b200 import workloads as wl  # noqa: E402

NG = wl.NG


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_case(ndim, n, periodic_dims):
    prob, q = wl.random_state(ndim, n, 2, seed=17, periodic=True)
    bc = tuple(wl.BC_PERIODIC if d in periodic_dims else wl.BC_EXTRAP for d in range(3))
    import dataclasses
    prob = dataclasses.replace(prob, bc_lo=bc, bc_hi=bc)
    core = q[prob.interior()]
    pads = [(0, 0)] + [(NG, NG) if (2 - ax) < ndim else (0, 0) for ax in range(3)]
    ref = core
    for d in range(ndim):                                   # x, then y, then z over the full padded extents: numpy.pad per axis
        ax = 3 - d
        p = [(0, 0)] * 4
        p[ax] = (NG, NG)
        ref = np.pad(ref, p, mode="wrap" if d in periodic_dims else "edge")
    return prob, q, ref


def _worker(rank, world, port, dims, ndim, n, periodic_dims, out):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        prob, q, ref = _global_case(ndim, n, periodic_dims)
        dec = halo.Decomposition(dims, prob.bc_lo, prob.bc_hi)
        local, ql = halo.split_problem(prob, q, dec, rank)
        rng = np.random.default_rng(100 + rank)
        core = ql[local.interior()].copy()
        ql[...] = rng.normal(size=ql.shape)                 # garbage in the ghosts
        ql[local.interior()] = core
        t = torch.from_numpy(ql)
        halo.fill_ghosts(t, ndim, dec, rank)
        cells = dec.local_cells(rank, prob.n)
        win = [slice(None)] + [slice(cells[d][0], cells[d][1] + 2 * NG) if d < ndim else slice(0, 1) for d in (2, 1, 0)]
        out.put((rank, bool(np.array_equal(t.numpy(), ref[tuple(win)])), local.n))
    finally:
        dist.destroy_process_group()


CASES = [
    # dims, ndim, n, periodic dimensions
    ((2, 1, 1), 1, (23,), ()),
    ((2, 1, 1), 1, (24,), (0,)),                # two blocks in a periodic dimension: each is the other's neighbour on both sides
    ((2, 1, 1), 2, (17, 9), (0, 1)),
    ((1, 2, 1), 2, (11, 14), (1,)),             # periodic in the split dimension, extrapolation in x (local fill)
    ((1, 2, 1), 3, (7, 13, 6), (0, 2)),         # split in y (extrapolation), periodic x and z wrap locally
    ((1, 1, 2), 3, (8, 7, 12), (0, 1, 2)),
    ((2, 1, 1), 3, (12, 6, 7), ()),
    ((2, 2, 1), 3, (10, 9, 5), (0, 1, 2)),      # four ranks: corners travel through two exchanges
    ((2, 1, 2), 3, (9, 5, 10), (1,)),
]


@pytest.mark.parametrize("dims,ndim,n,periodic_dims", CASES)
def test_blocks_after_exchange_equal_the_global_ghost_fill(dims, ndim, n, periodic_dims):
    import torch.multiprocessing as mp
    world = dims[0] * dims[1] * dims[2]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, dims, ndim, n, periodic_dims, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[0] for g in got] == list(range(world))
    assert all(g[1] for g in got), got
    for d in range(ndim):                                   # the blocks tile the domain
        assert sum(g[2][d] for g in got if all(halo.Decomposition(dims, (1,) * 3, (1,) * 3).coords(g[0])[e] == 0 for e in range(3) if e != d)) == n[d]


def test_decomposition_rank_maps():
    dec = halo.Decomposition((3, 2, 2), (0, 1, 0), (0, 1, 0))
    assert dec.world == 12
    for r in range(12):
        assert dec.rank_of(dec.coords(r)) == r
    assert dec.coords(7) == (1, 0, 1)
    assert dec.neighbour(0, 0, 0) == 2 and dec.neighbour(2, 0, 1) == 0       # periodic wrap in x
    assert dec.neighbour(0, 1, 0) is None and dec.neighbour(3, 1, 1) is None  # extrapolation in y: physical boundary
    assert dec.neighbour(0, 1, 1) == 3 and dec.neighbour(0, 2, 0) == 6 and dec.neighbour(6, 2, 1) == 0
    one = halo.Decomposition((1, 1, 1), (0, 0, 0), (0, 0, 0))
    assert one.neighbour(0, 0, 0) == 0 and one.neighbour(0, 2, 1) == 0       # its own periodic neighbour
    cells = [dec.local_cells(r, (10, 7, 4)) for r in range(12)]
    assert [c[0] for c in cells[:3]] == [(0, 4), (4, 7), (7, 10)] and cells[3][1] == (4, 7) and cells[6][2] == (2, 4)


def test_single_block_fill_is_the_plain_ghost_fill():
    """world = 1: periodic sides wrap locally, extrapolation sides copy the edge -- numpy.pad again, no process group."""
    import torch
    prob, q, ref = _global_case(3, (9, 8, 7), (0, 2))
    dec = halo.Decomposition((1, 1, 1), prob.bc_lo, prob.bc_hi)
    t = torch.from_numpy(q.copy())
    halo.fill_ghosts(t, 3, dec, 0)
    assert np.array_equal(t.numpy(), ref)


# ---------------------------------------------------------------------------------------------
# the in-process fill (all blocks of a decomposition in one process: what the one-GPU decomposition tests use) moves the
# same slabs as the P2P exchange: held to the same reference
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,ndim,n,periodic_dims", [
    ((2, 1, 1), 3, (9, 7, 8), (0, 1, 2)),
    ((2, 1, 1), 3, (9, 7, 8), ()),
    ((1, 2, 2), 3, (8, 9, 11), (0, 2)),
    ((2, 2, 2), 3, (10, 9, 11), (1,)),
    ((3, 2, 1), 2, (13, 9), (0,)),
    ((4, 1, 1), 1, (23,), (0,)),
])
def test_in_process_fill_matches_numpy_pad_of_the_global_array(dims, ndim, n, periodic_dims):
    import torch
    prob, q, ref = _global_case(ndim, n, periodic_dims)
    dec = halo.Decomposition(dims, prob.bc_lo, prob.bc_hi)
    blocks, locals_ = [], []
    for rank in range(dec.world):
        local, ql = halo.split_problem(prob, q, dec, rank)
        core = ql[local.interior()].copy()
        ql[...] = np.random.default_rng(100 + rank).normal(size=ql.shape)      # garbage in the ghosts
        ql[local.interior()] = core
        blocks.append(torch.from_numpy(ql))
        locals_.append(local)
    halo.fill_ghosts_in_process(blocks, ndim, dec)
    for rank, (local, t) in enumerate(zip(locals_, blocks)):
        cells = dec.local_cells(rank, prob.n)
        sl = [slice(None)]
        for ax, d in ((1, 2), (2, 1), (3, 0)):
            sl.append(slice(cells[d][0], cells[d][1] + 2 * NG) if d < ndim else slice(0, 1))
        assert np.array_equal(t.numpy(), ref[tuple(sl)]), rank


def test_blocks_of_a_split_problem_carry_the_global_reciprocal_width():
    prob, q, _ = _global_case(3, (10, 9, 11), ())
    dec = halo.Decomposition((2, 2, 2), prob.bc_lo, prob.bc_hi)
    want = tuple(float(prob.n[d]) / (prob.hi[d] - prob.lo[d]) for d in range(3))
    for rank in range(dec.world):
        local, _ = halo.split_problem(prob, q, dec, rank)
        assert local.inv_dx == want
