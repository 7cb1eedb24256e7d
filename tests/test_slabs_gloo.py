"""CPU test (gloo, world_size 2 and 3) of the inter-rank schedule of the slab decomposition
(paper_1011_2613_b200.slabs.RankSlab): which buffer goes to which neighbour, the two
messages of a 2-slab periodic ring, walls, and the integer all-reduce of the force sums.  The lattice is a stand-in
that only implements the pack / unpack / export / import contract of include/lbmimb.h on numpy arrays -- the CUDA
library cannot run here; its side of the contract is tested on the GPU in tests/test_gpu_slabs.py."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1011_2613_b200 import slabs


def test_decomposition_and_messages():
    assert slabs.decompose(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert slabs.decompose(1008, 8)[-1] == (882, 126)
    with pytest.raises(ValueError):
        slabs.decompose(3, 4)
    assert slabs.halo_messages(3, False) == [(0, 1, 1, 0), (1, 0, 0, 1), (1, 1, 2, 0), (2, 0, 1, 1)]
    assert slabs.halo_messages(2, True) == [(0, 0, 1, 1), (0, 1, 1, 0), (1, 0, 0, 1), (1, 1, 0, 0)]
    assert slabs.halo_messages(1, True) == [(0, 0, 0, 1), (0, 1, 0, 0)] and slabs.halo_messages(1, False) == []
    assert list(slabs.stored_rows(0, 4, 10, True)) == [9, 0, 1, 2, 3, 4]
    assert list(slabs.stored_rows(0, 4, 10, False)) == [0, 1, 2, 3, 4]
    assert list(slabs.stored_rows(7, 3, 10, False)) == [6, 7, 8, 9]


class ToyLattice:
    """Rows of a global field f[row][col] (value = 100 * global row + col + 0.25 * side-dependent marker), ghost rows
    included, with the halo contract: pack(side) = first / last owned row, unpack(side) = ghost row of that side."""

    def __init__(self, y0, rows, ny, periodic, ncol=5, P=3):
        self.rows_global = slabs.stored_rows(y0, rows, ny, periodic)
        self.glo = 1 if (periodic or y0 > 0) else 0
        self.ghi = 1 if (periodic or y0 + rows < ny) else 0
        self.n_own = rows
        self.f = np.full((len(self.rows_global), ncol), -1.0)
        own = slice(self.glo, self.glo + rows)
        self.f[own] = 100.0 * self.rows_global[own, None] + np.arange(ncol)[None, :]
        self.ncol = ncol
        self.sums = torch.arange(P * 6, dtype=torch.int64) * (y0 + 1)      # stands for this slab's partial sums

    def halo_count(self):
        return self.ncol

    def pack_halo(self, side, t):
        row = self.glo if side == 0 else self.glo + self.n_own - 1
        t.copy_(torch.from_numpy(self.f[row] + (0.25 if side == 0 else 0.5)))

    def unpack_halo(self, side, t):
        row = 0 if side == 0 else len(self.f) - 1
        assert (side == 0 and self.glo) or (side == 1 and self.ghi)
        self.f[row] = t.numpy()

    def force_sums_count(self):
        return int(self.sums.numel())

    def export_force_sums_dev(self, t):
        t.copy_(self.sums)

    def import_force_sums_dev(self, t):
        self.sums = t.clone()


def _worker(rank, world, port, periodic, ny, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        y0, rows = slabs.decompose(ny, world)[rank]
        lat = ToyLattice(y0, rows, ny, periodic)
        rs = slabs.RankSlab(lat, rank, world, periodic, "cpu", pointers=False)
        rs.exchange_halos()
        rs.combine_force_sums()
        out.put((rank, lat.f.copy(), lat.rows_global.copy(), lat.glo, lat.ghi, lat.sums.numpy().copy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True), (3, False)])
def test_rank_schedule_over_gloo(world, periodic):
    ny = 11
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, periodic, ny, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    parts = slabs.decompose(ny, world)
    want_sum = sum(np.arange(18, dtype=np.int64) * (y0 + 1) for (y0, _) in parts)
    for rank, f, rows_g, glo, ghi, sums in res:
        y0, rows = parts[rank]
        assert np.array_equal(sums, want_sum)                                   # integer all-reduce
        if glo:     # lower ghost row holds the LAST owned row of the slab below, packed with side 1 (+0.5)
            assert np.array_equal(f[0], 100.0 * rows_g[0] + np.arange(5) + 0.5)
            assert rows_g[0] == (y0 - 1) % ny
        if ghi:     # upper ghost row holds the FIRST owned row of the slab above, packed with side 0 (+0.25)
            assert np.array_equal(f[-1], 100.0 * rows_g[-1] + np.arange(5) + 0.25)
            assert rows_g[-1] == (y0 + rows) % ny
        assert (glo, ghi) == ((1, 1) if periodic else (int(rank > 0), int(rank < world - 1)))
