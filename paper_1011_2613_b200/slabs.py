"""Slab decomposition along y over several lattices (Fig. 2).

Host-side plumbing only: which rows a slab owns, which buffer goes to which neighbour, and the calls of the C-ABI
(include/lbmimb.h "Slabs") in their order.  Every number is computed by the library's kernels; the transport is
torch (device-to-device copies inside one process, torch.distributed send/recv + all_reduce between ranks).

    decompose(ny, k)            rows of the k slabs
    halo_messages(k, periodic)  the messages of one exchange: (src slab, src side, dst slab, dst side)
    LocalSlabs                  all slabs in THIS process on one device (how the decomposition is tested on one GPU)
    RankSlab                    one slab per torch.distributed rank (one process per GPU)

UNMEASURED ACROSS GPUs: this round had one GPU per call.
"""
import numpy as np


def decompose(ny, nslabs):
    """[(y0, rows)] of `nslabs` slabs covering 0..ny, sizes differing by at most one row."""
    if not 1 <= nslabs <= ny:
        raise ValueError("need 1 <= nslabs <= ny")
    base, extra = divmod(ny, nslabs)
    out, y0 = [], 0
    for k in range(nslabs):
        rows = base + (1 if k < extra else 0)
        out.append((y0, rows))
        y0 += rows
    return out


def neighbour(k, side, nslabs, periodic):
    """Slab across the lower (side 0) / upper (side 1) end of slab k, or None at a wall of the global lattice."""
    j = k - 1 if side == 0 else k + 1
    if 0 <= j < nslabs:
        return j
    return j % nslabs if periodic else None


def halo_messages(nslabs, periodic):
    """One halo exchange: every slab sends the populations leaving through each of its non-wall ends to the slab
    across that end, which stores them in its ghost row of the opposite side."""
    msgs = []
    for k in range(nslabs):
        for side in (0, 1):
            j = neighbour(k, side, nslabs, periodic)
            if j is not None:
                msgs.append((k, side, j, 1 - side))
    return msgs


def stored_rows(y0, rows, ny, periodic):
    """Global row indices a slab stores, ghost rows included (what lbmimb_set_distributions expects)."""
    lo = y0 - 1 if (periodic or y0 > 0) else y0
    hi = y0 + rows + 1 if (periodic or y0 + rows < ny) else y0 + rows
    return np.arange(lo, hi) % ny


class LocalSlabs:
    """All slabs of one lattice as separate handles in this process, on one device."""

    def __init__(self, lb, dim, n, bc, tau, g_fluid, subsamples, nslabs, max_particles=0, device=0, flags=0):
        import torch
        self.lb, self.torch = lb, torch
        self.dim, self.n, self.bc = dim, tuple(n), tuple(bc)
        self.periodic = bc[1] == 0
        self.parts = decompose(n[1], nslabs)
        self.lat = []
        for (y0, rows) in self.parts:
            nn = list(n)
            nn[1] = rows
            self.lat.append(lb.Lattice(dim, nn, bc, tau, g_fluid, subsamples, max_particles=max_particles, device=device,
                                       flags=flags, slab=(y0, n[1])))
        self.msgs = halo_messages(nslabs, self.periodic)
        dev = "cuda:%d" % device
        self.halo = {m: torch.empty(self.lat[m[0]].halo_count(), dtype=torch.float64, device=dev) for m in self.msgs}
        self.dev = dev
        self.sums = None

    def close(self):
        for l in self.lat:
            l.close()

    def set_particles(self, pos, vel, omega, radius, mass):
        for l in self.lat:                       # particles are replicated: global coordinates on every slab
            l.set_particles(pos, vel, omega, radius, mass)

    def set_distributions(self, f):
        """f[Q][nz][ny][nx] of the global lattice."""
        for l, (y0, rows) in zip(self.lat, self.parts):
            l.set_distributions(np.ascontiguousarray(f[:, :, stored_rows(y0, rows, self.n[1], self.periodic), :]))

    def map_particles(self):
        for l in self.lat:
            l.map_particles()

    def exchange_halos(self):
        for m in self.msgs:                      # pack everything first: an unpack must not overtake a pack
            self.lat[m[0]].pack_halo(m[1], self.halo[m].data_ptr())
        for m in self.msgs:
            self.lat[m[2]].unpack_halo(m[3], self.halo[m].data_ptr())

    def step(self, nsteps=1):
        for _ in range(nsteps):
            for l in self.lat:
                l.step(1)
            self.exchange_halos()

    def combine_force_sums(self):
        torch = self.torch
        cnt = self.lat[0].force_sums_count()
        if cnt == 0:
            return
        bufs = [torch.empty(cnt, dtype=torch.int64, device=self.dev) for _ in self.lat]
        for l, b in zip(self.lat, bufs):
            l.export_force_sums_dev(b.data_ptr())
        total = bufs[0].clone()
        for b in bufs[1:]:
            total += b                           # integer addition: exact, order-free
        for l in self.lat:
            l.import_force_sums_dev(total.data_ptr())
        self.sums = total

    def reduce_particle_forces(self):
        self.combine_force_sums()
        out = [l.reduce_particle_forces() for l in self.lat]
        return out[0], out

    def dem_step(self, kn, restitution, g_particle, dt=1.0):
        for l in self.lat:
            l.dem_step(kn, restitution, g_particle, dt)

    def get_particles(self):
        return self.lat[0].get_particles()

    def fetch_fields(self, what):
        """The owned rows of all slabs put together: the field of the global lattice."""
        parts = [l.fetch_fields(what) for l in self.lat]
        return np.concatenate(parts, axis=parts[0].ndim - 2)

    def synchronize(self):
        for l in self.lat:
            l.synchronize()


class RankSlab:
    """One slab per torch.distributed rank (launch with torchrun, one process per GPU).  `lat` is anything with the
    binding's pack_halo / unpack_halo / halo_count / export_force_sums_dev / import_force_sums_dev /
    force_sums_count methods; buffers are torch tensors on `device` ("cuda:k" with the nccl backend, "cpu" with
    gloo, where `lat` takes tensors instead of pointers: see tests/test_slabs_gloo.py)."""

    def __init__(self, lat, rank, world, periodic, device, pointers=True):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.lat, self.rank, self.world, self.periodic = lat, rank, world, periodic
        self.device, self.pointers = device, pointers
        self.send = {m: torch.empty(lat.halo_count(), dtype=torch.float64, device=device)
                     for m in halo_messages(world, periodic) if m[0] == rank}
        self.recv = {m: torch.empty(lat.halo_count(), dtype=torch.float64, device=device)
                     for m in halo_messages(world, periodic) if m[2] == rank}

    def _arg(self, t):
        return t.data_ptr() if self.pointers else t

    def exchange_halos(self):
        dist = self.dist
        for m, buf in self.send.items():
            self.lat.pack_halo(m[1], self._arg(buf))
        if self.pointers:
            self.torch.cuda.current_stream().synchronize()       # the packs ran on the lattice's stream
        ops = []
        # tags tell the two messages of a 2-slab periodic ring apart (same pair of ranks in both directions)
        for m, buf in self.send.items():
            if m[2] == self.rank:                                # a single periodic slab feeds itself
                self.recv[m].copy_(buf)
            else:
                ops.append(dist.P2POp(dist.isend, buf, m[2], tag=m[1]))
        for m, buf in self.recv.items():
            if m[0] != self.rank:
                ops.append(dist.P2POp(dist.irecv, buf, m[0], tag=m[1]))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        for m, buf in self.recv.items():
            self.lat.unpack_halo(m[3], self._arg(buf))

    def combine_force_sums(self):
        cnt = self.lat.force_sums_count()
        if cnt == 0:
            return None
        buf = self.torch.empty(cnt, dtype=self.torch.int64, device=self.device)
        self.lat.export_force_sums_dev(self._arg(buf))
        if self.world > 1:
            self.dist.all_reduce(buf, op=self.dist.ReduceOp.SUM)
        self.lat.import_force_sums_dev(self._arg(buf))
        return buf
