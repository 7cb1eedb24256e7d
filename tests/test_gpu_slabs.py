"""NEXT-4 (Fig. 2): the lattice cut into y-slabs, each its own handle, halo rows and
per-slab force sums exchanged through the C-ABI (include/lbmimb.h "Slabs").  `-m gpu`, ONE GPU: the slabs are
separate handles on the same device and the transport is a device-to-device copy (paper_1011_2613_b200.slabs.LocalSlabs);
the inter-rank schedule is covered on CPU by tests/test_slabs_gloo.py.  Reference: the CPU oracle on the UNDIVIDED
lattice, usual tolerances; plus bitwise equality with the undivided CUDA lattice (the decomposition changes no
arithmetic and the force sums are order-free integers)."""
import numpy as np
import pytest

from paper_1011_2613_b200 import inputs, slabs
from parity_util import assert_fields_close, assert_forces_close, force_floor, gpu_run, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available()
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def _slabs_for(lb, w, nslabs, bc=None):
    s = slabs.LocalSlabs(lb, w.dim, w.n, bc or w.bc, w.tau, w.g_fluid, w.subsamples, nslabs, max_particles=w.P)
    s.set_particles(w.pos, w.vel, w.omega, w.radius, w.mass)
    return s


@pytest.mark.parametrize("name,nslabs,periodic_y", [("C3", 2, False), ("C3", 3, False), ("C2", 3, False), ("C4", 3, False),
                                                    ("P3D", 4, True), ("P3D", 1, True), ("P2D", 4, True)])
def test_fixed_particles_slabs_against_the_undivided_lattice(orc, lb, name, nslabs, periodic_y):
    """Reduced cuts (particles cut by the slab faces, walls or a periodic seam in y): maps bit-exact, f <= 1e-12 and
    forces <= 1e-10 against the oracle; everything bitwise equal to the undivided CUDA lattice."""
    w = inputs.reduced(name)
    rng = np.random.default_rng(11)
    w.omega = rng.uniform(-1e-3, 1e-3, size=w.omega.shape)
    assert (w.bc[1] == 0) == periodic_y
    steps = 12
    ref = oracle_run(orc, w, steps)
    one, got1 = gpu_run(lb, w, steps, exchange_field=False)
    s = _slabs_for(lb, w, nslabs)
    cut = [y0 for (y0, _) in s.parts[1:]]
    if cut:                                       # some particle really straddles a face
        assert any(((w.pos[1] - w.radius < c) & (w.pos[1] + w.radius > c)).any() for c in cut)
    s.map_particles()
    s.step(steps)
    (F, T), every = s.reduce_particle_forces()
    eps, pid, f = s.fetch_fields(lb.FIELD_EPS_CNT), s.fetch_fields(lb.FIELD_PID), s.fetch_fields(lb.FIELD_F)
    assert np.array_equal(eps, ref["eps"]) and np.array_equal(pid, ref["pid"])
    assert_fields_close(f, ref["f"])
    assert_forces_close(F, T, ref)
    assert np.array_equal(f, got1["f"])
    assert np.array_equal(F, got1["force"]) and np.array_equal(T, got1["torque"])
    for Fk, Tk in every:                          # every slab ends up with the same, complete sums
        assert np.array_equal(Fk, F) and np.array_equal(Tk, T)
    assert np.array_equal(s.fetch_fields(lb.FIELD_RHO), got1["rho"])
    s.close()
    one.close()


@pytest.mark.parametrize("name,nslabs", [("C5", 2), ("P3D", 4)])
def test_coupled_windows_on_slabs(orc, lb, name, nslabs):
    """The coupled protocol (oracle.coupled_step leads, shared state at every window start) with the lattice in
    slabs: map -> step -> halo exchange -> force sums across slabs -> reduce -> DEM on every slab."""
    w = inputs.reduced(name)
    d = w.dem
    dargs = (d["kn"], d["restitution"], d["g_particle"], d["dt"])
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    s = slabs.LocalSlabs(lb, w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, nslabs, max_particles=w.P)
    for k in range(3):
        s.set_distributions(f)
        s.set_particles(pos, vel, om, w.radius, w.mass)
        for it in range(6):
            f, pos, vel, om, ref = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                    w.radius, w.mass, *dargs)
            s.map_particles()
            if it == 0:
                assert np.array_equal(s.fetch_fields(lb.FIELD_EPS_CNT), ref["eps"])
                assert np.array_equal(s.fetch_fields(lb.FIELD_PID), ref["pid"])
            s.step(1)
            (F, T), _ = s.reduce_particle_forces()
            ref.update(floor=force_floor(ref["pid"], w.P), radius=w.radius)
            assert_forces_close(F, T, ref)
            s.dem_step(*dargs)
        assert_fields_close(s.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = s.get_particles()
        assert np.abs(pg - pos).max() < 1e-10
        assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max() + 1e-18
        for l in s.lat[1:]:                       # the replicated particles stay bit-identical on every slab
            p2, v2, o2 = l.get_particles()
            assert np.array_equal(p2, pg) and np.array_equal(v2, vg) and np.array_equal(o2, og)
    s.close()


def test_slab_diagnostics_add_up_and_errors(orc, lb):
    w = inputs.reduced("C3")
    s = _slabs_for(lb, w, 3)
    s.map_particles()
    s.step(5)
    one, _ = gpu_run(lb, w, 5, exchange_field=False)
    whole = one.diagnostics()
    parts = [l.diagnostics() for l in s.lat]
    assert abs(sum(p["mass"] for p in parts) - whole["mass"]) < 1e-9 * whole["mass"]
    assert abs(sum(p["gas_area"] for p in parts) - whole["gas_area"]) < 1e-9 * whole["gas_area"]
    mom = sum(p["fluid_momentum"] for p in parts)
    assert np.abs(mom - whole["fluid_momentum"]).max() < 1e-12 * w.nodes
    assert s.lat[0].slab_ghost_rows(0) == 0 and s.lat[0].slab_ghost_rows(1) == 1     # walls in y: no ghost at the wall
    assert s.lat[1].slab_ghost_rows(0) == 1 and s.lat[2].slab_ghost_rows(1) == 0
    import torch
    buf = torch.empty(s.lat[0].halo_count(), dtype=torch.float64, device="cuda")
    with pytest.raises(lb.LbmimbError) as ei:
        s.lat[0].pack_halo(0, buf.data_ptr())                    # the lower end of slab 0 is a wall
    assert ei.value.status == lb.ESTATE
    with pytest.raises(lb.LbmimbError) as ei:
        one.pack_halo(1, buf.data_ptr())                         # not a slab
    assert ei.value.status == lb.ESTATE
    d = inputs.reduced("C5").dem
    with pytest.raises(lb.LbmimbError) as ei:
        s.lat[1].run_coupled(2, d["kn"], d["restitution"], d["g_particle"], d["dt"])
    assert ei.value.status == lb.ESTATE
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(3, (16, 8, 16), (0, 0, 0), 0.8, (0, 0, 0), 4, streaming=lb.STREAM_AA, slab=(0, 16))
    assert ei.value.status == lb.EINVAL
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(3, (16, 8, 16), (0, 0, 0), 0.8, (0, 0, 0), 4, slab=(10, 16))      # rows 10..18 of 16
    assert ei.value.status == lb.EINVAL
    s.close()
    one.close()


@pytest.mark.parametrize("dim,n,bc,nslabs", [(2, (37, 8), (0, 0), 8), (2, (130, 6), (1, 1), 3), (3, (9, 5, 4), (0, 0, 0), 5),
                                             (3, (6, 7, 3), (1, 1, 1), 2)])
def test_degenerate_slabs_random_state_no_particles(orc, lb, dim, n, bc, nslabs):
    """Slabs of a single owned row (every row is a first AND a last row: both ghosts feed it), walls on every axis,
    no particles: a random non-equilibrium state stepped on the slabs equals the oracle on the undivided lattice."""
    rng = np.random.default_rng(21)
    _, wq, _ = orc.velocity_set(dim)
    shape = (len(wq),) + tuple(reversed(tuple(n) + (1,) * (3 - len(n))))
    f0 = wq.reshape((-1, 1, 1, 1)) * (1 + 0.05 * rng.standard_normal(shape))
    g = (1e-5, -2e-5, 3e-5)[:dim]
    s = slabs.LocalSlabs(lb, dim, n, bc, 0.63, g, 8 if dim == 2 else 4, nslabs)
    s.set_distributions(f0)
    assert np.array_equal(s.fetch_fields(lb.FIELD_F), f0)
    f = f0
    for _ in range(9):
        f = orc.step(dim, n, bc, 0.63, g, 8, f)
    s.step(9)
    assert_fields_close(s.fetch_fields(lb.FIELD_F), f)
    s.close()


def test_c3_full_size_two_slabs_bitwise_and_halo_cost(lb):
    """BASELINE.json configs[2] at its full size (256 x 1008 x 256, 24,600 spheres) as two slabs of 504 rows on ONE
    GPU against the undivided lattice: density, maps and every per-particle force / torque bit for bit after 6 steps
    (the oracle covers the undivided lattice at this size in tests/test_gpu_fullsize.py).  Prints what a halo
    exchange costs on the device (pack + unpack of 256 x 256 x 5 doubles per face)."""
    import torch
    w = inputs.c3()
    steps = 6
    one = lb.from_workload(w)
    one.map_particles()
    one.step(steps)
    F1, T1 = one.reduce_particle_forces()
    rho1 = one.fetch_fields(lb.FIELD_RHO)
    eps1 = one.fetch_fields(lb.FIELD_EPS_CNT)
    pid1 = one.fetch_fields(lb.FIELD_PID)
    one.close()
    del one
    torch.cuda.empty_cache()
    s = slabs.LocalSlabs(lb, w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, 2, max_particles=w.P)
    s.set_particles(w.pos, w.vel, w.omega, w.radius, w.mass)
    s.map_particles()
    s.step(steps)
    (F, T), _ = s.reduce_particle_forces()
    assert np.array_equal(F, F1) and np.array_equal(T, T1)
    assert np.array_equal(s.fetch_fields(lb.FIELD_EPS_CNT), eps1) and np.array_equal(s.fetch_fields(lb.FIELD_PID), pid1)
    assert np.array_equal(s.fetch_fields(lb.FIELD_RHO), rho1)
    cut = s.parts[1][0]
    assert ((w.pos[1] - w.radius < cut) & (w.pos[1] + w.radius > cut)).sum() > 50      # spheres cut by the face
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(20):
        s.exchange_halos()
    b.record()
    torch.cuda.synchronize()
    print("halo exchange of a C3 face pair (2 packs + 2 unpacks of %d doubles, device-to-device): %.3f ms"
          % (s.lat[0].halo_count(), a.elapsed_time(b) / 20))
    s.close()


def test_rank_slab_with_the_real_library_one_rank(lb):
    """slabs.RankSlab (the one-slab-per-rank plumbing, otherwise tested over gloo with a stand-in lattice) driving the
    real library through device pointers: world_size 1, periodic in y, so the rank's single slab feeds its own ghost
    rows and the force sums need no reduction.  Bitwise equal to the undivided lattice."""
    import os
    import torch
    import torch.distributed as dist
    w = inputs.reduced("P3D")
    steps = 7
    one, got1 = gpu_run(lb, w, steps, exchange_field=False)
    created = False
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29591")
        dist.init_process_group("gloo", rank=0, world_size=1)
        created = True
    try:
        lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P, slab=(0, w.n[1]))
        lat.set_particles(w.pos, w.vel, w.omega, w.radius, w.mass)
        rs = slabs.RankSlab(lat, 0, 1, True, "cuda:0", pointers=True)
        assert lat.slab_ghost_rows(0) == 1 and lat.slab_ghost_rows(1) == 1
        lat.map_particles()
        for _ in range(steps):
            lat.step(1)
            rs.exchange_halos()
        rs.combine_force_sums()
        F, T = lat.reduce_particle_forces()
        assert np.array_equal(F, got1["force"]) and np.array_equal(T, got1["torque"])
        assert np.array_equal(lat.fetch_fields(lb.FIELD_F), got1["f"])
        assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), got1["pid"])
        lat.close()
    finally:
        if created:
            dist.destroy_process_group()
    one.close()
