"""lbmimb_run_coupled (the coupled loop replayed from a CUDA graph) against the same loop made of the four
entry points, bit for bit, and against the oracle at the usual tolerances.  `-m gpu` only."""
import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import assert_fields_close

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def loop(lat, d, n):
    for _ in range(n):
        lat.map_particles()
        lat.step(1)
        lat.reduce_particle_forces(to_host=False)
        lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])


def same_state(lb, a, b):
    assert np.array_equal(a.fetch_fields(lb.FIELD_F), b.fetch_fields(lb.FIELD_F))
    for x, y in zip(a.get_particles(), b.get_particles()):
        assert np.array_equal(x, y)
    assert a.time() == b.time()


@pytest.mark.parametrize("name,streaming,verlet", [("C5", 0, False), ("C5", 1, True), ("P2D", 0, True), ("P3D", 1, False)])
def test_run_coupled_equals_the_explicit_loop(lb, name, streaming, verlet):
    w = inputs.reduced(name)
    d = dict(w.dem)
    if name == "C5":
        d["kn"] = 50.0                                        # contacts that matter
    a = lb.from_workload(w, streaming=streaming)
    b = lb.from_workload(w, streaming=streaming)
    if verlet:
        a.set_neighbor_mode(lb.NEIGHBOR_VERLET, 0.5, 3)       # age rule fires inside the replayed steps
        b.set_neighbor_mode(lb.NEIGHBOR_VERLET, 0.5, 3)
    args = (d["kn"], d["restitution"], d["g_particle"], d["dt"])
    l0a, l0b = a.launch_count(), b.launch_count()
    loop(a, d, 9)
    b.run_coupled(9, *args)                                   # 1 plain step + 4 replays of the pair
    same_state(lb, a, b)
    # the launch counter counts replayed kernels too; with the cell list run_coupled folds the conversion of the
    # force sums into its DEM kernels, which saves the explicit loop's one reduce launch per step
    assert (a.launch_count() - l0a) - (b.launch_count() - l0b) == (0 if verlet else 9)
    loop(a, d, 4)
    b.run_coupled(4, *args)                                   # starts on the other parity: second graph
    same_state(lb, a, b)
    loop(a, d, 6)
    b.run_coupled(1, *args)
    b.run_coupled(0, *args)
    b.run_coupled(5, *args)
    same_state(lb, a, b)
    if verlet:
        assert a.fetch_neighbor_list()[2] == b.fetch_neighbor_list()[2]
        sa, ia, _ = a.fetch_neighbor_list()
        sb, ib, _ = b.fetch_neighbor_list()
        assert np.array_equal(sa, sb) and np.array_equal(ia, ib)
    # new positions in the same buffers: the captured launches still apply
    pos, vel, om = a.get_particles()
    pos2 = pos.copy()
    pos2[0] = np.mod(pos2[0] + 0.125, w.n[0])
    for lat in (a, b):
        lat.set_particles(pos2, vel, om, w.radius, w.mass)
    loop(a, d, 5)
    b.run_coupled(5, *args)
    same_state(lb, a, b)
    # other DEM parameters are kernel arguments: the pair is captured again
    d2 = dict(d)
    d2["kn"] = 2.0 * d["kn"]
    loop(a, d2, 5)
    b.run_coupled(5, d2["kn"], d2["restitution"], d2["g_particle"], d2["dt"])
    same_state(lb, a, b)
    a.close()
    b.close()


def test_run_coupled_against_the_oracle(orc, lb):
    w = inputs.reduced("C5")
    d = w.dem
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    n = 8
    for _ in range(n):
        f, pos, vel, om, _ = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                              w.radius, w.mass, d["kn"], d["restitution"], d["g_particle"], d["dt"])
    lat = lb.from_workload(w)
    lat.run_coupled(n, d["kn"], d["restitution"], d["g_particle"], d["dt"])
    assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
    pg, vg, og = lat.get_particles()
    assert np.abs(pg - pos).max() < 1e-10
    assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max() + 1e-18
    assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
    lat.close()


def test_run_coupled_without_particles_and_errors(lb):
    lat = lb.Lattice(2, (32, 24), (0, 1), 0.8, (0.0, -1e-6), 8, max_particles=4)
    ref = lb.Lattice(2, (32, 24), (0, 1), 0.8, (0.0, -1e-6), 8, max_particles=4)
    lat.run_coupled(7, 1.0, 0.9, (0, 0), 1.0)
    ref.step(7)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_F), ref.fetch_fields(lb.FIELD_F)) and lat.time() == 7
    for bad in ((-1, 1.0, 0.9), (3, 0.0, 0.9), (3, 1.0, 1.5)):
        with pytest.raises(lb.LbmimbError) as ei:
            lat.run_coupled(bad[0], bad[1], bad[2], (0, 0), 1.0)
        assert ei.value.status == lb.EINVAL
    lat.close()
    ref.close()
