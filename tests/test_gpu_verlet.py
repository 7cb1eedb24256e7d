"""GPU-vs-oracle parity of the Verlet neighbour-list mode of a4 (R19) through the
C-ABI (lbmimb_set_neighbor_mode / lbmimb_dem_step / lbmimb_fetch_neighbor_list).  `-m gpu` only.

Lists and rebuild counts are integer results: bit-exact against the oracle's definition.  Trajectories and
coupled runs: the tolerances of tests/parity_util.py.  No expected value comes from the CUDA path."""
import math

import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import assert_fields_close, assert_forces_close, force_floor

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def dense_set(dim, n, P, seed, rlo=1.0, rhi=2.5):
    rng = np.random.default_rng(seed)
    pos = rng.random((dim, P)) * (np.array(n)[:, None] - 5.0) + 2.0
    vel = rng.uniform(-0.02, 0.02, size=(dim, P))
    om = rng.uniform(-1e-3, 1e-3, size=(1 if dim == 2 else 3, P))
    radius = rlo + (rhi - rlo) * rng.random(P)
    mass = 50.0 + 100.0 * rng.random(P)
    return pos, vel, om, radius, mass


CASES = [(3, (30, 26, 22), (0, 1, 0), 150, 0.75), (2, (40, 33), (1, 0), 90, 1.0), (3, (14, 9, 11), (0, 0, 0), 60, 0.5),
         (2, (300, 17), (0, 0), 400, 1.5), (3, (64, 40, 7), (1, 1, 0), 500, 0.25)]


@pytest.mark.parametrize("dim,n,bc,P,skin", CASES)
def test_list_is_bit_exact_against_the_definition(orc, lb, dim, n, bc, P, skin):
    """Overlapping polydisperse random sets; walls and periodic seams; domains with fewer than three grid
    cells on a periodic axis.  The list the first contact evaluation builds is the list of the positions
    that were set."""
    pos, vel, om, radius, mass = dense_set(dim, n, P, 40 + P)
    lat = lb.Lattice(dim, n, bc, 0.8, (0,) * dim, 8 if dim == 2 else 4, max_particles=P + 7)
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, skin, 100)
    lat.set_particles(pos, vel, om, radius, mass)
    start, items, info = lat.fetch_neighbor_list()
    assert not info["valid"] and items.size == 0 and (start == 0).all()
    lat.dem_step(0.05, 0.85, (0,) * dim, 1.0)                   # soft spring: nobody moves farther than skin/2
    start, items, info = lat.fetch_neighbor_list()
    s_o, i_o = orc.verlet_build(dim, n, bc, pos, radius, skin)
    assert info == {"valid": True, "age": 1, "builds": 1}      # |v| dt = 0.03 << skin/2: one build
    assert np.array_equal(start, s_o) and np.array_equal(items, i_o)
    assert items.size > 2 * P                                   # the lists are not trivial
    lat.synchronize()
    lat.close()


@pytest.mark.parametrize("dim,bc", [(2, (0, 1)), (3, (0, 1, 0))])
def test_colliding_trajectory_and_rebuild_count_against_oracle(orc, lb, dim, bc):
    """Fast colliding particles: many contacts and many displacement-triggered rebuilds (the run of
    tests/test_oracle_verlet_pins.py's exactness pin).  Same number of builds, same final lists,
    trajectories within the DEM tolerances."""
    n = (36, 30) if dim == 2 else (24, 20, 18)
    P = 40 if dim == 2 else 70
    rng = np.random.default_rng(21 + dim)
    pos = np.zeros((dim, 0))
    while pos.shape[1] < P:                                     # random sequential addition, distance >= 3
        c = rng.uniform(0, 1, size=(dim, 1)) * np.array(n, dtype=float)[:, None]
        d = pos - c
        for a in range(dim):
            d[a] -= n[a] * np.round(d[a] / n[a])
        if pos.shape[1] == 0 or (d * d).sum(axis=0).min() >= 9.0:
            pos = np.concatenate([pos, c], axis=1)
    vel = rng.uniform(-0.15, 0.15, size=(dim, P))
    for a in range(dim):
        if bc[a]:
            pos[a] = 2.5 + pos[a] * (n[a] - 6.0) / n[a]
    R, m = np.full(P, 1.4), np.full(P, 50.0)
    om = np.zeros((1 if dim == 2 else 3, P))
    fh, th = np.zeros((dim, P)), np.zeros_like(om)
    gp = (0.0, -1e-3, 0.0)[:dim]
    kn = (np.pi ** 2 + np.log(0.9) ** 2) * 25.0 / 8.0 ** 2
    vs = orc.VerletState(dim, P, skin=0.6, every=100)
    lat = lb.Lattice(dim, n, bc, 0.8, (0,) * dim, 8 if dim == 2 else 4, max_particles=P)
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, 0.6, 100)
    lat.set_particles(pos, vel, om, R, m)
    x, v, o = pos.copy(), vel.copy(), om.copy()
    for it in range(120):
        x, v, o = orc.dem_step_verlet(dim, n, bc, x, v, o, R, m, fh, th, kn, 0.9, gp, vs)
        lat.dem_step(kn, 0.9, gp, 1.0)
        if it % 40 == 39:
            xg, vg, og = lat.get_particles()
            assert np.abs(xg - x).max() < 1e-10 and np.abs(vg - v).max() < 1e-11
            start, items, info = lat.fetch_neighbor_list()
            s_o, i_o = vs.lists()
            assert info == {"valid": True, "age": vs.age, "builds": vs.builds}
            assert np.array_equal(start, s_o) and np.array_equal(items, i_o)
    assert 10 < vs.builds < 120
    lat.close()


def test_rebuild_rule_closed_forms(orc, lb):
    """SURVEY/R19 closed forms (tests/test_oracle_verlet_pins.py): uniform motion at |v| = 1/8 with skin 1
    rebuilds every 5 steps of travel (builds = 1 + N // 5); particles at rest rebuild by age only."""
    n, bc = (64, 64), (0, 0)
    pos = np.array([[5.0, 30.0, 50.0], [5.0, 30.0, 50.0]])
    vel = np.array([[0.125, 0.0, -0.125], [0.0, 0.125, 0.0]])
    R, m = np.ones(3), np.ones(3)
    lat = lb.Lattice(2, n, bc, 0.8, (0, 0), 8, max_particles=3)
    for N in (4, 5, 23, 61):
        lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, 1.0, 10 ** 6)
        lat.set_particles(pos, vel, None, R, m)
        for _ in range(N):
            lat.dem_step(1.0, 0.9, (0, 0), 1.0)
        assert lat.fetch_neighbor_list()[2]["builds"] == 1 + N // 5
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, 1.0, 10)
    lat.set_particles(pos, np.zeros((2, 3)), None, R, m)
    for _ in range(35):
        lat.dem_step(1.0, 0.9, (0, 0), 1.0)
    info = lat.fetch_neighbor_list()[2]
    assert info["builds"] == 4 and info["age"] == 5
    # replacing the velocities keeps the list, replacing the positions drops it
    lat.set_particle_velocities(np.zeros((2, 3)), None)
    lat.dem_step(1.0, 0.9, (0, 0), 1.0)
    assert lat.fetch_neighbor_list()[2]["builds"] == 4
    lat.set_particles(pos, np.zeros((2, 3)), None, R, m)
    assert not lat.fetch_neighbor_list()[2]["valid"]
    lat.dem_step(1.0, 0.9, (0, 0), 1.0)
    assert lat.fetch_neighbor_list()[2]["builds"] == 5
    lat.close()


def test_two_sphere_bounce_restitution_with_lists(orc, lb):
    """SURVEY P11 (tests/golden/survey_bounce_values.txt): t_c = 50 steps, e = 0.9 -> v_out/v_in = 0.90370."""
    m, R, tc, e = 1000.0, 5.0, 50.0, 0.9
    kn = (math.pi ** 2 + math.log(e) ** 2) * (m / 2) / tc ** 2
    pos = np.array([[32 - 5.05, 32 + 5.05], [8.0, 8.0], [8.0, 8.0]])
    vel = np.array([[0.01, -0.01], [0, 0], [0, 0.0]])
    lat = lb.Lattice(3, (64, 16, 16), (0, 0, 0), 0.8, (0, 0, 0), 4, max_particles=2)
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, 0.5, 100)
    lat.set_particles(pos, vel, None, np.full(2, R), np.full(2, m))
    for _ in range(700):
        lat.dem_step(kn, e, (0, 0, 0), 1.0)
    _, v, _ = lat.get_particles()
    assert abs(-v[0, 0] / 0.01 - 0.90370) < 1e-5
    lat.close()


def test_coupled_reduced_c5_windows_with_lists(orc, lb):
    """The C5 protocol (oracle leads, shared state at every window start) with the neighbour-list DEM step on
    both sides: map -> step -> reduce -> dem.  A stiffer spring than C5's makes the contacts matter."""
    w = inputs.reduced("C5")
    d = dict(w.dem)
    d["kn"] = 50.0
    skin, every = 0.5, 7
    win, nwin = 10, 3
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    vs = orc.VerletState(w.dim, w.P, skin=skin, every=every)
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P)
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, skin, every)
    for k in range(nwin):
        lat.set_distributions(f)
        lat.set_particles(pos, vel, om, w.radius, w.mass)
        vs.state[0] = 0                                      # shared state: both sides start the window without a list
        b0 = vs.builds
        g0 = lat.fetch_neighbor_list()[2]["builds"]
        for it in range(win):
            f, pos, vel, om, ref = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                    w.radius, w.mass, d["kn"], d["restitution"], d["g_particle"], d["dt"],
                                                    verlet=vs)
            ref.update(floor=force_floor(ref["pid"], w.P), radius=w.radius)
            lat.map_particles()
            lat.step(1)
            gF, gT = lat.reduce_particle_forces()
            assert_forces_close(gF, gT, ref)
            lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])
        assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = lat.get_particles()
        assert np.abs(pg - pos).max() < 1e-10
        assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max() + 1e-18
        assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
        start, items, info = lat.fetch_neighbor_list()
        s_o, i_o = vs.lists()
        assert info["builds"] - g0 == vs.builds - b0 == 2 and info["age"] == vs.age     # window of 10, every = 7
        assert np.array_equal(start, s_o) and np.array_equal(items, i_o)
    lat.close()


def test_paper_scale_2d_cut_lists_and_cell_mode_agree(orc, lb):
    """Reduced cut of the paper's 2D suspension (Table 2 parameters): the list of the
    lattice-like arrangement against the definition, and a neighbour-list run against the cell-list run of
    the same library (sums differ in order only)."""
    w = inputs.reduced("P2D")
    d = w.dem
    lat_c = lb.from_workload(w)
    lat_v = lb.from_workload(w)
    lat_v.set_neighbor_mode(lb.NEIGHBOR_VERLET, 1.0, 100)
    for _ in range(25):
        for lat in (lat_c, lat_v):
            lat.map_particles()
            lat.step(1)
            lat.reduce_particle_forces(to_host=False)
            lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])
    start, items, info = lat_v.fetch_neighbor_list()
    assert info["valid"] and info["builds"] >= 1
    xc, vc, oc = lat_c.get_particles()
    xv, vv, ov = lat_v.get_particles()
    assert np.abs(xc - xv).max() < 1e-11 and np.abs(vc - vv).max() <= 1e-11 * np.abs(vc).max()
    s_o, i_o = orc.verlet_build(w.dim, w.n, w.bc, w.pos, w.radius, 1.0)
    if info["builds"] == 1:
        assert np.array_equal(start, s_o) and np.array_equal(items, i_o)
    lat_c.close()
    lat_v.close()


def test_neighbor_mode_errors(lb):
    lat = lb.Lattice(2, (32, 32), (0, 0), 0.8, (0, 0), 8, max_particles=64)
    for args in ((7, 1.0, 10), (lb.NEIGHBOR_VERLET, 0.0, 10), (lb.NEIGHBOR_VERLET, -1.0, 10),
                 (lb.NEIGHBOR_VERLET, float("nan"), 10), (lb.NEIGHBOR_VERLET, 1.0, 0)):
        with pytest.raises(lb.LbmimbError) as ei:
            lat.set_neighbor_mode(*args)
        assert ei.value.status == lb.EINVAL
    with pytest.raises(lb.LbmimbError) as ei:                   # cell mode has no lists
        lat.fetch_neighbor_list()
    assert ei.value.status == lb.ESTATE
    # 40 disks piled on one spot: more neighbours than the packing bound allows for -> ESTATE, not garbage
    rng = np.random.default_rng(3)
    P = 40
    pos = 16.0 + 0.2 * rng.random((2, P))
    lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, 0.5, 10)
    lat.set_particles(pos, np.zeros((2, P)), None, np.ones(P), np.ones(P))
    lat.dem_step(1e-3, 0.9, (0, 0), 1.0)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.synchronize()
    assert ei.value.status == lb.ESTATE and "neighbour list" in str(ei.value)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.fetch_neighbor_list()
    assert ei.value.status == lb.ESTATE
    # back to the cell list: the same pile is fine
    lat.set_neighbor_mode(lb.NEIGHBOR_CELLS)
    lat.set_particles(pos, np.zeros((2, P)), None, np.ones(P), np.ones(P))
    lat.dem_step(1e-3, 0.9, (0, 0), 1.0)
    lat.synchronize()
    lat.close()
