"""GPU-vs-oracle parity through the C-ABI (binding -> liblbmimb.so).  `-m gpu` only.

Every comparison runs the CUDA path and the CPU oracle on the same seeded inputs
(paper_1011_2613_b200.inputs) and compares element by element with the tolerances
of tests/parity_util.py.  No expected value comes from the CUDA path.
"""
import math

import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import (F_TOL, assert_fields_close, assert_forces_close, force_floor, gpu_run, oracle_run)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


# ----------------------------------------------------------------------------- fixed particles
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_reduced_configs_fields_maps_forces(orc, lb, name):
    """C1 in full (128x128, 100 steps) and the reduced cuts of C2..C5 (ragged tails: nx not a
    multiple of the 128-node tile, several tiles per row, odd row counts)."""
    w = inputs.reduced(name)
    ref = oracle_run(orc, w, w.steps)
    lat, got = gpu_run(lb, w, w.steps)
    assert np.array_equal(got["eps"], ref["eps"]), "eps_cnt is not bit-exact"
    assert np.array_equal(got["pid"], ref["pid"]), "pid is not bit-exact"
    assert_fields_close(got["f"], ref["f"], "f")
    assert_fields_close(got["rho"], ref["rho"], "rho")
    assert np.abs(got["u"] - ref["u"]).max() <= F_TOL * max(np.abs(ref["f"]).max(), np.abs(ref["u"]).max())
    # s is a sum of f-sized terms that cancel (sum_i Omega_i c_i): its rounding scale is that of f
    assert np.abs(got["s"] - ref["s"]).max() <= F_TOL * np.abs(ref["f"]).max()
    assert_forces_close(got["force"], got["torque"], ref)
    assert lat.time() == w.steps
    lat.close()


@pytest.mark.parametrize("dim,n,bc", [(2, (130, 7), (0, 0)), (2, (257, 5), (1, 1)), (2, (3, 4), (1, 0)),
                                      (3, (129, 5, 4), (0, 1, 0)), (3, (6, 5, 3), (1, 1, 1)),
                                      (3, (2, 2, 2), (0, 0, 0)), (2, (1, 1), (0, 0)), (3, (1, 3, 1), (0, 1, 0))])
def test_pure_lbgk_random_state(orc, lb, dim, n, bc):
    """No particles: set a random non-equilibrium state, step, compare (walls, periodic seams,
    degenerate 1-node axes, two tiles per row)."""
    rng = np.random.default_rng(5)
    _, wq, _ = orc.velocity_set(dim)
    shape = (len(wq),) + tuple(reversed(tuple(n) + (1,) * (3 - len(n))))
    f0 = wq.reshape((-1, 1, 1, 1)) * (1 + 0.05 * rng.standard_normal(shape))
    g = (1e-5, -2e-5, 3e-5)[:dim]
    lat = lb.Lattice(dim, n, bc, 0.63, g, 8 if dim == 2 else 4)
    lat.set_distributions(f0)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_F), f0)       # set/fetch is an exact permutation round trip
    f = f0
    for _ in range(7):
        f = orc.step(dim, n, bc, 0.63, g, 8, f)
    lat.step(7)
    assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
    rho, u = orc.macros(dim, f)
    assert_fields_close(lat.fetch_fields(lb.FIELD_RHO), rho, "rho")
    assert np.abs(lat.fetch_fields(lb.FIELD_U) - u).max() < 1e-13
    lat.close()


def test_rest_state_and_mass_conservation(lb):
    lat = lb.Lattice(3, (70, 9, 11), (0, 1, 0), 0.8, (0, 0, 0), 4)
    lat.step(20)
    f = lat.fetch_fields(lb.FIELD_F)
    rho = lat.fetch_fields(lb.FIELD_RHO)
    assert np.abs(rho - 1).max() < 1e-14 and np.abs(lat.fetch_fields(lb.FIELD_U)).max() < 1e-15
    assert abs(f.sum() - 70 * 9 * 11) < 1e-9
    lat.close()


def test_sub_box_fetch(orc, lb):
    w = inputs.reduced("C3")
    lat, got = gpu_run(lb, w, 5)
    lo, hi = (3, 70, 1), (72, 90, 30)
    sl = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    for what, key in ((lb.FIELD_F, "f"), (lb.FIELD_U, "u"), (lb.FIELD_S, "s")):
        assert np.array_equal(lat.fetch_fields(what, lo, hi), got[key][(slice(None),) + sl])
    for what, key in ((lb.FIELD_RHO, "rho"), (lb.FIELD_EPS_CNT, "eps"), (lb.FIELD_PID, "pid")):
        assert np.array_equal(lat.fetch_fields(what, lo, hi), got[key][sl])
    lat.close()


# ----------------------------------------------------------------------------- mapping edge cases
def _map_both(orc, lb, dim, n, bc, S, pos, radius):
    P = pos.shape[1]
    lat = lb.Lattice(dim, n, bc, 0.8, (0,) * dim, S, max_particles=P)
    lat.set_particles(pos, np.zeros((dim, P)), None, radius, np.ones(P))
    lat.map_particles()
    e, p = lat.fetch_fields(lb.FIELD_EPS_CNT), lat.fetch_fields(lb.FIELD_PID)
    lat.synchronize()
    lat.close()
    eo, po = orc.map_particles(dim, n, bc, S, pos, radius)
    assert np.array_equal(e, eo), "eps_cnt differs at %d nodes" % (e != eo).sum()
    assert np.array_equal(p, po), "pid differs at %d nodes" % (p != po).sum()
    return e, p


@pytest.mark.parametrize("dim,S", [(2, 8), (2, 5), (2, 15), (3, 4), (3, 6), (3, 3), (2, 1), (3, 1)])
def test_map_overlapping_seam_and_unquantised(orc, lb, dim, S):
    """Overlapping particles (contested nodes, ties), particles across the periodic seam and at
    walls, radii from 0.4 to 9, centres that are NOT multiples of 2^-16, S not a power of two."""
    rng = np.random.default_rng(100 * dim + S)
    n = (67, 45) if dim == 2 else (35, 22, 27)
    bc = (0, 1) if dim == 2 else (0, 1, 0)
    P = 40
    pos = rng.random((dim, P)) * np.array(n)[:, None]
    radius = 0.4 + 5.0 * rng.random(P) ** 2
    radius[0] = 9.0
    pos[:, 1] = pos[:, 0] + 0.37             # heavy overlap
    pos[:, 2] = pos[:, 3]                    # identical centres, tie -> lowest index
    radius[2] = radius[3]
    pos[0, 4] = 0.01                         # across the periodic seam in x
    pos[0, 5] = n[0] - 0.3
    for a in range(dim):
        if bc[a]:
            pos[a] = np.clip(pos[a], 0.0, n[a] - 1.0)
        else:
            pos[a] = np.mod(pos[a], n[a])
    e, p = _map_both(orc, lb, dim, n, bc, S, pos, radius)
    assert (p >= 0).sum() > 50 and e.max() == S ** dim


def test_map_box_wider_than_the_periodic_domain(orc, lb):
    _map_both(orc, lb, 2, (9, 7), (0, 0), 8, np.array([[4.2, 1.0], [3.3, 6.5]]), np.array([5.5, 1.2]))
    _map_both(orc, lb, 3, (6, 5, 7), (0, 0, 0), 4, np.array([[3.1], [2.2], [3.3]]), np.array([4.0]))


@pytest.mark.parametrize("dim", [2, 3])
def test_big_particles_many_row_chunks_map_table_and_forces(orc, lb, dim):
    """Particles whose bounding box has more rows than a thread group (several row chunks and several
    candidate passes of the dense box walk), next to small ones, across a seam and against a wall:
    sampled map and table map bit-exact, fields and forces at the usual tolerances."""
    if dim == 2:
        n, bc, S = (150, 131), (0, 1), 8
        pos = np.array([[60.3, 140.2, 20.7, 100.1], [66.6, 30.4, 100.9, 110.3]])
        radius = np.array([40.25, 17.5, 3.0, 16.0])
    else:
        n, bc, S = (61, 50, 57), (0, 1, 0), 4
        pos = np.array([[25.3, 55.2, 50.7], [24.6, 12.4, 40.9], [30.1, 50.3, 8.2]])
        radius = np.array([20.5, 6.25, 9.0])
    P = radius.size
    _map_both(orc, lb, dim, n, bc, S, pos, radius)
    rng = np.random.default_rng(5 + dim)
    w = inputs.Workload("big", dim, n, bc, 0.8, (0.0, -1e-5, 0.0)[:dim], S, 5, pos, rng.uniform(-0.01, 0.01, (dim, P)),
                        rng.uniform(-1e-3, 1e-3, (1 if dim == 2 else 3, P)), radius, np.full(P, 100.0))
    ref = oracle_run(orc, w, 5)
    lat, got = gpu_run(lb, w, 5)
    assert np.array_equal(got["eps"], ref["eps"]) and np.array_equal(got["pid"], ref["pid"])
    assert_fields_close(got["f"], ref["f"])
    assert_forces_close(got["force"], got["torque"], ref)
    lat.close()
    # the paper's table look-up needs one radius
    rad1 = np.full(P, radius[0] / 2)
    lat = lb.Lattice(dim, n, bc, 0.8, (0,) * dim, S, max_particles=P)
    lat.set_mapping_mode(lb.MAP_TABLE)
    lat.set_particles(pos, np.zeros((dim, P)), None, rad1, np.ones(P))
    lat.map_particles()
    eo, po = orc.map_particles_table(dim, n, bc, pos, rad1)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eo)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), po)
    lat.close()


def test_map_is_translation_invariant_on_the_gpu_too(orc, lb):
    w = inputs.reduced("C2")
    e0, p0 = _map_both(orc, lb, w.dim, w.n, (0, 0), 8, w.pos, w.radius)
    pos = w.pos + np.array([[17.0], [-5.0]])
    pos = np.mod(pos, np.array(w.n)[:, None])
    e1, p1 = _map_both(orc, lb, w.dim, w.n, (0, 0), 8, pos, w.radius)
    assert np.array_equal(np.roll(e0, (-5, 17), axis=(1, 2)), e1)


def test_remap_after_moving_particles_and_no_particles(orc, lb):
    w = inputs.reduced("C2")
    lat = lb.from_workload(w)
    lat.map_particles()
    pos2 = np.mod(w.pos + 3.25, np.array(w.n)[:, None] - 12.0) + 6.0
    lat.set_particles(pos2, w.vel, w.omega, w.radius, w.mass)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.step(1)
    assert ei.value.status == lb.ESTATE
    lat.map_particles()
    eo, po = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, pos2, w.radius)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eo)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), po)
    lat.set_particles(None, None, None, None, None)          # P = 0
    lat.step(2)
    assert lat.fetch_fields(lb.FIELD_EPS_CNT).max() == 0 and lat.fetch_fields(lb.FIELD_PID).max() == -1
    lat.close()


# ----------------------------------------------------------------------------- forces
def test_force_reduction_is_reproducible_and_matches_spinning_overlapping_set(orc, lb):
    rng = np.random.default_rng(77)
    w = inputs.reduced("C3")
    w.omega = rng.uniform(-2e-3, 2e-3, size=(3, w.P))
    w.pos[:, 1] = w.pos[:, 0] + np.array([5.0, 2.0, 1.0])      # overlapping pair: shared nodes
    ref = oracle_run(orc, w, 6)
    lat, got = gpu_run(lb, w, 6)
    assert np.array_equal(got["pid"], ref["pid"])
    assert_forces_close(got["force"], got["torque"], ref)
    again = lat.reduce_particle_forces()
    assert np.array_equal(again[0], got["force"]) and np.array_equal(again[1], got["torque"])
    lat.close()


def test_prescribed_velocity_update_keeps_the_map(orc, lb):
    w = inputs.reduced("C2")
    lat = lb.from_workload(w)
    lat.map_particles()
    lat.step(3)
    vel2, om2 = -0.5 * w.vel, 2.0 * w.omega
    lat.set_particle_velocities(vel2, om2)
    lat.step(2)
    ref = oracle_run(orc, w, 3)
    ref2 = oracle_run(orc, w, 2, f0=ref["f"], vel=vel2, omega=om2)
    assert_fields_close(lat.fetch_fields(lb.FIELD_F), ref2["f"])
    F, T = lat.reduce_particle_forces()
    assert_forces_close(F, T, ref2)
    lat.close()


# ----------------------------------------------------------------------------- DEM
def test_dem_contact_and_integration_against_oracle(orc, lb):
    """Dense overlapping random set, walls + periodic axes, prescribed hydrodynamic loads = 0."""
    rng = np.random.default_rng(9)
    for dim, n, bc in ((3, (30, 26, 22), (0, 1, 0)), (2, (40, 33), (1, 0)), (3, (14, 9, 11), (0, 0, 0))):
        P = 150 if dim == 3 else 90
        pos = rng.random((dim, P)) * (np.array(n)[:, None] - 5.0) + 2.0
        vel = rng.uniform(-0.02, 0.02, size=(dim, P))
        om = rng.uniform(-1e-3, 1e-3, size=(1 if dim == 2 else 3, P))
        radius = 1.0 + 1.5 * rng.random(P)
        mass = 50.0 + 100.0 * rng.random(P)
        kn, e, gp = 3.0, 0.85, (1e-4, -2e-4, 5e-5)[:dim]
        lat = lb.Lattice(dim, n, bc, 0.8, (0,) * dim, 8 if dim == 2 else 4, max_particles=P)
        lat.set_particles(pos, vel, om, radius, mass)
        z = np.zeros((dim, P))
        zt = np.zeros_like(om)
        p_o, v_o, o_o = pos, vel, om
        for _ in range(12):
            lat.dem_step(kn, e, gp, 1.0)
            p_o, v_o, o_o = orc.dem_step(dim, n, bc, p_o, v_o, o_o, radius, mass, z, zt, kn, e, gp, 1.0)
        p_g, v_g, o_g = lat.get_particles()
        fc = orc.contact_forces(dim, n, bc, p_o, v_o, radius, mass, kn, e)
        assert (np.abs(fc).max(axis=0) > 0).sum() > P // 4          # contacts are really exercised
        assert np.abs(p_g - p_o).max() < 1e-11
        assert np.abs(v_g - v_o).max() < 1e-12 * max(1.0, np.abs(v_o).max() / 1e-2)
        assert np.array_equal(o_g, o_o)
        lat.close()


def test_dem_two_sphere_bounce_matches_oracle_and_restitution(orc, lb):
    m, R, tc, e = 1000.0, 5.0, 50.0, 0.9
    kn = (math.pi ** 2 + math.log(e) ** 2) * (m / 2) / tc ** 2
    n = (64, 16, 16)
    pos = np.array([[32 - 5.05, 32 + 5.05], [8.0, 8.0], [8.0, 8.0]])
    vel = np.array([[0.01, -0.01], [0, 0], [0, 0.0]])
    lat = lb.Lattice(3, n, (0, 0, 0), 0.8, (0, 0, 0), 4, max_particles=2)
    lat.set_particles(pos, vel, None, np.full(2, R), np.full(2, m))
    for _ in range(700):
        lat.dem_step(kn, e, (0, 0, 0), 1.0)
    _, v, _ = lat.get_particles()
    assert abs(-v[0, 0] / 0.01 - 0.90370) < 1e-5                 # SURVEY P11, tests/golden/survey_bounce_values.txt
    lat.close()


# ----------------------------------------------------------------------------- coupled run
def test_coupled_reduced_c5_windows(orc, lb):
    """C5 protocol on the reduced cut: the oracle leads; at the start of every window the CUDA
    path is set to the oracle's state (f, x, v, omega), both run `win` coupled steps
    (map -> step -> reduce -> dem), and are compared at the end of the window."""
    w = inputs.reduced("C5")
    d = w.dem
    win, nwin = 10, 4
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P)
    moved = 0.0
    for k in range(nwin):
        lat.set_distributions(f)
        lat.set_particles(pos, vel, om, w.radius, w.mass)
        for it in range(win):
            f, pos, vel, om, ref = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                    w.radius, w.mass, d["kn"], d["restitution"], d["g_particle"], d["dt"])
            eps, pid = ref["eps"], ref["pid"]
            ref.update(floor=force_floor(pid, w.P), radius=w.radius)
            lat.map_particles()
            if it == 0:
                assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eps)
                assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), pid)
            lat.step(1)
            gF, gT = lat.reduce_particle_forces()
            assert_forces_close(gF, gT, ref)
            lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])
        assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = lat.get_particles()
        assert np.abs(pg - pos).max() < 1e-10
        assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max() + 1e-18
        assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
        moved = max(moved, np.abs(vel).max())
    assert moved > 1e-6
    lat.close()


# ----------------------------------------------------------------------------- device-pointer variants
def test_device_pointer_variants_match_the_host_variants(orc, lb):
    """lbmimb_set_particles_dev / lbmimb_reduce_particle_forces_dev with torch tensors (plumbing only) give
    bit for bit what the host-pointer calls give, and the oracle agrees."""
    import torch
    w = inputs.reduced("C3")
    ref = oracle_run(orc, w, 4)
    lat_h, got = gpu_run(lb, w, 4)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    tp, tv, to, tr, tm = dev(w.pos), dev(w.vel), dev(w.omega), dev(w.radius), dev(w.mass)
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P)
    lat.set_particles_dev(w.P, tp.data_ptr(), tv.data_ptr(), to.data_ptr(), tr.data_ptr(), tm.data_ptr())
    lat.map_particles()
    lat.step(4)
    tF = torch.zeros((w.dim, w.P), dtype=torch.float64, device="cuda")
    tT = torch.zeros((3, w.P), dtype=torch.float64, device="cuda")
    lat.reduce_particle_forces_dev(tF.data_ptr(), tT.data_ptr())
    lat.synchronize()
    assert np.array_equal(tF.cpu().numpy(), got["force"]) and np.array_equal(tT.cpu().numpy(), got["torque"])
    assert np.array_equal(lat.fetch_fields(lb.FIELD_F), got["f"])
    assert_forces_close(tF.cpu().numpy(), tT.cpu().numpy(), ref)
    pg, vg, og = lat.get_particles()
    assert np.array_equal(pg, w.pos) and np.array_equal(vg, w.vel) and np.array_equal(og, w.omega)
    lat.close()
    lat_h.close()


# ----------------------------------------------------------------------------- errors
def test_error_behaviour(lb):
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(2, (16, 16), (0, 0), 0.5, (0, 0), 8)
    assert ei.value.status == lb.EINVAL
    with pytest.raises(lb.LbmimbError):
        lb.Lattice(3, (8, 8, 8), (0, 0, 0), 0.8, (0, 0, 0), 7)          # 7^3 > 255
    lat = lb.Lattice(2, (16, 16), (0, 0), 0.8, (0, 0), 8, max_particles=2)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.set_particles(np.zeros((2, 3)) + 4, np.zeros((2, 3)), None, np.ones(3), np.ones(3))
    assert ei.value.status == lb.EINVAL
    with pytest.raises(lb.LbmimbError):
        lat.set_particles(np.array([[40.0], [3.0]]), np.zeros((2, 1)), None, np.ones(1), np.ones(1))  # outside
    lat.set_particles(np.array([[4.0], [3.0]]), np.zeros((2, 1)), None, np.ones(1), np.ones(1))
    lat.map_particles()
    with pytest.raises(lb.LbmimbError) as ei:
        lat.reduce_particle_forces()                                     # no step yet
    assert ei.value.status == lb.ESTATE
    with pytest.raises(lb.LbmimbError):
        lat.fetch_fields(lb.FIELD_F, (0, 0, 0), (17, 16, 1))
    lat.step(1)
    F, T = lat.reduce_particle_forces()
    assert F.shape == (2, 1) and T.shape == (1, 1)
    assert lat.launch_count() > 3
    lat.close()


# ----------------------------------------------------------------------------- in-kernel force sums
def test_in_kernel_force_sums_reproducible_and_independent_of_the_exchange_field(orc, lb):
    """a3 is summed inside the fused step with fixed-point integer atomics: two lattices give bit-identical
    forces, with or without the per-node exchange field, in either streaming mode; FIELD_S needs the flag;
    sums of a step that was never reduced do not leak into the next one."""
    w = inputs.reduced("C3")
    rng = np.random.default_rng(3)
    w.omega = rng.uniform(-2e-3, 2e-3, size=(3, w.P))
    ref = oracle_run(orc, w, 5)
    res = []
    for streaming in (lb.STREAM_AB, lb.STREAM_AA):
        for flags in (0, lb.FLAG_EXCHANGE_FIELD, 0):
            lat = lb.from_workload(w, streaming=streaming, flags=flags)
            lat.map_particles()
            lat.step(3)
            lat.step(1)                          # emits sums nobody reduces ...
            lat.step(1)                          # ... which must not be added to these
            res.append(lat.reduce_particle_forces())
            if not flags:
                with pytest.raises(lb.LbmimbError) as ei:
                    lat.fetch_fields(lb.FIELD_S)
                assert ei.value.status == lb.ESTATE
            lat.close()
    for F, T in res[1:]:
        assert np.array_equal(F, res[0][0]) and np.array_equal(T, res[0][1])
    assert_forces_close(res[0][0], res[0][1], ref)


def test_particle_limit_is_24_bits(lb):
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(2, (16, 16), (0, 0), 0.8, (0, 0), 8, max_particles=(1 << 24) + 1)
    assert ei.value.status == lb.EINVAL


def test_device_side_overflow_surfaces_in_every_synchronous_call_and_clears(orc, lb):
    """12 coincident disks of radius 110 put ~11 x 38,000 entries on the list of shared nodes of a 1024 x 1024
    lattice (capacity N/4 + 65536): the overflow is raised by the map kernel and must come back as ESTATE from
    the calls that synchronise, not as a wrong map; a valid particle set afterwards clears it."""
    n, P = (1024, 1024), 12
    lat = lb.Lattice(2, n, (0, 0), 0.8, (0, 0), 8, max_particles=P)
    pos = np.full((2, P), 500.25)
    lat.set_particles(pos, np.zeros((2, P)), None, np.full(P, 110.0), np.ones(P))
    lat.map_particles()
    for call in (lambda: lat.fetch_fields(lb.FIELD_EPS_CNT, (0, 0, 0), (8, 8, 1)), lat.get_particles, lat.synchronize,
                 lat.diagnostics):
        with pytest.raises(lb.LbmimbError) as ei:
            call()
        assert ei.value.status == lb.ESTATE and "overflow" in str(ei.value)
    lat.step(1)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.reduce_particle_forces()
    assert ei.value.status == lb.ESTATE
    pos2 = np.array([[100.5, 400.25], [300.0, 700.75]])
    rad2 = np.array([20.0, 30.5])
    lat.set_particles(pos2, np.zeros((2, 2)), None, rad2, np.ones(2))
    lat.map_particles()
    eo, po = orc.map_particles(2, n, (0, 0), 8, pos2, rad2)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT)[0], eo[0])
    assert np.array_equal(lat.fetch_fields(lb.FIELD_PID)[0], po[0])
    lat.synchronize()
    lat.close()


def test_set_particles_dev_rejects_bad_input_without_touching_the_handle(orc, lb):
    import torch
    w = inputs.reduced("C2")
    lat = lb.from_workload(w)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    bad_pos = w.pos.copy()
    bad_pos[1, 7] = w.n[1] + 3.0                                   # outside the domain
    bad_mass = w.mass.copy()
    bad_mass[3] = 0.0
    for p_, m_ in ((bad_pos, w.mass), (w.pos, bad_mass)):
        tp, tv, to, tr, tm = dev(p_), dev(w.vel), dev(w.omega), dev(w.radius), dev(m_)
        with pytest.raises(lb.LbmimbError) as ei:
            lat.set_particles_dev(w.P, tp.data_ptr(), tv.data_ptr(), to.data_ptr(), tr.data_ptr(), tm.data_ptr())
        assert ei.value.status == lb.EINVAL
    pg, vg, og = lat.get_particles()                              # still the set from_workload installed
    assert np.array_equal(pg, w.pos) and np.array_equal(vg, w.vel)
    lat.map_particles()
    eo, po = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, w.pos, w.radius)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eo)
    lat.close()


@pytest.mark.parametrize("n,region,rlo,rhi", [((420, 380), None, 0.8, 2.0), ((1600, 1500), 300.0, 0.3, 0.5)])
def test_dem_large_set_thread_per_particle_path_against_oracle(orc, lb, n, region, rlo, rhi):
    """More than 16,384 particles: the DEM step takes its thread-per-particle kernels (smaller sets: a warp per
    particle).  20,000 overlapping disks, walls in x and a periodic seam in y, against the oracle's all-pairs step.
    First case: the single-block cell-list kernel (4,410 cells); second case: small disks crowded into a corner of
    a large lattice, 284,000 cells, i.e. the multi-kernel counting sort inside the DEM step."""
    rng = np.random.default_rng(12)
    dim, bc, P = 2, (1, 0), 20000
    if region is None:
        pos = rng.random((dim, P)) * (np.array(n)[:, None] - 6.0) + 2.5
    else:
        pos = rng.random((dim, P)) * region + np.array([[1.0], [n[1] - region / 2]])     # across the y seam
        pos[1] = np.mod(pos[1], n[1])
    vel = rng.uniform(-0.02, 0.02, size=(dim, P))
    om = rng.uniform(-1e-3, 1e-3, size=(1, P))
    radius = rlo + (rhi - rlo) * rng.random(P)
    mass = 50.0 + 100.0 * rng.random(P)
    kn, e, gp = 3.0, 0.85, (1e-4, -2e-4)
    lat = lb.Lattice(dim, n, bc, 0.8, (0, 0), 8, max_particles=P)
    lat.set_particles(pos, vel, om, radius, mass)
    z, zt = np.zeros((dim, P)), np.zeros((1, P))
    p_o, v_o, o_o = pos, vel, om
    for _ in range(4):
        lat.dem_step(kn, e, gp, 1.0)
        p_o, v_o, o_o = orc.dem_step(dim, n, bc, p_o, v_o, o_o, radius, mass, z, zt, kn, e, gp, 1.0)
    p_g, v_g, o_g = lat.get_particles()
    fc = orc.contact_forces(dim, n, bc, p_o, v_o, radius, mass, kn, e)
    assert (np.abs(fc).max(axis=0) > 0).sum() > P // 4          # contacts are really exercised
    assert np.abs(p_g - p_o).max() < 1e-11
    assert np.abs(v_g - v_o).max() < 1e-12 * max(1.0, np.abs(v_o).max() / 1e-2)
    assert np.array_equal(o_g, o_o)
    lat.close()
