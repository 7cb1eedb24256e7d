"""GPU-vs-oracle parity of the TABLE mapping mode (NEXT-1: the paper's own eps method, PAPER.md:71-77
eq. (6), discretisation DESIGN.md R17) through the C-ABI.  `-m gpu` only.  The table, the code map and
the particle-id map are integer work: bit-exact.  Fields and forces: the tolerances of parity_util."""
import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import F_TOL, assert_fields_close, assert_forces_close, force_floor

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def _lattice(lb, dim, n, bc, pos, radius, tau=0.8):
    P = pos.shape[1]
    lat = lb.Lattice(dim, n, bc, tau, (0,) * dim, 8 if dim == 2 else 4, max_particles=P)
    lat.set_mapping_mode(lb.MAP_TABLE)
    lat.set_particles(pos, np.zeros((dim, P)), None, radius, np.ones(P))
    return lat


@pytest.mark.parametrize("dim,R", [(2, 4.0), (2, 6.0), (2, 1.0), (3, 4.0), (3, 5.0), (3, 2.37)])
def test_table_is_bit_exact(orc, lb, dim, R):
    n = (32, 32) if dim == 2 else (24, 24, 24)
    lat = _lattice(lb, dim, n, (0,) * dim, np.full((dim, 1), 12.3), np.array([R]))
    tab = lat.fetch_eps_table()
    ref = orc.eps_table(dim, R)
    assert tab.shape == ref.shape and lb.TABLE_SHAPE[dim] == ref.shape
    assert np.array_equal(tab, ref), "%d table entries differ" % (tab != ref).sum()
    lat.close()


@pytest.mark.parametrize("dim", [2, 3])
def test_table_map_overlapping_seam_walls(orc, lb, dim):
    """Shared nodes (touching and overlapping particles, identical centres -> tie), particles across
    the periodic seam and next to walls, centres that are not multiples of 2^-16."""
    rng = np.random.default_rng(300 + dim)
    n = (67, 45) if dim == 2 else (35, 22, 27)
    bc = (0, 1) if dim == 2 else (0, 1, 0)
    P = 40
    R = 3.3
    pos = rng.random((dim, P)) * np.array(n)[:, None]
    pos[:, 1] = pos[:, 0] + 0.37
    pos[:, 2] = pos[:, 3]
    pos[0, 4] = 0.01
    pos[0, 5] = n[0] - 0.3
    pos[:, 7] = pos[:, 6] + np.array([2 * R + 0.3, 0.0, 0.0])[:dim]          # touching pair: codes add
    for a in range(dim):
        pos[a] = np.clip(pos[a], 0.0, n[a] - 1.0) if bc[a] else np.mod(pos[a], n[a])
    radius = np.full(P, R)
    lat = _lattice(lb, dim, n, bc, pos, radius)
    lat.map_particles()
    e, p = lat.fetch_fields(lb.FIELD_EPS_CNT), lat.fetch_fields(lb.FIELD_PID)
    lat.synchronize()
    eo, po = orc.map_particles_table(dim, n, bc, pos, radius)
    assert np.array_equal(e, eo), "codes differ at %d nodes" % (e != eo).sum()
    assert np.array_equal(p, po), "pid differs at %d nodes" % (p != po).sum()
    assert e.max() == 255 and (p >= 0).sum() > 50
    lat.close()


def test_table_map_box_wider_than_the_periodic_domain(orc, lb):
    for dim, n, c, R in ((2, (9, 7), (4.2, 3.3), 5.5), (3, (6, 5, 7), (3.1, 2.2, 3.3), 4.0)):
        pos = np.array(c).reshape(dim, 1)
        lat = _lattice(lb, dim, n, (0,) * dim, pos, np.array([R]))
        lat.map_particles()
        eo, po = orc.map_particles_table(dim, n, (0,) * dim, pos, np.array([R]))
        assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eo)
        assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), po)
        lat.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_reduced_configs_in_table_mode(orc, lb, name):
    """The fixed-particle runs of the reduced configurations with the table map: maps bit-exact,
    fields <= 1e-12, forces <= 1e-10 (eps = code/255 in beta on both sides)."""
    w = inputs.reduced(name)
    steps = min(w.steps, 20)
    eps, pid = orc.map_particles_table(w.dim, w.n, w.bc, w.pos, w.radius)
    f = orc.init(w.dim, w.n)
    for it in range(steps):
        f, s = orc.step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, eps_cnt=eps, pid=pid, pos=w.pos,
                        vel=w.vel, omega=w.omega, want_s=True, eps_den=orc.TABLE_DEN)
    F, T, aF, aT = orc.forces(w.dim, w.n, w.bc, s, pid, w.pos)
    lat = lb.from_workload(w, map_mode=lb.MAP_TABLE, flags=lb.FLAG_EXCHANGE_FIELD)
    lat.map_particles()
    lat.step(steps)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eps)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), pid)
    assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
    assert np.abs(lat.fetch_fields(lb.FIELD_S) - s).max() <= F_TOL * np.abs(f).max()
    gF, gT = lat.reduce_particle_forces()
    ref = dict(force=F, torque=T, abs_f=aF, abs_t=aT, floor=force_floor(pid, w.P), radius=w.radius)
    assert_forces_close(gF, gT, ref)
    lat.close()


def test_mode_switch_and_errors(orc, lb):
    w = inputs.reduced("C2")
    lat = lb.from_workload(w)
    lat.map_particles()
    e_s = lat.fetch_fields(lb.FIELD_EPS_CNT)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.fetch_eps_table()                                  # sampling mode: no table
    assert ei.value.status == lb.ESTATE
    lat.set_mapping_mode(lb.MAP_TABLE)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.step(1)                                            # mode change invalidates the map
    assert ei.value.status == lb.ESTATE
    lat.map_particles()
    e_t = lat.fetch_fields(lb.FIELD_EPS_CNT)
    assert np.array_equal(e_t, orc.map_particles_table(w.dim, w.n, w.bc, w.pos, w.radius)[0])
    # the two methods describe the same solids: the coverage agrees to the accuracy of either
    assert abs(e_t.sum() / 255.0 - e_s.sum() / 64.0) / (e_s.sum() / 64.0) < 5e-3
    lat.set_mapping_mode(lb.MAP_SAMPLING)
    lat.map_particles()
    assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), e_s)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.set_mapping_mode(7)
    assert ei.value.status == lb.EINVAL
    # two radii: the table is for "a solid particle with a given radius"
    lat.set_mapping_mode(lb.MAP_TABLE)
    rad = w.radius.copy()
    rad[0] += 0.5
    lat.set_particles(w.pos, w.vel, w.omega, rad, w.mass)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.map_particles()
    assert ei.value.status == lb.ESTATE
    lat.close()
