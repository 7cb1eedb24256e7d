"""GPU-vs-oracle parity of the in-place AA-pattern streaming mode (LBMIMB_STREAM_AA) through the
C-ABI.  `-m gpu` only.  The oracle is the same two-buffer definition of eq. (1):
the streaming scheme is an implementation choice that must not change the result beyond rounding.
Odd AND even step counts are compared because the stored array alternates between two layouts.
"""
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


@pytest.mark.parametrize("name,steps", [("C1", 100), ("C1", 7), ("C2", 20), ("C2", 21), ("C3", 10), ("C3", 11),
                                        ("C4", 9), ("C4", 10), ("C5", 5), ("C5", 6)])
def test_aa_reduced_configs_fields_maps_forces(orc, lb, name, steps):
    w = inputs.reduced(name)
    ref = oracle_run(orc, w, steps)
    lat, got = gpu_run(lb, w, steps, streaming=lb.STREAM_AA)
    assert np.array_equal(got["eps"], ref["eps"]) and np.array_equal(got["pid"], ref["pid"])
    assert_fields_close(got["f"], ref["f"], "f")
    assert_fields_close(got["rho"], ref["rho"], "rho")
    assert np.abs(got["u"] - ref["u"]).max() <= F_TOL * max(np.abs(ref["f"]).max(), np.abs(ref["u"]).max())
    assert np.abs(got["s"] - ref["s"]).max() <= F_TOL * np.abs(ref["f"]).max()
    assert_forces_close(got["force"], got["torque"], ref)
    assert lat.time() == steps
    lat.close()


@pytest.mark.parametrize("dim,n,bc", [(2, (130, 7), (0, 0)), (2, (257, 5), (1, 1)), (2, (3, 4), (1, 0)),
                                      (3, (129, 5, 4), (0, 1, 0)), (3, (6, 5, 3), (1, 1, 1)),
                                      (3, (2, 2, 2), (0, 0, 0)), (2, (1, 1), (0, 0)), (3, (1, 3, 1), (0, 1, 0)),
                                      (3, (2, 1, 2), (1, 0, 1)), (2, (2, 2), (1, 1))])
def test_aa_pure_lbgk_random_state(orc, lb, dim, n, bc):
    """Walls on every axis combination, periodic seams, degenerate 1- and 2-node axes (where a node is
    its own neighbour and the in-place update must still be a permutation), two tiles per row."""
    rng = np.random.default_rng(6)
    _, wq, _ = orc.velocity_set(dim)
    shape = (len(wq),) + tuple(reversed(tuple(n) + (1,) * (3 - len(n))))
    f0 = wq.reshape((-1, 1, 1, 1)) * (1 + 0.05 * rng.standard_normal(shape))
    g = (1e-5, -2e-5, 3e-5)[:dim]
    lat = lb.Lattice(dim, n, bc, 0.63, g, 8 if dim == 2 else 4, streaming=lb.STREAM_AA)
    lat.set_distributions(f0)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_F), f0)
    f = f0
    done = 0
    for nst in (1, 1, 5, 4):          # compare in both layouts (after odd and even totals)
        for _ in range(nst):
            f = orc.step(dim, n, bc, 0.63, g, 8, f)
        lat.step(nst)
        done += nst
        assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        rho, u = orc.macros(dim, f)
        assert_fields_close(lat.fetch_fields(lb.FIELD_RHO), rho, "rho")
        assert np.abs(lat.fetch_fields(lb.FIELD_U) - u).max() < 1e-13
    # set_distributions in the swapped layout (odd total) must reset the layout
    assert done % 2 == 1
    lat.set_distributions(f0)
    assert np.array_equal(lat.fetch_fields(lb.FIELD_F), f0)
    lat.step(1)
    assert_fields_close(lat.fetch_fields(lb.FIELD_F), orc.step(dim, n, bc, 0.63, g, 8, f0))
    lat.close()


def test_aa_matches_ab_bitwise_and_halves_the_footprint(lb):
    """Both schemes run the same node arithmetic on the same values: identical bits, one array."""
    w = inputs.reduced("C3")
    la, ga = gpu_run(lb, w, 5, streaming=lb.STREAM_AA)
    lb_, gb = gpu_run(lb, w, 5, streaming=lb.STREAM_AB)
    for key in ("f", "s", "force", "torque", "eps", "pid"):
        assert np.array_equal(ga[key], gb[key]), key
    need_aa = lb.workspace_bytes(la.params, w.P)
    need_ab = lb.workspace_bytes(lb_.params, w.P)
    assert need_ab - need_aa >= w.Q * w.nodes * 8
    la.close()
    lb_.close()


def test_aa_sub_box_fetch_in_both_layouts(orc, lb):
    w = inputs.reduced("C3")
    for steps in (4, 5):
        lat, got = gpu_run(lb, w, steps, streaming=lb.STREAM_AA)
        lo, hi = (3, 70, 1), (72, 90, 30)
        sl = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        for what, key in ((lb.FIELD_F, "f"), (lb.FIELD_U, "u"), (lb.FIELD_S, "s")):
            assert np.array_equal(lat.fetch_fields(what, lo, hi), got[key][(slice(None),) + sl])
        for what, key in ((lb.FIELD_RHO, "rho"), (lb.FIELD_EPS_CNT, "eps"), (lb.FIELD_PID, "pid")):
            assert np.array_equal(lat.fetch_fields(what, lo, hi), got[key][sl])
        lat.close()


def test_aa_coupled_reduced_c5_windows(orc, lb):
    """C5 protocol (map -> step -> reduce -> dem, resynchronised per window) in AA mode, with an odd
    window length so that windows start in either layout before set_distributions resets it."""
    w = inputs.reduced("C5")
    d = w.dem
    win, nwin = 7, 3
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P, streaming=lb.STREAM_AA)
    for k in range(nwin):
        lat.set_distributions(f)
        lat.set_particles(pos, vel, om, w.radius, w.mass)
        for it in range(win):
            f, pos, vel, om, ref = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                    w.radius, w.mass, d["kn"], d["restitution"], d["g_particle"], d["dt"])
            eps, pid = ref["eps"], ref["pid"]
            ref.update(floor=force_floor(pid, w.P), radius=w.radius)
            lat.map_particles()
            lat.step(1)
            gF, gT = lat.reduce_particle_forces()
            assert_forces_close(gF, gT, ref)
            lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])
        assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = lat.get_particles()
        assert np.abs(pg - pos).max() < 1e-10
        assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max() + 1e-18
    lat.close()


def test_aa_rejects_bad_streaming_value(lb):
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(2, (16, 16), (0, 0), 0.8, (0, 0), 8, streaming=7)
    assert ei.value.status == lb.EINVAL
