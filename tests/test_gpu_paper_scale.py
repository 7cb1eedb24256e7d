"""GPU-vs-oracle parity of the NEXT-2 pieces (`-m gpu`): the paper-parameter suspensions P2D / P3D
(Table 2; reduced cuts here, full size in test_gpu_fullsize.py) run as coupled
LBM-IMB-DEM windows, and the suspension diagnostics of Figs. 5/7 (lbmimb_diagnostics, R18).
"""
import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import assert_fields_close, assert_forces_close, force_floor, gpu_run, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def assert_diag_close(got, ref, nodes, P, fscale, vscale):
    """Sums of N terms, reduced in different orders, of fields that agree to 1e-12 * max|f| (u = sum f c / rho
    cancels f-sized terms, so its rounding scale is that of f: `fscale` = max(|f|, |u|), as for u in
    test_gpu_parity): |diff| <= 1e-12 * N * scale; the averaged entries divide that by the weight sum."""
    g, r = got["vector"], ref["vector"]
    assert abs(g[0] - r[0]) <= 1e-12 * nodes and abs(g[1] - r[1]) <= 1e-12 * nodes
    assert np.abs(g[2:5] - r[2:5]).max() <= 1e-12 * max(fscale, np.abs(r[2:5]).max())
    assert np.abs(g[14:17] - r[14:17]).max() <= 1e-12 * nodes * fscale
    if P:
        assert np.abs(g[5:8] - r[5:8]).max() <= 1e-12 * vscale
        assert np.abs(g[8:11] - r[8:11]).max() <= 1e-12 * max(vscale, fscale)
        assert np.abs(g[17:20] - r[17:20]).max() <= 1e-12 * np.abs(r[17:20]).max() + 1e-12 * P * vscale * got["mscale"]
        assert np.abs(g[11:14] - r[11:14]).max() <= got["fptol"]     # mean of the per-particle force tolerances (R12)


@pytest.mark.parametrize("name,streaming", [("C2", 0), ("C3", 1), ("C1", 1), ("P2D", 0), ("P3D", 1)])
def test_diagnostics_match_the_oracle(orc, lb, name, streaming):
    w = inputs.reduced(name)
    steps = 9
    ref = oracle_run(orc, w, steps)
    lat, got = gpu_run(lb, w, steps, streaming=streaming)
    d_ref = orc.diagnostics(w.dim, ref["f"], ref["eps"], w.subsamples ** w.dim, w.vel, w.radius, w.mass, ref["force"])
    d = lat.diagnostics()
    d["mscale"] = float(w.mass.max())
    nF = np.sqrt((ref["force"] ** 2).sum(axis=0))
    d["fptol"] = float((1e-10 * np.maximum(nF, 1e-3 * ref["abs_f"]) + ref["floor"]).mean())
    fscale = float(max(np.abs(ref["f"]).max(), np.abs(ref["u"]).max()))
    assert_diag_close(d, d_ref, w.nodes, w.P, fscale, float(np.abs(w.vel).max()) + 1e-30)
    again = lat.diagnostics()
    assert np.array_equal(again["vector"], d["vector"])              # deterministic reduction
    lat.close()


def test_diagnostics_without_particles_and_in_table_mode(orc, lb):
    rng = np.random.default_rng(8)
    n = (37, 21, 9)
    _, wq, _ = orc.velocity_set(3)
    f0 = wq.reshape((-1, 1, 1, 1)) * (1 + 0.05 * rng.standard_normal((19, 9, 21, 37)))
    lat = lb.Lattice(3, n, (0, 1, 0), 0.7, (0, 0, 0), 4)
    lat.set_distributions(f0)
    d = lat.diagnostics()
    r = orc.diagnostics(3, f0)
    assert d["gas_area"] == 37 * 21 * 9 and abs(d["mass"] - r["mass"]) < 1e-10
    assert np.abs(d["gas_velocity"] - r["gas_velocity"]).max() < 1e-13
    assert np.abs(d["fluid_momentum"] - r["fluid_momentum"]).max() < 1e-10
    assert np.all(d["vector"][5:8] == 0) and np.all(d["vector"][11:14] == 0) and np.all(d["vector"][17:] == 0)
    lat.close()
    # table mode: eps = code / 255
    w = inputs.reduced("C2")
    lat = lb.from_workload(w, map_mode=lb.MAP_TABLE)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.diagnostics()                                            # particles set, not mapped
    assert ei.value.status == lb.ESTATE
    lat.map_particles()
    lat.step(4)
    code = lat.fetch_fields(lb.FIELD_EPS_CNT)
    d = lat.diagnostics()
    r = orc.diagnostics(2, lat.fetch_fields(lb.FIELD_F), code, 255, w.vel, w.radius, w.mass)
    assert abs(d["gas_area"] - r["gas_area"]) < 1e-9 and np.abs(d["gas_velocity"] - r["gas_velocity"]).max() < 1e-15
    lat.close()


@pytest.mark.parametrize("name,streaming", [("P2D", 0), ("P2D", 1), ("P3D", 1), ("P3D", 0)])
def test_paper_suspension_coupled_windows(orc, lb, name, streaming):
    """C5 protocol on the reduced paper suspensions (fully periodic, Table 2 parameters, t_c = 10 steps):
    the oracle leads, the CUDA path is set to its state at each window start, both run `win` coupled steps."""
    w = inputs.reduced(name)
    d = w.dem
    win, nwin = 6, 3
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P, streaming=streaming)
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
        assert np.abs(vg - vel).max() <= 1e-10 * np.abs(vel).max()
        assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
        # diagnostics of the coupled state
        lat.map_particles()
        eps, pid = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, pos, w.radius)
        dg = lat.diagnostics()
        dr = orc.diagnostics(w.dim, f, eps, w.subsamples ** w.dim, vel, w.radius, w.mass, ref["force"])
        assert np.abs(dg["slip"] - dr["slip"]).max() <= 1e-10 * np.abs(dr["slip"]).max() + 1e-12 * np.abs(f).max()
        assert np.abs(dg["drag"] - dr["drag"]).max() <= 1e-10 * np.abs(dr["drag"]).max() + float((1e-10 * 1e-3 * ref["abs_f"] + ref["floor"]).mean())
    lat.close()
