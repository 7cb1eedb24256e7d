"""BASELINE.json's configurations run in FULL (whole lattice, the stated number of steps), CUDA path against
the CPU oracle element by element.  `-m gpu`, and opt-in: the oracle needs tens of minutes per configuration
(DESIGN.md section 14), so these run only with

    LBMIMB_FULL=C2,C3,C4,C5 [LBMIMB_FULL_WINDOWS=k] [LBMIMB_FULL_STEPS=n] python -m pytest tests/test_gpu_full_protocol.py -m gpu -s

Each test appends one JSON line with what it measured to gpurun_out/full_protocol.jsonl (if that folder
exists).  Tolerances: tests/parity_util.py (north star).  No expected value comes from the CUDA path."""
import json
import os
import time

import numpy as np
import pytest

from paper_1011_2613_b200 import inputs
from parity_util import F_TOL, assert_fields_close, assert_forces_close, force_floor, gpu_run, oracle_run

pytestmark = [pytest.mark.gpu, pytest.mark.slow]
WANTED = [s for s in os.environ.get("LBMIMB_FULL", "").split(",") if s]
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def need(name):
    if name not in WANTED:
        pytest.skip("full-protocol run of %s not requested (LBMIMB_FULL=%s)" % (name, ",".join(WANTED)))


def record(**kw):
    out = os.path.join(ROOT, "gpurun_out")
    print(json.dumps(kw))
    if os.path.isdir(out):
        with open(os.path.join(out, "full_protocol.jsonl"), "a") as fh:
            fh.write(json.dumps(kw) + "\n")


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_fixed_particle_config_in_full(orc, lb, name):
    """BASELINE.json configs[1] / configs[2] / configs[3]: the whole lattice for the stated number of steps with the
    particles held fixed; f, rho, u, the maps and the per-particle force / torque are compared."""
    need(name)
    w = inputs.FULL[name]()
    steps = int(os.environ.get("LBMIMB_FULL_STEPS", w.steps))      # a cap, for a box with a time limit per call
    t0 = time.time()
    lat, g = gpu_run(lb, w, steps)
    t1 = time.time()
    ref = oracle_run(orc, w, steps)
    t2 = time.time()
    assert np.array_equal(g["eps"], ref["eps"]) and np.array_equal(g["pid"], ref["pid"])
    ef = assert_fields_close(g["f"], ref["f"], "f")
    assert_fields_close(g["rho"], ref["rho"], "rho")
    eu = np.abs(g["u"] - ref["u"]).max()
    assert eu <= F_TOL * max(1.0, np.abs(ref["u"]).max() / 1e-2)
    rF, rT = assert_forces_close(g["force"], g["torque"], ref)
    assert np.abs(ref["u"]).max() > 1e-4                           # the flow has developed
    record(config=name, lattice=list(w.n), particles=int(w.P), steps=steps, steps_of_config=int(w.steps), max_rel_f_err=float(ef),
           max_abs_u_err=float(eu), force_worst_ratio_of_tolerance=rF, torque_worst_ratio_of_tolerance=rT,
           gpu_seconds=round(t1 - t0, 2), oracle_seconds=round(t2 - t1, 1), oracle_threads=orc.num_threads())
    lat.close()


def test_c5_coupled_in_full(orc, lb):
    """BASELINE.json configs[4]: 128 x 512 x 128, 4,096 spheres, map -> fused step -> force/torque reduction ->
    DEM step per step; the oracle leads and the CUDA path is set to its state at the start of every 100-step
    window and compared at the end of it.  LBMIMB_FULL_WINDOWS limits the number of windows (default: all 20)."""
    need("C5")
    w = inputs.c5()
    d = w.dem
    win = 100
    nwin = int(os.environ.get("LBMIMB_FULL_WINDOWS", w.steps // win))
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P)
    for k in range(nwin):
        t0 = time.time()
        lat.set_distributions(f)
        lat.set_particles(pos, vel, om, w.radius, w.mass)
        worst_f = 0.0
        for it in range(win):
            eps, pid = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, pos, w.radius)
            f, s = orc.step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, eps_cnt=eps, pid=pid, pos=pos,
                            vel=vel, omega=om, want_s=True)
            F, T, aF, aT = orc.forces(w.dim, w.n, w.bc, s, pid, pos)
            pos, vel, om = orc.dem_step(w.dim, w.n, w.bc, pos, vel, om, w.radius, w.mass, F, T, d["kn"],
                                        d["restitution"], d["g_particle"], d["dt"])
            lat.map_particles()
            lat.step(1)
            if it % 25 == 24 or it == 0:                     # forces and maps inside the window as well
                assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), eps)
                assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), pid)
                gF, gT = lat.reduce_particle_forces()
                ref = dict(force=F, torque=T, abs_f=aF, abs_t=aT, floor=force_floor(pid, w.P), radius=w.radius)
                worst_f = max(worst_f, assert_forces_close(gF, gT, ref)[0])
            else:
                lat.reduce_particle_forces(to_host=False)
            lat.dem_step(d["kn"], d["restitution"], d["g_particle"], d["dt"])
        ef = assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = lat.get_particles()
        ex = np.abs(pg - pos).max()
        ev = np.abs(vg - vel).max() / np.abs(vel).max()
        assert ex < 1e-10 and ev <= 1e-10
        assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
        record(config="C5", window=k, steps=[k * win, (k + 1) * win], max_rel_f_err=float(ef), max_abs_x_err=float(ex),
               max_rel_v_err=float(ev), force_worst_ratio_of_tolerance=worst_f, max_speed=float(np.abs(vel).max()),
               seconds=round(time.time() - t0, 1), oracle_threads=orc.num_threads())
    lat.close()
