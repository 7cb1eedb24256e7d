"""BASELINE.json's configurations run in FULL (whole lattice, the stated number of steps), CUDA path against
the CPU oracle element by element.  `-m gpu`, and opt-in: the oracle needs tens of minutes per configuration
on the GPU box's 16 host threads and one call on the box is limited to an hour, so these run only with

    LBMIMB_FULL=C2,C3,C4,C5 python -m pytest tests/test_gpu_full_protocol.py -m gpu -s
      LBMIMB_FULL_STEPS=n        C2/C3/C4: cap of the step count (default: the configuration's)
      LBMIMB_FULL_SLAB=k/K       C4: compare the k-th of K y-slabs in this call (default: all K = 4, one after the other)
      LBMIMB_FULL_WINDOWS=a:b    C5: run windows a .. b-1 of the 20 (default 0:20)
      LBMIMB_FULL_CKPT=dir       C5: where the ORACLE's state (f, x, v, omega; 1.3 GB) at a window boundary is kept
                                 so that the next call continues the run (default <tmp>/lbmimb_ckpt)

C4 (268 M nodes, 37 s of oracle per step) is compared slab by slab: the CUDA path runs the WHOLE lattice for
the 200 steps; the oracle runs a y-slab of it (all of x, the rows to compare plus a rim of steps + 2R + 3 rows
on every side that is not a true wall, the same particles translated exactly: inputs.y_slab).  After n steps
the state of a node depends only on the initial state within n nodes of it, so inside the compared rows the
slab run IS the whole-lattice oracle run; K overlapping slabs cover every row and every particle.

C5 (coupled; the oracle leads): the oracle's state at the end of each window is written to the checkpoint
folder by THIS test from oracle arrays only; a later call reloads it and goes on.  If the checkpoint is
missing the oracle replays the earlier windows by itself.  The CUDA path is set from the oracle's state at
every window start, never the other way round.

Each test appends one JSON line per result to gpurun_out/full_protocol.jsonl (if that folder exists).
Tolerances: tests/parity_util.py (north star; forces against the plain R12 bound first, the ratio to it is recorded).  No expected value comes
from the CUDA path."""
import json
import os
import tempfile
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
    print(json.dumps(kw), flush=True)
    if os.path.isdir(out):
        with open(os.path.join(out, "full_protocol.jsonl"), "a") as fh:
            fh.write(json.dumps(kw) + "\n")


def force_fields(chk):
    """The per-particle force / torque result of assert_forces_close as record fields."""
    return dict(force_worst_ratio_of_tolerance=chk[0], torque_worst_ratio_of_tolerance=chk[1],
                force_worst_ratio_no_floor=chk.no_floor[0], torque_worst_ratio_no_floor=chk.no_floor[1],
                force_used_floor=bool(chk.used_floor[0]), torque_used_floor=bool(chk.used_floor[1]),
                force_worst_rel_err=chk.rel[0], torque_worst_rel_err=chk.rel[1])


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_fixed_particle_config_in_full(orc, lb, name):
    """BASELINE.json configs[1] / configs[2]: the whole lattice for the stated number of steps with the
    particles held fixed; f, rho, u, the maps and the per-particle force / torque are compared."""
    need(name)
    w = inputs.FULL[name]()
    steps = int(os.environ.get("LBMIMB_FULL_STEPS", w.steps))      # a cap, for a box with a time limit per call
    t0 = time.time()
    lat, g = gpu_run(lb, w, steps, exchange_field=False)
    t1 = time.time()
    ref = oracle_run(orc, w, steps)
    t2 = time.time()
    assert np.array_equal(g["eps"], ref["eps"]) and np.array_equal(g["pid"], ref["pid"])
    ef = assert_fields_close(g["f"], ref["f"], "f")
    assert_fields_close(g["rho"], ref["rho"], "rho")
    eu = np.abs(g["u"] - ref["u"]).max()
    assert eu <= F_TOL * max(1.0, np.abs(ref["u"]).max() / 1e-2)
    chk = assert_forces_close(g["force"], g["torque"], ref)
    assert np.abs(ref["u"]).max() > 1e-4                           # the flow has developed
    record(config=name, lattice=list(w.n), particles=int(w.P), steps=steps, steps_of_config=int(w.steps),
           max_rel_f_err=float(ef), max_abs_u_err=float(eu), gpu_seconds=round(t1 - t0, 2),
           oracle_seconds=round(t2 - t1, 1), oracle_threads=orc.num_threads(), version=lb.version(), **force_fields(chk))
    lat.close()


def slab_bounds(ny, k, K, overlap):
    """Rows [y0, y1) compared by slab k of K: equal parts of the lattice, widened by `overlap` rows on the inner
    sides so that every particle lies wholly inside some slab."""
    h = (ny + K - 1) // K
    return max(0, k * h - overlap), min(ny, (k + 1) * h + overlap)


def test_c4_in_full_by_slabs(orc, lb):
    """BASELINE.json configs[3]: 8192 x 32768 D2Q9, 1,166,400 disks, 200 steps.  See the module text."""
    need("C4")
    w = inputs.c4()
    steps = int(os.environ.get("LBMIMB_FULL_STEPS", w.steps))
    spec = os.environ.get("LBMIMB_FULL_SLAB", "")
    K = int(spec.split("/")[1]) if spec else 4
    todo = [int(spec.split("/")[0])] if spec else list(range(K))
    R = float(w.radius.max())
    rim = steps + int(2 * R) + 3
    nx, ny = w.n
    t0 = time.time()
    lat = lb.from_workload(w)
    lat.map_particles()
    lat.step(steps)
    gF, gT = lat.reduce_particle_forces()
    lat.synchronize()
    gpu_s = time.time() - t0
    for k in todo:
        y0, y1 = slab_bounds(ny, k, K, int(2 * R) + 6)
        lo, hi = max(0, y0 - rim), min(ny, y1 + rim)
        pos, vel, om, rad, mass, idx = inputs.y_slab(w, lo, hi)
        sub_n, sub_bc = (nx, hi - lo), (w.bc[0], 1)
        t1 = time.time()
        eps, pid = orc.map_particles(2, sub_n, sub_bc, w.subsamples, pos, rad)
        f = orc.init(2, sub_n)
        part = dict(eps_cnt=eps, pid=pid, pos=pos, vel=vel, omega=om)
        for it in range(steps - 1):
            f = orc.step(2, sub_n, sub_bc, w.tau, w.g_fluid, w.subsamples, f, **part)
        f, s = orc.step(2, sub_n, sub_bc, w.tau, w.g_fluid, w.subsamples, f, want_s=True, **part)
        t2 = time.time()
        rows = slice(y0 - lo, y1 - lo)
        box = ((0, y0, 0), (nx, y1, 1))
        assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT, *box)[0], eps[0, rows]), "eps_cnt"
        opid = np.where(pid >= 0, idx[np.maximum(pid, 0)], -1).astype(np.int32)
        assert np.array_equal(lat.fetch_fields(lb.FIELD_PID, *box)[0], opid[0, rows]), "pid"
        ef = assert_fields_close(lat.fetch_fields(lb.FIELD_F, *box)[:, 0], f[:, 0, rows], "f")
        rho, u = orc.macros(2, f)
        assert_fields_close(lat.fetch_fields(lb.FIELD_RHO, *box)[0], rho[0, rows], "rho")
        eu = np.abs(lat.fetch_fields(lb.FIELD_U, *box)[:, 0] - u[:, 0, rows]).max()
        assert eu <= F_TOL * max(1.0, np.abs(u[:, 0, rows]).max() / 1e-2)
        assert np.abs(u[:, 0, rows]).max() > 1e-4                                  # the flow has developed
        # particles that lie wholly inside the compared rows
        F, T, aF, aT = orc.forces(2, sub_n, sub_bc, s, pid, pos)
        gy = pos[1] + lo
        keep = ((gy - rad - 2 >= y0) | (y0 == 0)) & ((gy + rad + 2 <= y1 - 1) | (y1 == ny))   # true walls need no margin
        ref = dict(force=F[:, keep], torque=T[:, keep], abs_f=aF[keep], abs_t=aT[keep],
                   floor=force_floor(pid, pos.shape[1])[keep], radius=rad[keep])
        chk = assert_forces_close(gF[:, idx[keep]], gT[:, idx[keep]], ref)
        record(config="C4", lattice=list(w.n), particles=int(w.P), steps=steps, steps_of_config=int(w.steps),
               slab="%d/%d" % (k, K), rows_compared=[int(y0), int(y1)], oracle_rows=[int(lo), int(hi)],
               particles_compared=int(keep.sum()), max_rel_f_err=float(ef), max_abs_u_err=float(eu),
               gpu_seconds=round(gpu_s, 2), oracle_seconds=round(t2 - t1, 1), oracle_threads=orc.num_threads(),
               version=lb.version(), **force_fields(chk))
    lat.close()


def _ckpt_path(k):
    d = os.environ.get("LBMIMB_FULL_CKPT", os.path.join(tempfile.gettempdir(), "lbmimb_ckpt"))
    os.makedirs(d, exist_ok=True)
    return os.path.join(d, "c5_oracle_state_window_%02d.npz" % k)


def test_c5_coupled_in_full(orc, lb):
    """BASELINE.json configs[4]: 128 x 512 x 128, 4,096 spheres, map -> fused step -> force/torque reduction ->
    DEM step per step (oracle.coupled_step); the oracle leads and the CUDA path is set to its state at the start of
    every 100-step window and compared at the end of it (forces and maps at 5 steps inside the window too)."""
    need("C5")
    w = inputs.c5()
    d = w.dem
    win = 100
    spec = os.environ.get("LBMIMB_FULL_WINDOWS", "0:%d" % (w.steps // win))
    first, last = (int(v) for v in spec.split(":")) if ":" in spec else (0, int(spec))
    dargs = (d["kn"], d["restitution"], d["g_particle"], d["dt"])
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()
    start = 0
    for k in range(first, 0, -1):                     # newest oracle checkpoint at or before `first`
        if os.path.exists(_ckpt_path(k)):
            z = np.load(_ckpt_path(k))
            f, pos, vel, om, start = z["f"], z["pos"], z["vel"], z["omega"], k
            break
    for k in range(start, first):                     # no checkpoint: the oracle replays the windows by itself
        t0 = time.time()
        for it in range(win):
            f, pos, vel, om, _ = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                  w.radius, w.mass, *dargs)
        record(config="C5", window=k, oracle_only_replay=True, seconds=round(time.time() - t0, 1))
        np.savez(_ckpt_path(k + 1), f=f, pos=pos, vel=vel, omega=om)             # so that a later call need not replay
        if os.path.exists(_ckpt_path(k)):
            os.remove(_ckpt_path(k))
    lat = lb.Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, max_particles=w.P)
    for k in range(first, last):
        t0 = time.time()
        lat.set_distributions(f)
        lat.set_particles(pos, vel, om, w.radius, w.mass)
        worst = None
        for it in range(win):
            f, pos, vel, om, ref = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                    w.radius, w.mass, *dargs)
            lat.map_particles()
            lat.step(1)
            if it % 25 == 24 or it == 0:                     # forces and maps inside the window as well
                assert np.array_equal(lat.fetch_fields(lb.FIELD_EPS_CNT), ref["eps"])
                assert np.array_equal(lat.fetch_fields(lb.FIELD_PID), ref["pid"])
                gF, gT = lat.reduce_particle_forces()
                ref.update(floor=force_floor(ref["pid"], w.P), radius=w.radius)
                chk = assert_forces_close(gF, gT, ref)
                if worst is None or chk.no_floor[0] > worst.no_floor[0]:
                    worst = chk
            else:
                lat.reduce_particle_forces(to_host=False)
            lat.dem_step(*dargs)
        ef = assert_fields_close(lat.fetch_fields(lb.FIELD_F), f)
        pg, vg, og = lat.get_particles()
        ex = np.abs(pg - pos).max()
        ev = np.abs(vg - vel).max() / np.abs(vel).max()
        assert ex < 1e-10 and ev <= 1e-10
        assert np.abs(og - om).max() <= 1e-10 * np.abs(om).max() + 1e-18
        record(config="C5", window=k, steps=[k * win, (k + 1) * win], max_rel_f_err=float(ef), max_abs_x_err=float(ex),
               max_rel_v_err=float(ev), max_speed=float(np.abs(vel).max()), seconds=round(time.time() - t0, 1),
               oracle_threads=orc.num_threads(), version=lb.version(), **force_fields(worst))
        np.savez(_ckpt_path(k + 1), f=f, pos=pos, vel=vel, omega=om)             # oracle arrays only
        old = _ckpt_path(k)
        if os.path.exists(old):
            os.remove(old)
    lat.close()
