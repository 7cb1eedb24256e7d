"""Shared helpers of the GPU parity tests: run the CPU oracle and the CUDA path on
the same seeded workload and compare them with the tolerances BASELINE.json's
north_star states:
  lattice runs : max |f_gpu - f_cpu| <= 1e-12 * max |f|
  forces/torque: |F_gpu - F_cpu| <= 1e-10 * max(|F_cpu|, 1e-3 * A_p) + n_p * 1e-15   (R12)
                 (torque: the same with A_p = sum |r x s| and the floor times (R_p + 1))
  eps / pid    : bit-exact
"""
import numpy as np

F_TOL = 1e-12
FORCE_TOL = 1e-10


def oracle_run(orc, w, steps, f0=None, pos=None, vel=None, omega=None):
    """Fixed-particle oracle run: returns dict(f, rho, u, s, eps, pid, force, torque, abs_f, abs_t)."""
    pos = w.pos if pos is None else pos
    vel = w.vel if vel is None else vel
    omega = w.omega if omega is None else omega
    out = {}
    part = {}
    if pos.shape[1] > 0:
        eps, pid = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, pos, w.radius)
        part = dict(eps_cnt=eps, pid=pid, pos=pos, vel=vel, omega=omega)
        out["eps"], out["pid"] = eps, pid
    f = orc.init(w.dim, w.n) if f0 is None else f0
    s = None
    for it in range(steps):
        if it == steps - 1 and part:
            f, s = orc.step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, want_s=True, **part)
        else:
            f = orc.step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, **part)
    out["f"] = f
    out["rho"], out["u"] = orc.macros(w.dim, f)
    if s is not None:
        out["s"] = s
        out["force"], out["torque"], out["abs_f"], out["abs_t"] = orc.forces(w.dim, w.n, w.bc, s, out["pid"], pos)
        out["floor"] = force_floor(out["pid"], pos.shape[1])
        out["radius"] = w.radius
    return out


def assert_fields_close(gpu_f, cpu_f, what="f", tol=F_TOL):
    scale = np.abs(cpu_f).max()
    err = np.abs(gpu_f - cpu_f).max()
    assert err <= tol * scale, "%s: max abs diff %.3e > %.1e * %.3e" % (what, err, tol, scale)
    return err / scale


def force_floor(pid, P):
    """Absolute rounding floor of a per-particle sum of exchange vectors: the oracle's literal
    sum_i Omega_i c_i cancels f-sized terms (|f| <= 0.45), so each node's s carries an absolute
    rounding error of up to ~Q * 2^-53 * max|f| ~ 1e-15 whatever the size of s itself; a sum over
    the n_p nodes of particle p cannot be trusted below n_p * 1e-15."""
    n_p = np.bincount(pid[pid >= 0].ravel(), minlength=P).astype(float)
    return 1e-15 * n_p


def assert_forces_close(gF, gT, ref, tol=FORCE_TOL):
    """R12: per particle, |dF| <= tol * max(|F|, 1e-3 * sum_n |s_n|) + n_p * 1e-15; same for the torque
    with the floor scaled by the lever arm (R_p + 1)."""
    F, T, aF, aT = ref["force"], ref["torque"], ref["abs_f"], ref["abs_t"]
    floor = ref["floor"]
    dF = np.sqrt(((gF - F) ** 2).sum(axis=0))
    nF = np.sqrt((F ** 2).sum(axis=0))
    lim = tol * np.maximum(nF, 1e-3 * aF) + floor
    assert (dF <= lim + 1e-300).all(), "force: worst ratio %.3e" % (dF / (lim + 1e-300)).max()
    dT = np.sqrt(((gT - T) ** 2).sum(axis=0))
    nT = np.sqrt((T ** 2).sum(axis=0))
    limT = tol * np.maximum(nT, 1e-3 * aT) + floor * (ref["radius"] + 1.0)
    assert (dT <= limT + 1e-300).all(), "torque: worst ratio %.3e" % (dT / (limT + 1e-300)).max()
    return float((dF / (lim + 1e-300)).max()), float((dT / (limT + 1e-300)).max())


def gpu_run(lb, w, steps, f0=None, streaming=0):
    """Fixed-particle CUDA run through the C-ABI binding; returns (lattice, dict).
    streaming: lb.STREAM_AB (0) or lb.STREAM_AA (1)."""
    lat = lb.from_workload(w, streaming=streaming)
    if f0 is not None:
        lat.set_distributions(f0)
    if w.P:
        lat.map_particles()
    lat.step(steps)
    out = {"f": lat.fetch_fields(lb.FIELD_F), "rho": lat.fetch_fields(lb.FIELD_RHO),
           "u": lat.fetch_fields(lb.FIELD_U)}
    if w.P:
        out["eps"] = lat.fetch_fields(lb.FIELD_EPS_CNT)
        out["pid"] = lat.fetch_fields(lb.FIELD_PID)
        out["s"] = lat.fetch_fields(lb.FIELD_S)
        out["force"], out["torque"] = lat.reduce_particle_forces()
    lat.synchronize()
    return lat, out
