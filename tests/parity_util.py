"""Shared helpers of the GPU parity tests: run the CPU oracle and the CUDA path on the same seeded
workload and compare them with the tolerances BASELINE.json's north_star states:
  lattice runs : max |f_gpu - f_cpu| <= 1e-12 * max |f|
  forces/torque: |F_gpu - F_cpu| <= 1e-10 * max(|F_cpu|, 1e-3 * A_p)      (R12; A_p = sum_n |s_n| of particle p;
                 torque: A_p = sum |r x s|).  The oracle forms the exchange vectors and the per-particle sums in
                 long double, so it is itself far inside 1e-10.  The plain bound is tried first.  Where it is
                 exceeded, the rounding floor of f decides: both sides carry f to ~2^-53 max|f| per step, which the
                 north star's own field tolerance lets grow to 1e-12 max|f|; the velocity of a node is therefore
                 only known to ~1e-15, and a sum of beta rho (V_S - u) over the n_p nodes of a particle to
                 n_p * 1e-15 (torque: times the lever arm R_p + 1) -- which exceeds 1e-13 A_p whenever the slip
                 velocity is below ~1e-2 and the sum cancels (the torque on a non-rotating particle, a suspension
                 at rest).  Every result records which bound was used and the ratio to the plain one.
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
    """Rounding floor of a per-particle sum: f carries rounding noise of ~2^-53 max|f| per step on both sides,
    so the velocity of a node is only known to ~1e-15 and a sum of beta rho (V_S - u) over the n_p nodes of
    particle p to n_p * 1e-15 (module text)."""
    n_p = np.bincount(pid[pid >= 0].ravel(), minlength=P).astype(float)
    return 1e-15 * n_p


class ForceCheck(tuple):
    """(force ratio, torque ratio) of the worst particle against the asserted bound (with the floor where it was
    needed), plus .no_floor = the same two ratios against the plain R12 bound (no additive term), .used_floor =
    (bool, bool) whether the plain bound was exceeded and the floor decided, and .rel = worst |dF|/|F|, |dT|/|T|
    over the particles whose |F| (|T|) is above 1e-3 A_p."""
    def __new__(cls, rF, rT, no_floor, used_floor, rel):
        self = super().__new__(cls, (rF, rT))
        self.no_floor, self.used_floor, self.rel = no_floor, used_floor, rel
        return self


def assert_forces_close(gF, gT, ref, tol=FORCE_TOL, floor=True):
    """R12: per particle |dF| <= tol * max(|F|, 1e-3 * sum_n |s_n|), same for the torque with sum |r x s|.
    If (and only if) that plain bound is exceeded and floor=True, the bound with the rounding floor of f,
    + n_p * 1e-15 (torque: times R_p + 1), decides; the result says which bound was used."""
    F, T, aF, aT = ref["force"], ref["torque"], ref["abs_f"], ref["abs_t"]
    dF = np.sqrt(((gF - F) ** 2).sum(axis=0))
    nF = np.sqrt((F ** 2).sum(axis=0))
    lim0 = tol * np.maximum(nF, 1e-3 * aF) + 1e-300
    dT = np.sqrt(((gT - T) ** 2).sum(axis=0))
    nT = np.sqrt((T ** 2).sum(axis=0))
    limT0 = tol * np.maximum(nT, 1e-3 * aT) + 1e-300
    nfF, nfT = float((dF / lim0).max()), float((dT / limT0).max())
    rF, rT = nfF, nfT
    if floor and nfF > 1.0:
        rF = float((dF / (lim0 + ref["floor"])).max())
    if floor and nfT > 1.0:
        rT = float((dT / (limT0 + ref["floor"] * (ref["radius"] + 1.0))).max())
    assert rF <= 1.0, "force: worst ratio %.3e (%.3e without the floor)" % (rF, nfF)
    assert rT <= 1.0, "torque: worst ratio %.3e (%.3e without the floor)" % (rT, nfT)
    bigF, bigT = nF > 1e-3 * aF, nT > 1e-3 * aT
    rel = (float((dF[bigF] / nF[bigF]).max()) if bigF.any() else 0.0,
           float((dT[bigT] / nT[bigT]).max()) if bigT.any() else 0.0)
    return ForceCheck(rF, rT, (nfF, nfT), (nfF > 1.0, nfT > 1.0), rel)


def gpu_run(lb, w, steps, f0=None, streaming=0, exchange_field=True):
    """Fixed-particle CUDA run through the C-ABI binding; returns (lattice, dict).
    streaming: lb.STREAM_AB (0) or lb.STREAM_AA (1).  exchange_field: create the lattice with
    LBMIMB_FLAG_EXCHANGE_FIELD so that the per-node exchange vectors can be fetched and compared
    (the full-size runs switch it off: it is a diagnostic output, the forces do not need it)."""
    lat = lb.from_workload(w, streaming=streaming, flags=lb.FLAG_EXCHANGE_FIELD if exchange_field else 0)
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
        if exchange_field:
            out["s"] = lat.fetch_fields(lb.FIELD_S)
        out["force"], out["torque"] = lat.reduce_particle_forces()
    lat.synchronize()
    return lat, out
