"""Pins of the oracle's suspension diagnostics (oracle.diagnostics; Figs. 5/7; R18)
and of the paper-parameter input recipes.  CPU only.  Every expected value is a closed form, an exact
rational written out by hand, an invariant of the dynamics, or a number the paper prints.
"""
import math

import numpy as np
import pytest

from paper_1011_2613_b200 import inputs


def _golden(name):
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, *v = line.split()
                out[k] = [float(x) for x in v]
    return out


@pytest.mark.parametrize("dim", [2, 3])
def test_uniform_equilibrium_gives_its_own_velocity_mass_and_momentum(orc, dim):
    n = (5, 4) if dim == 2 else (5, 4, 3)
    N = int(np.prod(n))
    u0 = np.array([0.01, -0.02, 0.03][:dim])
    feq = orc.feq(dim, 1.25, u0)
    f = np.broadcast_to(feq.reshape((-1, 1, 1, 1)), (len(feq),) + tuple(reversed(n + (1,) * (3 - dim)))).copy()
    d = orc.diagnostics(dim, f)
    assert d["gas_area"] == N
    assert abs(d["mass"] - 1.25 * N) < 1e-12
    assert np.abs(d["gas_velocity"] - u0).max() < 1e-16
    assert np.abs(d["fluid_momentum"] - 1.25 * N * u0).max() < 1e-13
    assert np.abs(d["slip"] - u0).max() < 1e-16 and np.all(d["drag"] == 0)


def test_gas_average_is_weighted_by_the_gas_fraction_exact_rational(orc):
    """4 nodes with eps = 16/64 moving at u1 = (0.04, 0) and 12 nodes with eps = 0 at u2 = (0.01, 0.02):
    U_g = (4 * 3/4 * u1 + 12 * u2) / (4 * 3/4 + 12) = (0.016, 0.016); A_g = 15."""
    f = np.empty((9, 1, 4, 4))
    eps = np.zeros((1, 4, 4), dtype=np.uint8)
    f[:] = orc.feq(2, 1.0, np.array([0.01, 0.02])).reshape(9, 1, 1, 1)
    f[:, 0, 1, :] = orc.feq(2, 0.9, np.array([0.04, 0.0])).reshape(9, 1)
    eps[0, 1, :] = 16
    d = orc.diagnostics(2, f, eps, 64)
    assert d["gas_area"] == 15.0
    assert np.abs(d["gas_velocity"] - np.array([0.016, 0.016])).max() < 1e-16
    # mass and momentum are NOT eps-weighted
    assert abs(d["mass"] - (12 + 4 * 0.9)) < 1e-14
    assert np.abs(d["fluid_momentum"] - np.array([12 * 0.01 + 3.6 * 0.04, 12 * 0.02])).max() < 1e-15


def test_solid_average_is_volume_weighted_and_slip_sign(orc):
    """Radii 1 and 2: areas 1:4, volumes 1:8.  v_1 = e_x, v_2 = e_y."""
    for dim, w2 in ((2, 4.0), (3, 8.0)):
        n = (3, 3) if dim == 2 else (3, 3, 3)
        f = orc.init(dim, n)
        vel = np.zeros((dim, 2))
        vel[0, 0] = 1.0
        vel[1, 1] = 1.0
        force = np.zeros((dim, 2))
        force[1] = [3.0, -1.0]
        d = orc.diagnostics(dim, f, None, 1, vel, np.array([1.0, 2.0]), np.array([2.0, 5.0]), force)
        vs = np.zeros(dim)
        vs[0], vs[1] = 1.0 / (1.0 + w2), w2 / (1.0 + w2)
        assert np.abs(d["solid_velocity"] - vs).max() < 1e-16
        assert np.abs(d["slip"] + vs).max() < 1e-16            # gas at rest: slip = U_g - V_s = -V_s
        assert d["drag"][1] == 1.0 and d["drag"][0] == 0.0     # mean force per particle
        sm = np.zeros(dim)
        sm[0], sm[1] = 2.0, 5.0
        assert np.array_equal(d["solid_momentum"], sm)


def test_uniform_porous_medium_closed_form_P5(orc):
    """SURVEY P5 (tests/golden/survey_closed_forms.txt): periodic, uniform eps = 0.3, V_S = 0, g_y = -1e-6,
    tau = 0.8, 50 steps -> u_y = (g/beta)(1 - (1-beta)^n).  The gas-averaged velocity must be that value."""
    n, S = (6, 5), 10
    eps = np.full((1, 5, 6), 30, dtype=np.uint8)
    pid = np.zeros((1, 5, 6), dtype=np.int32)
    f = orc.init(2, n)
    z = np.zeros((2, 1))
    for _ in range(50):
        f = orc.step(2, n, (0, 0), 0.8, (0.0, -1e-6), S, f, eps_cnt=eps, pid=pid, pos=z + 2.0, vel=z,
                     omega=np.zeros((1, 1)))
    d = orc.diagnostics(2, f, eps, 100)
    beta = 0.3 * 0.3 / (0.7 + 0.3)
    closed = (-1e-6 / beta) * (1 - (1 - beta) ** 50)
    assert abs(closed - (-1.1011610188751e-05)) < 1e-18
    assert abs(d["gas_velocity"][1] - closed) < 1e-15 and abs(d["gas_velocity"][0]) < 1e-18
    assert abs(d["gas_area"] - 30 * 0.7) < 1e-13


def test_total_momentum_of_a_coupled_run_is_conserved_P8(orc):
    """No gravity, no body force, moving particles: what the fluid gains per step (sum_x s) is what eq. (3)
    takes from the particles, so fluid momentum + solid momentum changes only by rounding.
    Uses the diagnostics' two momentum sums, which pins them to the dynamics."""
    w = inputs.reduced("C5")
    rng = np.random.default_rng(3)
    vel = rng.uniform(-5e-3, 5e-3, size=(3, w.P))
    pos, om = w.pos.copy(), w.omega.copy()
    bc = (0, 0, 0)
    f = orc.init(3, w.n)
    tot = []
    for it in range(6):
        d = orc.diagnostics(3, f, None, 1, vel, w.radius, w.mass)
        tot.append(d["fluid_momentum"] + d["solid_momentum"])
        eps, pid = orc.map_particles(3, w.n, bc, 4, pos, w.radius)
        f, s = orc.step(3, w.n, bc, 0.6, (0, 0, 0), 4, f, eps_cnt=eps, pid=pid, pos=pos, vel=vel, omega=om, want_s=True)
        F, T, _, _ = orc.forces(3, w.n, bc, s, pid, pos)
        pos, vel, om = orc.dem_step(3, w.n, bc, pos, vel, om, w.radius, w.mass, F, T, 1e-9, 1.0, (0, 0, 0), 1.0)
    tot = np.array(tot)
    scale = np.abs(w.mass[0] * vel).sum()
    assert np.abs(tot[0]).max() > 1e-3 * scale / w.P              # there is momentum to conserve
    assert np.abs(tot - tot[0]).max() < 1e-12 * scale
    # and the fluid alone did change (the exchange is real)
    d0 = orc.diagnostics(3, orc.init(3, w.n))["fluid_momentum"]
    assert np.abs(orc.diagnostics(3, f)["fluid_momentum"] - d0).max() > 1e-6


def test_settling_suspension_slip_and_drag_have_the_physical_signs(orc):
    """Reduced paper suspension: particles fall (g_s < 0), the gas is pushed up (F_i > 0): after a few steps the
    slip U_g - V_s is positive in y and the mean drag on the particles points up."""
    w = inputs.reduced("P2D")
    f = orc.init(2, w.n)
    pos, vel, om = w.pos.copy(), np.zeros_like(w.vel), w.omega.copy()
    d = w.dem
    for _ in range(12):
        eps, pid = orc.map_particles(2, w.n, w.bc, w.subsamples, pos, w.radius)
        f, s = orc.step(2, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, eps_cnt=eps, pid=pid, pos=pos, vel=vel,
                        omega=om, want_s=True)
        F, T, _, _ = orc.forces(2, w.n, w.bc, s, pid, pos)
        pos, vel, om = orc.dem_step(2, w.n, w.bc, pos, vel, om, w.radius, w.mass, F, T, d["kn"], d["restitution"],
                                    d["g_particle"], d["dt"])
    eps, pid = orc.map_particles(2, w.n, w.bc, w.subsamples, pos, w.radius)
    dg = orc.diagnostics(2, f, eps, 64, vel, w.radius, w.mass, F)
    assert dg["slip"][1] > 0 and dg["drag"][1] > 0 and dg["solid_velocity"][1] < 0 < dg["gas_velocity"][1]


# ----------------------------------------------------------------------------- paper-parameter recipes
def test_paper_workloads_reproduce_table2_and_the_particle_counts():
    t2 = _golden("paper_table2.txt")
    for dim, col, make in ((2, 0, inputs.p2d), (3, 1, inputs.p3d)):
        t = inputs.TABLE2[dim]
        assert t["nu"] == t2["viscosity"][col] and t["kn"] == t2["stiffness"][col]
        assert t["body_force"] == t2["body_force"][col] and t["mass"] == t2["particle_mass"][col]
        assert int(np.prod(t["grid"])) == (1166400, 129024)[col]
        assert tuple(t["n"]) == ((15360, 61440), (512, 2016, 512))[col]
        vol = math.pi * 25 if dim == 2 else 4 / 3 * math.pi * 125
        phi = np.prod(t["grid"]) * vol / np.prod(t["n"], dtype=np.float64)
        assert abs(phi - t2["solid_fraction"][col]) < 4e-3                # 0.0971 vs 0.1, 0.1278 vs 0.128
        assert abs(t["mass"] / (inputs.PAPER_RHO_S * vol) - 1) < 1e-4     # m = rho_s * volume
    # the balance rule reproduces the 2D body force of Table 2 with the actual solid fraction
    phi2 = 1166400 * math.pi * 25 / (15360 * 61440)
    assert abs(inputs.balance_body_force(-1.176e-7, 692.3, phi2) / 8.753e-6 - 1) < 1e-4


def test_reduced_paper_workloads_are_well_formed():
    for name in ("P2D", "P3D"):
        w = inputs.reduced(name)
        assert w.bc == (0,) * w.dim and w.dem["kn"] == inputs.TABLE2[w.dim]["kn"]
        assert np.allclose(np.sqrt((w.vel ** 2).sum(axis=0)), 5.0e-3, rtol=1e-12)   # |v| = v_s0
        assert np.array_equal(w.pos, np.round(w.pos * 65536) / 65536)
        nn = np.array(w.n, dtype=float)[:, None, None]
        d = w.pos[:, :, None] - w.pos[:, None, :]
        d -= nn * np.round(d / nn)
        r = np.sqrt((d ** 2).sum(axis=0)) + 1e9 * np.eye(w.P)
        assert r.min() >= 10.0                                                      # no initial overlap (d = 10)
        w2 = inputs.reduced(name)
        assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.vel, w2.vel)
