"""CPU oracle of the LBM-IMB-DEM hot path -- TEST INFRASTRUCTURE ONLY.

numpy-facing wrappers (argument marshalling only) around
oracle/lbmimb_oracle.c, the plain fp64 restatement of PAPER.md eq. (1)-(5).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` leg may import this package; the product
(paper_1011_2613_b200) never does, and this package never imports the product.

Array conventions (identical to include/lbmimb.h so that the same seeded inputs
serve both sides): f[Q][nz][ny][nx] (x fastest), particle arrays [D][P],
omega [1][P] (2D) / [3][P] (3D), eps_cnt uint8[N], pid int32[N], s[D][N].
"""
import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_beta.restype = C.c_double
        _lib.orc_beta.argtypes = [C.c_double, C.c_double]
        _lib.orc_contact_duration.restype = C.c_double
        _lib.orc_contact_duration.argtypes = [C.c_double] * 4
        _lib.orc_damping.restype = C.c_double
        _lib.orc_damping.argtypes = [C.c_double] * 3
        _lib.orc_map.restype = C.c_int
        _lib.orc_eps_table.restype = C.c_int
        _lib.orc_map_table.restype = C.c_int
        _lib.orc_dem_step.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_verlet_build.restype = C.c_int64
        _lib.orc_verlet_max_disp2.restype = C.c_double
        _lib.orc_dem_step_verlet.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _n3(n):
    n = list(n) + [1] * (3 - len(n))
    return np.array(n, dtype=np.int64)


def _bc3(bc):
    bc = list(bc) + [0] * (3 - len(bc))
    return np.array(bc, dtype=np.int32)


def _g3(g):
    g = list(g) + [0.0] * (3 - len(g))
    return np.array(g, dtype=np.float64)


def nq(dim):
    return 9 if dim == 2 else 19


def num_threads():
    return int(lib().orc_num_threads())


def velocity_set(dim):
    Q = nq(dim)
    c = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q)
    o = np.zeros(Q, dtype=np.int32)
    lib().orc_velocity_set(C.c_int(dim), _p(c), _p(w), _p(o))
    return c, w, o


def feq(dim, rho, u):
    u = _g3(u)
    out = np.zeros(nq(dim))
    lib().orc_feq(C.c_int(dim), C.c_double(rho), _p(u), _p(out))
    return out


def beta(eps, tau):
    return float(lib().orc_beta(eps, tau))


def collide_node(dim, tau, g, f, beta_, vs):
    """-> (fstar[Q], s[3], rho, u[3]) of one node (eq. (1)-(2) before streaming)."""
    f = _f64(f)
    g = _g3(g)
    vs = _g3(vs)
    fstar = np.zeros(nq(dim))
    s = np.zeros(3)
    rho = C.c_double(0.0)
    u = np.zeros(3)
    lib().orc_collide_node(C.c_int(dim), C.c_double(tau), _p(g), _p(f),
                           C.c_double(beta_), _p(vs), _p(fstar), _p(s),
                           C.byref(rho), _p(u))
    return fstar, s, rho.value, u


def init(dim, n):
    n3 = _n3(n)
    N = int(n3.prod())
    f = np.empty((nq(dim), int(n3[2]), int(n3[1]), int(n3[0])))
    lib().orc_init(C.c_int(dim), C.c_int64(N), _p(f))
    return f


def macros(dim, f):
    """-> rho[nz,ny,nx], u[dim,nz,ny,nx] (bare u, R2)."""
    f = _f64(f)
    shp = f.shape[1:]
    N = int(np.prod(shp))
    rho = np.empty(shp)
    u = np.empty((dim,) + shp)
    lib().orc_macros(C.c_int(dim), C.c_int64(N), _p(f), _p(rho), _p(u))
    return rho, u


def map_particles(dim, n, bc, S, pos, radius):
    """-> eps_cnt uint8[nz,ny,nx], pid int32[nz,ny,nx]."""
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    radius = _f64(radius)
    P = pos.shape[1]
    shp = (int(n3[2]), int(n3[1]), int(n3[0]))
    eps = np.zeros(shp, dtype=np.uint8)
    pid = np.empty(shp, dtype=np.int32)
    rc = lib().orc_map(C.c_int(dim), _p(n3), _p(bc3), C.c_int(S), C.c_int64(P),
                       _p(pos), _p(radius), _p(eps), _p(pid))
    if rc != 0:
        raise RuntimeError("orc_map failed (S^D > 255 or out of memory)")
    return eps, pid


# discretisation of the eps table (R17): (Nd, Nt, St) per dimension; part of the ABI text
TABLE_DIMS = {2: (128, 32, 256), 3: (128, 16, 64)}
TABLE_DEN = 255


_tables = {}


def eps_table(dim, R, dims=None):
    """The paper's pre-calculated table gamma = phi(d, theta) as uint8 codes,
    shape [Nd, Nt] (2D) or [Nd, Nt, Nt] (3D); gamma = code / 255.  Computed once per (dim, R, dims)."""
    Nd, Nt, St = dims or TABLE_DIMS[dim]
    key = (dim, float(R), Nd, Nt, St)
    if key not in _tables:
        tab = np.zeros((Nd, Nt) if dim == 2 else (Nd, Nt, Nt), dtype=np.uint8)
        rc = lib().orc_eps_table(C.c_int(dim), C.c_double(R), C.c_int(Nd), C.c_int(Nt), C.c_int(St), _p(tab))
        if rc != 0:
            raise RuntimeError("orc_eps_table failed (R < 1 or bad sizes)")
        tab.setflags(write=False)
        _tables[key] = tab
    return _tables[key]


def map_particles_table(dim, n, bc, pos, radius, dims=None):
    """Table-mode map -> eps_code uint8[nz,ny,nx] (eps = code/255), pid int32[nz,ny,nx]."""
    Nd, Nt, St = dims or TABLE_DIMS[dim]
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    radius = _f64(radius)
    P = pos.shape[1]
    shp = (int(n3[2]), int(n3[1]), int(n3[0]))
    eps = np.zeros(shp, dtype=np.uint8)
    pid = np.empty(shp, dtype=np.int32)
    tab = eps_table(dim, radius[0], (Nd, Nt, St)) if P else np.zeros(1, dtype=np.uint8)
    rc = lib().orc_map_table(C.c_int(dim), _p(n3), _p(bc3), C.c_int(Nd), C.c_int(Nt), _p(tab),
                             C.c_int64(P), _p(pos), _p(radius), _p(eps), _p(pid))
    if rc != 0:
        raise RuntimeError("orc_map_table failed (%d: -2 = radii differ)" % rc)
    return eps, pid


def step(dim, n, bc, tau, g, S, f, eps_cnt=None, pid=None, pos=None, vel=None,
         omega=None, want_s=False, eps_den=None):
    """One step of eq. (1): returns f(t+1) (and s[dim,nz,ny,nx] if want_s).
    eps = eps_cnt / eps_den, eps_den = S^dim unless given (255 for the table map)."""
    n3, bc3, g3 = _n3(n), _bc3(bc), _g3(g)
    if eps_den is None:
        eps_den = S ** dim
    f = _f64(f)
    out = np.empty_like(f)
    shp = f.shape[1:]
    s = np.zeros((dim,) + shp) if want_s else None
    if eps_cnt is None:
        P = 0
        args = [None] * 5
    else:
        pos = _f64(pos).reshape(dim, -1)
        vel = _f64(vel).reshape(dim, -1)
        omega = _f64(omega).reshape(1 if dim == 2 else 3, -1)
        P = pos.shape[1]
        eps_cnt = np.ascontiguousarray(eps_cnt, dtype=np.uint8)
        pid = np.ascontiguousarray(pid, dtype=np.int32)
        args = [_p(eps_cnt), _p(pid), _p(pos), _p(vel), _p(omega)]
    lib().orc_step(C.c_int(dim), _p(n3), _p(bc3), C.c_double(tau), _p(g3),
                   C.c_int(eps_den), _p(f), _p(out), args[0], args[1], C.c_int64(P),
                   args[2], args[3], args[4], _p(s) if want_s else None)
    return (out, s) if want_s else out


def forces(dim, n, bc, s, pid, pos):
    """Literal eq. (3) with the sign of R6 -> force[dim,P], torque[1|3,P], abs_f[P], abs_t[P]."""
    n3, bc3 = _n3(n), _bc3(bc)
    s = _f64(s)
    pid = np.ascontiguousarray(pid, dtype=np.int32)
    pos = _f64(pos).reshape(dim, -1)
    P = pos.shape[1]
    force = np.zeros((dim, P))
    torque = np.zeros((1 if dim == 2 else 3, P))
    abs_f = np.zeros(P)
    abs_t = np.zeros(P)
    lib().orc_forces(C.c_int(dim), _p(n3), _p(bc3), _p(s), _p(pid), C.c_int64(P),
                     _p(pos), _p(force), _p(torque), _p(abs_f), _p(abs_t))
    return force, torque, abs_f, abs_t


def contact_duration(kn, e, mi, mj):
    return float(lib().orc_contact_duration(kn, e, mi, mj))


def damping(kn, e, meff):
    return float(lib().orc_damping(kn, e, meff))


def contact_forces(dim, n, bc, pos, vel, radius, mass, kn, e):
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    vel = _f64(vel).reshape(dim, -1)
    P = pos.shape[1]
    fc = np.zeros((dim, P))
    lib().orc_contact_forces(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(P), _p(pos),
                             _p(vel), _p(_f64(radius)), _p(_f64(mass)),
                             C.c_double(kn), C.c_double(e), _p(fc))
    return fc


def dem_step(dim, n, bc, pos, vel, omega, radius, mass, fh, th, kn, e, gp, dt=1.0):
    """One velocity-Verlet DEM step (R11); returns new (pos, vel, omega) copies."""
    n3, bc3, gp3 = _n3(n), _bc3(bc), _g3(gp)
    pos = _f64(pos).reshape(dim, -1).copy()
    vel = _f64(vel).reshape(dim, -1).copy()
    omega = _f64(omega).reshape(1 if dim == 2 else 3, -1).copy()
    P = pos.shape[1]
    rc = lib().orc_dem_step(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(P), _p(pos),
                            _p(vel), _p(omega), _p(_f64(radius)), _p(_f64(mass)),
                            _p(_f64(fh)), _p(_f64(th)), C.c_double(kn),
                            C.c_double(e), _p(gp3), C.c_double(dt))
    if rc != 0:
        raise RuntimeError("orc_dem_step failed")
    return pos, vel, omega


def coupled_step(dim, n, bc, tau, g, S, f, pos, vel, omega, radius, mass, kn, e, gp, dt=1.0, verlet=None):
    """One coupled step of the method in the order BASELINE.json configs[4] fixes (R11):
         1. map      eps, pid at the CURRENT positions x(t)
         2. LBM step f(t) -> f(t+1) with V_S from the CURRENT v(t), omega(t); the exchange vectors s are
                     those of this collision, i.e. they come from the PRE-collision state f(t)
         3. forces   F_h, T_h = eq. (3) over s
         4. DEM step x, v, omega advance by dt with F_h, T_h held constant over the step
       (`verlet`: a VerletState -> the neighbour-list variant of step 4, R19).
    Returns (f, pos, vel, omega, info) with info = dict(eps, pid, s, force, torque, abs_f, abs_t) of this step."""
    eps, pid = map_particles(dim, n, bc, S, pos, radius)
    f, s = step(dim, n, bc, tau, g, S, f, eps_cnt=eps, pid=pid, pos=pos, vel=vel, omega=omega, want_s=True)
    F, T, aF, aT = forces(dim, n, bc, s, pid, pos)
    if verlet is None:
        pos, vel, omega = dem_step(dim, n, bc, pos, vel, omega, radius, mass, F, T, kn, e, gp, dt)
    else:
        pos, vel, omega = dem_step_verlet(dim, n, bc, pos, vel, omega, radius, mass, F, T, kn, e, gp, verlet, dt)
    return f, pos, vel, omega, dict(eps=eps, pid=pid, s=s, force=F, torque=T, abs_f=aF, abs_t=aT)


def verlet_build(dim, n, bc, pos, radius, skin):
    """The neighbour lists by their definition (R19): CSR (start[P+1] int64, items int32), j ascending."""
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    P = pos.shape[1]
    start = np.zeros(P + 1, dtype=np.int64)
    cap = max(64 * P, 1)
    while True:
        items = np.zeros(cap, dtype=np.int32)
        t = int(lib().orc_verlet_build(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(P), _p(pos), _p(_f64(radius)),
                                       C.c_double(skin), _p(start), _p(items), C.c_int64(cap)))
        if t >= 0:
            return start, items[:t].copy()
        cap = -t


def verlet_max_disp2(dim, n, bc, pos, pos_ref):
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    ref = _f64(pos_ref).reshape(dim, -1)
    return float(lib().orc_verlet_max_disp2(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(pos.shape[1]), _p(pos), _p(ref)))


def contact_forces_list(dim, n, bc, pos, vel, radius, mass, kn, e, start, items):
    n3, bc3 = _n3(n), _bc3(bc)
    pos = _f64(pos).reshape(dim, -1)
    vel = _f64(vel).reshape(dim, -1)
    P = pos.shape[1]
    fc = np.zeros((dim, P))
    start = np.ascontiguousarray(start, dtype=np.int64)
    items = np.ascontiguousarray(items, dtype=np.int32)
    lib().orc_contact_forces_list(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(P), _p(pos), _p(vel), _p(_f64(radius)),
                                  _p(_f64(mass)), C.c_double(kn), C.c_double(e), _p(start), _p(items), _p(fc))
    return fc


class VerletState:
    """What the neighbour-list variant of the DEM step carries from step to step (R19)."""

    def __init__(self, dim, P, skin, every, cap_per_particle=128):
        self.skin, self.every = float(skin), int(every)
        self.state = np.zeros(3, dtype=np.int64)          # valid, age (steps), number of builds
        self.x_ref = np.zeros((dim, P))
        self.start = np.zeros(P + 1, dtype=np.int64)
        self.items = np.zeros(max(cap_per_particle * P, 1), dtype=np.int32)

    valid = property(lambda self: bool(self.state[0]))
    age = property(lambda self: int(self.state[1]))
    builds = property(lambda self: int(self.state[2]))

    def lists(self):
        return self.start.copy(), self.items[:self.start[-1]].copy()


def dem_step_verlet(dim, n, bc, pos, vel, omega, radius, mass, fh, th, kn, e, gp, vs, dt=1.0):
    """One DEM step (R11) with the neighbour list `vs` (VerletState, updated in place) and the rebuild rule
    R19; returns new (pos, vel, omega) copies."""
    n3, bc3, gp3 = _n3(n), _bc3(bc), _g3(gp)
    pos = _f64(pos).reshape(dim, -1).copy()
    vel = _f64(vel).reshape(dim, -1).copy()
    omega = _f64(omega).reshape(1 if dim == 2 else 3, -1).copy()
    P = pos.shape[1]
    rc = lib().orc_dem_step_verlet(C.c_int(dim), _p(n3), _p(bc3), C.c_int64(P), _p(pos), _p(vel), _p(omega),
                                   _p(_f64(radius)), _p(_f64(mass)), _p(_f64(fh)), _p(_f64(th)), C.c_double(kn),
                                   C.c_double(e), _p(gp3), C.c_double(dt), C.c_double(vs.skin),
                                   C.c_int64(vs.every), _p(vs.state), _p(vs.x_ref), _p(vs.start), _p(vs.items),
                                   C.c_int64(vs.items.size))
    if rc != 0:
        raise RuntimeError("orc_dem_step_verlet failed (list capacity?)")
    return pos, vel, omega


DIAG_LEN = 20


def diagnostics(dim, f, eps_cnt=None, eps_den=1, vel=None, radius=None, mass=None, force=None):
    """Area/volume-averaged suspension diagnostics of PAPER.md:154 and Figs. 5/7 ("area-averaged inter-phase
    slip velocity V_ry and drag force F_dy"); the paper prints no formula, the reading is DESIGN.md R18:
      eps_x = eps_cnt_x / eps_den, u = bare velocity of `macros` (R2),
      gas area       A_g = sum_x (1 - eps_x)
      gas velocity   U_g = sum_x (1 - eps_x) u_x / A_g
      solid velocity V_s = sum_p vol_p v_p / sum_p vol_p,  vol_p = pi R^2 (2D) or 4/3 pi R^3 (3D)
      slip           V_r = U_g - V_s
      drag           F_d = sum_p F_p / P        (mean hydrodynamic force per particle, eq. (3))
    plus the fluid mass sum_x rho, fluid momentum sum_x rho u and solid momentum sum_p m_p v_p.
    Returns a dict and, under "vector", the 20 doubles in the layout of lbmimb_diagnostics:
      [0] A_g [1] mass [2:5] U_g [5:8] V_s [8:11] V_r [11:14] F_d [14:17] fluid momentum [17:20] solid momentum
    (unused z components are 0).  Plain numpy sums in fp64."""
    rho, u = macros(dim, f)
    if eps_cnt is None:
        gas = np.ones(rho.shape)
    else:
        gas = 1.0 - np.asarray(eps_cnt, dtype=np.float64).reshape(rho.shape) / float(eps_den)
    out = np.zeros(DIAG_LEN)
    A_g = gas.sum()
    out[0] = A_g
    out[1] = rho.sum()
    for a in range(dim):
        out[2 + a] = (gas * u[a]).sum() / A_g
        out[14 + a] = (rho * u[a]).sum()
    P = 0 if radius is None else int(np.asarray(radius).shape[0])
    if P > 0:
        radius = _f64(radius)
        vel = _f64(vel).reshape(dim, P)
        vol = np.pi * radius ** 2 if dim == 2 else 4.0 / 3.0 * np.pi * radius ** 3
        for a in range(dim):
            out[5 + a] = (vol * vel[a]).sum() / vol.sum()
            out[17 + a] = (_f64(mass) * vel[a]).sum()
            if force is not None:
                out[11 + a] = _f64(force).reshape(dim, P)[a].sum() / P
    out[8:11] = out[2:5] - out[5:8]
    return {"gas_area": out[0], "mass": out[1], "gas_velocity": out[2:2 + dim], "solid_velocity": out[5:5 + dim],
            "slip": out[8:8 + dim], "drag": out[11:11 + dim], "fluid_momentum": out[14:14 + dim],
            "solid_momentum": out[17:17 + dim], "vector": out}
