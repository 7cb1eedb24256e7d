"""Seeded synthetic workloads C1..C5 (BASELINE.json:configs[0..4]).

This module is the ONE thing the CUDA path's tests/bench and the CPU oracle
share: it only draws random particle sets and names parameters.  It holds none
of the method's arithmetic (no f^eq, no beta, no mapping, no forces) and
imports neither `oracle` nor the CUDA binding.

The paper measures on no public dataset; its two production runs (PAPER.md:117,
Table 2) are a fully periodic 2D suspension (15360x61440 nodes, 1,166,400 disks
of d = 10) and a 3D one (512x2016x512, 129,024 spheres).  C1..C5 are synthetic
stand-ins of the same shape (aspect ratios, solid fraction 0.1-0.26, d/l = 8-12,
random velocities of a few 1e-3), generated here with numpy's PCG64,
seed = 10112613 + k for config k = 1..5.

Every particle centre is rounded to a multiple of 2**-16 so that translating a
particle set by whole nodes is exact in fp64 (used by the sub-box parity tests;
DESIGN.md "Input recipe").
"""
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

SEED0 = 10112613
_QUANT = 65536.0


@dataclass
class Workload:
    name: str
    dim: int
    n: Tuple[int, ...]              # nodes per axis, x first (x is the fastest-varying axis)
    bc: Tuple[int, ...]             # per axis: 0 periodic, 1 half-way bounce-back walls
    tau: float
    g_fluid: Tuple[float, ...]
    subsamples: int                 # S per axis (8 in 2D, 4 in 3D)
    steps: int
    pos: np.ndarray                 # [D][P]
    vel: np.ndarray                 # [D][P]
    omega: np.ndarray               # [1][P] (2D) or [3][P] (3D)
    radius: np.ndarray              # [P]
    mass: np.ndarray                # [P]
    dem: Optional[dict] = None      # kn, restitution, g_particle, dt (C5 only)
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def P(self):
        return int(self.pos.shape[1])

    @property
    def nodes(self):
        return int(np.prod(self.n))

    @property
    def Q(self):
        return 9 if self.dim == 2 else 19


def _quantise(x):
    return np.round(np.asarray(x, dtype=np.float64) * _QUANT) / _QUANT


def _place_random(rng, dim, n, bc, P, R, wall_lo, wall_hi, max_tries=2000000):
    """Random sequential addition of P equal balls of radius R, centre distance
    >= 2R (periodic axes: minimum image).  Wall axes: centre in [wall_lo, n-1-wall_hi]
    measured in node coordinates.  Hash grid of edge >= 2R keeps it O(P)."""
    n = np.asarray(n, dtype=np.int64)
    ncell = np.maximum((n // (2 * R)).astype(np.int64), 1)
    edge = n / ncell
    grid = {}
    out = np.empty((dim, P))
    lo = np.array([wall_lo if bc[a] else 0.0 for a in range(dim)])
    hi = np.array([n[a] - 1 - wall_hi if bc[a] else float(n[a]) for a in range(dim)])
    offs = np.array(np.meshgrid(*([[-1, 0, 1]] * dim), indexing="ij")).reshape(dim, -1).T
    placed = 0
    tries = 0
    d2min = (2.0 * R) ** 2
    while placed < P:
        tries += 1
        if tries > max_tries:
            raise RuntimeError("random sequential addition did not converge")
        c = _quantise(lo + rng.random(dim) * (hi - lo))
        for a in range(dim):
            if not bc[a] and c[a] >= n[a]:
                c[a] -= n[a]
        cell = np.minimum((c / edge).astype(np.int64), ncell - 1)
        ok = True
        seen = set()
        for o in offs:
            cc = cell + o
            key = []
            for a in range(dim):
                v = int(cc[a])
                if bc[a]:
                    if v < 0 or v >= ncell[a]:
                        key = None
                        break
                else:
                    v %= int(ncell[a])
                key.append(v)
            if key is None:
                continue
            key = tuple(key)
            if key in seen:
                continue
            seen.add(key)
            for q in grid.get(key, ()):
                d = c - out[:, q]
                for a in range(dim):
                    if not bc[a]:
                        if d[a] > 0.5 * n[a]:
                            d[a] -= n[a]
                        elif d[a] < -0.5 * n[a]:
                            d[a] += n[a]
                if float(d @ d) < d2min:
                    ok = False
                    break
            if not ok:
                break
        if ok:
            out[:, placed] = c
            grid.setdefault(tuple(int(v) for v in cell), []).append(placed)
            placed += 1
    return out


def _ball_mass(dim, R, density):
    R = np.asarray(R, dtype=np.float64)
    return density * (np.pi * R ** 2 if dim == 2 else 4.0 / 3.0 * np.pi * R ** 3)


def c1(n=(128, 128), P=16, R=6.0, steps=100, seed=SEED0 + 1):
    """C1: D2Q9, periodic box, 16 fixed disks of radius 6 at rest."""
    rng = np.random.default_rng(seed)
    pos = _place_random(rng, 2, n, (0, 0), P, R, 0.0, 0.0)
    radius = np.full(P, R)
    return Workload("C1", 2, tuple(n), (0, 0), 0.8, (0.0, -1e-6), 8, steps, pos,
                    np.zeros((2, P)), np.zeros((1, P)), radius,
                    _ball_mass(2, radius, 1000.0))


def c2(n=(1024, 4096), P=14000, R=4.0, steps=1000, seed=SEED0 + 2):
    """C2: D2Q9, x periodic, walls in y, tau=0.6, disks with prescribed v, omega."""
    rng = np.random.default_rng(seed)
    pos = _place_random(rng, 2, n, (0, 1), P, R, R + 0.5, R + 0.5)
    vel = rng.uniform(-0.01, 0.01, size=(2, P))
    omega = rng.uniform(-1e-3, 1e-3, size=(1, P))
    radius = np.full(P, R)
    return Workload("C2", 2, tuple(n), (0, 1), 0.6, (0.0, -1e-6), 8, steps, pos, vel,
                    omega, radius, _ball_mass(2, radius, 1000.0))


def c3(n=(256, 1008, 256), P=24600, R=4.0, steps=500, seed=SEED0 + 3):
    """C3: D3Q19, x,z periodic, walls in y, tau=0.7, spheres with prescribed v."""
    rng = np.random.default_rng(seed)
    pos = _place_random(rng, 3, n, (0, 1, 0), P, R, R + 0.5, R + 0.5)
    vel = rng.uniform(-0.005, 0.005, size=(3, P))
    radius = np.full(P, R)
    return Workload("C3", 3, tuple(n), (0, 1, 0), 0.7, (0.0, -1e-6, 0.0), 4, steps, pos,
                    vel, np.zeros((3, P)), radius, _ball_mass(3, radius, 1000.0))


def c4(n=(8192, 32768), grid=(540, 2160), R=4.0, steps=200, seed=SEED0 + 4):
    """C4: D2Q9 throughput lattice, jittered grid of disks (jitter +-1 lu)."""
    rng = np.random.default_rng(seed)
    gx, gy = grid
    px, py = n[0] / gx, n[1] / gy
    a, b = np.meshgrid(np.arange(gx), np.arange(gy), indexing="ij")
    P = gx * gy
    cx = (a.reshape(-1) + 0.5) * px + rng.uniform(-1.0, 1.0, size=P)
    cy = (b.reshape(-1) + 0.5) * py + rng.uniform(-1.0, 1.0, size=P)
    pos = _quantise(np.stack([cx, cy]))
    vel = rng.uniform(-0.01, 0.01, size=(2, P))
    radius = np.full(P, R)
    return Workload("C4", 2, tuple(n), (0, 1), 0.55, (0.0, -1e-6), 8, steps, pos, vel,
                    np.zeros((1, P)), radius, _ball_mass(2, radius, 1000.0))


def c5(n=(128, 512, 128), P=4096, R=5.0, steps=2000, seed=SEED0 + 5, kn=1e-2):
    """C5: coupled run, D3Q19, spheres at rest, gravity on the particles only."""
    rng = np.random.default_rng(seed)
    pos = _place_random(rng, 3, n, (0, 1, 0), P, R, R + 2.0, R + 2.0)
    radius = np.full(P, R)
    dem = {"kn": kn, "restitution": 0.9, "g_particle": (0.0, -1e-6, 0.0), "dt": 1.0}
    return Workload("C5", 3, tuple(n), (0, 1, 0), 0.6, (0.0, 0.0, 0.0), 4, steps, pos,
                    np.zeros((3, P)), np.zeros((3, P)), radius,
                    _ball_mass(3, radius, 1000.0), dem=dem)


FULL = {"C1": c1, "C2": c2, "C3": c3, "C4": c4, "C5": c5}


# ---------------------------------------------------------------------------------------------
# Paper-scale, paper-parameter suspensions (PAPER.md:117 and Table 2).
# Everything below is a parameter the paper prints (tests/golden/paper_table2.txt) or a placement
# recipe (R19); none of it is arithmetic of the method.
# ---------------------------------------------------------------------------------------------
TABLE2 = {
    2: dict(nu=0.1231, body_force=8.753e-6, g_s=-1.176e-7, mass=54373.0, kn=2686.0, n=(15360, 61440),
            grid=(540, 2160)),
    3: dict(nu=0.2462, body_force=4.04e-5, g_s=-4.704e-7, mass=362491.0, kn=17892.0, n=(512, 2016, 512),
            grid=(32, 126, 32)),
}
PAPER_R, PAPER_E, PAPER_VS0, PAPER_RHO_S = 5.0, 0.9, 5.0e-3, 692.3


def balance_body_force(g_s, rho_s, phi, rho_g=1.0):
    """The body force per unit gas mass that balances the weight of the solids ("A body force
    F_i is exerted on the gas phase to balance the gravity on solid particles"): the gas occupies the
    fraction 1 - phi of the domain, the solids phi, so  F rho_g (1 - phi) = |g_s| rho_s phi.
    Table 2's 2D entry 8.753e-6 follows from it with the actual phi = 0.09707."""
    return abs(g_s) * rho_s * phi / ((1.0 - phi) * rho_g)


def _paper_suspension(name, dim, n, grid, seed, jitter=2.0, steps=1000):
    t = TABLE2[dim]
    rng = np.random.default_rng(seed)
    pitch = [n[a] / grid[a] for a in range(dim)]
    idx = np.meshgrid(*[np.arange(g) for g in grid], indexing="ij")
    P = int(np.prod(grid))
    pos = np.stack([(idx[a].reshape(-1) + 0.5) * pitch[a] + rng.uniform(-jitter, jitter, size=P) for a in range(dim)])
    pos = _quantise(np.mod(pos, np.array(n, dtype=np.float64)[:, None]))
    d = rng.standard_normal((dim, P))
    vel = PAPER_VS0 * d / np.sqrt((d * d).sum(axis=0))          # random direction, magnitude v_s0
    radius = np.full(P, PAPER_R)
    mass = np.full(P, t["mass"])
    gf = [0.0] * dim
    gf[1] = t["body_force"]                                      # on the gas, upwards: balances the solids' weight
    gp = [0.0] * 3
    gp[1] = t["g_s"]
    dem = {"kn": t["kn"], "restitution": PAPER_E, "g_particle": tuple(gp), "dt": 1.0}
    return Workload(name, dim, tuple(n), (0,) * dim, 3.0 * t["nu"] + 0.5, tuple(gf), 8 if dim == 2 else 4, steps,
                    pos, vel, np.zeros((1 if dim == 2 else 3, P)), radius, mass, dem=dem,
                    note="PAPER.md:117 / Table 2 suspension, jittered %s lattice of d = 10 particles" %
                    "x".join(str(g) for g in grid))


def p2d(n=None, grid=None, steps=1000, seed=SEED0 + 12):
    """The paper's 2D suspension: 15360 x 61440 D2Q9, fully periodic, 1,166,400 disks of d = 10
    (540 x 2160 jittered lattice, solid fraction 0.0971), Table 2 parameters, coupled LBM-IMB-DEM."""
    t = TABLE2[2]
    return _paper_suspension("P2D", 2, n or t["n"], grid or t["grid"], seed, steps=steps)


def p3d(n=None, grid=None, steps=1000, seed=SEED0 + 13):
    """The paper's 3D suspension: 512 x 2016 x 512 D3Q19, fully periodic, 129,024 spheres of d = 10
    (32 x 126 x 32 jittered lattice, solid fraction 0.128), Table 2 parameters, coupled LBM-IMB-DEM."""
    t = TABLE2[3]
    return _paper_suspension("P3D", 3, n or t["n"], grid or t["grid"], seed, steps=steps)


FULL.update({"P2D": p2d, "P3D": p3d})


def reduced(name):
    """Cuts of C1..C5 the oracle finishes in seconds: same recipe and solid
    fraction, lattice sizes that are NOT multiples of the kernel tiles (ragged
    tails in x, odd row counts)."""
    if name == "C1":
        return c1()
    if name == "C2":
        w = c2(n=(200, 333), P=220, steps=60)
    elif name == "C3":
        w = c3(n=(72, 90, 44), P=105, steps=30)
    elif name == "C4":
        w = c4(n=(455, 606), grid=(30, 40), steps=40)
    elif name == "C5":
        w = c5(n=(40, 84, 36), P=58, steps=40, kn=50.0)
        w.extra["note"] = "stiffer k_n so that contacts act within the short run"
    elif name == "P2D":
        w = p2d(n=(313, 270), grid=(11, 9), steps=30)            # pitch 28.45 x 30 as in the paper's 28.44
    elif name == "P3D":
        w = p3d(n=(70, 96, 52), grid=(4, 6, 3), steps=20)        # pitch 17.5 x 16 x 17.3 (paper: 16)
    else:
        raise KeyError(name)
    w.name = name + "-reduced"
    return w


def sub_box(w, lo, size):
    """Particle set of workload w seen from the all-periodic box [lo, lo+size):
    every particle (and periodic image) whose bounding box touches the box,
    translated by -lo (exact, centres are multiples of 2**-16).  Returns
    (pos, vel, omega, radius, mass, idx) for a lattice of `size` nodes; idx = original particle indices."""
    dim = w.dim
    lo = np.asarray(lo, dtype=np.float64)
    size = np.asarray(size, dtype=np.float64)
    keep_pos, keep_idx = [], []
    shifts = [[0.0] if w.bc[a] else [-float(w.n[a]), 0.0, float(w.n[a])] for a in range(dim)]
    grids = np.array(np.meshgrid(*shifts, indexing="ij")).reshape(dim, -1).T
    for sh in grids:
        c = w.pos + sh[:, None] - lo[:, None]
        m = np.ones(w.P, dtype=bool)
        for a in range(dim):
            m &= (c[a] + w.radius + 2.0 >= 0.0) & (c[a] - w.radius - 2.0 <= size[a] - 1.0)
        idx = np.nonzero(m)[0]
        keep_pos.append(c[:, idx])
        keep_idx.append(idx)
    idx = np.concatenate(keep_idx)
    pos = np.concatenate(keep_pos, axis=1)
    return pos, w.vel[:, idx].copy(), w.omega[:, idx].copy(), w.radius[idx].copy(), w.mass[idx].copy(), idx


def y_slab(w, y_lo, y_hi):
    """Particle set of workload w seen from the rows [y_lo, y_hi) of its lattice, all other axes kept whole:
    every particle whose bounding box (centre +- (R + 2)) touches the slab, translated by -y_lo along y
    (exact: centres are multiples of 2**-16, y_lo is an integer).  For a lattice of (n_x, y_hi - y_lo[, n_z]) nodes
    whose y edges are walls.  The order of the particles is kept, so that "ties -> lowest index" picks the same
    particle in the slab as in the whole lattice.  Returns (pos, vel, omega, radius, mass, idx)."""
    y = w.pos[1]
    m = (y + w.radius + 2.0 >= float(y_lo)) & (y - w.radius - 2.0 <= float(y_hi) - 1.0)
    idx = np.nonzero(m)[0]
    pos = w.pos[:, idx].copy()
    pos[1] -= float(y_lo)
    return pos, w.vel[:, idx].copy(), w.omega[:, idx].copy(), w.radius[idx].copy(), w.mass[idx].copy(), idx
