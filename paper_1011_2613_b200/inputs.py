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
