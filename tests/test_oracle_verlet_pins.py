"""Pins of the oracle's Verlet neighbour list ("The neighbor-list of each solid particle is
established roughly every 100th time step"; R19).  CPU only.

What fixes it, other than itself: lists enumerated by hand, closed-form neighbour counts of regular
lattices, the symmetry of the definition, the theorem that makes the list exact (a trajectory computed with
lists equals the all-pairs trajectory of orc_dem_step BITWISE, because a pair that does not touch adds nothing
to either sum and both sum in ascending j), and closed-form rebuild counts for uniformly moving particles."""
import numpy as np
import pytest

import oracle as orc


def lists_of(start, items):
    return [items[start[i]:start[i + 1]].tolist() for i in range(len(start) - 1)]


def test_hand_enumerated_lists_periodic_and_walled():
    # 20 x 20 box, R = 1, skin = 1.5: members are closer than 3.5.  0-1: 3.  0-2: 3 through the periodic seam in x
    # (17 directly).  1-2: 6 through the seam.  3 is far from everyone.  4 sits at exactly 3.5 from 3: strict "<".
    pos = np.array([[2.0, 5.0, 19.0, 10.0, 10.0], [2.0, 2.0, 2.0, 10.0, 13.5]])
    R = np.ones(5)
    start, items = orc.verlet_build(2, (20, 20), (0, 0), pos, R, 1.5)
    assert lists_of(start, items) == [[1, 2], [0], [0], [], []]
    # with walls in x there is no image: 0-2 are 17 apart
    start, items = orc.verlet_build(2, (20, 20), (1, 0), pos, R, 1.5)
    assert lists_of(start, items) == [[1], [0], [], [], []]
    # a hair more skin lets the pair at 3.5 in
    start, items = orc.verlet_build(2, (20, 20), (0, 0), pos, R, 1.5 + 2.0 ** -40)
    assert lists_of(start, items)[3] == [4] and lists_of(start, items)[4] == [3]
    # radii enter as R_i + R_j: a big particle 3 (R = 4.6) reaches 0 (distance sqrt(128) = 11.31 > 4.6+1+1.5) no,
    # but reaches 4 and nothing else
    R2 = np.array([1.0, 1.0, 1.0, 4.6, 1.0])
    start, items = orc.verlet_build(2, (20, 20), (0, 0), pos, R2, 1.5)
    assert lists_of(start, items)[3] == [4]


@pytest.mark.parametrize("dim,skin,expect", [(2, 2.5, 4), (2, 4.0, 8), (3, 2.5, 6), (3, 4.0, 18), (3, 5.0, 26)])
def test_lattice_neighbour_counts_closed_form(dim, skin, expect):
    # simple square / cubic lattice of spacing 4 (periodic), R = 1: shells at 4 (2D 4, 3D 6), 4 sqrt2 = 5.66
    # (2D 4, 3D 12), 4 sqrt3 = 6.93 (3D 8), 8.  Cut-off 2 + skin: 4.5 -> first shell, 6 -> two shells, 7 -> three.
    m = 5
    g = np.meshgrid(*[np.arange(m) * 4.0 + 1.0] * dim, indexing="ij")
    pos = np.stack([a.reshape(-1) for a in g])
    P = pos.shape[1]
    start, items = orc.verlet_build(dim, (4 * m,) * dim, (0,) * dim, pos, np.ones(P), skin)
    assert (np.diff(start) == expect).all()
    assert items.size == expect * P


def random_gas(dim, n, P, R, seed, vmax):
    rng = np.random.default_rng(seed)
    pos = np.zeros((dim, 0))
    while pos.shape[1] < P:                                  # random sequential addition, periodic distance >= 2R
        c = rng.uniform(0, 1, size=(dim, 1)) * np.array(n, dtype=float)[:, None]
        d = pos - c
        for a in range(dim):
            d[a] -= n[a] * np.round(d[a] / n[a])
        if pos.shape[1] == 0 or (d * d).sum(axis=0).min() >= (2 * R) ** 2:
            pos = np.concatenate([pos, c], axis=1)
    vel = rng.uniform(-vmax, vmax, size=(dim, P))
    return pos, vel


@pytest.mark.parametrize("dim", [2, 3])
def test_list_is_symmetric_sorted_and_matches_numpy_distances(dim):
    n = (48, 40) if dim == 2 else (30, 26, 22)
    pos, _ = random_gas(dim, n, 60, 1.5, 5, 0.0)
    R = np.random.default_rng(1).uniform(1.0, 1.5, size=60)
    start, items = orc.verlet_build(dim, n, (0,) * dim, pos, R, 1.25)
    L = lists_of(start, items)
    for i, li in enumerate(L):
        assert li == sorted(li) and i not in li
        for j in li:
            assert i in L[j]
    # against a vectorised restatement in exact rational-free form: same comparison on numpy's own distances
    d = pos[:, :, None] - pos[:, None, :]
    for a in range(dim):
        d[a] -= n[a] * np.round(d[a] / n[a])
    dist = np.sqrt((d * d).sum(axis=0))
    cut = R[:, None] + R[None, :] + 1.25
    member = (dist < cut - 1e-9) & ~np.eye(60, dtype=bool)   # away from the knife edge both must agree
    doubtful = np.abs(dist - cut) <= 1e-9
    got = np.zeros((60, 60), dtype=bool)
    for i, li in enumerate(L):
        got[i, li] = True
    assert (got[~doubtful] == member[~doubtful]).all()


def test_zero_skin_list_is_the_touching_pairs_and_forces_are_bitwise_equal():
    dim, n = 3, (16, 16, 16)
    pos, vel = random_gas(dim, n, 40, 1.5, 11, 0.01)
    R = np.full(40, 1.6)                                     # placed at >= 3.0 apart, R_i + R_j = 3.2: some touch
    m = np.full(40, 10.0)
    start, items = orc.verlet_build(dim, n, (0, 0, 0), pos, R, 0.0)
    assert items.size > 0
    a = orc.contact_forces(dim, n, (0, 0, 0), pos, vel, R, m, 0.5, 0.9)
    b = orc.contact_forces_list(dim, n, (0, 0, 0), pos, vel, R, m, 0.5, 0.9, start, items)
    assert np.array_equal(a, b)
    touching = (np.abs(a).sum(axis=0) > 0)
    assert (np.diff(start)[touching] > 0).all()


@pytest.mark.parametrize("dim,bc", [(2, (0, 1)), (3, (0, 1, 0))])
def test_trajectory_with_lists_equals_all_pairs_trajectory_bitwise(dim, bc):
    """The exactness theorem of R19, over a run with many collisions and many rebuilds."""
    n = (36, 30) if dim == 2 else (24, 20, 18)
    P = 40 if dim == 2 else 70
    pos, vel = random_gas(dim, n, P, 1.5, 21 + dim, 0.15)
    for a in range(dim):                                     # keep clear of the walls at the start
        if bc[a]:
            pos[a] = 2.5 + pos[a] * (n[a] - 6.0) / n[a]
    R = np.full(P, 1.4)
    m = np.full(P, 50.0)
    om = np.zeros((1 if dim == 2 else 3, P))
    fh = np.zeros((dim, P))
    th = np.zeros_like(om)
    gp = (0.0, -1e-3, 0.0)
    kn = (np.pi ** 2 + np.log(0.9) ** 2) * 25.0 / 8.0 ** 2  # contact lasts 8 steps
    vs = orc.VerletState(dim, P, skin=0.6, every=100)
    xa, va, oa = pos.copy(), vel.copy(), om.copy()
    xb, vb, ob = pos.copy(), vel.copy(), om.copy()
    contacts = 0
    for _ in range(300):
        contacts += int((np.abs(orc.contact_forces(dim, n, bc, xa, va, R, m, kn, 0.9)).sum(axis=0) > 0).sum())
        xa, va, oa = orc.dem_step(dim, n, bc, xa, va, oa, R, m, fh, th, kn, 0.9, gp)
        xb, vb, ob = orc.dem_step_verlet(dim, n, bc, xb, vb, ob, R, m, fh, th, kn, 0.9, gp, vs)
        assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    assert contacts > 100 and vs.builds > 10                 # the run exercised both
    assert vs.builds < 300                                   # and the list was reused


def test_fixed_interval_alone_misses_contacts():
    """Why R19 adds the displacement rule to the paper's "roughly every 100th step": a list built while two
    particles are apart knows nothing of their contact 50 steps later."""
    n, bc = (40, 40), (0, 0)
    pos = np.array([[10.0, 20.0], [10.0, 10.0]])
    vel = np.array([[0.1, -0.1], [0.0, 0.0]])
    R, m = np.ones(2), np.ones(2)
    start, items = orc.verlet_build(2, n, bc, pos, R, 1.0)   # cut-off 3 < 10: empty lists
    assert items.size == 0
    later = pos + 41 * vel                                   # centres 1.8 apart: touching
    stale = orc.contact_forces_list(2, n, bc, later, vel, R, m, 1.0, 0.9, start, items)
    true = orc.contact_forces(2, n, bc, later, vel, R, m, 1.0, 0.9)
    assert np.abs(stale).max() == 0.0 and np.abs(true).max() > 0.1
    assert orc.verlet_max_disp2(2, n, bc, later, pos) > 0.5 ** 2   # the displacement rule would have fired


def test_rebuild_counts_closed_form():
    # uniform motion, nobody touches: displacement after k steps is k |v|.  |v| = 1/8 (exact), skin = 1: the rule
    # fires when k/8 > 1/2, i.e. every 5 steps of travel; positions x_0 .. x_N are visited, so builds = 1 + N // 5.
    n, bc = (64, 64), (0, 0)
    pos = np.array([[5.0, 30.0, 50.0], [5.0, 30.0, 50.0]])
    vel = np.array([[0.125, 0.0, -0.125], [0.0, 0.125, 0.0]])
    R, m = np.ones(3), np.ones(3)
    z = np.zeros((2, 3))
    for N in (4, 5, 23, 61):
        vs = orc.VerletState(2, 3, skin=1.0, every=10 ** 6)
        x, v, o = pos.copy(), vel.copy(), np.zeros((1, 3))
        for _ in range(N):
            x, v, o = orc.dem_step_verlet(2, n, bc, x, v, o, R, m, z, np.zeros((1, 3)), 1.0, 0.9, (0, 0, 0), vs)
        assert vs.builds == 1 + N // 5
    # particles at rest: only the age rule acts.  every = 10, 35 steps: builds at steps 0, 10, 20, 30
    vs = orc.VerletState(2, 3, skin=1.0, every=10)
    x, v, o = pos.copy(), np.zeros((2, 3)), np.zeros((1, 3))
    for _ in range(35):
        x, v, o = orc.dem_step_verlet(2, n, bc, x, v, o, R, m, z, np.zeros((1, 3)), 1.0, 0.9, (0, 0, 0), vs)
    assert vs.builds == 4 and vs.age == 5


def test_displacement_uses_the_minimum_image():
    n = (20, 20)
    ref = np.array([[19.9, 3.0], [5.0, 5.0]])
    now = np.array([[0.1, 3.0], [5.0, 5.25]])
    d2 = orc.verlet_max_disp2(2, n, (0, 0), now, ref)
    assert abs(d2 - 0.25 ** 2) < 1e-15                       # the seam crossing moved 0.2, the other 0.25
    d2 = orc.verlet_max_disp2(2, n, (1, 0), now, ref)        # with walls in x there is no image
    assert abs(d2 - 19.8 ** 2) < 1e-12
