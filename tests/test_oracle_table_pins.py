"""Pins of the oracle's table-look-up eps method (NEXT-1; eq. (6); R17).

The table is an approximation ("slightly less accurate but faster"), so the oracle follows the
algorithm step by step; what pins it is the quantity the table approximates: the area / volume of the
cell covered by the particle.  The covered fraction is computed here by quadrature of the
chord length (no sub-cell points, no code of the oracle), and the map is checked against the sampled map
of orc_map, against the particle's area/volume, and against the lattice symmetries.
"""
import numpy as np
import pytest


def _cell_centre(dim, R, dims, k, m1, m2=0):
    """Cell centre of table entry (k, m1[, m2]) relative to the particle centre (R17)."""
    Nd, Nt, _ = dims
    sq = np.sqrt(dim)
    dk = (R - 0.5 * sq) + (k + 0.5) * sq / Nd
    t1 = (m1 + 0.5) / Nt
    t2 = (m2 + 0.5) / Nt if dim == 3 else 0.0
    v = np.array([1.0, t1, t2])
    return dk * v / np.linalg.norm(v)


def _covered_fraction_2d(r, R, n=40001):
    """Area of the unit square centred at r inside the disk |x| <= R: integral of the chord overlap."""
    x = np.linspace(r[0] - 0.5, r[0] + 0.5, n)
    h = np.sqrt(np.maximum(R * R - x * x, 0.0))
    ov = np.clip(np.minimum(h, r[1] + 0.5) - np.maximum(-h, r[1] - 0.5), 0.0, None)
    ov[R * R - x * x < 0] = 0.0
    return float(np.sum((ov[1:] + ov[:-1]) * 0.5) * (x[1] - x[0]))


def _covered_fraction_3d(r, R, n=600):
    """Volume of the unit cube centred at r inside the sphere: midpoint rule over (x,y) of the z overlap."""
    xs = r[0] - 0.5 + (np.arange(n) + 0.5) / n
    ys = r[1] - 0.5 + (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    h2 = R * R - X * X - Y * Y
    h = np.sqrt(np.maximum(h2, 0.0))
    ov = np.clip(np.minimum(h, r[2] + 0.5) - np.maximum(-h, r[2] - 0.5), 0.0, None)
    ov[h2 < 0] = 0.0
    return float(ov.mean())


@pytest.mark.parametrize("R", [4.0, 6.0])
def test_table_entries_are_the_covered_area_2d(orc, R):
    dims = orc.TABLE_DIMS[2]
    tab = orc.eps_table(2, R)
    rng = np.random.default_rng(7)
    worst = 0.0
    for k, m in zip(rng.integers(0, dims[0], 80), rng.integers(0, dims[1], 80)):
        exact = _covered_fraction_2d(_cell_centre(2, R, dims, k, m), R)
        worst = max(worst, abs(tab[k, m] / 255.0 - exact))
    # 8-bit code (0.5/255) + midpoint sampling on a 256^2 grid (a whole row of points flips at once when
    # the boundary is almost parallel to an axis: 1/256) + quadrature
    assert worst <= 0.5 / 255 + 1.0 / 256 + 1e-4, worst


def test_table_entries_are_the_covered_volume_3d(orc):
    R = 4.0
    dims = orc.TABLE_DIMS[3]
    tab = orc.eps_table(3, R)
    rng = np.random.default_rng(8)
    worst = 0.0
    for k, m1, m2 in zip(rng.integers(0, dims[0], 40), rng.integers(0, dims[1], 40), rng.integers(0, dims[1], 40)):
        exact = _covered_fraction_3d(_cell_centre(3, R, dims, k, m1, m2), R)
        worst = max(worst, abs(tab[k, m1, m2] / 255.0 - exact))
    assert worst <= 0.5 / 255 + 1.0 / 64 + 2e-3, worst          # 64^3 sample points per entry


@pytest.mark.parametrize("dim,R", [(2, 4.0), (3, 4.0)])
def test_table_limits_and_monotone_in_d(orc, dim, R):
    tab = orc.eps_table(dim, R).astype(int)
    assert tab[0].min() >= 253 and tab[-1].max() <= 2          # fully inside / outside at the ends of the d range
    assert (np.diff(tab, axis=0) <= 0).all()                    # farther away => never more covered
    assert tab.min() == 0 and tab.max() == 255


def test_table_rejects_small_radius(orc):
    with pytest.raises(RuntimeError):
        orc.eps_table(2, 0.5)


@pytest.mark.parametrize("dim,n,R,c", [(2, (24, 24), 4.0, (11.3, 12.7)), (2, (30, 30), 6.0, (15.0, 14.5)),
                                       (3, (16, 16, 16), 4.0, (7.3, 8.1, 7.6)), (3, (18, 18, 18), 5.0, (9.0, 8.5, 9.2))])
def test_table_map_area_and_agreement_with_fine_sampling(orc, dim, n, R, c):
    """Sum of eps over the nodes = area / volume of the particle (P10's statement for the table map), and
    node by node the table map agrees with a fine sampled map (S^D <= 255 points per cell) to the accuracy
    the discretisation allows."""
    pos = np.array(c, dtype=float).reshape(dim, 1)
    rad = np.array([R])
    bc = (0,) * dim
    code, pid = orc.map_particles_table(dim, n, bc, pos, rad)
    S = 15 if dim == 2 else 6
    cnt, pid_s = orc.map_particles(dim, n, bc, S, pos, rad)
    eps_t, eps_s = code / 255.0, cnt / float(S ** dim)
    vol = np.pi * R * R if dim == 2 else 4.0 / 3.0 * np.pi * R ** 3
    assert abs(eps_t.sum() - vol) / vol < 5e-3
    diff = np.abs(eps_t - eps_s)
    assert diff.max() < 0.05 and diff[(eps_s > 0) & (eps_s < 1)].mean() < 0.012
    # same interior; the covered sets differ only in cells the particle barely touches
    assert ((eps_t == 1) <= (eps_s > 0.97)).all() and ((eps_s == 1) <= (eps_t > 0.97)).all()
    assert (eps_s[eps_t == 0] < 0.03).all() and (eps_t[eps_s == 0] < 0.03).all()
    assert ((pid == 0) == (code > 0)).all()


def test_table_map_symmetries_and_translation(orc):
    """A particle centred on a node has a map with the symmetries of the square / cube; shifting the
    centre by whole nodes shifts the map (centres are multiples of 1/64, so the shift is exact)."""
    R = 4.0
    code, _ = orc.map_particles_table(2, (21, 21), (0, 0), np.array([[10.0], [10.0]]), np.array([R]))
    c2 = code[0]
    assert np.array_equal(c2, c2[::-1, :]) and np.array_equal(c2, c2[:, ::-1]) and np.array_equal(c2, c2.T)
    code3, _ = orc.map_particles_table(3, (13, 13, 13), (0, 0, 0), np.array([[6.0], [6.0], [6.0]]), np.array([R]))
    for perm in ((1, 0, 2), (0, 2, 1), (2, 1, 0)):
        assert np.array_equal(code3, code3.transpose(perm))
    assert np.array_equal(code3, code3[::-1]) and np.array_equal(code3, code3[:, ::-1]) and np.array_equal(code3, code3[:, :, ::-1])
    a, _ = orc.map_particles_table(2, (32, 32), (0, 0), np.array([[9.171875], [12.40625]]), np.array([R]))
    b, _ = orc.map_particles_table(2, (32, 32), (0, 0), np.array([[9.171875 + 5], [12.40625 + 30]]), np.array([R]))
    assert np.array_equal(np.roll(a, (30, 5), axis=(1, 2)), b)      # wraps through the periodic seam in y


def test_table_map_two_particles_share_a_node(orc):
    """R5 for the table map: codes of the two particles add (saturating at 255), the covering particle is
    the one with the larger code, ties -> lowest index."""
    R = 4.0
    n = (32, 16)
    one = lambda x, y: orc.map_particles_table(2, n, (0, 0), np.array([[x], [y]]), np.array([R]))[0].astype(int)
    xa, xb = 10.0, 18.3                                            # gap 0.3: both reach the cell of node 14
    both, pid = orc.map_particles_table(2, n, (0, 0), np.array([[xa, xb], [8.0, 8.0]]), np.array([R, R]))
    ca, cb = one(xa, 8.0), one(xb, 8.0)
    assert np.array_equal(both, np.minimum(ca + cb, 255))
    shared = (ca > 0) & (cb > 0)
    assert shared.any()
    assert np.array_equal(pid[shared], np.where(cb[shared] > ca[shared], 1, 0))
    # mirror-symmetric pair: equal codes on the shared nodes of the mid-plane -> lowest index wins
    both2, pid2 = orc.map_particles_table(2, n, (0, 0), np.array([[9.75, 18.25], [8.0, 8.0]]), np.array([R, R]))
    ca2, cb2 = one(9.75, 8.0), one(18.25, 8.0)
    tie = (ca2 > 0) & (ca2 == cb2)
    assert tie.any() and (pid2[tie] == 0).all()


def test_table_map_needs_one_radius(orc):
    with pytest.raises(RuntimeError):
        orc.map_particles_table(2, (32, 32), (0, 0), np.array([[8.0, 20.0], [8.0, 20.0]]), np.array([4.0, 5.0]))


def test_step_uses_the_table_denominator(orc):
    """eps = code/255 in the collision: uniform code c on every node, V_S = 0, uniform g reproduces the
    porous-medium closed form P5, u_n = (g/beta)(1 - (1-beta)^n), with beta(c/255, tau)."""
    n, tau, g, c = (6, 5), 0.8, (0.0, -1e-6), 77
    eps = c / 255.0
    beta = eps * (tau - 0.5) / ((1 - eps) + (tau - 0.5))
    f = orc.init(2, n)
    code = np.full((1, 5, 6), c, dtype=np.uint8)
    pid = np.zeros((1, 5, 6), dtype=np.int32)
    z = np.zeros((2, 1))
    for _ in range(40):
        f = orc.step(2, n, (0, 0), tau, g, 8, f, eps_cnt=code, pid=pid, pos=z, vel=z, omega=np.zeros((1, 1)),
                     eps_den=orc.TABLE_DEN)
    _, u = orc.macros(2, f)
    assert np.abs(u[1] - (g[1] / beta) * (1 - (1 - beta) ** 40)).max() < 1e-15
