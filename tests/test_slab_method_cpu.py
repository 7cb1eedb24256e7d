"""CPU check of the method behind the slab-wise full-protocol run of C4 (tests/test_gpu_full_protocol.py) and the
sampled boxes of tests/test_gpu_fullsize.py: the oracle on a y-slab (rows to compare + a rim of steps + 2R + 3 rows,
particles translated by inputs.y_slab) gives, inside the compared rows, bit for bit what the oracle gives on the whole
lattice -- maps, distributions, exchange vectors and the forces of the particles that lie wholly inside."""
import numpy as np

from paper_1011_2613_b200 import inputs
from test_gpu_full_protocol import slab_bounds


def test_slab_oracle_equals_whole_lattice_oracle_in_the_compared_rows(orc):
    w = inputs.c4(n=(150, 420), grid=(10, 28), steps=25)
    steps, K = w.steps, 3
    R = float(w.radius.max())
    rim = steps + int(2 * R) + 3
    nx, ny = w.n
    eps_w, pid_w = orc.map_particles(2, w.n, w.bc, w.subsamples, w.pos, w.radius)
    part = dict(eps_cnt=eps_w, pid=pid_w, pos=w.pos, vel=w.vel, omega=w.omega)
    fw = orc.init(2, w.n)
    for it in range(steps):
        fw, sw = orc.step(2, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, fw, want_s=True, **part)
    Fw, Tw, _, _ = orc.forces(2, w.n, w.bc, sw, pid_w, w.pos)
    covered_rows = np.zeros(ny, dtype=bool)
    covered_particles = np.zeros(w.P, dtype=bool)
    for k in range(K):
        y0, y1 = slab_bounds(ny, k, K, int(2 * R) + 6)
        lo, hi = max(0, y0 - rim), min(ny, y1 + rim)
        assert hi - lo < ny                                      # a real cut, with artificial edges
        pos, vel, om, rad, mass, idx = inputs.y_slab(w, lo, hi)
        sn, sbc = (nx, hi - lo), (w.bc[0], 1)
        eps, pid = orc.map_particles(2, sn, sbc, w.subsamples, pos, rad)
        f = orc.init(2, sn)
        for it in range(steps):
            f, s = orc.step(2, sn, sbc, w.tau, w.g_fluid, w.subsamples, f, eps_cnt=eps, pid=pid, pos=pos, vel=vel,
                            omega=om, want_s=True)
        rows = slice(y0 - lo, y1 - lo)
        assert np.array_equal(eps[0, rows], eps_w[0, y0:y1])
        assert np.array_equal(np.where(pid >= 0, idx[np.maximum(pid, 0)], -1)[0, rows], pid_w[0, y0:y1])
        assert np.array_equal(f[:, 0, rows], fw[:, 0, y0:y1])
        assert np.array_equal(s[:, 0, rows], sw[:, 0, y0:y1])
        assert not np.array_equal(f[:, 0, :3], fw[:, 0, lo:lo + 3]) or lo == 0      # the artificial edge does differ
        F, T, _, _ = orc.forces(2, sn, sbc, s, pid, pos)
        gy = pos[1] + lo
        keep = ((gy - rad - 2 >= y0) | (y0 == 0)) & ((gy + rad + 2 <= y1 - 1) | (y1 == ny))   # true walls need no margin
        assert np.array_equal(F[:, keep], Fw[:, idx[keep]]) and np.array_equal(T[:, keep], Tw[:, idx[keep]])
        covered_rows[y0:y1] = True
        covered_particles[idx[keep]] = True
    assert covered_rows.all() and covered_particles.all()
