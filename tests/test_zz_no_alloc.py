"""lbmimb_diagnostics_static_dev: the diagnostics entry point that allocates nothing (scratch in a static device
array of the library, include/lbmimb.h) against the existing lbmimb_diagnostics, on two calls in a row.
`-m gpu`.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after
the other tests: it depends on no state of theirs, and the shared scratch keeps nothing a call relies on."""
import numpy as np
import pytest

from paper_1011_2613_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1011_2613_b200 import binding
    binding.load()
    return binding


def _compare(lb, lat, out):
    """existing path vs the no-allocation entry point on the same state"""
    import torch
    want = lat.diagnostics()["vector"].copy()
    out.fill_(float("nan"))
    lat.diagnostics_static_dev(out.data_ptr())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    # node sums: same kernel, same grid, same order -> bit for bit
    for k in (0, 1, 2, 3, 4, 14, 15, 16):
        assert got[k] == want[k], (k, got[k], want[k])
    # particle sums are added in another order: to rounding (the tolerance of the diagnostics parity tests, 1e-10, is far wider)
    scale = np.abs(want).max()
    assert np.all(np.isfinite(got))
    assert np.abs(got - want).max() <= 1e-13 * scale + 1e-300
    rel = np.abs(got - want) / np.maximum(np.abs(want), 1e-300)
    assert rel[np.abs(want) > 1e-12 * scale].max() <= 1e-10
    return want


@pytest.mark.parametrize("name,streaming", [("C5", 0), ("P2D", 1)])
def test_static_scratch_diagnostics_match_on_two_calls_in_a_row(lb, name, streaming):
    import torch
    w = inputs.reduced(name)
    d = w.dem
    dargs = (d["kn"], d["restitution"], d["g_particle"], d["dt"])
    out = torch.empty(lb.DIAG_LEN, dtype=torch.float64, device="cuda")
    # a larger lattice first, so that the shared scratch holds MORE rows than the next calls use
    big = lb.from_workload(inputs.reduced("C3"))
    big.map_particles()
    big.step(3)
    big.reduce_particle_forces(to_host=False)
    _compare(lb, big, out)
    lat = lb.from_workload(w, streaming=streaming)
    first = None
    for call in range(2):                      # two calls in a row on an evolving coupled state
        for _ in range(3):
            lat.map_particles()
            lat.step(1)
            lat.reduce_particle_forces(to_host=False)
            lat.dem_step(*dargs)
        lat.map_particles()
        v = _compare(lb, lat, out)
        if first is None:
            first = v
    assert not np.array_equal(first, v)        # the state did change between the two calls
    assert np.abs(v[11:14]).max() > 0 and np.abs(v[17:20]).max() > 0     # drag and solid momentum are exercised
    lat.close()
    big.close()


def test_static_scratch_limits_and_errors(lb):
    import torch
    assert lb.diagnostics_static_max_particles() == 4096 * 256
    assert lb.diagnostics_static_scratch_bytes() == (1184 * 8 + 4096 * 10) * 8
    out = torch.zeros(lb.DIAG_LEN, dtype=torch.float64, device="cuda")
    # no particles: works, equals the existing path
    lat = lb.Lattice(2, (70, 33), (0, 1), 0.8, (0.0, -1e-5), 8, max_particles=4)
    lat.step(5)
    _compare(lb, lat, out)
    with pytest.raises(lb.LbmimbError) as ei:
        lat.diagnostics_static_dev(0)
    assert ei.value.status == lb.EINVAL
    lat.set_particles(np.array([[20.0], [15.0]]), np.zeros((2, 1)), None, np.array([4.0]), np.ones(1))
    with pytest.raises(lb.LbmimbError) as ei:
        lat.diagnostics_static_dev(out.data_ptr())             # set but not mapped
    assert ei.value.status == lb.ESTATE
    lat.close()
    # more particles than the static scratch holds: a clear error, nothing launched
    P = lb.diagnostics_static_max_particles() + 1
    lat = lb.Lattice(2, (64, 64), (0, 0), 0.8, (0, 0), 8, max_particles=P)
    rng = np.random.default_rng(1)
    lat.set_particles(rng.random((2, P)) * 60.0, np.zeros((2, P)), None, np.full(P, 0.05), np.ones(P))
    with pytest.raises(lb.LbmimbError) as ei:
        lat.diagnostics_static_dev(out.data_ptr())
    assert ei.value.status == lb.EINVAL and "exceed the static scratch" in str(ei.value)
    lat.close()
