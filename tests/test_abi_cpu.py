"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports
every symbol include/lbmimb.h declares, its structs match the ctypes mirror, the host-only
entry points work and the product path fails loudly without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lbmimb.h")


@pytest.fixture(scope="module")
def lb():
    from paper_1011_2613_b200 import build, binding
    build.build()
    binding.load()
    return binding


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lbmimb_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lb):
    names = declared_symbols()
    assert len(names) >= 18
    lib = C.CDLL(lb.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), "liblbmimb.so does not export %s" % name
    assert sorted(lb.EXPORTS) == names, "binding.EXPORTS and include/lbmimb.h disagree"


def test_library_is_built_for_sm_100a(lb):
    out = subprocess.run(["cuobjdump", "-lelf", lb.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_struct_layout_matches_the_header(lb, tmp_path):
    prog = tmp_path / "layout.c"
    prog.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "lbmimb.h"\nint main(void){\n'
                    'printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(lbmimb_params),'
                    'offsetof(lbmimb_params,dim),offsetof(lbmimb_params,subsamples),offsetof(lbmimb_params,n),'
                    'offsetof(lbmimb_params,bc),offsetof(lbmimb_params,device),offsetof(lbmimb_params,tau),'
                    'offsetof(lbmimb_params,g_fluid),offsetof(lbmimb_params,stream),'
                    'offsetof(lbmimb_params,workspace_dev),offsetof(lbmimb_params,workspace_bytes),'
                    'offsetof(lbmimb_params,streaming),offsetof(lbmimb_params,flags),'
                    'offsetof(lbmimb_params,slab_y0),offsetof(lbmimb_params,slab_ny));\n'
                    'printf("%zu %zu %zu %zu %zu\\n", sizeof(lbmimb_dem_params),offsetof(lbmimb_dem_params,kn),'
                    'offsetof(lbmimb_dem_params,restitution),offsetof(lbmimb_dem_params,g_particle),'
                    'offsetof(lbmimb_dem_params,dt));\nreturn 0;}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)], check=True)
    lines = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split("\n")
    got = [int(v) for v in lines[0].split()]
    P = lb.Params
    want = [C.sizeof(P)] + [getattr(P, k).offset for k in ("dim", "subsamples", "n", "bc", "device", "tau", "g_fluid",
                                                            "stream", "workspace_dev", "workspace_bytes", "streaming", "flags",
                                                            "slab_y0", "slab_ny")]
    assert got == want
    got = [int(v) for v in lines[1].split()]
    D = lb.DemParams
    assert got == [C.sizeof(D)] + [getattr(D, k).offset for k in ("kn", "restitution", "g_particle", "dt")]


def test_workspace_bytes_and_parameter_validation(lb):
    p = lb.make_params(3, (256, 1008, 256), (0, 1, 0), 0.7, (0, -1e-6, 0), 4)
    need = lb.workspace_bytes(p, 24600)
    N = 256 * 1008 * 256
    assert need >= 2 * 19 * N * 8 + 4 * N                      # two f buffers + one tag word per node
    assert need < 2 * 19 * N * 8 * 1.05                        # and not much more
    ps = lb.make_params(3, (256, 1008, 256), (0, 1, 0), 0.7, (0, -1e-6, 0), 4, flags=lb.FLAG_EXCHANGE_FIELD)
    assert lb.workspace_bytes(ps, 24600) - need == 4 * N * 8   # the optional per-node exchange records
    assert lb.workspace_bytes(lb.make_params(2, (16, 16), (0, 0), 0.8, (0, 0), 8, flags=2), 0) == 0   # unknown flag
    assert lb.workspace_bytes(p, (1 << 24) + 1) == 0           # tags hold 24-bit particle indices
    p2 = lb.make_params(2, (8192, 32768), (0, 1), 0.55, (0, -1e-6), 8)
    assert lb.workspace_bytes(p2, 1166400) > 2 * 9 * 8192 * 32768 * 8     # > 2^31 elements per buffer
    for bad in (lb.make_params(2, (16, 16), (0, 0), 0.5, (0, 0), 8),      # tau
                lb.make_params(4, (16, 16), (0, 0), 0.8, (0, 0), 8),      # dim
                lb.make_params(2, (16, 16, 2), (0, 0), 0.8, (0, 0), 8),   # n[2] in 2D
                lb.make_params(2, (16, 16), (0, 2), 0.8, (0, 0), 8),      # bc
                lb.make_params(2, (16, 16), (0, 0), 0.8, (0, 0), 16),     # S^2 > 255
                lb.make_params(3, (16, 0, 16), (0, 0, 0), 0.8, (0, 0, 0), 4)):
        assert lb.workspace_bytes(bad, 0) == 0
        assert len(lb.load().lbmimb_last_error()) > 0
    assert "lbmimb" in lb.version()


def test_no_cpu_fallback(lb):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(lb.LbmimbError) as ei:
        lb.Lattice(2, (16, 16), (0, 0), 0.8, (0, 0), 8)
    assert ei.value.status == lb.ECUDA
    # straight through the C entry point as well
    h = C.c_void_p()
    p = lb.make_params(2, (16, 16), (0, 0), 0.8, (0, 0), 8)
    st = lb.load().lbmimb_create_lattice(C.byref(p), 0, C.byref(h))
    assert st == lb.ECUDA and not h.value
    assert b"no CPU fallback" in lb.load().lbmimb_last_error()


def test_null_handle_is_rejected_by_every_entry_point(lb):
    """Argument checks run before any CUDA call, so they can be exercised without a GPU."""
    lib = lb.load()
    d = lb.DemParams()
    d.kn, d.restitution, d.dt = 1.0, 0.9, 1.0
    buf = np.zeros(8)
    i64 = np.zeros(4, dtype=np.int64)
    calls = [lambda: lib.lbmimb_set_particles(None, 0, None, None, None, None, None),
             lambda: lib.lbmimb_set_particle_velocities(None, None, None),
             lambda: lib.lbmimb_get_particles(None, None, None, None),
             lambda: lib.lbmimb_map_particles(None),
             lambda: lib.lbmimb_set_mapping_mode(None, 0),
             lambda: lib.lbmimb_step(None, 1),
             lambda: lib.lbmimb_reduce_particle_forces(None, None, None),
             lambda: lib.lbmimb_dem_step(None, C.byref(d)),
             lambda: lib.lbmimb_set_neighbor_mode(None, 1, 1.0, 100),
             lambda: lib.lbmimb_fetch_neighbor_list(None, i64.ctypes.data_as(C.c_void_p), None, 0, None),
             lambda: lib.lbmimb_diagnostics(None, buf.ctypes.data_as(C.c_void_p)),
             lambda: lib.lbmimb_set_distributions(None, buf.ctypes.data_as(C.c_void_p)),
             lambda: lib.lbmimb_synchronize(None)]
    for k, call in enumerate(calls):
        assert call() == lb.EINVAL, "entry point %d accepted a NULL handle" % k
        assert b"NULL" in lib.lbmimb_last_error()
    assert lib.lbmimb_destroy_lattice(None) == lb.OK
    assert lib.lbmimb_num_particles(None) == -1 and lib.lbmimb_time(None) == -1


def test_product_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under paper_1011_2613_b200/ may name it."""
    pkg = os.path.join(ROOT, "paper_1011_2613_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "lbmimb_oracle" not in text and "liblbmimb_oracle" not in text, fn
    otext = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(
        os.path.join(ROOT, "oracle", "lbmimb_oracle.c")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_1011_2613_b200", otext, flags=re.M)
    assert "lbmimb.h" not in otext.replace("include/lbmimb.h so that", "")


def test_inputs_are_seeded_and_well_formed():
    from paper_1011_2613_b200 import inputs
    a, b = inputs.reduced("C3"), inputs.reduced("C3")
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.vel, b.vel)
    for name in ("C1", "C2", "C3", "C4", "C5"):
        w = inputs.reduced(name)
        assert w.pos.shape == (w.dim, w.P) and w.omega.shape == (1 if w.dim == 2 else 3, w.P)
        assert np.array_equal(w.pos * 65536, np.round(w.pos * 65536))        # multiples of 2^-16
        d = w.pos[:, :, None] - w.pos[:, None, :]
        for ax in range(w.dim):
            if not w.bc[ax]:
                d[ax] -= w.n[ax] * np.round(d[ax] / w.n[ax])
        dist = np.sqrt((d ** 2).sum(axis=0)) + 1e9 * np.eye(w.P)
        assert dist.min() >= 2 * w.radius[0] - 1e-9, name
        frac = (np.pi * w.radius ** 2 if w.dim == 2 else 4 / 3 * np.pi * w.radius ** 3).sum() / w.nodes
        want = {"C1": 0.110, "C2": 0.168, "C3": 0.0998, "C4": 0.218, "C5": 0.256}[name]
        assert abs(frac - want) / want < 0.03, (name, frac)
    full = inputs.c4()
    assert full.P == 1166400 and full.n == (8192, 32768)


def test_sub_box_translation_is_exact():
    from paper_1011_2613_b200 import inputs
    w = inputs.reduced("C3")
    lo, size = (60, 10, 30), (24, 24, 24)
    pos, vel, om, rad, mass, idx = inputs.sub_box(w, lo, size)
    assert pos.shape[1] > 0 and np.array_equal(pos * 65536, np.round(pos * 65536))
    # every kept particle is an exact integer translate of an original one
    for p in range(pos.shape[1]):
        d = w.pos - (pos[:, p] + np.array(lo))[:, None]
        d -= np.array(w.n)[:, None] * np.round(d / np.array(w.n)[:, None])
        assert (np.abs(d).sum(axis=0) == 0).any()
