"""Thin ctypes binding of the C-ABI library include/lbmimb.h (liblbmimb.so).

Same names as the C entry points, argument marshalling only: every step of the
path runs in the CUDA kernels.  PyTorch supplies the device workspace buffer and
the stream (plumbing); numpy arrays are the host buffers.  There is NO CPU
fallback: if the built library is missing, loading raises; if no CUDA device is
present, create_lattice fails with LBMIMB_ECUDA.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblbmimb.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = range(5)
FIELD_F, FIELD_RHO, FIELD_U, FIELD_EPS_CNT, FIELD_PID, FIELD_S = range(6)
MAP_SAMPLING, MAP_TABLE = 0, 1
STREAM_AB, STREAM_AA = 0, 1
FLAG_EXCHANGE_FIELD = 1
NEIGHBOR_CELLS, NEIGHBOR_VERLET = 0, 1
TABLE_DEN = 255
TABLE_SHAPE = {2: (128, 32), 3: (128, 16, 16)}      # LBMIMB_TABLE_ND/NT_* of include/lbmimb.h

EXPORTS = [
    "lbmimb_workspace_bytes", "lbmimb_create_lattice", "lbmimb_destroy_lattice", "lbmimb_set_particles",
    "lbmimb_set_particle_velocities", "lbmimb_get_particles", "lbmimb_num_particles", "lbmimb_map_particles",
    "lbmimb_step", "lbmimb_reduce_particle_forces", "lbmimb_dem_step", "lbmimb_fetch_fields",
    "lbmimb_set_distributions", "lbmimb_set_particles_dev", "lbmimb_reduce_particle_forces_dev",
    "lbmimb_synchronize", "lbmimb_time", "lbmimb_launch_count", "lbmimb_last_error", "lbmimb_version",
    "lbmimb_set_mapping_mode", "lbmimb_fetch_eps_table", "lbmimb_diagnostics",
    "lbmimb_set_neighbor_mode", "lbmimb_fetch_neighbor_list", "lbmimb_run_coupled",
    "lbmimb_halo_count", "lbmimb_slab_ghost_rows", "lbmimb_pack_halo", "lbmimb_unpack_halo",
    "lbmimb_force_sums_count", "lbmimb_export_force_sums_dev", "lbmimb_import_force_sums_dev",
    "lbmimb_diagnostics_static_dev", "lbmimb_diagnostics_static_max_particles",
    "lbmimb_diagnostics_static_scratch_bytes",
]
DIAG_LEN = 20


class Params(C.Structure):
    _fields_ = [("dim", C.c_int32), ("subsamples", C.c_int32), ("n", C.c_int64 * 3), ("bc", C.c_int32 * 3),
                ("device", C.c_int32), ("tau", C.c_double), ("g_fluid", C.c_double * 3), ("stream", C.c_void_p),
                ("workspace_dev", C.c_void_p), ("workspace_bytes", C.c_uint64), ("streaming", C.c_int32),
                ("flags", C.c_int32), ("slab_y0", C.c_int64), ("slab_ny", C.c_int64)]


class DemParams(C.Structure):
    _fields_ = [("kn", C.c_double), ("restitution", C.c_double), ("g_particle", C.c_double * 3),
                ("dt", C.c_double)]


class LbmimbError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("lbmimb status %d: %s" % (status, msg))
        self.status = status


_lib = None


def load():
    """Loads liblbmimb.so (fails loudly when it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_1011_2613_b200.build` (nvcc, sm_100a); "
                          "there is no CPU fallback" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, dp = C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_double)
    lib.lbmimb_workspace_bytes.restype = C.c_uint64
    lib.lbmimb_workspace_bytes.argtypes = [C.POINTER(Params), i64]
    lib.lbmimb_create_lattice.argtypes = [C.POINTER(Params), i64, C.POINTER(vp)]
    lib.lbmimb_destroy_lattice.argtypes = [vp]
    lib.lbmimb_set_particles.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    lib.lbmimb_set_particles_dev.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    lib.lbmimb_set_particle_velocities.argtypes = [vp, vp, vp]
    lib.lbmimb_get_particles.argtypes = [vp, vp, vp, vp]
    lib.lbmimb_num_particles.restype = i64
    lib.lbmimb_num_particles.argtypes = [vp]
    lib.lbmimb_map_particles.argtypes = [vp]
    lib.lbmimb_set_mapping_mode.argtypes = [vp, i32]
    lib.lbmimb_fetch_eps_table.argtypes = [vp, vp, i64]
    lib.lbmimb_step.argtypes = [vp, i32]
    lib.lbmimb_reduce_particle_forces.argtypes = [vp, vp, vp]
    lib.lbmimb_reduce_particle_forces_dev.argtypes = [vp, vp, vp]
    lib.lbmimb_dem_step.argtypes = [vp, C.POINTER(DemParams)]
    lib.lbmimb_run_coupled.argtypes = [vp, C.POINTER(DemParams), i32]
    lib.lbmimb_set_neighbor_mode.argtypes = [vp, i32, C.c_double, i64]
    lib.lbmimb_fetch_neighbor_list.argtypes = [vp, vp, vp, i64, vp]
    lib.lbmimb_fetch_fields.argtypes = [vp, i32, C.POINTER(i64), C.POINTER(i64), vp]
    lib.lbmimb_set_distributions.argtypes = [vp, vp]
    lib.lbmimb_diagnostics.argtypes = [vp, vp]
    lib.lbmimb_diagnostics_static_dev.argtypes = [vp, vp]
    lib.lbmimb_diagnostics_static_max_particles.restype = i64
    lib.lbmimb_diagnostics_static_max_particles.argtypes = []
    lib.lbmimb_diagnostics_static_scratch_bytes.restype = i64
    lib.lbmimb_diagnostics_static_scratch_bytes.argtypes = []
    lib.lbmimb_halo_count.restype = i64
    lib.lbmimb_halo_count.argtypes = [vp]
    lib.lbmimb_slab_ghost_rows.restype = i32
    lib.lbmimb_slab_ghost_rows.argtypes = [vp, i32]
    lib.lbmimb_pack_halo.argtypes = [vp, i32, vp]
    lib.lbmimb_unpack_halo.argtypes = [vp, i32, vp]
    lib.lbmimb_force_sums_count.restype = i64
    lib.lbmimb_force_sums_count.argtypes = [vp]
    lib.lbmimb_export_force_sums_dev.argtypes = [vp, vp]
    lib.lbmimb_import_force_sums_dev.argtypes = [vp, vp]
    lib.lbmimb_synchronize.argtypes = [vp]
    lib.lbmimb_time.restype = i64
    lib.lbmimb_time.argtypes = [vp]
    lib.lbmimb_launch_count.restype = i64
    lib.lbmimb_launch_count.argtypes = [vp]
    lib.lbmimb_last_error.restype = C.c_char_p
    lib.lbmimb_version.restype = C.c_char_p
    for name in EXPORTS:
        fn = getattr(lib, name)
        if fn.restype is C.c_int:       # lbmimb_status
            fn.restype = C.c_int
    _lib = lib
    return lib


def _check(st):
    if st != OK:
        raise LbmimbError(st, load().lbmimb_last_error().decode())


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def version():
    return load().lbmimb_version().decode()


def diagnostics_static_max_particles():
    return int(load().lbmimb_diagnostics_static_max_particles())


def diagnostics_static_scratch_bytes():
    return int(load().lbmimb_diagnostics_static_scratch_bytes())


def make_params(dim, n, bc, tau, g_fluid, subsamples, device=0, stream=0, workspace_dev=0, workspace_bytes=0,
                streaming=STREAM_AB, flags=0, slab=None):
    """slab = (y0, global_ny): this lattice owns rows [y0, y0 + n[1]) of a global lattice of global_ny rows."""
    p = Params()
    p.dim = dim
    p.subsamples = subsamples
    n = list(n) + [1] * (3 - len(n))
    bc = list(bc) + [0] * (3 - len(bc))
    g = list(g_fluid) + [0.0] * (3 - len(g_fluid))
    for a in range(3):
        p.n[a] = int(n[a])
        p.bc[a] = int(bc[a])
        p.g_fluid[a] = float(g[a])
    p.device = device
    p.tau = tau
    p.stream = stream or None
    p.workspace_dev = workspace_dev or None
    p.workspace_bytes = workspace_bytes
    p.streaming = streaming
    p.flags = flags
    p.slab_y0, p.slab_ny = (int(slab[0]), int(slab[1])) if slab else (0, 0)
    return p


def workspace_bytes(params, max_particles):
    return int(load().lbmimb_workspace_bytes(C.byref(params), max_particles))


class Lattice:
    """Owner of one lbmimb_lattice handle.  Method names = C entry points without the prefix."""

    def __init__(self, dim, n, bc, tau, g_fluid, subsamples, max_particles=0, device=0, use_torch=True,
                 streaming=STREAM_AB, flags=0, slab=None):
        self.lib = load()
        self.dim = dim
        self.n = tuple(int(v) for v in n) + (1,) * (3 - len(n))
        self.Q = 9 if dim == 2 else 19
        self.nt = 1 if dim == 2 else 3
        self._ws = None
        stream = 0
        ws_ptr, ws_bytes = 0, 0
        probe = make_params(dim, n, bc, tau, g_fluid, subsamples, device, streaming=streaming, flags=flags, slab=slab)
        if use_torch:
            import torch
            if not torch.cuda.is_available():
                raise LbmimbError(ECUDA, "no CUDA device: the lbmimb path has no CPU fallback")
            need = workspace_bytes(probe, max_particles)
            if need == 0:
                _check(EINVAL)
            with torch.cuda.device(device):
                stream = torch.cuda.current_stream().cuda_stream
                self._ws = torch.empty(need + 256, dtype=torch.uint8, device="cuda:%d" % device)
            ws_ptr = (self._ws.data_ptr() + 255) & ~255
            ws_bytes = need
        self.params = make_params(dim, n, bc, tau, g_fluid, subsamples, device, stream, ws_ptr, ws_bytes, streaming, flags,
                                  slab)
        h = C.c_void_p()
        _check(self.lib.lbmimb_create_lattice(C.byref(self.params), max_particles, C.byref(h)))
        self.h = h

    # -- lifetime ---------------------------------------------------------
    def destroy_lattice(self):
        if getattr(self, "h", None):
            self.lib.lbmimb_destroy_lattice(self.h)
            self.h = None
            self._ws = None

    close = destroy_lattice

    def __del__(self):
        try:
            self.destroy_lattice()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy_lattice()

    # -- particles ----------------------------------------------------------
    def set_particles(self, pos, vel, omega, radius, mass):
        pos, vel, omega, radius, mass = map(_f64, (pos, vel, omega, radius, mass))
        P = 0 if radius is None else int(radius.shape[0])
        self._keep = (pos, vel, omega, radius, mass)
        _check(self.lib.lbmimb_set_particles(self.h, P, _hp(pos), _hp(vel), _hp(omega), _hp(radius), _hp(mass)))

    def set_particles_dev(self, P, pos, vel, omega, radius, mass):
        """Device pointers (ints), e.g. torch tensors' data_ptr()."""
        _check(self.lib.lbmimb_set_particles_dev(self.h, P, pos, vel, omega or None, radius, mass))

    def set_particle_velocities(self, vel, omega):
        vel, omega = _f64(vel), _f64(omega)
        _check(self.lib.lbmimb_set_particle_velocities(self.h, _hp(vel), _hp(omega)))

    def num_particles(self):
        return int(self.lib.lbmimb_num_particles(self.h))

    def get_particles(self):
        P = self.num_particles()
        pos, vel, om = np.empty((self.dim, P)), np.empty((self.dim, P)), np.empty((self.nt, P))
        _check(self.lib.lbmimb_get_particles(self.h, _hp(pos), _hp(vel), _hp(om)))
        return pos, vel, om

    # -- the path -----------------------------------------------------------
    def set_mapping_mode(self, mode):
        _check(self.lib.lbmimb_set_mapping_mode(self.h, mode))

    def fetch_eps_table(self):
        out = np.empty(TABLE_SHAPE[self.dim], dtype=np.uint8)
        _check(self.lib.lbmimb_fetch_eps_table(self.h, _hp(out), out.nbytes))
        return out

    def map_particles(self):
        _check(self.lib.lbmimb_map_particles(self.h))

    def step(self, nsteps=1):
        _check(self.lib.lbmimb_step(self.h, nsteps))

    def reduce_particle_forces(self, to_host=True, out=None):
        if not to_host:
            _check(self.lib.lbmimb_reduce_particle_forces(self.h, None, None))
            return None
        P = self.num_particles()
        if out is None:
            out = (np.empty((self.dim, P)), np.empty((self.nt, P)))
        _check(self.lib.lbmimb_reduce_particle_forces(self.h, _hp(out[0]), _hp(out[1])))
        return out

    def reduce_particle_forces_dev(self, force_ptr, torque_ptr):
        _check(self.lib.lbmimb_reduce_particle_forces_dev(self.h, force_ptr or None, torque_ptr or None))

    @staticmethod
    def _dem_params(kn, restitution, g_particle, dt):
        d = DemParams()
        d.kn, d.restitution, d.dt = kn, restitution, dt
        g = list(g_particle) + [0.0] * (3 - len(g_particle))
        for a in range(3):
            d.g_particle[a] = g[a]
        return d

    def dem_step(self, kn, restitution, g_particle, dt=1.0):
        _check(self.lib.lbmimb_dem_step(self.h, C.byref(self._dem_params(kn, restitution, g_particle, dt))))

    def run_coupled(self, nsteps, kn, restitution, g_particle, dt=1.0):
        _check(self.lib.lbmimb_run_coupled(self.h, C.byref(self._dem_params(kn, restitution, g_particle, dt)), nsteps))

    def set_neighbor_mode(self, mode, skin=0.0, every=0):
        _check(self.lib.lbmimb_set_neighbor_mode(self.h, mode, float(skin), int(every)))

    def fetch_neighbor_list(self):
        """(start[P+1] int64, items int32, info) with info = dict(valid, age, builds)."""
        P = self.num_particles()
        start = np.zeros(P + 1, dtype=np.int64)
        info = np.zeros(4, dtype=np.int64)
        items = np.zeros(max(16 * P, 1), dtype=np.int32)
        st = self.lib.lbmimb_fetch_neighbor_list(self.h, _hp(start), _hp(items), items.size, _hp(info))
        if st == EINVAL and info[3] > items.size:      # grow to the size the library reported
            items = np.zeros(int(info[3]), dtype=np.int32)
            st = self.lib.lbmimb_fetch_neighbor_list(self.h, _hp(start), _hp(items), items.size, _hp(info))
        _check(st)
        return start, items[:int(start[-1])].copy(), {"valid": bool(info[0]), "age": int(info[1]), "builds": int(info[2])}

    def fetch_fields(self, what, lo=None, hi=None, out=None):
        lo = [0, 0, 0] if lo is None else list(lo) + [0] * (3 - len(lo))
        hi = list(self.n) if hi is None else list(hi) + [1] * (3 - len(hi))
        ext = tuple(hi[a] - lo[a] for a in (2, 1, 0))
        comps, dt = {FIELD_F: (self.Q, np.float64), FIELD_RHO: (0, np.float64), FIELD_U: (self.dim, np.float64),
                     FIELD_EPS_CNT: (0, np.uint8), FIELD_PID: (0, np.int32), FIELD_S: (self.dim, np.float64)}[what]
        shape = ((comps,) if comps else ()) + ext
        if out is None:
            out = np.empty(shape, dtype=dt)
        assert out.shape == shape and out.dtype == dt and out.flags.c_contiguous
        _check(self.lib.lbmimb_fetch_fields(self.h, what, (C.c_int64 * 3)(*lo), (C.c_int64 * 3)(*hi), _hp(out)))
        return out

    def set_distributions(self, f):
        f = _f64(f)
        rows = self.n[1] + (self.slab_ghost_rows(0) + self.slab_ghost_rows(1) if self.params.slab_ny else 0)
        assert f.size == self.Q * self.n[0] * rows * self.n[2]      # a slab takes its STORED rows (ghosts included)
        _check(self.lib.lbmimb_set_distributions(self.h, _hp(f)))

    def diagnostics(self):
        """The 20 doubles of lbmimb_diagnostics and the same named views as a dict."""
        out = np.zeros(DIAG_LEN)
        _check(self.lib.lbmimb_diagnostics(self.h, _hp(out)))
        D = self.dim
        return {"gas_area": out[0], "mass": out[1], "gas_velocity": out[2:2 + D], "solid_velocity": out[5:5 + D],
                "slip": out[8:8 + D], "drag": out[11:11 + D], "fluid_momentum": out[14:14 + D],
                "solid_momentum": out[17:17 + D], "vector": out}

    def diagnostics_static_dev(self, out_ptr):
        """The 20 doubles of lbmimb_diagnostics into a DEVICE buffer; no allocation, no synchronisation."""
        _check(self.lib.lbmimb_diagnostics_static_dev(self.h, out_ptr))

    # -- slabs (NEXT-4): device pointers in, device pointers out ------------------------------------
    def halo_count(self):
        return int(self.lib.lbmimb_halo_count(self.h))

    def slab_ghost_rows(self, side):
        return int(self.lib.lbmimb_slab_ghost_rows(self.h, side))

    def pack_halo(self, side, dst_ptr):
        _check(self.lib.lbmimb_pack_halo(self.h, side, dst_ptr))

    def unpack_halo(self, side, src_ptr):
        _check(self.lib.lbmimb_unpack_halo(self.h, side, src_ptr))

    def force_sums_count(self):
        return int(self.lib.lbmimb_force_sums_count(self.h))

    def export_force_sums_dev(self, dst_ptr):
        _check(self.lib.lbmimb_export_force_sums_dev(self.h, dst_ptr))

    def import_force_sums_dev(self, src_ptr):
        _check(self.lib.lbmimb_import_force_sums_dev(self.h, src_ptr))

    def synchronize(self):
        _check(self.lib.lbmimb_synchronize(self.h))

    def time(self):
        return int(self.lib.lbmimb_time(self.h))

    def launch_count(self):
        return int(self.lib.lbmimb_launch_count(self.h))


def from_workload(w, device=0, max_particles=None, map_mode=MAP_SAMPLING, streaming=STREAM_AB, flags=0):
    """Lattice for a paper_1011_2613_b200.inputs.Workload with its particles set (not yet mapped)."""
    lat = Lattice(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples,
                  max_particles=w.P if max_particles is None else max_particles, device=device, streaming=streaming,
                  flags=flags)
    if map_mode != MAP_SAMPLING:
        lat.set_mapping_mode(map_mode)
    if w.P:
        lat.set_particles(w.pos, w.vel, w.omega, w.radius, w.mass)
    return lat
