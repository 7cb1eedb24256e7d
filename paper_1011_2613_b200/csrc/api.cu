// C-ABI entry points of liblbmimb.so (include/lbmimb.h): argument checks, device
// memory layout, state machine.  All per-node and per-particle arithmetic of the method runs
// in the kernels of lattice.cu / particles.cu.  The host evaluates parameters only: 1/tau and
// tau g (collide.cuh), the cell-list geometry, and the 256-entry table beta(n_s / S^D, tau) of
// PAPER.md:41 (fill_beta_table below), which is uploaded once per lattice / mapping mode.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "lbmimb_internal.cuh"

namespace lbmimb {

static thread_local char g_err[512] = "";

lbmimb_status fail(lbmimb_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}

lbmimb_status cuda_fail(cudaError_t e, const char *what) {
  snprintf(g_err, sizeof(g_err), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  return e == cudaErrorMemoryAllocation ? LBMIMB_ENOMEM : LBMIMB_ECUDA;
}

static uint64_t align_up(uint64_t v) { return (v + 255) & ~(uint64_t)255; }

static bool valid_params(const lbmimb_params *p, int64_t maxp) {
  if (!p) return fail(LBMIMB_EINVAL, "params is NULL"), false;
  if (p->dim != 2 && p->dim != 3) return fail(LBMIMB_EINVAL, "dim must be 2 or 3"), false;
  for (int a = 0; a < 3; ++a) {
    if (p->n[a] < 1 || p->n[a] > 0x7fffffff) return fail(LBMIMB_EINVAL, "n[%d] out of range", a), false;
    if (p->bc[a] != 0 && p->bc[a] != 1) return fail(LBMIMB_EINVAL, "bc[%d] must be 0 or 1", a), false;
  }
  if (p->dim == 2 && p->n[2] != 1) return fail(LBMIMB_EINVAL, "n[2] must be 1 in 2D"), false;
  if (!(p->tau > 0.5) || !std::isfinite(p->tau)) return fail(LBMIMB_EINVAL, "tau must be > 0.5"), false;
  for (int a = 0; a < 3; ++a)
    if (!std::isfinite(p->g_fluid[a])) return fail(LBMIMB_EINVAL, "g_fluid not finite"), false;
  int64_t sd = 1;
  if (p->subsamples < 1) return fail(LBMIMB_EINVAL, "subsamples must be >= 1"), false;
  for (int a = 0; a < p->dim; ++a) sd *= p->subsamples;
  if (sd > 255) return fail(LBMIMB_EINVAL, "subsamples^dim must be <= 255"), false;
  if (p->streaming != LBMIMB_STREAM_AB && p->streaming != LBMIMB_STREAM_AA)
    return fail(LBMIMB_EINVAL, "streaming must be LBMIMB_STREAM_AB or LBMIMB_STREAM_AA"), false;
  if ((p->flags & ~LBMIMB_FLAG_EXCHANGE_FIELD) != 0) return fail(LBMIMB_EINVAL, "unknown bit in flags"), false;
  if (p->slab_ny != 0) {
    if (p->slab_ny < 0 || p->slab_ny > 0x7fffffff || p->slab_y0 < 0 || p->slab_y0 + p->n[1] > p->slab_ny)
      return fail(LBMIMB_EINVAL, "slab rows [%lld, %lld) do not fit a lattice of %lld rows", (long long)p->slab_y0,
                  (long long)(p->slab_y0 + p->n[1]), (long long)p->slab_ny), false;
    if (p->streaming != LBMIMB_STREAM_AB)
      return fail(LBMIMB_EINVAL, "slab lattices stream with two arrays (LBMIMB_STREAM_AB)"), false;
  } else if (p->slab_y0 != 0) {
    return fail(LBMIMB_EINVAL, "slab_y0 without slab_ny"), false;
  }
  if (maxp < 0 || maxp > kMaxParticles)
    return fail(LBMIMB_EINVAL, "max_particles out of range (node tags hold 24-bit particle indices)"), false;
  double nn = (double)p->n[0] * (double)p->n[1] * (double)p->n[2];
  if (nn > 4.0e12) return fail(LBMIMB_EINVAL, "lattice too large"), false;
  return true;
}

// Rows a lattice stores and how they map to the global lattice (lbmimb_internal.cuh: SlabRows).
static SlabRows slab_rows(const lbmimb_params *p) {
  SlabRows s;
  if (p->slab_ny == 0) {
    s.ny_stored = s.gny = (int)p->n[1];
    s.oy = 0;
    s.own_lo = 0;
    s.own_hi = (int)p->n[1];
    s.wall_lo = s.wall_hi = p->bc[1];
    return s;
  }
  const int ghost_lo = !(p->bc[1] == 1 && p->slab_y0 == 0);
  const int ghost_hi = !(p->bc[1] == 1 && p->slab_y0 + p->n[1] == p->slab_ny);
  s.ny_stored = (int)p->n[1] + ghost_lo + ghost_hi;
  s.gny = (int)p->slab_ny;
  s.oy = (int)p->slab_y0 - ghost_lo;
  s.own_lo = ghost_lo;
  s.own_hi = ghost_lo + (int)p->n[1];
  s.wall_lo = !ghost_lo;
  s.wall_hi = !ghost_hi;
  return s;
}

// One place that decides the device memory layout; used for sizing and for carving.
struct Layout {
  uint64_t off_f[2], off_tag, off_s, off_facc, off_beta, off_contested, off_counters, off_table, off_diag;
  uint64_t off_pos, off_vel, off_omega, off_radius, off_mass, off_force, off_torque, off_fc, off_prec, off_pos2, off_vel2;
  uint64_t off_count, off_start, off_fill, off_items, off_cell_of, off_bsums;
  uint64_t total;
  int64_t N, contested_cap, ncells_max;
};

static Layout make_layout(const lbmimb_params *p, int64_t maxp) {
  Layout L;
  memset(&L, 0, sizeof(L));
  int Q = p->dim == 2 ? 9 : 19;
  const SlabRows sr = slab_rows(p);
  L.N = p->n[0] * (int64_t)sr.ny_stored * p->n[2];
  int64_t pm = maxp > 0 ? maxp : 1;
  L.contested_cap = L.N / 4 + 65536;
  L.ncells_max = 1;
  for (int a = 0; a < p->dim; ++a) {   // the particles live in the GLOBAL lattice
    const int64_t na = a == 1 ? sr.gny : p->n[a];
    L.ncells_max *= (na / 2 > 0 ? na / 2 : 1);
  }
  uint64_t o = 0;
  auto take = [&](uint64_t bytes) {
    uint64_t r = o;
    o = align_up(o + bytes);
    return r;
  };
  L.off_f[0] = take((uint64_t)Q * L.N * 8);
  L.off_f[1] = p->streaming == LBMIMB_STREAM_AA ? L.off_f[0] : take((uint64_t)Q * L.N * 8);
  L.off_tag = take((uint64_t)L.N * 4);
  L.off_counters = take(64);   // directly behind the tags: one memset clears the map and its counters
  L.off_s = (p->flags & LBMIMB_FLAG_EXCHANGE_FIELD) ? take((uint64_t)exchange_stride(p->dim) * L.N * 8) : 0;
  L.off_facc = take((uint64_t)pm * force_values(p->dim) * 16);
  L.off_beta = take(256 * 8);
  L.off_contested = take((uint64_t)L.contested_cap * 8);
  L.off_table = take((uint64_t)eps_table_entries(p->dim));
  L.off_diag = take((uint64_t)(kDiagBlocksMax * 8 + 32) * 8);
  L.off_pos = take((uint64_t)3 * pm * 8);
  L.off_vel = take((uint64_t)3 * pm * 8);
  L.off_omega = take((uint64_t)3 * pm * 8);
  L.off_radius = take((uint64_t)pm * 8);
  L.off_mass = take((uint64_t)pm * 8);
  L.off_force = take((uint64_t)3 * pm * 8);
  L.off_torque = take((uint64_t)3 * pm * 8);
  L.off_fc = take((uint64_t)3 * pm * 8);
  L.off_prec = take((uint64_t)10 * pm * 8);
  L.off_pos2 = take((uint64_t)3 * pm * 8);
  L.off_vel2 = take((uint64_t)3 * pm * 8);
  L.off_count = take((uint64_t)(L.ncells_max + 1) * 4);
  L.off_start = take((uint64_t)(L.ncells_max + 1) * 4);
  L.off_fill = take((uint64_t)(L.ncells_max + 1) * 4);
  L.off_items = take((uint64_t)pm * 4);
  L.off_cell_of = take((uint64_t)pm * 4);
  L.off_bsums = take((uint64_t)((L.ncells_max + 1) / 1024 + 2) * 4);
  L.total = o;
  return L;
}

static lbmimb_status copy_in(lbmimb_lattice *h, void *dst, const void *src, uint64_t bytes) {
  LBMIMB_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, h->stream));
  return LBMIMB_OK;
}

static lbmimb_status use_device(const lbmimb_lattice *h) {
  LBMIMB_CUDA(cudaSetDevice(h->prm.device));
  return LBMIMB_OK;
}

// Host-side refresh of the beta table: beta(n_s/S^D, tau).  Plain IEEE
// + - * / in the paper's order (it is a parameter table, like tau itself).
static void fill_beta_table(double tau, int SD, double *tab) {
  for (int c = 0; c < 256; ++c) {
    double eps = c <= SD ? (double)c / (double)SD : 1.0;
    tab[c] = eps * (tau - 0.5) / ((1.0 - eps) + (tau - 0.5));
  }
}

}  // namespace lbmimb

using namespace lbmimb;

extern "C" {

const char *lbmimb_last_error(void) { return g_err; }
const char *lbmimb_version(void) { return "lbmimb 0.4 (sm_100a, fused collide-stream + in-kernel force sums: pull A-B and in-place AA; DEM: cell list or Verlet lists)"; }

uint64_t lbmimb_workspace_bytes(const lbmimb_params *params, int64_t max_particles) {
  if (!valid_params(params, max_particles)) return 0;
  return make_layout(params, max_particles).total;
}

lbmimb_status lbmimb_create_lattice(const lbmimb_params *params, int64_t max_particles, lbmimb_lattice **out) {
  if (!out) return fail(LBMIMB_EINVAL, "out is NULL");
  *out = nullptr;
  if (!valid_params(params, max_particles)) return LBMIMB_EINVAL;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0)
    return fail(LBMIMB_ECUDA, "no CUDA device available (%s); this library has no CPU fallback",
                cudaGetErrorString(e));
  if (params->device < 0 || params->device >= ndev) return fail(LBMIMB_EINVAL, "device ordinal out of range");
  LBMIMB_CUDA(cudaSetDevice(params->device));

  lbmimb_lattice *h = new (std::nothrow) lbmimb_lattice;
  if (!h) return fail(LBMIMB_ENOMEM, "host allocation failed");
  memset(h, 0, sizeof(*h));
  h->prm = *params;
  h->sl = slab_rows(params);
  h->is_slab = params->slab_ny != 0;
  h->g.dim = params->dim;
  h->g.nx = (int)params->n[0];
  h->g.ny = h->sl.ny_stored;
  h->g.nz = (int)params->n[2];
  h->g.bcx = params->bc[0];
  h->g.bcy = params->bc[1];
  h->g.bcz = params->dim == 3 ? params->bc[2] : 0;
  h->g.N = params->n[0] * (int64_t)h->sl.ny_stored * params->n[2];
  h->gp = h->g;
  h->gp.ny = h->sl.gny;
  h->gp.N = params->n[0] * (int64_t)h->sl.gny * params->n[2];
  h->Q = params->dim == 2 ? 9 : 19;
  h->SD = 1;
  for (int a = 0; a < params->dim; ++a) h->SD *= params->subsamples;
  h->stream = (cudaStream_t)params->stream;
  h->Pmax = max_particles;

  Layout L = make_layout(params, max_particles);
  if (params->workspace_dev) {
    if (params->workspace_bytes < L.total || ((uintptr_t)params->workspace_dev & 255)) {
      delete h;
      return fail(LBMIMB_ENOMEM, "workspace too small (%llu < %llu bytes) or not 256-byte aligned",
                  (unsigned long long)params->workspace_bytes, (unsigned long long)L.total);
    }
    h->ws = (char *)params->workspace_dev;
    h->owns_ws = false;
  } else {
    void *p = nullptr;
    e = cudaMalloc(&p, L.total);
    if (e != cudaSuccess) {
      delete h;
      return cuda_fail(e, "cudaMalloc(workspace)");
    }
    h->ws = (char *)p;
    h->owns_ws = true;
  }
  h->ws_bytes = L.total;
  h->f[0] = (double *)(h->ws + L.off_f[0]);
  h->f[1] = (double *)(h->ws + L.off_f[1]);
  h->tag = (uint32_t *)(h->ws + L.off_tag);
  h->keep_s = (params->flags & LBMIMB_FLAG_EXCHANGE_FIELD) != 0;
  h->s = h->keep_s ? (double *)(h->ws + L.off_s) : nullptr;
  h->facc = (long long *)(h->ws + L.off_facc);
  h->beta_tab = (double *)(h->ws + L.off_beta);
  h->contested = (int64_t *)(h->ws + L.off_contested);
  h->contested_cap = L.contested_cap;
  h->counters = (int32_t *)(h->ws + L.off_counters);
  h->eps_table = (uint8_t *)(h->ws + L.off_table);
  h->diag_partial = (double *)(h->ws + L.off_diag);
  h->diag_out = h->diag_partial + (size_t)kDiagBlocksMax * 8;
  h->map_mode = LBMIMB_MAP_SAMPLING;
  h->table_R = -1.0;
  h->pos = (double *)(h->ws + L.off_pos);
  h->vel = (double *)(h->ws + L.off_vel);
  h->omega = (double *)(h->ws + L.off_omega);
  h->radius = (double *)(h->ws + L.off_radius);
  h->mass = (double *)(h->ws + L.off_mass);
  h->force = (double *)(h->ws + L.off_force);
  h->torque = (double *)(h->ws + L.off_torque);
  h->fc = (double *)(h->ws + L.off_fc);
  h->prec = (double *)(h->ws + L.off_prec);
  h->pos2 = (double *)(h->ws + L.off_pos2);
  h->vel2 = (double *)(h->ws + L.off_vel2);
  h->cl.count = (int32_t *)(h->ws + L.off_count);
  h->cl.start = (int32_t *)(h->ws + L.off_start);
  h->cl.fill = (int32_t *)(h->ws + L.off_fill);
  h->cl.items = (int32_t *)(h->ws + L.off_items);
  h->cl.cell_of = (int32_t *)(h->ws + L.off_cell_of);
  h->cl.block_sums = (int32_t *)(h->ws + L.off_bsums);
  h->cl.ncells_max = L.ncells_max;

  lbmimb_status st = LBMIMB_OK;
  double tab[256];
  fill_beta_table(params->tau, h->SD, tab);
  auto body = [&]() -> lbmimb_status {
    LBMIMB_CUDA(cudaMemcpyAsync(h->beta_tab, tab, sizeof(tab), cudaMemcpyHostToDevice, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->tag, 0, (size_t)h->g.N * 4, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->facc, 0, (size_t)(h->Pmax > 0 ? h->Pmax : 1) * force_values(h->g.dim) * 16, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->counters, 0, 64, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->force, 0, (size_t)3 * (h->Pmax > 0 ? h->Pmax : 1) * 8, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->torque, 0, (size_t)3 * (h->Pmax > 0 ? h->Pmax : 1) * 8, h->stream));
    lbmimb_status s2 = launch_init_rest(h);
    if (s2 != LBMIMB_OK) return s2;
    LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
    return LBMIMB_OK;
  };
  st = body();
  if (st != LBMIMB_OK) {
    if (h->owns_ws) cudaFree(h->ws);
    delete h;
    return st;
  }
  h->cur = 0;
  h->aa = params->streaming == LBMIMB_STREAM_AA;
  h->aa_swapped = false;
  h->P = 0;
  h->map_valid = true;  // no particles: the all-zero map is the map
  h->s_valid = false;
  h->forces_valid = false;
  h->t = 0;
  *out = h;
  return LBMIMB_OK;
}

static void coupled_graph_drop(lbmimb_lattice *h);
static lbmimb_status sync_and_check(lbmimb_lattice *h);

lbmimb_status lbmimb_destroy_lattice(lbmimb_lattice *h) {
  if (!h) return LBMIMB_OK;
  cudaSetDevice(h->prm.device);
  cudaStreamSynchronize(h->stream);
  coupled_graph_drop(h);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  neighbor_list_release(h);
  if (h->fetch_stage) cudaFree(h->fetch_stage);
  if (h->owns_ws) cudaFree(h->ws);
  delete h;
  return LBMIMB_OK;
}

static lbmimb_status after_particles_changed(lbmimb_lattice *h, bool positions) {
  if (positions) {
    h->map_valid = (h->P == 0);
    h->cl_valid = false;
    h->s_valid = false;
    h->forces_valid = false;
    if (h->acc_dirty) {   // sums of a step nobody reduced: the particle set they belong to is gone
      LBMIMB_CUDA(cudaMemsetAsync(h->facc, 0, (size_t)(h->Pmax > 0 ? h->Pmax : 1) * force_values(h->g.dim) * 16, h->stream));
      h->acc_dirty = false;
    }
    lbmimb_status st = neighbor_list_invalidate(h);
    if (st != LBMIMB_OK) return st;
  }
  if (h->P > 0) return launch_pack_records(h);
  return LBMIMB_OK;
}

lbmimb_status lbmimb_set_particles(lbmimb_lattice *h, int64_t P, const double *pos, const double *vel,
                                   const double *omega, const double *radius, const double *mass) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (P < 0 || P > h->Pmax) return fail(LBMIMB_EINVAL, "P = %lld exceeds max_particles = %lld", (long long)P,
                                        (long long)h->Pmax);
  if (P > 0 && (!pos || !vel || !radius || !mass)) return fail(LBMIMB_EINVAL, "NULL particle array");
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  double rmax = 0.0, rmin = INFINITY;
  for (int64_t p = 0; p < P; ++p) {
    if (radius[p] < rmin) rmin = radius[p];
    if (!(radius[p] > 0.0) || !(mass[p] > 0.0) || !std::isfinite(radius[p]) || !std::isfinite(mass[p]))
      return fail(LBMIMB_EINVAL, "particle %lld: radius and mass must be positive and finite", (long long)p);
    for (int a = 0; a < D; ++a) {
      double x = pos[(int64_t)a * P + p];
      const double na = a == 1 ? (double)h->gp.ny : (double)h->prm.n[a];
      if (!(x >= -0.5) || !(x < na))  // [ -1/2, n ) accepted (DEM wraps into [0,n))
        return fail(LBMIMB_EINVAL, "particle %lld: centre outside the domain on axis %d", (long long)p, a);
    }
    if (radius[p] > rmax) rmax = radius[p];
  }
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  if (P > 0) {
    if ((st = copy_in(h, h->pos, pos, (uint64_t)D * P * 8)) != LBMIMB_OK) return st;
    if ((st = copy_in(h, h->vel, vel, (uint64_t)D * P * 8)) != LBMIMB_OK) return st;
    if (omega) {
      if ((st = copy_in(h, h->omega, omega, (uint64_t)nt * P * 8)) != LBMIMB_OK) return st;
    } else {
      LBMIMB_CUDA(cudaMemsetAsync(h->omega, 0, (size_t)nt * P * 8, h->stream));
    }
    if ((st = copy_in(h, h->radius, radius, (uint64_t)P * 8)) != LBMIMB_OK) return st;
    if ((st = copy_in(h, h->mass, mass, (uint64_t)P * 8)) != LBMIMB_OK) return st;
    LBMIMB_CUDA(cudaMemsetAsync(h->force, 0, (size_t)D * P * 8, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->torque, 0, (size_t)nt * P * 8, h->stream));
  }
  h->P = P;
  h->rmax = rmax;
  h->rmin = P > 0 ? rmin : 0.0;
  if (P == 0) LBMIMB_CUDA(cudaMemsetAsync(h->tag, 0, (size_t)h->g.N * 4, h->stream));
  st = after_particles_changed(h, true);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  return LBMIMB_OK;
}

lbmimb_status lbmimb_set_particles_dev(lbmimb_lattice *h, int64_t P, const double *pos_dev, const double *vel_dev,
                                       const double *omega_dev, const double *radius_dev, const double *mass_dev) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (P < 0 || P > h->Pmax) return fail(LBMIMB_EINVAL, "P exceeds max_particles");
  if (P > 0 && (!pos_dev || !vel_dev || !radius_dev || !mass_dev)) return fail(LBMIMB_EINVAL, "NULL particle array");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  double rmax = 0.0, rmin = INFINITY;
  if (P > 0) {
    // checked on the device before anything is committed: on EINVAL the handle is unchanged
    if ((st = validate_particles_dev(h, P, pos_dev, radius_dev, mass_dev, &rmax, &rmin)) != LBMIMB_OK) return st;
    auto d2d = [&](void *dst, const void *src, uint64_t bytes) -> lbmimb_status {
      LBMIMB_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, h->stream));
      return LBMIMB_OK;
    };
    if ((st = d2d(h->pos, pos_dev, (uint64_t)D * P * 8)) != LBMIMB_OK) return st;
    if ((st = d2d(h->vel, vel_dev, (uint64_t)D * P * 8)) != LBMIMB_OK) return st;
    if (omega_dev) {
      if ((st = d2d(h->omega, omega_dev, (uint64_t)nt * P * 8)) != LBMIMB_OK) return st;
    } else {
      LBMIMB_CUDA(cudaMemsetAsync(h->omega, 0, (size_t)nt * P * 8, h->stream));
    }
    if ((st = d2d(h->radius, radius_dev, (uint64_t)P * 8)) != LBMIMB_OK) return st;
    if ((st = d2d(h->mass, mass_dev, (uint64_t)P * 8)) != LBMIMB_OK) return st;
    LBMIMB_CUDA(cudaMemsetAsync(h->force, 0, (size_t)D * P * 8, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->torque, 0, (size_t)nt * P * 8, h->stream));
  }
  h->P = P;
  h->rmax = rmax;
  h->rmin = P > 0 ? rmin : 0.0;
  if (P == 0) LBMIMB_CUDA(cudaMemsetAsync(h->tag, 0, (size_t)h->g.N * 4, h->stream));
  return after_particles_changed(h, true);
}

lbmimb_status lbmimb_set_particle_velocities(lbmimb_lattice *h, const double *vel, const double *omega) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (h->P == 0) return LBMIMB_OK;
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  if (vel && (st = copy_in(h, h->vel, vel, (uint64_t)D * h->P * 8)) != LBMIMB_OK) return st;
  if (omega && (st = copy_in(h, h->omega, omega, (uint64_t)nt * h->P * 8)) != LBMIMB_OK) return st;
  st = after_particles_changed(h, false);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  return LBMIMB_OK;
}

lbmimb_status lbmimb_get_particles(lbmimb_lattice *h, double *pos, double *vel, double *omega) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  if (h->P > 0) {
    if (pos) LBMIMB_CUDA(cudaMemcpyAsync(pos, h->pos, (size_t)D * h->P * 8, cudaMemcpyDeviceToHost, h->stream));
    if (vel) LBMIMB_CUDA(cudaMemcpyAsync(vel, h->vel, (size_t)D * h->P * 8, cudaMemcpyDeviceToHost, h->stream));
    if (omega)
      LBMIMB_CUDA(cudaMemcpyAsync(omega, h->omega, (size_t)nt * h->P * 8, cudaMemcpyDeviceToHost, h->stream));
  }
  return sync_and_check(h);
}

int64_t lbmimb_num_particles(const lbmimb_lattice *h) { return h ? h->P : -1; }
int64_t lbmimb_time(const lbmimb_lattice *h) { return h ? h->t : -1; }
int64_t lbmimb_launch_count(const lbmimb_lattice *h) { return h ? h->launches : -1; }

// Waits for the handle's stream and reads the error flags kernels raise on the device: overflow of the
// shared-node list of the map, of a neighbour list or of a cell of its build grid.  Every call that
// synchronises anyway ends with this, so that a result is never handed out next to a silent overflow.
static lbmimb_status sync_and_check(lbmimb_lattice *h) {
  int32_t c[4] = {0, 0, 0, 0}, s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  LBMIMB_CUDA(cudaMemcpyAsync(c, h->counters, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
  if (h->nl.mem) LBMIMB_CUDA(cudaMemcpyAsync(s, h->nl.state, sizeof(s), cudaMemcpyDeviceToHost, h->stream));
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  if (c[1] != 0)
    return fail(LBMIMB_ESTATE, "particle map: the list of nodes shared by several particles overflowed (%lld entries; "
                               "particles overlap too much)", (long long)h->contested_cap);
  if (s[4] != 0 || s[5] != 0)
    return fail(LBMIMB_ESTATE, "neighbour list: %s overflowed (particles overlap more deeply than the sizing allows)",
                s[4] ? "a particle's list" : "a cell of the build grid");
  return LBMIMB_OK;
}

lbmimb_status lbmimb_synchronize(lbmimb_lattice *h) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  return sync_and_check(h);
}

// Bodies of the four calls of a coupled step: launches and state machine only (no argument checks, no
// cudaSetDevice), shared by the entry points and by the graph capture of lbmimb_run_coupled.
static lbmimb_status map_body(lbmimb_lattice *h) {
  if (h->P > 0) {
    lbmimb_status st = launch_map(h);
    if (st != LBMIMB_OK) return st;
  }
  h->map_valid = true;
  h->s_valid = false;
  h->forces_valid = false;
  return LBMIMB_OK;
}

lbmimb_status lbmimb_map_particles(lbmimb_lattice *h) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  return map_body(h);
}

lbmimb_status lbmimb_set_mapping_mode(lbmimb_lattice *h, int32_t mode) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (mode != LBMIMB_MAP_SAMPLING && mode != LBMIMB_MAP_TABLE) return fail(LBMIMB_EINVAL, "unknown mapping mode %d", mode);
  if (mode == h->map_mode) return LBMIMB_OK;
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  // eps = eps_cnt / S^D (sampling) or code / 255 (table): refresh beta(eps, tau)
  double tab[256];
  fill_beta_table(h->prm.tau, mode == LBMIMB_MAP_TABLE ? LBMIMB_TABLE_DEN : h->SD, tab);
  LBMIMB_CUDA(cudaMemcpyAsync(h->beta_tab, tab, sizeof(tab), cudaMemcpyHostToDevice, h->stream));
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));  // tab lives on this stack frame
  h->map_mode = mode;
  h->map_valid = (h->P == 0);
  h->s_valid = false;
  h->forces_valid = false;
  return LBMIMB_OK;
}

lbmimb_status lbmimb_fetch_eps_table(lbmimb_lattice *h, uint8_t *dst, int64_t capacity) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!dst) return fail(LBMIMB_EINVAL, "dst is NULL");
  if (h->map_mode != LBMIMB_MAP_TABLE) return fail(LBMIMB_ESTATE, "table mapping mode is not selected");
  if (h->P == 0) return fail(LBMIMB_ESTATE, "no particles: the table is built for the particles' radius");
  const int64_t bytes = eps_table_entries(h->g.dim);
  if (capacity < bytes) return fail(LBMIMB_EINVAL, "dst holds %lld bytes, the table has %lld", (long long)capacity, (long long)bytes);
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  if ((st = ensure_eps_table(h)) != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaMemcpyAsync(dst, h->eps_table, (size_t)bytes, cudaMemcpyDeviceToHost, h->stream));
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  return LBMIMB_OK;
}

static lbmimb_status step_body(lbmimb_lattice *h, int32_t nsteps) {
  lbmimb_status st;
  for (int32_t it = 0; it < nsteps; ++it) {
    bool emit = (h->P > 0) && (it == nsteps - 1);
    if (emit && h->acc_dirty) {   // sums of an earlier step that no reduce_particle_forces consumed
      LBMIMB_CUDA(cudaMemsetAsync(h->facc, 0, (size_t)h->P * force_values(h->g.dim) * 16, h->stream));
      h->acc_dirty = false;
    }
    if ((st = launch_collide_stream(h, emit)) != LBMIMB_OK) return st;
    if (emit) h->acc_dirty = true;
    if (h->aa)
      h->aa_swapped = !h->aa_swapped;
    else
      h->cur ^= 1;
    h->t += 1;
    if (emit) h->s_valid = true;
    h->forces_valid = false;
  }
  return LBMIMB_OK;
}

lbmimb_status lbmimb_step(lbmimb_lattice *h, int32_t nsteps) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (nsteps < 0) return fail(LBMIMB_EINVAL, "nsteps < 0");
  if (!h->map_valid) return fail(LBMIMB_ESTATE, "particles were set or moved but not mapped: call lbmimb_map_particles first");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  return step_body(h, nsteps);
}

static lbmimb_status reduce_body(lbmimb_lattice *h) {
  if (h->P > 0 && !h->s_valid)
    return fail(LBMIMB_ESTATE, "no exchange vectors: call lbmimb_step after lbmimb_map_particles first");
  if (h->P > 0 && !h->forces_valid) {   // (a repeated call finds force / torque already in place)
    lbmimb_status st = launch_finish_forces(h);
    if (st != LBMIMB_OK) return st;
    h->acc_dirty = false;
  }
  h->forces_valid = true;
  return LBMIMB_OK;
}

static lbmimb_status reduce_common(lbmimb_lattice *h) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  return reduce_body(h);
}

lbmimb_status lbmimb_reduce_particle_forces(lbmimb_lattice *h, double *force, double *torque) {
  lbmimb_status st = reduce_common(h);
  if (st != LBMIMB_OK) return st;
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  if (h->P > 0 && (force || torque)) {
    if (force) LBMIMB_CUDA(cudaMemcpyAsync(force, h->force, (size_t)D * h->P * 8, cudaMemcpyDeviceToHost, h->stream));
    if (torque)
      LBMIMB_CUDA(cudaMemcpyAsync(torque, h->torque, (size_t)nt * h->P * 8, cudaMemcpyDeviceToHost, h->stream));
    return sync_and_check(h);
  }
  return LBMIMB_OK;
}

lbmimb_status lbmimb_reduce_particle_forces_dev(lbmimb_lattice *h, double *force_dev, double *torque_dev) {
  lbmimb_status st = reduce_common(h);
  if (st != LBMIMB_OK) return st;
  int D = h->g.dim, nt = D == 2 ? 1 : 3;
  if (h->P > 0) {
    if (force_dev)
      LBMIMB_CUDA(cudaMemcpyAsync(force_dev, h->force, (size_t)D * h->P * 8, cudaMemcpyDeviceToDevice, h->stream));
    if (torque_dev)
      LBMIMB_CUDA(cudaMemcpyAsync(torque_dev, h->torque, (size_t)nt * h->P * 8, cudaMemcpyDeviceToDevice, h->stream));
  }
  return LBMIMB_OK;
}

static lbmimb_status check_dem_params(const lbmimb_dem_params *dem) {
  if (!dem) return fail(LBMIMB_EINVAL, "dem params is NULL");
  if (!(dem->kn > 0.0) || !(dem->restitution > 0.0) || !(dem->restitution <= 1.0) || !(dem->dt > 0.0))
    return fail(LBMIMB_EINVAL, "dem params: need kn > 0, 0 < restitution <= 1, dt > 0");
  return LBMIMB_OK;
}

static lbmimb_status dem_body(lbmimb_lattice *h, const lbmimb_dem_params *dem, bool finish) {
  if (h->P == 0) return LBMIMB_OK;
  lbmimb_status st;
  const bool cells = dem_can_finish(h);   // cell-list mode: the second-half kernel packs the records itself
  if ((st = launch_dem(h, dem, finish)) != LBMIMB_OK) return st;
  // positions moved: the map and the exchange vectors are stale; the cell list was rebuilt at
  // the new positions inside the step and stays valid; force/torque stay "the last reduction"
  h->map_valid = false;
  h->s_valid = false;
  return cells ? LBMIMB_OK : launch_pack_records(h);
}

lbmimb_status lbmimb_dem_step(lbmimb_lattice *h, const lbmimb_dem_params *dem) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = check_dem_params(dem);
  if (st != LBMIMB_OK) return st;
  if (h->P == 0) return LBMIMB_OK;
  if ((st = use_device(h)) != LBMIMB_OK) return st;
  return dem_body(h, dem, false);
}

// ---- lbmimb_run_coupled: the coupled loop with its launches replayed from a CUDA graph ----
static lbmimb_status coupled_step_body(lbmimb_lattice *h, const lbmimb_dem_params *dem) {
  lbmimb_status st;
  if ((st = map_body(h)) != LBMIMB_OK) return st;
  if ((st = step_body(h, 1)) != LBMIMB_OK) return st;
  if (h->P > 0 && dem_can_finish(h)) {   // a3's conversion of the sums rides in the first DEM kernel
    h->forces_valid = true;
    h->acc_dirty = false;
    return dem_body(h, dem, true);
  }
  if ((st = reduce_body(h)) != LBMIMB_OK) return st;
  return dem_body(h, dem, false);
}

static bool coupled_graph_matches(const lbmimb_lattice *h, const CoupledGraph &g, const lbmimb_dem_params *dem) {
  return g.valid && g.P == h->P && g.rmax == h->rmax && g.rmin == h->rmin && g.table_R == h->table_R &&
         g.map_mode == h->map_mode && g.nl_mode == h->nl.mode && g.nl_skin == h->nl.skin &&
         g.nl_every == h->nl.every && g.nl_mem == h->nl.mem && memcmp(&g.dem, dem, sizeof(*dem)) == 0;
}

static void coupled_graph_drop(lbmimb_lattice *h) {
  for (int k = 0; k < 2; ++k) {
    if (h->cg[k].exec) cudaGraphExecDestroy(h->cg[k].exec);
    h->cg[k].exec = nullptr;
    h->cg[k].valid = false;
  }
}

// Captures two consecutive coupled steps (both parities of the distribution arrays) on the private stream.
// The handle must be in the steady state of the loop (one plain step has run): then the host-side state
// machine ends the pair exactly where it started, and only t and the launch counter are put back.
static lbmimb_status coupled_graph_capture(lbmimb_lattice *h, const lbmimb_dem_params *dem, CoupledGraph &g) {
  if (g.exec) cudaGraphExecDestroy(g.exec);
  g.exec = nullptr;
  g.valid = false;
  if (!h->cap_stream) LBMIMB_CUDA(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
  const cudaStream_t user = h->stream;
  const int64_t t0 = h->t, l0 = h->launches;
  // the host-side state machine as it stands: a capture that fails half way has executed nothing on the
  // device, so everything the captured calls toggled is put back
  const int cur0 = h->cur;
  const bool swapped0 = h->aa_swapped, map0 = h->map_valid, s0 = h->s_valid, forces0 = h->forces_valid;
  const bool cl0 = h->cl_valid, dirty0 = h->acc_dirty, clean0 = h->cl.count_clean;
  const double table0 = h->table_R;
  LBMIMB_CUDA(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
  h->stream = h->cap_stream;
  lbmimb_status st = coupled_step_body(h, dem);
  if (st == LBMIMB_OK) st = coupled_step_body(h, dem);
  h->stream = user;
  cudaGraph_t graph = nullptr;
  const cudaError_t e = cudaStreamEndCapture(h->cap_stream, &graph);
  g.launches = h->launches - l0;
  h->launches = l0;
  h->t = t0;
  if (st != LBMIMB_OK || e != cudaSuccess || !graph) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    h->cur = cur0;
    h->aa_swapped = swapped0;
    h->map_valid = map0;
    h->s_valid = s0;
    h->forces_valid = forces0;
    h->cl_valid = cl0;
    h->acc_dirty = dirty0;
    h->cl.count_clean = clean0;
    h->table_R = table0;
    return st != LBMIMB_OK ? st : cuda_fail(e, "cudaStreamEndCapture(coupled steps)");
  }
  const cudaError_t e2 = cudaGraphInstantiate(&g.exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e2 != cudaSuccess) {
    g.exec = nullptr;
    return cuda_fail(e2, "cudaGraphInstantiate(coupled steps)");
  }
  g.valid = true;
  g.P = h->P;
  g.rmax = h->rmax;
  g.rmin = h->rmin;
  g.table_R = h->table_R;
  g.map_mode = h->map_mode;
  g.nl_mode = h->nl.mode;
  g.nl_skin = h->nl.skin;
  g.nl_every = h->nl.every;
  g.nl_mem = h->nl.mem;
  g.dem = *dem;
  return LBMIMB_OK;
}

static bool coupled_graphs_enabled() {
  static int v = -1;
  if (v < 0) {
    const char *e = getenv("LBMIMB_NO_GRAPH");
    v = (e && atoi(e) != 0) ? 0 : 1;
  }
  return v == 1;
}

lbmimb_status lbmimb_run_coupled(lbmimb_lattice *h, const lbmimb_dem_params *dem, int32_t nsteps) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  lbmimb_status st = check_dem_params(dem);
  if (st != LBMIMB_OK) return st;
  if (nsteps < 0) return fail(LBMIMB_EINVAL, "nsteps < 0");
  if (h->is_slab)
    return fail(LBMIMB_ESTATE, "run_coupled is not available on a slab lattice: the force sums cross slabs inside the step");
  if ((st = use_device(h)) != LBMIMB_OK) return st;
  if (h->P == 0) return step_body(h, nsteps);   // no particles: the other three calls are no-ops
  int32_t left = nsteps;
  if (left > 0) {   // the first step also (re)builds whatever the steady loop takes for granted
    if ((st = coupled_step_body(h, dem)) != LBMIMB_OK) return st;
    --left;
  }
  if (left >= 2 && coupled_graphs_enabled() && !h->cg_broken) {
    CoupledGraph &g = h->cg[h->aa ? (h->aa_swapped ? 1 : 0) : h->cur];
    if (!coupled_graph_matches(h, g, dem) && coupled_graph_capture(h, dem, g) != LBMIMB_OK) h->cg_broken = true;
    if (g.valid) {
      for (; left >= 2; left -= 2) {
        if (cudaGraphLaunch(g.exec, h->stream) != cudaSuccess) {   // nothing was enqueued: go on call by call
          cudaGetLastError();
          h->cg_broken = true;
          break;
        }
        h->t += 2;
        h->launches += g.launches;
      }
    }
  }
  for (; left > 0; --left)
    if ((st = coupled_step_body(h, dem)) != LBMIMB_OK) return st;
  return LBMIMB_OK;
}

lbmimb_status lbmimb_set_neighbor_mode(lbmimb_lattice *h, int32_t mode, double skin, int64_t every) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (mode != LBMIMB_NEIGHBOR_CELLS && mode != LBMIMB_NEIGHBOR_VERLET)
    return fail(LBMIMB_EINVAL, "unknown neighbour mode %d", mode);
  if (mode == LBMIMB_NEIGHBOR_VERLET && (!(skin > 0.0) || !std::isfinite(skin) || every < 1))
    return fail(LBMIMB_EINVAL, "neighbour lists need skin > 0 and every >= 1");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  neighbor_list_release(h);
  h->nl.mode = mode;
  h->nl.skin = mode == LBMIMB_NEIGHBOR_VERLET ? skin : 0.0;
  h->nl.every = mode == LBMIMB_NEIGHBOR_VERLET ? (int)(every > 0x7fffffff ? 0x7fffffff : every) : 0;
  return LBMIMB_OK;
}

lbmimb_status lbmimb_fetch_neighbor_list(lbmimb_lattice *h, int64_t *start, int32_t *items, int64_t capacity,
                                         int64_t *info) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!start || (capacity > 0 && !items) || capacity < 0) return fail(LBMIMB_EINVAL, "NULL output / negative capacity");
  if (h->nl.mode != LBMIMB_NEIGHBOR_VERLET) return fail(LBMIMB_ESTATE, "neighbour-list mode is not selected");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  const int64_t P = h->P;
  int32_t s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  if (h->nl.mem) LBMIMB_CUDA(cudaMemcpy(s, h->nl.state, sizeof(s), cudaMemcpyDeviceToHost));
  if (s[4] != 0 || s[5] != 0)
    return fail(LBMIMB_ESTATE, "neighbour list: %s overflowed (particles overlap more deeply than the sizing allows)",
                s[4] ? "a particle's list" : "a cell of the build grid");
  if (info) {
    info[0] = s[0];
    info[1] = s[1];
    info[2] = s[2];
    info[3] = 0;
  }
  if (!s[0] || P == 0) {   // no valid list: all lists empty
    for (int64_t p = 0; p <= P; ++p) start[p] = 0;
    return LBMIMB_OK;
  }
  // marshalling only: the device keeps K slots per particle (slot-major); the ABI speaks CSR
  std::vector<int32_t> cnt((size_t)P), slots((size_t)h->nl.K * P);
  LBMIMB_CUDA(cudaMemcpy(cnt.data(), h->nl.count, (size_t)P * 4, cudaMemcpyDeviceToHost));
  LBMIMB_CUDA(cudaMemcpy2D(slots.data(), (size_t)P * 4, h->nl.items, (size_t)h->nl.Pcap * 4, (size_t)P * 4,
                           (size_t)h->nl.K, cudaMemcpyDeviceToHost));
  int64_t total = 0;
  for (int64_t p = 0; p < P; ++p) total += cnt[p];
  if (info) info[3] = total;
  if (capacity < total)
    return fail(LBMIMB_EINVAL, "items holds %lld entries, the lists have %lld", (long long)capacity, (long long)total);
  int64_t o = 0;
  for (int64_t p = 0; p < P; ++p) {
    start[p] = o;
    for (int k = 0; k < cnt[p]; ++k) items[o++] = slots[(size_t)k * P + p];
  }
  start[P] = o;
  return LBMIMB_OK;
}

lbmimb_status lbmimb_fetch_fields(lbmimb_lattice *h, int32_t what, const int64_t lo[3], const int64_t hi[3], void *dst) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!lo || !hi || !dst) return fail(LBMIMB_EINVAL, "NULL argument");
  int64_t box = 1;
  for (int a = 0; a < 3; ++a) {
    int64_t na = a == 0 ? h->g.nx : (a == 1 ? h->sl.own_hi - h->sl.own_lo : h->g.nz);   // rows: the owned ones
    if (lo[a] < 0 || hi[a] > na || lo[a] >= hi[a]) return fail(LBMIMB_EINVAL, "box out of range on axis %d", a);
    box *= hi[a] - lo[a];
  }
  int comps;
  size_t esz;
  switch (what) {
    case LBMIMB_FIELD_F: comps = h->Q; esz = 8; break;
    case LBMIMB_FIELD_RHO: comps = 1; esz = 8; break;
    case LBMIMB_FIELD_U: comps = h->g.dim; esz = 8; break;
    case LBMIMB_FIELD_EPS_CNT: comps = 1; esz = 1; break;
    case LBMIMB_FIELD_PID: comps = 1; esz = 4; break;
    case LBMIMB_FIELD_S: comps = h->g.dim; esz = 8; break;
    default: return fail(LBMIMB_EINVAL, "unknown field selector %d", what);
  }
  if ((what == LBMIMB_FIELD_EPS_CNT || what == LBMIMB_FIELD_PID) && !h->map_valid)
    return fail(LBMIMB_ESTATE, "particle map is stale");
  if (what == LBMIMB_FIELD_S && !h->keep_s)
    return fail(LBMIMB_ESTATE, "per-node exchange vectors are kept only by a lattice created with LBMIMB_FLAG_EXCHANGE_FIELD");
  if (what == LBMIMB_FIELD_S && h->P > 0 && !h->s_valid) return fail(LBMIMB_ESTATE, "no exchange vectors yet");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  // A-B: the idle distribution buffer is the staging area (every field of a sub-box fits in Q*N
  // doubles).  AA has no idle buffer: a grow-only staging buffer owned by the handle.
  void *stage = h->f[h->cur ^ 1];
  const size_t bytes = (size_t)comps * box * esz;
  if (h->aa) {
    if (bytes > h->fetch_stage_bytes) {
      LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
      if (h->fetch_stage) cudaFree(h->fetch_stage);
      h->fetch_stage = nullptr;
      h->fetch_stage_bytes = 0;
      cudaError_t e = cudaMalloc(&h->fetch_stage, bytes);
      if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(fetch staging, AA mode)");
      h->fetch_stage_bytes = bytes;
    }
    stage = h->fetch_stage;
  }
  if ((st = launch_fetch(h, what, lo, hi, stage)) != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaMemcpyAsync(dst, stage, bytes, cudaMemcpyDeviceToHost, h->stream));
  return sync_and_check(h);
}

lbmimb_status lbmimb_diagnostics(lbmimb_lattice *h, double *out) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!out) return fail(LBMIMB_EINVAL, "out is NULL");
  if (h->P > 0 && !h->map_valid) return fail(LBMIMB_ESTATE, "particle map is stale: call lbmimb_map_particles first");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  const double den = h->map_mode == LBMIMB_MAP_TABLE ? (double)LBMIMB_TABLE_DEN : (double)h->SD;
  if ((st = launch_diagnostics(h, den)) != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaMemcpyAsync(out, h->diag_out, LBMIMB_DIAG_LEN * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  return sync_and_check(h);
}

// The same diagnostics without any allocation or synchronisation: scratch in a static device array (lattice.cu).
int64_t lbmimb_diagnostics_static_max_particles(void) { return diagnostics_static_max_particles(); }
int64_t lbmimb_diagnostics_static_scratch_bytes(void) { return diagnostics_static_scratch_bytes(); }

lbmimb_status lbmimb_diagnostics_static_dev(lbmimb_lattice *h, double *out_dev) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!out_dev) return fail(LBMIMB_EINVAL, "out_dev is NULL");
  if (h->P > diagnostics_static_max_particles())
    return fail(LBMIMB_EINVAL, "lbmimb_diagnostics_static_dev: %lld particles exceed the static scratch (at most %lld); "
                               "use lbmimb_diagnostics", (long long)h->P, (long long)diagnostics_static_max_particles());
  if (h->P > 0 && !h->map_valid) return fail(LBMIMB_ESTATE, "particle map is stale: call lbmimb_map_particles first");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  const double den = h->map_mode == LBMIMB_MAP_TABLE ? (double)LBMIMB_TABLE_DEN : (double)h->SD;
  return launch_diagnostics_static(h, den, out_dev);
}

// ---- slab decomposition (NEXT-4): halo pack / unpack and the per-slab force sums ----
int64_t lbmimb_halo_count(const lbmimb_lattice *h) { return h ? halo_doubles(h) : -1; }

int32_t lbmimb_slab_ghost_rows(const lbmimb_lattice *h, int32_t side) {
  if (!h || (side != 0 && side != 1)) return -1;
  return side == 0 ? h->sl.own_lo : h->sl.ny_stored - h->sl.own_hi;
}

static lbmimb_status halo_common(lbmimb_lattice *h, int32_t side, double *buf_dev, bool pack) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (side != 0 && side != 1) return fail(LBMIMB_EINVAL, "side must be 0 (lower y end) or 1 (upper y end)");
  if (!buf_dev) return fail(LBMIMB_EINVAL, "buffer is NULL");
  if (!h->is_slab) return fail(LBMIMB_ESTATE, "not a slab lattice (params.slab_ny = 0)");
  if (lbmimb_slab_ghost_rows(h, side) == 0)
    return fail(LBMIMB_ESTATE, "the %s end of this slab is a wall of the global lattice: nothing crosses it",
                side == 0 ? "lower" : "upper");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  return launch_halo(h, side, buf_dev, pack);
}

lbmimb_status lbmimb_pack_halo(lbmimb_lattice *h, int32_t side, double *dst_dev) {
  return halo_common(h, side, dst_dev, true);
}

lbmimb_status lbmimb_unpack_halo(lbmimb_lattice *h, int32_t side, const double *src_dev) {
  return halo_common(h, side, const_cast<double *>(src_dev), false);
}

int64_t lbmimb_force_sums_count(const lbmimb_lattice *h) { return h ? h->P * force_values(h->g.dim) * 2 : -1; }

lbmimb_status lbmimb_export_force_sums_dev(lbmimb_lattice *h, int64_t *dst_dev) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!dst_dev) return fail(LBMIMB_EINVAL, "dst_dev is NULL");
  if (h->P > 0 && (!h->s_valid || h->forces_valid))
    return fail(LBMIMB_ESTATE, "no unreduced force sums: call after lbmimb_step and before lbmimb_reduce_particle_forces");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaMemcpyAsync(dst_dev, h->facc, (size_t)lbmimb_force_sums_count(h) * 8, cudaMemcpyDeviceToDevice, h->stream));
  return LBMIMB_OK;
}

lbmimb_status lbmimb_import_force_sums_dev(lbmimb_lattice *h, const int64_t *src_dev) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!src_dev) return fail(LBMIMB_EINVAL, "src_dev is NULL");
  if (h->P > 0 && (!h->s_valid || h->forces_valid))
    return fail(LBMIMB_ESTATE, "no unreduced force sums: call after lbmimb_step and before lbmimb_reduce_particle_forces");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  LBMIMB_CUDA(cudaMemcpyAsync(h->facc, src_dev, (size_t)lbmimb_force_sums_count(h) * 8, cudaMemcpyDeviceToDevice, h->stream));
  return LBMIMB_OK;
}

lbmimb_status lbmimb_set_distributions(lbmimb_lattice *h, const double *f) {
  if (!h) return fail(LBMIMB_EINVAL, "handle is NULL");
  if (!f) return fail(LBMIMB_EINVAL, "f is NULL");
  lbmimb_status st = use_device(h);
  if (st != LBMIMB_OK) return st;
  if (h->aa) {   // the AA natural layout IS f_i(x,t)
    LBMIMB_CUDA(cudaMemcpyAsync(h->f[0], f, (size_t)h->Q * h->g.N * 8, cudaMemcpyHostToDevice, h->stream));
    h->aa_swapped = false;
  } else {
    double *stage = h->f[h->cur ^ 1];
    LBMIMB_CUDA(cudaMemcpyAsync(stage, f, (size_t)h->Q * h->g.N * 8, cudaMemcpyHostToDevice, h->stream));
    if ((st = launch_unstream(h, stage, h->f[h->cur])) != LBMIMB_OK) return st;
  }
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  h->t = 0;
  h->s_valid = false;
  h->forces_valid = false;
  return LBMIMB_OK;
}

}  // extern "C"
