// Internal declarations of the lbmimb CUDA library (sm_100a).  Not part of the ABI.
// Shares nothing with oracle/ (the tests' CPU oracle): tables, helpers and kernels
// here are written independently from PAPER.md / DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lbmimb.h"

namespace lbmimb {

// ---------------------------------------------------------------------------
// Velocity sets (R1, ABI order of include/lbmimb.h).  constexpr
// functions so that every use in a fully unrolled loop folds to an immediate.
// ---------------------------------------------------------------------------
template <int D>
struct Lat;

template <>
struct Lat<2> {
  static constexpr int Q = 9;
  __host__ __device__ static constexpr int cx(int q) {
    constexpr int t[9] = {0, 1, -1, 0, 0, 1, -1, 1, -1};
    return t[q];
  }
  __host__ __device__ static constexpr int cy(int q) {
    constexpr int t[9] = {0, 0, 0, 1, -1, 1, -1, -1, 1};
    return t[q];
  }
  __host__ __device__ static constexpr int cz(int) { return 0; }
  __host__ __device__ static constexpr double w(int q) {
    return q == 0 ? 4.0 / 9.0 : (q < 5 ? 1.0 / 9.0 : 1.0 / 36.0);
  }
};

template <>
struct Lat<3> {
  static constexpr int Q = 19;
  __host__ __device__ static constexpr int cx(int q) {
    constexpr int t[19] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
    return t[q];
  }
  __host__ __device__ static constexpr int cy(int q) {
    constexpr int t[19] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
    return t[q];
  }
  __host__ __device__ static constexpr int cz(int q) {
    constexpr int t[19] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
    return t[q];
  }
  __host__ __device__ static constexpr double w(int q) {
    return q == 0 ? 1.0 / 3.0 : (q < 7 ? 1.0 / 18.0 : 1.0 / 36.0);
  }
};

__host__ __device__ constexpr int opposite(int q) { return q == 0 ? 0 : ((q & 1) ? q + 1 : q - 1); }

// Packed per-particle record the fused kernel gathers on covered nodes.
//   3D: x y z vx vy vz wx wy wz R   (10 doubles)      2D: x y vx vy w R (6 doubles)
__host__ __device__ constexpr int prec_stride(int dim) { return dim == 3 ? 10 : 6; }

// Exchange vectors s (kept per node only with LBMIMB_FLAG_EXCHANGE_FIELD) are stored as one record per
// node: [N][2] in 2D, [N][4] in 3D (4th slot unused).
__host__ __device__ constexpr int exchange_stride(int dim) { return dim == 3 ? 4 : 2; }

// Node tag: one 32-bit word per node = (covering particle << 8) | inside-sample count (or table code).
// 0 = uncovered (the particle bits are meaningless when the count is 0), so one memset clears the map and
// the fused kernel reads one word per node.  Particle indices are 24 bits: max_particles <= 2^24.
constexpr int kTagPidShift = 8;
constexpr int64_t kMaxParticles = (int64_t)1 << 24;
__host__ __device__ constexpr uint32_t make_tag(int32_t p, int cnt) {
  return cnt > 0 ? ((uint32_t)p << kTagPidShift) | (uint32_t)cnt : 0u;
}
__host__ __device__ constexpr int tag_cnt(uint32_t t) { return (int)(t & 0xffu); }
__host__ __device__ constexpr int32_t tag_pid(uint32_t t) { return (t & 0xffu) ? (int32_t)(t >> kTagPidShift) : -1; }

// Per-particle force / torque accumulators of the fused step: NV = 3 (2D: Fx Fy Tz) or 6 (3D: F, T) values,
// each a pair of 64-bit fixed-point words (value = hi 2^-40 + lo 2^-91), added with integer atomics: the
// sum does not depend on the order in which warps arrive (collide.cuh: reduce_runs).
__host__ __device__ constexpr int force_values(int dim) { return dim == 3 ? 6 : 3; }

struct Geom {
  int dim;
  int nx, ny, nz;   // nodes per axis (each < 2^31)
  int bcx, bcy, bcz;  // 0 periodic, 1 walls
  int64_t N;        // nx*ny*nz
};

// Slab decomposition along y (include/lbmimb.h "Slabs").  A slab lattice stores its owned rows
// plus one ghost row on every side that is not a wall of the global lattice.  Two geometries describe it:
//   the STORED lattice (lbmimb_lattice::g): ny = stored rows; what the lattice kernels index;
//   the GLOBAL lattice (lbmimb_lattice::gp): ny = rows of the whole lattice; what the particle-side
//   kernels compute in (particle coordinates are global, so every inside test, minimum image and
//   contact is the same arithmetic as on the undivided lattice).
// SlabRows connects them: stored row jl <-> global row jg = jl + oy (mod gny).
struct SlabRows {
  int ny_stored;      // rows in memory (owned + ghosts)
  int gny;            // rows of the global lattice
  int oy;             // global row of stored row 0 (-1 for the lower ghost of the first periodic slab)
  int own_lo, own_hi; // stored rows [own_lo, own_hi) are owned; the others are ghosts
  int wall_lo, wall_hi;  // is the lower / upper end of the STORED lattice a wall (else: ghost row or periodic wrap)
};

__host__ __device__ __forceinline__ int slab_global_row(const SlabRows &s, int jl) {
  int jg = jl + s.oy;
  if (jg < 0) jg += s.gny;
  else if (jg >= s.gny) jg -= s.gny;
  return jg;
}
// stored row of global row jg, or -1 if this slab does not store it
__host__ __device__ __forceinline__ int slab_stored_row(const SlabRows &s, int jg) {
  int jl = jg - s.oy;
  if (jl < 0) jl += s.gny;
  else if (jl >= s.gny) jl -= s.gny;
  return jl < s.ny_stored ? jl : -1;
}

// Cell list over the particles (mapping fix-up pass and DEM contacts).
struct CellList {
  int ncx, ncy, ncz;     // cells per axis
  double inv_ex, inv_ey, inv_ez;  // 1 / cell edge
  int64_t ncells;
  int32_t *count;   // [ncells_max + 1]
  int32_t *start;   // [ncells_max + 1] exclusive scan of count
  int32_t *fill;    // [ncells_max]
  int32_t *items;   // [Pmax] particle indices, ascending inside a cell
  int32_t *cell_of; // [Pmax]
  int32_t *block_sums;  // scan scratch
  int64_t ncells_max;
  bool count_clean;     // count[] is all zero (the DEM first half adds to it; cl_small_kernel leaves it zeroed)
};

// Verlet neighbour lists of a4 (R19).  Library-allocated (sized from the radii).
//   items [K][Pcap] slot-major (thread i reading slot k is coalesced), count [Pcap], x_ref [3][Pcap];
//   build grid: cells of edge >= 2 R_max + skin with C slots each (gcount [ncells], gitems [ncells][C]);
//   state (device): [0] valid [1] age in dem_steps [2] builds [3] displacement flag
//                   [4] list overflow [5] grid overflow.
struct NeighborList {
  int mode;            // LBMIMB_NEIGHBOR_*
  double skin;
  int every;
  void *mem;           // one cudaMalloc holding everything below
  int64_t Pcap;
  int K, C;
  int32_t *items, *count, *state, *gcount, *gitems;
  double *x_ref;
  int nc[3];
  double inv_e[3];
  int64_t ncells;
  double rmax, rmin;   // radii the storage was sized for
};

// One instantiated CUDA graph of TWO consecutive coupled steps (lbmimb_run_coupled) and everything its
// launches were captured with: it is replayed only while all of this still holds.
struct CoupledGraph {
  cudaGraphExec_t exec;
  bool valid;
  int64_t launches;   // kernels per replay
  int64_t P;
  double rmax, rmin, table_R, nl_skin;
  int map_mode, nl_mode, nl_every;
  const void *nl_mem;
  lbmimb_dem_params dem;
};

}  // namespace lbmimb

struct lbmimb_lattice {
  lbmimb_params prm;
  lbmimb::Geom g;      // the STORED lattice (ny = owned rows + ghost rows)
  lbmimb::Geom gp;     // the GLOBAL lattice the particles live in (= g unless this is a slab)
  lbmimb::SlabRows sl;
  bool is_slab;
  int Q;
  int SD;            // S^dim
  cudaStream_t stream;
  bool owns_ws;
  char *ws;
  uint64_t ws_bytes;

  // lattice state.  f[cur] holds the POST-COLLISION distributions f*(x, t-1) of the last step
  // ("pull" representation): f_i(x,t) = f*_i(x - c_i) or, through a wall, f*_{-i}(x).
  // In AA mode (prm.streaming == LBMIMB_STREAM_AA) there is one array f[0]; aa_swapped tells which of
  // the two AA layouts it is in (lattice.cu: collide_stream_aa_kernel).
  double *f[2];
  int cur;
  bool aa, aa_swapped;
  uint32_t *tag;      // [N] node tags (make_tag)
  double *s;          // [N][exchange_stride] exchange vectors of the last step; NULL unless keep_s
  bool keep_s;        // LBMIMB_FLAG_EXCHANGE_FIELD
  long long *facc;    // [Pmax][force_values][2] fixed-point force / torque sums of the last emitting step
  bool acc_dirty;     // facc holds sums that have not been folded into force / torque (or discarded) yet
  double *beta_tab;   // [256] beta(n_s / S^D, tau)
  int64_t *contested; // mapping fix-up list
  int64_t contested_cap;
  int32_t *counters;  // [16]: [0] shared-node count, [1] its overflow flag, [8..13] result of validate_particles_dev
  void *fetch_stage;     // AA mode: grow-only staging buffer of fetch_fields (library-allocated)
  size_t fetch_stage_bytes;
  double *diag_partial;  // [kDiagBlocksMax][8] stage-1 sums of lbmimb_diagnostics
  double *diag_out;      // [20]

  // particles (SoA, device)
  int64_t Pmax, P;
  double *pos, *vel, *omega, *radius, *mass, *force, *torque, *fc, *prec;
  double *pos2, *vel2;   // state after the first half of a DEM step (double buffer, cell-list mode)
  double rmax, rmin;  // largest / smallest radius of the current set
  int map_mode;       // LBMIMB_MAP_SAMPLING or LBMIMB_MAP_TABLE
  uint8_t *eps_table; // table of map mode TABLE (R17), built for radius table_R
  double table_R;
  lbmimb::CellList cl;
  bool cl_valid;
  lbmimb::NeighborList nl;
  lbmimb::CoupledGraph cg[2];   // indexed by the distribution-array parity at the start of the pair
  cudaStream_t cap_stream;      // private stream the pair is captured on
  bool cg_broken;               // a capture failed once: keep to plain launches

  bool map_valid;     // eps_cnt/pid match the particle positions
  bool s_valid;       // the last step ran under the current map and left its force sums (and s, if kept)
  bool forces_valid;  // force/torque hold the reduction of s
  int64_t t;
  int64_t launches;
};

namespace lbmimb {

lbmimb_status fail(lbmimb_status st, const char *fmt, ...);
lbmimb_status cuda_fail(cudaError_t e, const char *what);

#define LBMIMB_CUDA(call)                                            \
  do {                                                               \
    cudaError_t e__ = (call);                                        \
    if (e__ != cudaSuccess) return ::lbmimb::cuda_fail(e__, #call);  \
  } while (0)

#define LBMIMB_LAUNCH_CHECK(h, name)                                 \
  do {                                                               \
    (h)->launches += 1;                                              \
    cudaError_t e__ = cudaGetLastError();                            \
    if (e__ != cudaSuccess) return ::lbmimb::cuda_fail(e__, name);   \
  } while (0)

// kernels.cu entry points used by api.cu
lbmimb_status launch_init_rest(lbmimb_lattice *h);
lbmimb_status launch_collide_stream(lbmimb_lattice *h, bool emit);
lbmimb_status launch_unstream(lbmimb_lattice *h, const double *f_pre, double *f_post);
lbmimb_status launch_fetch(lbmimb_lattice *h, int what, const int64_t lo[3], const int64_t hi[3], void *dst_dev);
lbmimb_status launch_pack_records(lbmimb_lattice *h);
lbmimb_status validate_particles_dev(lbmimb_lattice *h, int64_t P, const double *pos_dev, const double *radius_dev,
                                     const double *mass_dev, double *rmax, double *rmin);
lbmimb_status build_cell_list(lbmimb_lattice *h);
lbmimb_status launch_map(lbmimb_lattice *h);
lbmimb_status ensure_eps_table(lbmimb_lattice *h);
int64_t eps_table_entries(int dim);
lbmimb_status launch_finish_forces(lbmimb_lattice *h);   // facc -> force / torque, clears facc
lbmimb_status launch_dem(lbmimb_lattice *h, const lbmimb_dem_params *dem, bool finish);
bool dem_can_finish(const lbmimb_lattice *h);
lbmimb_status neighbor_list_prepare(lbmimb_lattice *h);   // (re)allocates the list storage for the current radii
void neighbor_list_release(lbmimb_lattice *h);
lbmimb_status neighbor_list_invalidate(lbmimb_lattice *h);  // positions were replaced
lbmimb_status launch_diagnostics(lbmimb_lattice *h, double eps_den);
lbmimb_status launch_diagnostics_static(lbmimb_lattice *h, double eps_den, double *out_dev);   // scratch: a static device array
int64_t diagnostics_static_max_particles();
int64_t diagnostics_static_scratch_bytes();
lbmimb_status launch_halo(lbmimb_lattice *h, int side, double *buf_dev, bool pack);
int64_t halo_doubles(const lbmimb_lattice *h);
constexpr int kDiagBlocksMax = 148 * 8;

}  // namespace lbmimb
