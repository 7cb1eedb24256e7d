// Verlet neighbour lists for the DEM contacts (a4): the paper's scheme of PAPER.md:69 ("The
// neighbor-list of each solid particle is established roughly every 100th time step"), reading
// DESIGN.md R19 (text in include/lbmimb.h).  Included by particles.cu after CellGeom / cell_coord.
//
// Everything that decides list membership or a rebuild is a separate IEEE operation
// (__dadd_rn / __dsub_rn / __dmul_rn): integer results, bit-exact against the definition.
//
// The rebuild decision lives on the device: every contact evaluation launches the three build
// kernels below, and each of them returns at once unless nl_need(state) holds.  The state is
// committed by the contact kernel that follows them in stream order (dem_contact_list_kernel),
// the displacement flag is raised by the drift kernel, the age advances in the final kick.
#pragma once
// (included inside namespace lbmimb, after CellGeom / cell_coord / min_image_d / wrap_i / off_lo / off_hi)

enum { NL_VALID = 0, NL_AGE = 1, NL_BUILDS = 2, NL_DISP = 3, NL_OVF_LIST = 4, NL_OVF_GRID = 5, NL_STATE_WORDS = 16 };

__device__ __forceinline__ bool nl_need(const int32_t *st, int every) {
  return st[NL_VALID] == 0 || st[NL_AGE] >= every || st[NL_DISP] != 0;
}

struct VerletArgs {
  Geom g;
  CellGeom cg;       // build grid: cells of edge >= 2 R_max + skin
  int64_t P, Pcap, ncells;
  const double *pos, *radius;
  double skin;
  int every, K, C;
  int32_t *items, *count, *state, *gcount, *gitems;
  double *x_ref;
};

__global__ void verlet_clear_kernel(const VerletArgs a) {
  if (!nl_need(a.state, a.every)) return;
  for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < a.ncells; c += (int64_t)gridDim.x * blockDim.x)
    a.gcount[c] = 0;
}

// particles -> grid cells with C slots each (order inside a cell is arbitrary: the lists are sorted)
template <int D>
__global__ void verlet_bin_kernel(const VerletArgs a) {
  if (!nl_need(a.state, a.every)) return;
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= a.P) return;
  const int cx = cell_coord(a.pos[p], a.cg, 0);
  const int cy = cell_coord(a.pos[a.P + p], a.cg, 1);
  const int cz = D == 3 ? cell_coord(a.pos[2 * a.P + p], a.cg, 2) : 0;
  const int64_t c = ((int64_t)cz * a.cg.nc[1] + cy) * a.cg.nc[0] + cx;
  const int slot = atomicAdd(a.gcount + c, 1);
  if (slot < a.C) a.gitems[c * a.C + slot] = (int32_t)p;
  else a.state[NL_OVF_GRID] = 1;
}

// L(i) by its definition over the 3^D cells around particle i, kept in ascending j; also
// records the build positions x_ref.
template <int D>
__global__ void verlet_list_kernel(const VerletArgs a) {
  if (!nl_need(a.state, a.every)) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.P) return;
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  const bool per[3] = {!a.g.bcx, !a.g.bcy, !a.g.bcz};
  double xi[3] = {0.0, 0.0, 0.0};
  int cc[3] = {0, 0, 0};
  for (int q = 0; q < D; ++q) {
    xi[q] = a.pos[(int64_t)q * a.P + i];
    a.x_ref[(int64_t)q * a.Pcap + i] = xi[q];
    cc[q] = cell_coord(xi[q], a.cg, q);
  }
  const double Ri = a.radius[i];
  const int nc0 = a.cg.nc[0], nc1 = a.cg.nc[1], nc2 = D == 3 ? a.cg.nc[2] : 1;
  int32_t *mine = a.items + i;   // slot k at mine[k * Pcap]
  int cnt = 0;
  bool overflow = false;
  for (int oz = D == 3 ? off_lo(nc2, a.cg.periodic[2]) : 0; oz <= (D == 3 ? off_hi(nc2, a.cg.periodic[2]) : 0); ++oz)
    for (int oy = off_lo(nc1, a.cg.periodic[1]); oy <= off_hi(nc1, a.cg.periodic[1]); ++oy)
      for (int ox = off_lo(nc0, a.cg.periodic[0]); ox <= off_hi(nc0, a.cg.periodic[0]); ++ox) {
        int ex = cc[0] + ox, ey = cc[1] + oy, ez = cc[2] + oz;
        if (a.cg.periodic[0]) ex = wrap_i(ex, nc0);
        else if (ex < 0 || ex >= nc0) continue;
        if (a.cg.periodic[1]) ey = wrap_i(ey, nc1);
        else if (ey < 0 || ey >= nc1) continue;
        if (D == 3) {
          if (a.cg.periodic[2]) ez = wrap_i(ez, nc2);
          else if (ez < 0 || ez >= nc2) continue;
        }
        const int64_t c = ((int64_t)ez * nc1 + ey) * nc0 + ex;
        int m = a.gcount[c];
        m = m < a.C ? m : a.C;
        for (int it = 0; it < m; ++it) {
          const int j = a.gitems[c * a.C + it];
          if (j == (int)i) continue;
          double dist2 = 0.0;
          for (int q = 0; q < D; ++q) {
            double d = __dsub_rn(xi[q], a.pos[(int64_t)q * a.P + j]);
            if (per[q]) d = min_image_d(d, n[q]);
            dist2 = __dadd_rn(dist2, __dmul_rn(d, d));
          }
          const double Rc = __dadd_rn(__dadd_rn(Ri, a.radius[j]), a.skin);
          if (!(dist2 < __dmul_rn(Rc, Rc))) continue;
          if (cnt >= a.K) {
            overflow = true;
            continue;
          }
          int q = cnt - 1;
          while (q >= 0 && mine[(int64_t)q * a.Pcap] > j) {
            mine[(int64_t)(q + 1) * a.Pcap] = mine[(int64_t)q * a.Pcap];
            --q;
          }
          mine[(int64_t)(q + 1) * a.Pcap] = j;
          ++cnt;
        }
      }
  a.count[i] = cnt;
  if (overflow) a.state[NL_OVF_LIST] = 1;
}

// squared displacement of a particle from its build position, as the rebuild rule states it
template <int D>
__device__ __forceinline__ double verlet_disp2(const double *x, const double *x_ref, int64_t Pcap, int64_t p,
                                               const int *n, const bool *per) {
  double d2 = 0.0;
  for (int q = 0; q < D; ++q) {
    double d = __dsub_rn(x[q], x_ref[(int64_t)q * Pcap + p]);
    if (per[q]) d = min_image_d(d, n[q]);
    d2 = __dadd_rn(d2, __dmul_rn(d, d));
  }
  return d2;
}

