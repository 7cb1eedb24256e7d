// a1 in TABLE mode (NEXT-1): the paper's own way to get the solid fraction, gamma = phi(d, theta)
// looked up in a pre-calculated table (eq. (6)); included by particles.cu.
//
// Discretisation (R17; Fig. 1 of the paper is not available): distance bins over
// [R - sqrt(D)/2, R + sqrt(D)/2) (outside that range a cell is full or empty), orientation as the ratios
// t1 = b/a, t2 = c/a of the sorted absolute displacement components a >= b >= c (t1 = tan(theta) in 2D),
// so that no transcendental function enters an index and the look-up is reproducible bit for bit.
// Entry = 8-bit code of the fraction of St^D sub-cell points of the cell inside the particle.
// The paper keeps the table in constant memory (Fermi: broadcast reads); neighbouring lanes look up
// different entries, which constant memory serialises, so here it is a 4-32 KB global array read
// through the L1 read-only path.
#pragma once
// (included inside namespace lbmimb, after MapArgs / bbox_axis / min_image_d / wrap_i / sub_offset /
//  map_pass1.cuh / CellGeom)

struct TableGeom {
  int Nd, Nt, St;
  double R, d0, inv_dd, dd;
  double full2, none2;  // d^2 below / above which a node is surely full / empty (1e-9 margin): skips the sqrt
  const uint8_t *tab;
};

// ---------------------------------------------------------------------------
// Table construction: one block per entry.  Same point set and inside test as the sampled map (R4):
// every operation is a separate IEEE operation, no FMA.
// ---------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256) build_eps_table_kernel(TableGeom t, uint8_t *__restrict__ out) {
  __shared__ double px2[256], py2[256], pz2[256];
  __shared__ unsigned long long total_in;
  const int Nt2 = D == 3 ? t.Nt : 1;
  const int e = blockIdx.x;
  const int m2 = e % Nt2, r = e / Nt2;
  const int m1 = r % t.Nt, k = r / t.Nt;
  const double dk = __dadd_rn(t.d0, __dmul_rn(__dadd_rn((double)k, 0.5), t.dd));
  const double t1 = __ddiv_rn(__dadd_rn((double)m1, 0.5), (double)t.Nt);
  const double t2 = D == 3 ? __ddiv_rn(__dadd_rn((double)m2, 0.5), (double)t.Nt) : 0.0;
  double nrm2 = __dadd_rn(1.0, __dmul_rn(t1, t1));
  if (D == 3) nrm2 = __dadd_rn(nrm2, __dmul_rn(t2, t2));
  const double rx = __ddiv_rn(dk, __dsqrt_rn(nrm2));
  const double ry = __dmul_rn(rx, t1);
  const double rz = __dmul_rn(rx, t2);
  if (threadIdx.x == 0) total_in = 0ull;
  for (int a = threadIdx.x; a < t.St; a += blockDim.x) {
    const double off = sub_offset(a, t.St);
    const double x = __dadd_rn(rx, off), y = __dadd_rn(ry, off), z = __dadd_rn(rz, off);
    px2[a] = __dmul_rn(x, x);
    py2[a] = __dmul_rn(y, y);
    pz2[a] = __dmul_rn(z, z);
  }
  __syncthreads();
  const double R2 = __dmul_rn(t.R, t.R);
  const int rows = D == 3 ? t.St * t.St : t.St;
  unsigned long long cnt = 0;
  for (int row = threadIdx.x; row < rows; row += blockDim.x) {
    const int ay = row % t.St, az = row / t.St;
    const double y2 = py2[ay], z2 = pz2[az];
    for (int ax = 0; ax < t.St; ++ax) {
      double d2 = __dadd_rn(px2[ax], y2);
      if (D == 3) d2 = __dadd_rn(d2, z2);
      cnt += d2 <= R2 ? 1ull : 0ull;
    }
  }
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(&total_in, cnt);
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long total = (unsigned long long)t.St * t.St * (D == 3 ? t.St : 1);
    out[e] = (uint8_t)((255ull * total_in + total / 2) / total);
  }
}

// ---------------------------------------------------------------------------
// Look-up of one node from its displacement (minimum image already applied).
// ---------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ int table_code(const TableGeom &t, double dx, double dy, double dz) {
  double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
  if (D == 3) d2 = __dadd_rn(d2, __dmul_rn(dz, dz));
  if (d2 < t.full2) return 255;
  if (d2 > t.none2) return 0;
  const double d = __dsqrt_rn(d2);
  if (d < t.d0) return 255;
  const double u = __dmul_rn(__dsub_rn(d, t.d0), t.inv_dd);
  if (u >= (double)t.Nd) return 0;
  const int k = (int)u;
  double a = fabs(dx), b = fabs(dy), c = D == 3 ? fabs(dz) : 0.0, s;
  if (a < b) { s = a; a = b; b = s; }
  if (D == 3) {
    if (b < c) { s = b; b = c; c = s; }
    if (a < b) { s = a; a = b; b = s; }
  }
  int m1 = (int)__dmul_rn(__ddiv_rn(b, a), (double)t.Nt);
  if (m1 > t.Nt - 1) m1 = t.Nt - 1;
  int idx = k * t.Nt + m1;
  if (D == 3) {
    int m2 = (int)__dmul_rn(__ddiv_rn(c, a), (double)t.Nt);
    if (m2 > t.Nt - 1) m2 = t.Nt - 1;
    idx = idx * t.Nt + m2;
  }
  return (int)__ldg(t.tab + idx);
}

// ---------------------------------------------------------------------------
// pass 1: one group of G threads per particle, one look-up per candidate node.  Dense walk of the bounding
// box (map_pass1.cuh): a node can have a non-zero code only if d^2 <= none2, so every row (j,k) contributes
// the columns with |dx| <= sqrt(none2 - dy^2 - dz^2) (+ margin: a superset) and the group walks the
// concatenated intervals.  The look-up itself is unchanged.  Shared nodes are detected like in the sampled
// map (exchange on the node tag, examined one commit later).
// ---------------------------------------------------------------------------
template <int D, int G>
__global__ void __launch_bounds__(128) map_table_kernel(const MapArgs a, const TableGeom t) {
  constexpr int groups = 128 / G;
  constexpr int NW = G >= 32 ? G / 32 : 1;
  __shared__ int pre[groups][G + 1];
  __shared__ int beg[groups][G];
  __shared__ int wtot[groups][NW];
  const int grp = threadIdx.x / G, gl = threadIdx.x % G;
  const int64_t p = (int64_t)blockIdx.x * groups + grp;
  const bool active = p < a.P;
  double cx = 0.0, cy = 0.0, cz = 0.0;
  const double R = t.R;
  int lo[3] = {0, 0, 0}, ext[3] = {0, 1, 1};
  bool wx = false, wy = false, wz = false;
  if (active) {
    cx = a.pos[p];
    cy = a.pos[a.P + p];
    cz = D == 3 ? a.pos[2 * a.P + p] : 0.0;
    bbox_axis(cx, R, a.g.nx, a.g.bcx, lo[0], ext[0]);
    bbox_axis(cy, R, a.g.ny, a.g.bcy, lo[1], ext[1]);
    if (D == 3) bbox_axis(cz, R, a.g.nz, a.g.bcz, lo[2], ext[2]);
    wx = crosses_seam(cx, R, a.g.nx, a.g.bcx);
    wy = crosses_seam(cy, R, a.g.ny, a.g.bcy);
    wz = D == 3 && crosses_seam(cz, R, a.g.nz, a.g.bcz);
  }
  int nrows = 0;
  if (active && ext[0] > 0) {
    const int64_t r64 = (int64_t)ext[1] * ext[2];
    nrows = r64 > (1 << 24) ? (1 << 24) : (int)r64;
  }
  const int nrows_u = group_uniform_max<G>(nrows);
  const float inv1 = 1.0f / (float)(ext[1] > 0 ? ext[1] : 1);
  auto row_of = [&](int row, int &j, int &k) {
    int bk = 0, bj = row;
    if (D == 3) fast_divmod(row, ext[1], inv1, bk, bj);
    j = lo[1] + bj;
    k = lo[2] + bk;
    if (wy) j = wrap_i(j, a.g.ny);
    if (D == 3 && wz) k = wrap_i(k, a.g.nz);
  };
  int64_t pend_x = -1;
  uint32_t pend_old = 0;
  auto settle = [&]() {
    if (pend_x >= 0 && pend_old != 0u && tag_pid(pend_old) != (int32_t)p) {
      const int slot = atomicAdd(a.counters, 1);
      if (slot < a.contested_cap) a.contested[slot] = pend_x;
      else a.counters[1] = 1;
    }
    pend_x = -1;
  };
  for (int row0 = 0; row0 < nrows_u; row0 += G) {
    int b0 = 0, len = 0;
    if (row0 + gl < nrows) {
      int j, k;
      row_of(row0 + gl, j, k);
      double dy = (double)j - cy, dz = D == 3 ? (double)k - cz : 0.0;
      if (wy) dy = min_image_d(dy, a.g.ny);
      if (D == 3 && wz) dz = min_image_d(dz, a.g.nz);
      const double rad = t.none2 - dy * dy - dz * dz;
      if (rad > -1e-9 && slab_stored_row(a.sl, j) >= 0) {
        if (wx) len = ext[0];
        else clip_interval(cx, sqrt(fmax(rad, 0.0) + 1e-9) + 1e-9, lo[0], ext[0], b0, len);
      }
    }
    const int total = scan_row_intervals<G>(len, b0, gl, pre[grp], beg[grp], wtot[grp]);
    for (int c = gl; c < total; c += G) {
      const int r = interval_row<G>(pre[grp], c);
      int i = lo[0] + beg[grp][r] + (c - pre[grp][r]), j, k;
      row_of(row0 + r, j, k);
      if (wx) i = wrap_i(i, a.g.nx);
      double dx = __dsub_rn((double)i, cx), dy = __dsub_rn((double)j, cy), dz = D == 3 ? __dsub_rn((double)k, cz) : 0.0;
      if (wx) dx = min_image_d(dx, a.g.nx);
      if (wy) dy = min_image_d(dy, a.g.ny);
      if (D == 3 && wz) dz = min_image_d(dz, a.g.nz);
      const int code = table_code<D>(t, dx, dy, dz);
      if (code > 0) {
        const int64_t x = ((int64_t)k * a.sl.ny_stored + slab_stored_row(a.sl, j)) * a.g.nx + i;
        settle();
        pend_old = atomicExch(a.tag + x, make_tag((int32_t)p, code));
        pend_x = x;
      }
    }
    group_sync<G>();
  }
  settle();
}

// ---------------------------------------------------------------------------
// pass 2: nodes reached by more than one particle: code = min(255, sum of the particles' codes),
// covering particle = largest code, ties -> lowest index.  One warp per node, one candidate per lane.
// ---------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128) map_table_contested_kernel(const MapArgs a, const TableGeom t, const CellGeom cg,
                                                                  const int32_t *__restrict__ start,
                                                                  const int32_t *__restrict__ items) {
  int total = a.counters[0];
  if (total > a.contested_cap) total = (int)a.contested_cap;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const int lo0 = off_lo(cg.nc[0], cg.periodic[0]), n0 = off_hi(cg.nc[0], cg.periodic[0]) - lo0 + 1;
  const int lo1 = off_lo(cg.nc[1], cg.periodic[1]), n1 = off_hi(cg.nc[1], cg.periodic[1]) - lo1 + 1;
  const int lo2 = D == 3 ? off_lo(cg.nc[2], cg.periodic[2]) : 0;
  const int n2 = D == 3 ? off_hi(cg.nc[2], cg.periodic[2]) - lo2 + 1 : 1;
  const bool cell_lane = lane < n0 * n1 * n2;
  const int ox = lo0 + lane % n0, oy = lo1 + (lane / n0) % n1, oz = lo2 + lane / (n0 * n1);
  for (int e = wid; e < total; e += warps) {
    const int64_t x = a.contested[e];
    const int i = (int)(x % a.g.nx);
    const int64_t r = x / a.g.nx;
    const int j = slab_global_row(a.sl, (int)(r % a.sl.ny_stored)), k = (int)(r / a.sl.ny_stored);
    int b = 0, en = 0;
    if (cell_lane) {
      int cx_ = cell_coord((double)i, cg, 0) + ox, cy_ = cell_coord((double)j, cg, 1) + oy;
      int cz_ = D == 3 ? cell_coord((double)k, cg, 2) + oz : 0;
      bool ok = true;
      if (cg.periodic[0]) cx_ = wrap_i(cx_, cg.nc[0]);
      else ok = ok && cx_ >= 0 && cx_ < cg.nc[0];
      if (cg.periodic[1]) cy_ = wrap_i(cy_, cg.nc[1]);
      else ok = ok && cy_ >= 0 && cy_ < cg.nc[1];
      if (D == 3) {
        if (cg.periodic[2]) cz_ = wrap_i(cz_, cg.nc[2]);
        else ok = ok && cz_ >= 0 && cz_ < cg.nc[2];
      }
      if (ok) {
        const int c = (cz_ * cg.nc[1] + cy_) * cg.nc[0] + cx_;
        b = __ldg(start + c);
        en = __ldg(start + c + 1);
      }
    }
    int sum = 0, best_code = 0, best_p = -1;
    // each lane walks the particles of its own cell; lanes are combined afterwards
    for (int it = b; it < en; ++it) {
      const int p = __ldg(items + it);
      double dx = __dsub_rn((double)i, a.pos[p]), dy = __dsub_rn((double)j, a.pos[a.P + p]);
      double dz = D == 3 ? __dsub_rn((double)k, a.pos[2 * a.P + p]) : 0.0;
      if (!a.g.bcx) dx = min_image_d(dx, a.g.nx);
      if (!a.g.bcy) dy = min_image_d(dy, a.g.ny);
      if (D == 3 && !a.g.bcz) dz = min_image_d(dz, a.g.nz);
      const int code = table_code<D>(t, dx, dy, dz);
      sum += code;
      if (code > best_code || (code == best_code && code > 0 && p < best_p)) {
        best_code = code;
        best_p = p;
      }
    }
    for (int o = 16; o > 0; o >>= 1) {
      sum += __shfl_xor_sync(0xffffffffu, sum, o);
      const int oc = __shfl_xor_sync(0xffffffffu, best_code, o);
      const int op = __shfl_xor_sync(0xffffffffu, best_p, o);
      if (oc > best_code || (oc == best_code && oc > 0 && (best_p < 0 || op < best_p))) {
        best_code = oc;
        best_p = op;
      }
    }
    if (lane == 0) a.tag[x] = make_tag(best_p, sum > 255 ? 255 : sum);
  }
}
