// a1, pass 1 of the particle -> lattice mapping (included by particles.cu).
//
// One group of G threads per particle walks the particle's bounding box.
//   phase A: every row of the box gets the interval of columns that can hold a covered node and, inside it,
//            the interval of columns that are surely full (count = S^D) -- two square roots per row, no
//            per-node classification (dense walk, below);
//   phase B: one THREAD per boundary cell counts the inside samples.  The squared distance is
//            separable, d2 = (dx^2 + dy^2) + dz^2 with dx depending on (i, ax) only, so the S
//            values per axis are formed once (S*D subtract/multiply) and the S^D samples cost one
//            or two additions and a compare each.  Every operation is the same IEEE operation on
//            the same operands as in the definition (include/lbmimb.h a1), so the counts are
//            bit-exact; only the order in which samples are visited differs.
// Nodes reached by more than one particle are detected with an atomic exchange on the node tag and
// queued for pass 2 (map_contested_kernel), which recomputes them from the definition.
// (Measured and dropped: one thread per ROW that writes the full columns itself and lists only the
//  shell -- no per-node classification, but serial commits per thread: C3 0.325 -> 0.369 ms, C4 1.50 -> 1.73 ms.)
#pragma once
// (included inside namespace lbmimb, after MapArgs / bbox_axis / min_image_d / wrap_i / sub_offset)

// exact b / d and b % d for 0 <= b < 2^24, d >= 1, without the integer-division sequence
__device__ __forceinline__ void fast_divmod(int b, int d, float inv_d, int &q, int &r) {
  q = __float2int_rz((float)b * inv_d);
  r = b - q * d;
  if (r < 0) {
    --q;
    r += d;
  } else if (r >= d) {
    ++q;
    r -= d;
  }
}

// inside-sample count of one node, compile-time S (register arrays).  SEAM = false: the particle's box touches
// no periodic seam (all but a few particles), so the minimum-image steps are compiled out (16 conditionals per
// cell in 2D, 12 in 3D; the kernel is issue-bound).
template <int D, int S, bool SEAM>
__device__ __forceinline__ int thread_count_fixed(const Geom &g, const double *__restrict__ sub, int i, int j, int k,
                                                  double cx, double cy, double cz, double R2, bool wx, bool wy,
                                                  bool wz) {
  double dx2[S], dy2[S], dz2[S];
  const double di = (double)i, dj = (double)j, dk = (double)k;
#pragma unroll
  for (int a = 0; a < S; ++a) {
    const double so = sub[a];
    double dx = __dsub_rn(__dadd_rn(di, so), cx);
    double dy = __dsub_rn(__dadd_rn(dj, so), cy);
    if (SEAM && wx) dx = min_image_d(dx, g.nx);
    if (SEAM && wy) dy = min_image_d(dy, g.ny);
    dx2[a] = __dmul_rn(dx, dx);
    dy2[a] = __dmul_rn(dy, dy);
    if (D == 3) {
      double dz = __dsub_rn(__dadd_rn(dk, so), cz);
      if (SEAM && wz) dz = min_image_d(dz, g.nz);
      dz2[a] = __dmul_rn(dz, dz);
    } else {
      dz2[a] = 0.0;
    }
  }
  int cnt = 0;
#pragma unroll
  for (int ay = 0; ay < S; ++ay) {
#pragma unroll
    for (int ax = 0; ax < S; ++ax) {
      const double s2 = __dadd_rn(dx2[ax], dy2[ay]);
      if (D == 2) {
        cnt += s2 <= R2 ? 1 : 0;
      } else {
#pragma unroll
        for (int az = 0; az < S; ++az) cnt += __dadd_rn(s2, dz2[az]) <= R2 ? 1 : 0;
      }
    }
  }
  return cnt;
}

// inside-sample count of one node, run-time S
template <int D>
__device__ __forceinline__ int thread_count_generic(const Geom &g, int S, const double *__restrict__ sub, int i, int j,
                                                    int k, double cx, double cy, double cz, double R2, bool wx, bool wy,
                                                    bool wz) {
  const double di = (double)i, dj = (double)j, dk = (double)k;
  int cnt = 0;
  for (int az = 0; az < (D == 3 ? S : 1); ++az) {
    double dz2 = 0.0;
    if (D == 3) {
      double dz = __dsub_rn(__dadd_rn(dk, sub[az]), cz);
      if (wz) dz = min_image_d(dz, g.nz);
      dz2 = __dmul_rn(dz, dz);
    }
    for (int ay = 0; ay < S; ++ay) {
      double dy = __dsub_rn(__dadd_rn(dj, sub[ay]), cy);
      if (wy) dy = min_image_d(dy, g.ny);
      const double dy2 = __dmul_rn(dy, dy);
      for (int ax = 0; ax < S; ++ax) {
        double dx = __dsub_rn(__dadd_rn(di, sub[ax]), cx);
        if (wx) dx = min_image_d(dx, g.nx);
        double d2 = __dadd_rn(__dmul_rn(dx, dx), dy2);
        if (D == 3) d2 = __dadd_rn(d2, dz2);
        cnt += d2 <= R2 ? 1 : 0;
      }
    }
  }
  return cnt;
}

// does the bounding box of this particle touch the periodic seam of an axis (or cover it whole)?
__device__ __forceinline__ bool crosses_seam(double c, double R, int n, int bc) {
  if (bc) return false;
  const int l = (int)floor(c - R) - 1;
  const int h = (int)ceil(c + R) + 1;
  return l < 0 || h > n - 1;
}

// Group barrier: a warp (or part of one) synchronises with __syncwarp, larger groups with the block barrier
// (all groups of a block run the same number of chunk iterations: the count is the block maximum).
template <int G>
__device__ __forceinline__ void group_sync() {
  if (G <= 32) __syncwarp();
  else __syncthreads();
}

// ---- dense walks of a particle's bounding box (map pass 1, table map, force reduction) ----
// Each of the G threads of a group brings the candidate interval [b0, b0 + len) of columns of ONE row of the
// box; the intervals are concatenated: pre[r] = number of candidates in rows < r (exclusive scan), beg[r] =
// first column of row r.  Candidate t then sits in row interval_row<G>(pre, t) at column beg[r] + t - pre[r].
// Returns the number of candidates of the G rows.  Ends with a group barrier (pre / beg are readable).
// pre: [G + 1] ints, beg: [G], wtot: [G / 32] (groups of more than one warp), all in shared memory.
template <int G>
__device__ __forceinline__ int scan_row_intervals(int len, int b0, int gl, int *pre, int *beg, int *wtot) {
  constexpr int NW = G >= 32 ? G / 32 : 1;
  constexpr int SW = G < 32 ? G : 32;   // two groups share a warp when G = 16
  const int sl = gl % SW, wid = gl >> 5;
  int incl = len;
#pragma unroll
  for (int o = 1; o < SW; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, incl, o, SW);
    if (sl >= o) incl += t;
  }
  int off = 0, total;
  if (NW > 1) {
    if (sl == 31) wtot[wid] = incl;
    __syncthreads();
    total = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      if (w < wid) off += wtot[w];
      total += wtot[w];
    }
  } else {
    total = __shfl_sync(0xffffffffu, incl, SW - 1, SW);
  }
  pre[gl] = off + incl - len;
  beg[gl] = b0;
  group_sync<G>();
  return total;
}

// largest r in [0, G) with pre[r] <= t
template <int G>
__device__ __forceinline__ int interval_row(const int *pre, int t) {
  int r = 0;
#pragma unroll
  for (int step = G / 2; step > 0; step >>= 1)
    if (pre[r + step] <= t) r += step;
  return r;
}

// loop bounds of groups that share a warp (G < 32) must agree: they synchronise with __syncwarp
template <int G>
__device__ __forceinline__ int group_uniform_max(int v) {
  return G < 32 ? __reduce_max_sync(0xffffffffu, v) : v;
}

// candidate columns of a row: lattice columns i of the box [lo, lo + ext) with |i - c| <= half
__device__ __forceinline__ void clip_interval(double c, double half, int lo, int ext, int &b0, int &len) {
  int il = (int)ceil(c - half), ih = (int)floor(c + half);
  if (il < lo) il = lo;
  if (ih > lo + ext - 1) ih = lo + ext - 1;
  b0 = il - lo;
  len = ih >= il ? ih - il + 1 : 0;
}

// Dense walk of the bounding box.  A sphere fills a third of its box, so classifying every box node spends
// most of its time on nodes that are plainly empty; and classifying every candidate node one by one (round 1)
// still costs ~130 instructions per node.  Here every row (j,k) of the box gets TWO column intervals from
// two square roots:
//   candidates: nodes that can hold an inside sample,  |dx| <= hs + sqrt(r2_none - ny_^2 - nz_^2)  (+ margin),
//               ny_ = max(|dy| - hs, 0): the nearest point of the node's sample cloud is not outside;
//   full      : nodes whose whole sample cloud is inside,  |dx| <= sqrt(r2_full - fy^2 - fz^2) - hs  (- margin),
//               fy = |dy| + hs: the farthest corner of the cloud is inside.
// (hs = 1/2 - 1/(2S) is the half edge of the cloud; the margins, relative 1e-9, dwarf the rounding of either
// side, and erring towards "candidate but not full" only means a node is sampled that needed not be.)
// The full intervals of a chunk of G rows are concatenated (exclusive scan of their lengths) and committed with
// count S^D, one node per thread, coalesced along x; the boundary pieces (candidates left and right of the full
// interval) are concatenated the same way and sampled, one THREAD per boundary cell.  A particle whose box
// covers a whole periodic x axis has no unwrapped coordinate to take intervals in: all its columns are sampled.
template <int D, int G, int SFIX>
__global__ void __launch_bounds__(128) map_particles_kernel(const MapArgs a) {
  constexpr int groups = 128 / G;
  constexpr int NW = G >= 32 ? G / 32 : 1;
  __shared__ double sub[256];
  __shared__ int pre_b[groups][G + 1], pre_f[groups][G + 1];   // exclusive prefixes of the boundary / full lengths
  __shared__ int cbeg[groups][G], fbeg[groups][G], flen[groups][G], clen[groups][G];
  __shared__ int wtot[groups][NW];
  for (int t = threadIdx.x; t < a.S; t += blockDim.x) sub[t] = sub_offset(t, a.S);
  const int grp = threadIdx.x / G, gl = threadIdx.x % G;
  const int64_t p = (int64_t)blockIdx.x * groups + grp;
  const bool active = p < a.P;
  double cx = 0, cy = 0, cz = 0, R = 1;
  int lo[3] = {0, 0, 0}, ext[3] = {0, 1, 1};
  bool wx = false, wy = false, wz = false;
  if (active) {
    cx = a.pos[p];
    cy = a.pos[a.P + p];
    cz = D == 3 ? a.pos[2 * a.P + p] : 0.0;
    R = a.radius[p];
    bbox_axis(cx, R, a.g.nx, a.g.bcx, lo[0], ext[0]);
    bbox_axis(cy, R, a.g.ny, a.g.bcy, lo[1], ext[1]);
    if (D == 3) bbox_axis(cz, R, a.g.nz, a.g.bcz, lo[2], ext[2]);
    wx = crosses_seam(cx, R, a.g.nx, a.g.bcx);
    wy = crosses_seam(cy, R, a.g.ny, a.g.bcy);
    wz = D == 3 && crosses_seam(cz, R, a.g.nz, a.g.bcz);
  }
  const bool whole_x = wx && ext[0] >= a.g.nx;   // box covers the periodic x axis: no interval arithmetic
  int nrows = 0;
  if (active && ext[0] > 0) {
    const int64_t r64 = (int64_t)ext[1] * ext[2];
    nrows = r64 > (1 << 24) ? (1 << 24) : (int)r64;   // (a box of 16 M rows does not occur)
  }
  // groups that share a warp (G < 32) synchronise with __syncwarp: they run the same number of passes
  const int nrows_u = group_uniform_max<G>(nrows);
  const float inv1 = 1.0f / (float)(ext[1] > 0 ? ext[1] : 1);
  const double R2 = __dmul_rn(R, R);
  const double hs = a.hs;
  const double r2_full = R2 - 1e-9 * (R2 + 1.0), r2_none = R2 + 1e-9 * (R2 + 1.0);
  __syncthreads();

  auto row_of = [&](int row, int &j, int &k) {
    int bk = 0, bj = row;
    if (D == 3) fast_divmod(row, ext[1], inv1, bk, bj);
    j = lo[1] + bj;
    k = lo[2] + bk;
    if (wy) j = wrap_i(j, a.g.ny);
    if (D == 3 && wz) k = wrap_i(k, a.g.nz);
  };
  // The exchange on the node tag tells whether another particle reached the node first.  Its result is
  // looked at one commit later (or at the end), so that the round trip of the atomic is off the critical path.
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
  auto commit = [&](int i, int j, int k, int cnt) {
    const int jl = slab_stored_row(a.sl, j);   // (a slab stores only some rows of the global lattice)
    if (jl < 0) return;
    const int64_t x = ((int64_t)k * a.sl.ny_stored + jl) * a.g.nx + i;
    settle();
    pend_old = atomicExch(a.tag + x, make_tag((int32_t)p, cnt));
    pend_x = x;
  };

  for (int row0 = 0; row0 < nrows_u; row0 += G) {
    // ---- the two intervals of each row of this chunk
    int cb = 0, cl = 0, fb = 0, fl = 0;
    if (row0 + gl < nrows) {
      int j, k;
      row_of(row0 + gl, j, k);
      double dy = (double)j - cy, dz = D == 3 ? (double)k - cz : 0.0;
      if (wy) dy = min_image_d(dy, a.g.ny);
      if (D == 3 && wz) dz = min_image_d(dz, a.g.nz);
      const double ay = fabs(dy), az = fabs(dz);
      const double ny_ = fmax(ay - hs, 0.0), nz_ = D == 3 ? fmax(az - hs, 0.0) : 0.0;
      const double rad = r2_none - ny_ * ny_ - nz_ * nz_;
      if (rad > -1e-9 && slab_stored_row(a.sl, j) >= 0) {
        if (whole_x) {
          cl = ext[0];
        } else {
          clip_interval(cx, hs + sqrt(fmax(rad, 0.0) + 1e-9) + 1e-9, lo[0], ext[0], cb, cl);
          const double fy = ay + hs, fz = D == 3 ? az + hs : 0.0;
          const double radf = r2_full - fy * fy - fz * fz;
          if (radf > 0.0 && cl > 0) {
            const double wf = sqrt(radf) - hs - 1e-9;
            if (wf >= 0.0) {
              clip_interval(cx, wf, lo[0] + cb, cl, fb, fl);   // inside the candidate interval
              fb += cb;
            }
          }
        }
      }
    }
    clen[grp][gl] = cl;
    flen[grp][gl] = fl;
    const int totalF = scan_row_intervals<G>(fl, fb, gl, pre_f[grp], fbeg[grp], wtot[grp]);
    const int totalB = scan_row_intervals<G>(cl - fl, cb, gl, pre_b[grp], cbeg[grp], wtot[grp]);

    // ---- full nodes: commit S^D, consecutive columns of a row on consecutive threads
    for (int t = gl; t < totalF; t += G) {
      const int r = interval_row<G>(pre_f[grp], t);
      int i = lo[0] + fbeg[grp][r] + (t - pre_f[grp][r]), j, k;
      row_of(row0 + r, j, k);
      if (wx) i = wrap_i(i, a.g.nx);
      commit(i, j, k, a.SD);
    }
    // ---- boundary cells (left and right of the full interval): one thread samples one cell
    for (int t = gl; t < totalB; t += G) {
      const int r = interval_row<G>(pre_b[grp], t);
      const int o = t - pre_b[grp][r];
      const int cbr = cbeg[grp][r], fbr = fbeg[grp][r], flr = flen[grp][r];
      const int left = flr > 0 ? fbr - cbr : clen[grp][r];
      int i = lo[0] + (o < left ? cbr + o : fbr + flr + (o - left)), j, k;
      row_of(row0 + r, j, k);
      if (wx) i = wrap_i(i, a.g.nx);
      int cnt;
      if (SFIX > 0) {
        if (wx || wy || wz) cnt = thread_count_fixed<D, (SFIX > 0 ? SFIX : 1), true>(a.g, sub, i, j, k, cx, cy, cz, R2, wx, wy, wz);
        else cnt = thread_count_fixed<D, (SFIX > 0 ? SFIX : 1), false>(a.g, sub, i, j, k, cx, cy, cz, R2, false, false, false);
      } else {
        cnt = thread_count_generic<D>(a.g, a.S, sub, i, j, k, cx, cy, cz, R2, wx, wy, wz);
      }
      if (cnt > 0) commit(i, j, k, cnt);
    }
    group_sync<G>();
  }
  settle();
}
