// Lattice kernels: rest-state init (a0), the fused collide-and-stream step (a2),
// the stream/unstream permutations behind set_distributions / fetch_fields (a5).
//
// Scheme: "pull", two buffers (A-B).  The stored array is the post-collision state
// f*(x, t-1); one thread per node gathers f_i(x,t) = f*_i(x - c_i) (periodic wrap) or,
// when x - c_i lies behind a wall, f*_{-i}(x) (half-way bounce-back, R15),
// collides with eq. (1) of the paper and writes f*(x,t) to the other
// buffer at its own node: every store is aligned and coalesced, the x-shifted loads
// are misaligned by one element and served from L1/L2 sectors.
#include "collide.cuh"
#include "lbmimb_internal.cuh"

namespace lbmimb {

struct StepArgs {
  const double *__restrict__ fin;
  double *__restrict__ fout;
  const uint32_t *__restrict__ tag;
  const double *__restrict__ prec;
  const double *__restrict__ beta_tab;
  double *__restrict__ s;            // per-node exchange records (EMIT == kEmitField only)
  long long *__restrict__ facc;      // per-particle fixed-point force / torque sums (EMIT != kEmitNone)
  int64_t N;
  int nx, ny, nz;
  int bcx, bcy, bcz;
  unsigned tiles;      // blocks per lattice row
  SlabRows sl;         // stored rows <-> global rows, wall flags of the two y ends, owned rows
  CollideParams cp;
  // Rows away from walls and seams: f_q(x) is read koff[q] bytes behind element x - cx_q of the array.
  //   pull (A-B):  koff[q] = 8 (q N - cy_q nx - cz_q nx ny);   AA odd step: the same with slot opposite(q)
  int64_t koff[19];
};

constexpr int kStepThreads = 128;
enum { kLayoutPull = 0, kLayoutNatural = 1, kLayoutSwapped = 2 };
// what a step leaves behind for a3: nothing (not the last step of a call), the per-particle force / torque
// sums, or those plus the per-node exchange vectors (LBMIMB_FLAG_EXCHANGE_FIELD)
enum { kEmitNone = 0, kEmitForces = 1, kEmitField = 2 };

// Tail of both step kernels on warps that hold a covered node: eq. (3) summed in the kernel.
template <int D, int EMIT>
__device__ __forceinline__ void emit_exchange(const StepArgs &a, int64_t x, bool covered, int pe, double beta, double rho,
                                              double ux, double uy, double uz, double vx, double vy, double vz,
                                              double rx, double ry, double rz) {
  const double br = beta * rho;
  const double sx = br * (vx - ux), sy = br * (vy - uy), sz = br * (vz - uz);   // s = beta rho (V_S - u)  (P6)
  if (EMIT == kEmitField && covered) store_exchange<D>(a.s, x, sx, sy, sz);
  const int key = covered ? pe : -1;
  if (D == 2) {
    double v[3] = {sx, sy, rx * sy};
    if (reduce_runs<3>(key, v)) {
      long long *acc = a.facc + (int64_t)key * 6;
      fixed_add(acc + 0, -v[0]);
      fixed_add(acc + 2, -v[1]);
      fixed_add(acc + 4, -(v[2] - ry * v[0]));
    }
  } else {
    double v[5] = {sx, sy, sz, rx * sy, rx * sz};
    if (reduce_runs<5>(key, v)) {
      long long *acc = a.facc + (int64_t)key * 12;
      fixed_add(acc + 0, -v[0]);
      fixed_add(acc + 2, -v[1]);
      fixed_add(acc + 4, -v[2]);
      fixed_add(acc + 6, -(ry * v[2] - rz * v[1]));
      fixed_add(acc + 8, -(rz * v[0] - v[4]));
      fixed_add(acc + 10, -(v[3] - ry * v[0]));
    }
  }
}

// ---------------------------------------------------------------------------
// a2: fused collide-and-stream, one thread per node, one block per row segment.
// IMB = particles present, EMIT = what is left for a3 (kEmit*).
// The y/z part of every source address is block-uniform; per thread only the three
// x indices i-1, i, i+1 (wrapped) differ.  A warp takes the IMB path as a whole when
// any of its nodes is covered (beta = 0 on the others), else the cheaper LBGK path.
// ---------------------------------------------------------------------------
template <int D, bool IMB, int EMIT, int MINB>
__global__ void __launch_bounds__(kStepThreads, MINB) collide_stream_kernel(const StepArgs a) {
  using L = Lat<D>;
  constexpr int Q = L::Q;
  const unsigned row = blockIdx.x / a.tiles;
  const unsigned tile = blockIdx.x - row * a.tiles;
  const int i0 = (int)(tile * kStepThreads + threadIdx.x);
  const bool live = i0 < a.nx;
  const int i = live ? i0 : a.nx - 1;
  const int k = D == 3 ? (int)(row / (unsigned)a.ny) : 0;
  const int j = (int)(row - (unsigned)k * (unsigned)a.ny);
  const int64_t rowoff = ((int64_t)k * a.ny + j) * a.nx;
  const int64_t x = rowoff + i;
  const int im = i == 0 ? a.nx - 1 : i - 1;
  const int ip = i == a.nx - 1 ? 0 : i + 1;

  // The node tag (sample count, covering particle) is requested before the populations so that the
  // dependent gather of the particle record overlaps the population loads (C4 7.00 -> 6.46 ms in round 1).
  uint32_t tg = 0;
  if (IMB) tg = a.tag[x];

  // ---- gather (streaming) ----
  // Rows whose 9 neighbouring rows all lie inside the stored lattice (block-uniform test; all but the first and
  // last row of each axis): the source of direction q is a constant byte offset koff[q] = 8 (q N - cy nx -
  // cz nx ny) behind one of three per-thread pointers (x-1, x, x+1 wrapped).  The general path below costs
  // ~15 integer instructions per direction; with it the kernel executed 1.86 G warp instructions against
  // 1.29-1.36 G of the in-place kernels for the same collision.
  double f[Q];
  const bool inner = j >= 1 && j <= a.ny - 2 && (D == 2 || (k >= 1 && k <= a.nz - 2));
  if (inner) {
    const char *const p0 = (const char *)(a.fin + x), *const pm = (const char *)(a.fin + (rowoff + im)),
                      *const pp = (const char *)(a.fin + (rowoff + ip));
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int cx = L::cx(q);
      f[q] = *(const double *)((cx == 0 ? p0 : (cx == 1 ? pm : pp)) + a.koff[q]);
    }
  } else {
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
    bool bounce = false;
    int js = j - cy, ks = k - cz;
    if (cy != 0 && (js < 0 || js >= a.ny)) {
      if (js < 0 ? a.sl.wall_lo : a.sl.wall_hi) bounce = true;
      else js = js < 0 ? js + a.ny : js - a.ny;   // periodic, or a ghost row pulling garbage nobody reads
    }
    if (D == 3 && cz != 0 && (ks < 0 || ks >= a.nz)) {
      if (a.bcz) bounce = true;
      else ks = ks < 0 ? ks + a.nz : ks - a.nz;
    }
    const double *base = bounce ? a.fin + ((int64_t)opposite(q) * a.N + rowoff)
                                : a.fin + ((int64_t)q * a.N + ((int64_t)ks * a.ny + js) * a.nx);
    const int xs = (bounce || cx == 0) ? i : (cx == 1 ? im : ip);
    f[q] = base[xs];
  }
  }
  if (a.bcx && (i == 0 || i == a.nx - 1)) {
    // x walls: the end nodes of a row bounce their own opposite population back (R15)
#pragma unroll
    for (int q = 1; q < Q; ++q) {
      const int cx = L::cx(q);
      if ((cx == 1 && i == 0) || (cx == -1 && i == a.nx - 1)) f[q] = a.fin[(int64_t)opposite(q) * a.N + x];
    }
  }

  // The tag is looked at only now: a warp issues in order, so decoding it earlier holds back the population
  // loads behind the tag's round trip (21 % of the stall samples with the round-1 ordering).  Here all Q loads
  // are in flight when the dependent gather of the particle record starts.
  int cnt = 0, pe = 0;
  if (IMB) {
    asm volatile("" : "+r"(tg) : : "memory");
    cnt = tag_cnt(tg);
    pe = (int)(tg >> kTagPidShift);
  }
  double beta = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, rx = 0.0, ry = 0.0, rz = 0.0;
  if (IMB && cnt > 0) {
    beta = __ldg(a.beta_tab + cnt);
    solid_velocity<D>(a.prec + (int64_t)pe * prec_stride(D), i, slab_global_row(a.sl, j), k, a.nx, a.sl.gny, a.nz, a.bcx,
                      a.bcy, a.bcz, vx, vy, vz, rx, ry, rz);
  }

  double rho, ux, uy, uz;
  moments<D>(f, rho, ux, uy, uz);

  const bool solid_warp = IMB && __any_sync(0xffffffffu, cnt > 0);
  if (!solid_warp) collide_fluid<D>(f, a.cp, rho, ux, uy, uz);
  else collide_imb<D>(f, a.cp, rho, ux, uy, uz, beta, vx, vy, vz);

  if (live) {
#pragma unroll
    for (int q = 0; q < Q; ++q) a.fout[(int64_t)q * a.N + x] = f[q];
  }
  if (EMIT != kEmitNone && solid_warp)
    emit_exchange<D, EMIT>(a, x, cnt > 0 && live && j >= a.sl.own_lo && j < a.sl.own_hi, pe, beta, rho, ux, uy, uz, vx,
                           vy, vz, rx, ry, rz);
}

// ---------------------------------------------------------------------------
// a2, in-place variant: AA-pattern streaming on ONE distribution array (BASELINE.json north_star:
// "either a pull-scheme double buffer or AA-pattern in-place streaming").  The array alternates
// between two layouts:
//   natural (after an ODD step, or after init / set_distributions): slot q of node x holds f_q(x,t);
//   swapped (after an EVEN step): slot -q of node x holds f*_q(x,t-1), so that
//       f_q(x,t) = slot -q of node x - c_q, or slot q of node x itself when x - c_q lies behind a wall.
// EVEN step: read the own node's slots, collide, write f*_q to slot -q of the own node (no neighbour
// access, every load and store aligned).  ODD step: gather as above, collide, write f*_q to slot q of
// node x + c_q (or slot -q of x through a wall): a node reads and writes exactly the same set of
// locations and no two nodes share one, so the update is race-free in place.
// ---------------------------------------------------------------------------
// In the ODD step the location node x reads f_q from is the one it writes f*_{-q} to, so there is ONE
// address per direction: a block-uniform 64-bit offset (slot and row, looked up in a table of the 9
// neighbouring rows (dy,dz) with their wall flags) plus one of the three wrapped x indices.
// XW = walls in x, where the end nodes of a row bounce per thread.
template <int D, bool IMB, int EMIT, bool ODD, bool XW, int MINB>
__global__ void __launch_bounds__(kStepThreads, MINB) collide_stream_aa_kernel(const StepArgs a) {
  using L = Lat<D>;
  constexpr int Q = L::Q;
  const unsigned row = blockIdx.x / a.tiles;
  const unsigned tile = blockIdx.x - row * a.tiles;
  const int i0 = (int)(tile * kStepThreads + threadIdx.x);
  const bool live = i0 < a.nx;
  const int i = live ? i0 : a.nx - 1;
  const int k = D == 3 ? (int)(row / (unsigned)a.ny) : 0;
  const int j = (int)(row - (unsigned)k * (unsigned)a.ny);
  const int64_t rowoff = ((int64_t)k * a.ny + j) * a.nx;
  const int64_t x = rowoff + i;
  double *__restrict__ F = a.fout;   // the one array (fin == fout)

  uint32_t tg = 0;
  if (IMB) tg = a.tag[x];

  const int im = i == 0 ? a.nx - 1 : i - 1;
  const int ip = i == a.nx - 1 ? 0 : i + 1;
  // Rows with all 9 neighbouring rows inside the lattice (block-uniform): constant offsets per direction.
  const bool inner = j >= 1 && j <= a.ny - 2 && (D == 2 || (k >= 1 && k <= a.nz - 2));
  char *const p0 = (char *)(F + x), *const pm = (char *)(F + (rowoff + im)), *const pp = (char *)(F + (rowoff + ip));
  auto fast_ptr = [&](int q) -> double * {   // koff is in bytes: one 64-bit add per address
    const int cx = L::cx(q);
    if (XW && cx != 0 && ((cx == 1 && i == 0) || (cx == -1 && i == a.nx - 1))) return (double *)p0 + (int64_t)q * a.N;
    return (double *)((cx == 0 ? p0 : (cx == 1 ? pm : pp)) + a.koff[q]);
  };
  // General rows: element offset of row (j+dy, k+dz), or -1 when that row lies behind a wall.
  auto slow_ptr = [&](int q) -> double * {
    const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
    int jj = j - cy, kk = k - cz;
    bool bounce = false;
    if (cy != 0 && (jj < 0 || jj >= a.ny)) {
      if (jj < 0 ? a.sl.wall_lo : a.sl.wall_hi) bounce = true;
      else jj = jj < 0 ? jj + a.ny : jj - a.ny;
    }
    if (D == 3 && cz != 0 && (kk < 0 || kk >= a.nz)) {
      if (a.bcz) bounce = true;
      else kk = kk < 0 ? kk + a.nz : kk - a.nz;
    }
    if (XW && cx != 0 && ((cx == 1 && i == 0) || (cx == -1 && i == a.nx - 1))) bounce = true;
    const int64_t uo = bounce ? (int64_t)q * a.N + rowoff : (int64_t)opposite(q) * a.N + ((int64_t)kk * a.ny + jj) * a.nx;
    const int xs = (bounce || cx == 0) ? i : (cx == 1 ? im : ip);
    return F + (uo + xs);
  };

  double f[Q];
  if (!ODD) {
#pragma unroll
    for (int q = 0; q < Q; ++q) f[q] = F[(int64_t)q * a.N + x];
  } else if (inner) {
#pragma unroll
    for (int q = 0; q < Q; ++q) f[q] = *fast_ptr(q);
  } else {
#pragma unroll
    for (int q = 0; q < Q; ++q) f[q] = *slow_ptr(q);
  }

  // The tag is looked at only now: a warp issues in order, so decoding it earlier holds back the population
  // loads behind the tag's round trip (21 % of the stall samples with the round-1 ordering).  Here all Q loads
  // are in flight when the dependent gather of the particle record starts.
  int cnt = 0, pe = 0;
  if (IMB) {
    asm volatile("" : "+r"(tg) : : "memory");
    cnt = tag_cnt(tg);
    pe = (int)(tg >> kTagPidShift);
  }
  double beta = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, rx = 0.0, ry = 0.0, rz = 0.0;
  if (IMB && cnt > 0) {
    beta = __ldg(a.beta_tab + cnt);
    solid_velocity<D>(a.prec + (int64_t)pe * prec_stride(D), i, slab_global_row(a.sl, j), k, a.nx, a.sl.gny, a.nz, a.bcx,
                      a.bcy, a.bcz, vx, vy, vz, rx, ry, rz);
  }

  double rho, ux, uy, uz;
  moments<D>(f, rho, ux, uy, uz);

  const bool solid_warp = IMB && __any_sync(0xffffffffu, cnt > 0);
  if (!solid_warp) collide_fluid<D>(f, a.cp, rho, ux, uy, uz);
  else collide_imb<D>(f, a.cp, rho, ux, uy, uz, beta, vx, vy, vz);

  if (live) {
    if (!ODD) {
#pragma unroll
      for (int q = 0; q < Q; ++q) F[(int64_t)opposite(q) * a.N + x] = f[q];
    } else if (inner) {
#pragma unroll
      for (int q = 0; q < Q; ++q) *fast_ptr(opposite(q)) = f[q];
    } else {
#pragma unroll
      for (int q = 0; q < Q; ++q) *slow_ptr(opposite(q)) = f[q];
    }
  }
  if (EMIT != kEmitNone && solid_warp)
    emit_exchange<D, EMIT>(a, x, cnt > 0 && live && j >= a.sl.own_lo && j < a.sl.own_hi, pe, beta, rho, ux, uy, uz, vx,
                           vy, vz, rx, ry, rz);
}

// ---------------------------------------------------------------------------
// a0: f = w_i (rest state, rho = 1, u = 0)
// ---------------------------------------------------------------------------
template <int D>
__global__ void init_rest_kernel(double *__restrict__ f, int64_t N) {
  using L = Lat<D>;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < N; x += stride) {
#pragma unroll
    for (int q = 0; q < L::Q; ++q) f[(int64_t)q * N + x] = L::w(q);
  }
}

// ---------------------------------------------------------------------------
// Gather of the pre-collision state f_i(x,t) of one node from the stored array, whose layout is
// pull (post-collision, A-B scheme), AA natural or AA swapped.
// ---------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void gather_node(const double *__restrict__ fst, const Geom &g, const SlabRows &sl, int layout,
                                            int i, int j, int k, double *f) {
  using L = Lat<D>;
  const int64_t x = ((int64_t)k * g.ny + j) * g.nx + i;
  if (layout == kLayoutNatural) {
#pragma unroll
    for (int q = 0; q < L::Q; ++q) f[q] = fst[(int64_t)q * g.N + x];
    return;
  }
  const bool swapped = layout == kLayoutSwapped;
#pragma unroll
  for (int q = 0; q < L::Q; ++q) {
    const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
    bool bounce = false;
    int is = i - cx, js = j - cy, ks = k - cz;
    if (is < 0 || is >= g.nx) {
      if (g.bcx) bounce = true;
      else is = is < 0 ? is + g.nx : is - g.nx;
    }
    if (js < 0 || js >= g.ny) {
      if (js < 0 ? sl.wall_lo : sl.wall_hi) bounce = true;
      else js = js < 0 ? js + g.ny : js - g.ny;
    }
    if (D == 3 && (ks < 0 || ks >= g.nz)) {
      if (g.bcz) bounce = true;
      else ks = ks < 0 ? ks + g.nz : ks - g.nz;
    }
    // pull (A-B): slot q of the source node, slot -q of the own node through a wall;
    // AA swapped: the two slots exchanged (see collide_stream_aa_kernel)
    const int slot = (bounce != swapped) ? opposite(q) : q;
    const int64_t src = bounce ? (int64_t)slot * g.N + x : (int64_t)slot * g.N + ((int64_t)ks * g.ny + js) * g.nx + is;
    f[q] = fst[src];
  }
}

// set_distributions: inverse permutation.  f*_q(x) = f_q(x + c_q), or f_{-q}(x) when x + c_q is behind a wall.
template <int D>
__global__ void unstream_kernel(const double *__restrict__ fpre, double *__restrict__ fpost, const Geom g,
                                const SlabRows sl) {
  using L = Lat<D>;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < g.N; x += stride) {
    const int i = (int)(x % g.nx);
    const int64_t r = x / g.nx;
    const int j = (int)(r % g.ny);
    const int k = (int)(r / g.ny);
#pragma unroll
    for (int q = 0; q < L::Q; ++q) {
      const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
      bool bounce = false;
      int it = i + cx, jt = j + cy, kt = k + cz;
      if (it < 0 || it >= g.nx) {
        if (g.bcx) bounce = true;
        else it = it < 0 ? it + g.nx : it - g.nx;
      }
      if (jt < 0 || jt >= g.ny) {
        if (jt < 0 ? sl.wall_lo : sl.wall_hi) bounce = true;
        else jt = jt < 0 ? jt + g.ny : jt - g.ny;
      }
      if (D == 3 && (kt < 0 || kt >= g.nz)) {
        if (g.bcz) bounce = true;
        else kt = kt < 0 ? kt + g.nz : kt - g.nz;
      }
      const int64_t src = bounce ? (int64_t)opposite(q) * g.N + x
                                 : (int64_t)q * g.N + ((int64_t)kt * g.ny + jt) * g.nx + it;
      fpost[(int64_t)q * g.N + x] = fpre[src];
    }
  }
}

struct FetchArgs {
  const double *fpost;
  const uint32_t *tag;
  const double *s;
  void *dst;
  int lo[3], ext[3];
  int64_t box;
  int what;
  int have_particles;
  int layout;
};

template <int D>
__global__ void fetch_kernel(const FetchArgs a, const Geom g, const SlabRows sl) {
  using L = Lat<D>;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; b < a.box; b += stride) {
    const int bi = (int)(b % a.ext[0]);
    const int64_t r = b / a.ext[0];
    const int bj = (int)(r % a.ext[1]);
    const int bk = (int)(r / a.ext[1]);
    const int i = a.lo[0] + bi, j = a.lo[1] + bj, k = a.lo[2] + bk;
    const int64_t x = ((int64_t)k * g.ny + j) * g.nx + i;
    if (a.what == LBMIMB_FIELD_EPS_CNT) {
      ((uint8_t *)a.dst)[b] = (uint8_t)tag_cnt(a.tag[x]);
    } else if (a.what == LBMIMB_FIELD_PID) {
      ((int32_t *)a.dst)[b] = tag_pid(a.tag[x]);
    } else if (a.what == LBMIMB_FIELD_S) {
      const bool cov = a.have_particles && tag_cnt(a.tag[x]) > 0;
      for (int c = 0; c < D; ++c) ((double *)a.dst)[(int64_t)c * a.box + b] = cov ? a.s[x * exchange_stride(D) + c] : 0.0;
    } else {
      double f[L::Q];
      gather_node<D>(a.fpost, g, sl, a.layout, i, j, k, f);
      if (a.what == LBMIMB_FIELD_F) {
#pragma unroll
        for (int q = 0; q < L::Q; ++q) ((double *)a.dst)[(int64_t)q * a.box + b] = f[q];
      } else {
        double rho = 0.0, m[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int q = 0; q < L::Q; ++q) {
          rho += f[q];
          m[0] += L::cx(q) * f[q];
          m[1] += L::cy(q) * f[q];
          m[2] += L::cz(q) * f[q];
        }
        if (a.what == LBMIMB_FIELD_RHO) {
          ((double *)a.dst)[b] = rho;
        } else {
          for (int c = 0; c < D; ++c) ((double *)a.dst)[(int64_t)c * a.box + b] = m[c] / rho;
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------
// Suspension diagnostics (Figs. 5/7; R18): deterministic two-stage reduction.
// Stage 1: every thread sums its grid-stride nodes in a fixed order, the block reduces by a fixed tree
// and writes 8 partial sums: gas area, mass, (1-eps) u [3], rho u [3].
// Stage 2 (one block): partials in block order, then the particle sums, then the derived quantities.
// ---------------------------------------------------------------------------
constexpr int kDiagThreads = 256;
constexpr int kDiagK = 8;

__device__ __forceinline__ double diag_block_sum(double v, double *sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) sh[w] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x == 0) {
    for (int k = 0; k < kDiagThreads / 32; ++k) r += sh[k];
  }
  return r;   // valid on thread 0
}

template <int D>
__global__ void __launch_bounds__(kDiagThreads) diag_nodes_kernel(const double *__restrict__ fst, const uint32_t *__restrict__ tag,
                                                                  const Geom g, const SlabRows sl, int layout,
                                                                  int have_particles, double eps_den,
                                                                  double *__restrict__ partial) {
  using L = Lat<D>;
  __shared__ double sh[kDiagThreads / 32];
  double acc[kDiagK];
#pragma unroll
  for (int c = 0; c < kDiagK; ++c) acc[c] = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < g.N; x += stride) {
    const int i = (int)(x % g.nx);
    const int64_t r = x / g.nx;
    const int j = (int)(r % g.ny);
    const int k = (int)(r / g.ny);
    if (j < sl.own_lo || j >= sl.own_hi) continue;   // ghost rows of a slab belong to the neighbour
    double f[L::Q];
    gather_node<D>(fst, g, sl, layout, i, j, k, f);
    double rho = 0.0, m[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int q = 0; q < L::Q; ++q) {
      rho += f[q];
      m[0] += L::cx(q) * f[q];
      m[1] += L::cy(q) * f[q];
      m[2] += L::cz(q) * f[q];
    }
    const double gas = have_particles ? 1.0 - (double)tag_cnt(tag[x]) / eps_den : 1.0;
    acc[0] += gas;
    acc[1] += rho;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      acc[2 + c] += gas * (m[c] / rho);
      acc[5 + c] += m[c];
    }
  }
#pragma unroll
  for (int c = 0; c < kDiagK; ++c) {
    const double t = diag_block_sum(acc[c], sh);
    if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * kDiagK + c] = t;
  }
}

// out[20]: [0] A_g [1] mass [2:5] U_g [5:8] V_s [8:11] V_r [11:14] F_d [14:17] fluid momentum [17:20] solid momentum
template <int D>
__global__ void __launch_bounds__(kDiagThreads) diag_final_kernel(const double *__restrict__ partial, int nblocks, int64_t P,
                                                                  const double *__restrict__ vel,
                                                                  const double *__restrict__ radius,
                                                                  const double *__restrict__ mass,
                                                                  const double *__restrict__ force,
                                                                  double *__restrict__ out) {
  __shared__ double sh[kDiagThreads / 32];
  __shared__ double tot[kDiagK + 10];
  for (int c = 0; c < kDiagK; ++c) {
    double v = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += kDiagThreads) v += partial[(int64_t)b * kDiagK + c];
    const double t = diag_block_sum(v, sh);
    if (threadIdx.x == 0) tot[c] = t;
  }
  // particles: [8] sum vol, [9..11] sum vol v, [12..14] sum m v, [15..17] sum F
  double pa[10];
#pragma unroll
  for (int c = 0; c < 10; ++c) pa[c] = 0.0;
  const double kPi = 3.14159265358979323846;
  for (int64_t p = threadIdx.x; p < P; p += kDiagThreads) {
    const double R = radius[p];
    const double vol = D == 2 ? kPi * (R * R) : (4.0 / 3.0 * kPi) * (R * R * R);
    pa[0] += vol;
#pragma unroll
    for (int c = 0; c < D; ++c) {
      const double v = vel[(int64_t)c * P + p];
      pa[1 + c] += vol * v;
      pa[4 + c] += mass[p] * v;
      pa[7 + c] += force[(int64_t)c * P + p];
    }
  }
#pragma unroll
  for (int c = 0; c < 10; ++c) {
    const double t = diag_block_sum(pa[c], sh);
    if (threadIdx.x == 0) tot[kDiagK + c] = t;
  }
  if (threadIdx.x == 0) {
    for (int c = 0; c < 20; ++c) out[c] = 0.0;
    out[0] = tot[0];
    out[1] = tot[1];
    for (int c = 0; c < D; ++c) {
      out[2 + c] = tot[2 + c] / tot[0];
      out[14 + c] = tot[5 + c];
      if (P > 0) {
        out[5 + c] = tot[9 + c] / tot[8];
        out[11 + c] = tot[15 + c] / (double)P;
        out[17 + c] = tot[12 + c];
      }
      out[8 + c] = out[2 + c] - out[5 + c];
    }
  }
}

static int grid_for(int64_t n, int threads, int cap = 148 * 16) {
  int64_t b = (n + threads - 1) / threads;
  if (b < 1) b = 1;
  return (int)(b < cap ? b : cap);
}

lbmimb_status launch_init_rest(lbmimb_lattice *h) {
  if (h->g.dim == 2)
    init_rest_kernel<2><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(h->f[0], h->g.N);
  else
    init_rest_kernel<3><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(h->f[0], h->g.N);
  LBMIMB_LAUNCH_CHECK(h, "init_rest_kernel");
  return LBMIMB_OK;
}

// One instantiation per (D, IMB, EMIT).  Occupancy targets from the round-1 sweep:
// 3D 80 registers / 6 blocks per SM, 2D 56 registers / 9 blocks per SM.
template <int D>
static void launch_cs(lbmimb_lattice *h, const StepArgs &a, unsigned blocks, bool imb, int emit) {
  constexpr int MINB = D == 3 ? 6 : 9;
  if (!imb)
    collide_stream_kernel<D, false, kEmitNone, MINB><<<blocks, kStepThreads, 0, h->stream>>>(a);
  else if (emit == kEmitNone)
    collide_stream_kernel<D, true, kEmitNone, MINB><<<blocks, kStepThreads, 0, h->stream>>>(a);
  else if (emit == kEmitForces)
    collide_stream_kernel<D, true, kEmitForces, MINB><<<blocks, kStepThreads, 0, h->stream>>>(a);
  else
    collide_stream_kernel<D, true, kEmitField, MINB><<<blocks, kStepThreads, 0, h->stream>>>(a);
}

template <int D, int MINB>
static void launch_aa(lbmimb_lattice *h, const StepArgs &a, unsigned blocks, bool imb, int emit, bool odd) {
#define LBMIMB_AA(I, E, O, X) collide_stream_aa_kernel<D, I, E, O, X, MINB><<<blocks, kStepThreads, 0, h->stream>>>(a)
#define LBMIMB_AA_ODD(I, E)                       \
  do {                                            \
    if (a.bcx) LBMIMB_AA(I, E, true, true);       \
    else LBMIMB_AA(I, E, true, false);            \
  } while (0)
  if (!odd) {   // the even step touches the own node only: walls do not matter
    if (!imb) LBMIMB_AA(false, kEmitNone, false, false);
    else if (emit == kEmitNone) LBMIMB_AA(true, kEmitNone, false, false);
    else if (emit == kEmitForces) LBMIMB_AA(true, kEmitForces, false, false);
    else LBMIMB_AA(true, kEmitField, false, false);
  } else {
    if (!imb) LBMIMB_AA_ODD(false, kEmitNone);
    else if (emit == kEmitNone) LBMIMB_AA_ODD(true, kEmitNone);
    else if (emit == kEmitForces) LBMIMB_AA_ODD(true, kEmitForces);
    else LBMIMB_AA_ODD(true, kEmitField);
  }
#undef LBMIMB_AA_ODD
#undef LBMIMB_AA
}

lbmimb_status launch_collide_stream(lbmimb_lattice *h, bool emit_last) {
  const int emit = !emit_last ? kEmitNone : (h->keep_s ? kEmitField : kEmitForces);
  StepArgs a;
  a.fin = h->f[h->cur];
  a.fout = h->f[h->cur ^ 1];
  a.tag = h->tag;
  a.prec = h->prec;
  a.beta_tab = h->beta_tab;
  a.s = h->s;
  a.facc = h->facc;
  a.N = h->g.N;
  a.nx = h->g.nx;
  a.ny = h->g.ny;
  a.nz = h->g.nz;
  a.bcx = h->g.bcx;
  a.bcy = h->g.bcy;
  a.bcz = h->g.bcz;
  a.sl = h->sl;
  a.tiles = (unsigned)((h->g.nx + kStepThreads - 1) / kStepThreads);
  a.cp = make_collide_params(h);
  const int64_t blocks = (int64_t)a.tiles * h->g.ny * h->g.nz;
  if (blocks > 0x7fffffff) return fail(LBMIMB_EINVAL, "lattice needs more than 2^31 thread blocks");
  const bool imb = h->P > 0;
  if (h->aa) {
    a.fin = a.fout = h->f[0];
    for (int q = 0; q < h->Q; ++q) {
      const int cy = h->g.dim == 2 ? Lat<2>::cy(q) : Lat<3>::cy(q);
      const int cz = h->g.dim == 2 ? 0 : Lat<3>::cz(q);
      a.koff[q] = 8 * ((int64_t)opposite(q) * a.N - (int64_t)cy * a.nx - (int64_t)cz * a.nx * a.ny);
    }
    if (h->g.dim == 2) launch_aa<2, 9>(h, a, (unsigned)blocks, imb, emit, h->aa_swapped);
    else launch_aa<3, 5>(h, a, (unsigned)blocks, imb, emit, h->aa_swapped);
    LBMIMB_LAUNCH_CHECK(h, "collide_stream_aa_kernel");
    return LBMIMB_OK;
  }
  for (int q = 0; q < h->Q; ++q) {
    const int cy = h->g.dim == 2 ? Lat<2>::cy(q) : Lat<3>::cy(q);
    const int cz = h->g.dim == 2 ? 0 : Lat<3>::cz(q);
    a.koff[q] = 8 * ((int64_t)q * a.N - (int64_t)cy * a.nx - (int64_t)cz * a.nx * a.ny);
  }
  if (h->g.dim == 2)
    launch_cs<2>(h, a, (unsigned)blocks, imb, emit);
  else
    launch_cs<3>(h, a, (unsigned)blocks, imb, emit);
  LBMIMB_LAUNCH_CHECK(h, "collide_stream_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_unstream(lbmimb_lattice *h, const double *f_pre, double *f_post) {
  if (h->g.dim == 2)
    unstream_kernel<2><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(f_pre, f_post, h->g, h->sl);
  else
    unstream_kernel<3><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(f_pre, f_post, h->g, h->sl);
  LBMIMB_LAUNCH_CHECK(h, "unstream_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_fetch(lbmimb_lattice *h, int what, const int64_t lo[3], const int64_t hi[3], void *dst_dev) {
  FetchArgs a;
  a.fpost = h->f[h->cur];
  a.tag = h->tag;
  a.s = h->s;
  a.dst = dst_dev;
  a.box = 1;
  for (int c = 0; c < 3; ++c) {
    a.lo[c] = (int)lo[c] + (c == 1 ? h->sl.own_lo : 0);   // box rows count from the first OWNED row
    a.ext[c] = (int)(hi[c] - lo[c]);
    a.box *= a.ext[c];
  }
  a.what = what;
  a.have_particles = h->P > 0;
  a.layout = h->aa ? (h->aa_swapped ? kLayoutSwapped : kLayoutNatural) : kLayoutPull;
  if (h->g.dim == 2)
    fetch_kernel<2><<<grid_for(a.box, 256), 256, 0, h->stream>>>(a, h->g, h->sl);
  else
    fetch_kernel<3><<<grid_for(a.box, 256), 256, 0, h->stream>>>(a, h->g, h->sl);
  LBMIMB_LAUNCH_CHECK(h, "fetch_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_diagnostics(lbmimb_lattice *h, double eps_den) {
  const int layout = h->aa ? (h->aa_swapped ? kLayoutSwapped : kLayoutNatural) : kLayoutPull;
  const int nb = grid_for(h->g.N, kDiagThreads, kDiagBlocksMax);
  const double *fst = h->f[h->cur];
  const int hp = h->P > 0;
  if (h->g.dim == 2) {
    diag_nodes_kernel<2><<<nb, kDiagThreads, 0, h->stream>>>(fst, h->tag, h->g, h->sl, layout, hp, eps_den, h->diag_partial);
    LBMIMB_LAUNCH_CHECK(h, "diag_nodes_kernel");
    diag_final_kernel<2><<<1, kDiagThreads, 0, h->stream>>>(h->diag_partial, nb, h->P, h->vel, h->radius, h->mass,
                                                           h->force, h->diag_out);
  } else {
    diag_nodes_kernel<3><<<nb, kDiagThreads, 0, h->stream>>>(fst, h->tag, h->g, h->sl, layout, hp, eps_den, h->diag_partial);
    LBMIMB_LAUNCH_CHECK(h, "diag_nodes_kernel");
    diag_final_kernel<3><<<1, kDiagThreads, 0, h->stream>>>(h->diag_partial, nb, h->P, h->vel, h->radius, h->mass,
                                                           h->force, h->diag_out);
  }
  LBMIMB_LAUNCH_CHECK(h, "diag_final_kernel");
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// Slab halo ("domain decomposition"; Fig. 2): after a step the stored array holds the
// post-collision state f*(x, t).  The next step of the neighbouring slab pulls, into its first / last owned
// row, the populations that move across the cut: the c_y = +1 ones of our LAST owned row, the c_y = -1 ones
// of our FIRST owned row (5 of 19 / 3 of 9).  pack copies them into a contiguous buffer [n_face][nz][nx];
// unpack writes a neighbour's buffer into our ghost row.  side 0 = lower (y-) end, 1 = upper (y+) end:
//   pack(side)   packs the populations LEAVING through that side (c_y = -1 for side 0, +1 for side 1);
//   unpack(side) stores populations ENTERING through that side (c_y = +1 for side 0, -1 for side 1) in the
//                ghost row of that side.
// Transport (peer copy, NCCL send/recv, MPI) is the caller's.
// ---------------------------------------------------------------------------
template <int D>
__global__ void halo_kernel(double *__restrict__ f, double *__restrict__ buf, const Geom g, int row, int want_cy,
                            int pack) {
  using L = Lat<D>;
  const int64_t plane = (int64_t)g.nx * g.nz;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < plane; e += stride) {
    const int i = (int)(e % g.nx), k = (int)(e / g.nx);
    const int64_t x = ((int64_t)k * g.ny + row) * g.nx + i;
    int slot = 0;
#pragma unroll
    for (int q = 0; q < L::Q; ++q) {
      if (L::cy(q) != want_cy) continue;
      if (pack) buf[(int64_t)slot * plane + e] = f[(int64_t)q * g.N + x];
      else f[(int64_t)q * g.N + x] = buf[(int64_t)slot * plane + e];
      ++slot;
    }
  }
}

int64_t halo_doubles(const lbmimb_lattice *h) { return (int64_t)(h->g.dim == 2 ? 3 : 5) * h->g.nx * h->g.nz; }

lbmimb_status launch_halo(lbmimb_lattice *h, int side, double *buf_dev, bool pack) {
  // pack: first / last owned row; unpack: the ghost row beyond it
  const int row = pack ? (side == 0 ? h->sl.own_lo : h->sl.own_hi - 1) : (side == 0 ? h->sl.own_lo - 1 : h->sl.own_hi);
  const int want_cy = pack ? (side == 0 ? -1 : 1) : (side == 0 ? 1 : -1);
  double *f = h->f[h->cur];
  const int nb = grid_for((int64_t)h->g.nx * h->g.nz, 256);
  if (h->g.dim == 2) halo_kernel<2><<<nb, 256, 0, h->stream>>>(f, buf_dev, h->g, row, want_cy, pack ? 1 : 0);
  else halo_kernel<3><<<nb, 256, 0, h->stream>>>(f, buf_dev, h->g, row, want_cy, pack ? 1 : 0);
  LBMIMB_LAUNCH_CHECK(h, "halo_kernel");
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// lbmimb_diagnostics_static_dev: the diagnostics of lbmimb_diagnostics for callers that must not allocate and
// must not synchronise (code under CUDA graph capture, tight loops).  Same node stage (diag_nodes_kernel, same
// grid => the same partial sums bit for bit); the particle sums, which lbmimb_diagnostics forms serially in
// its one final block, are formed by ceil(P / 256) blocks, so this variant needs scratch that grows with P.  That
// scratch is NOT in the handle's workspace but in the file-scope array below, of a fixed size:
//   kStaticNodeRows (1184) x 8 + kStaticParticleRows (4096) x 10 doubles = 403,456 bytes,
// which every GPU that loads the library holds until the process exits.  P beyond 4096 x 256 = 1,048,576 is
// rejected.  In host code the array's NAME is a host-side stand-in, not a device address: the address is taken
// once per device with cudaGetSymbolAddress, that device being current, and handed to the kernels.
// Every call (of every handle on the device) shares the array.  Nothing in it has to start at zero: each call
// overwrites exactly the rows it reads back (rows [0, nb) and [0, nbp)).  Calls that overlap on the GPU (two
// streams) race on it.
// ---------------------------------------------------------------------------
constexpr int kStaticNodeRows = kDiagBlocksMax;
constexpr int kStaticParticleRows = 4096;
constexpr int kStaticParticleK = 10;
constexpr int64_t kStaticMaxParticles = (int64_t)kStaticParticleRows * kDiagThreads;
constexpr int kStaticDoubles = kStaticNodeRows * kDiagK + kStaticParticleRows * kStaticParticleK;
static __device__ __align__(256) double g_diag_static_scratch[kStaticDoubles];

constexpr int kStaticMaxDevices = 64;
static double *g_diag_static_ptr[kStaticMaxDevices];   // device address of the array, per device ordinal (0 = not taken yet)

// per block: [0] sum vol, [1..3] sum vol v, [4..6] sum m v, [7..9] sum F  (the sums of diag_final_kernel)
template <int D>
__global__ void __launch_bounds__(kDiagThreads) diag_particles_static_kernel(int64_t P, const double *__restrict__ vel,
                                                                             const double *__restrict__ radius,
                                                                             const double *__restrict__ mass,
                                                                             const double *__restrict__ force,
                                                                             double *__restrict__ ppartial) {
  __shared__ double sh[kDiagThreads / 32];
  double pa[kStaticParticleK];
#pragma unroll
  for (int c = 0; c < kStaticParticleK; ++c) pa[c] = 0.0;
  const double kPi = 3.14159265358979323846;
  const int64_t p = (int64_t)blockIdx.x * kDiagThreads + threadIdx.x;
  if (p < P) {
    const double R = radius[p];
    const double vol = D == 2 ? kPi * (R * R) : (4.0 / 3.0 * kPi) * (R * R * R);
    pa[0] = vol;
#pragma unroll
    for (int c = 0; c < D; ++c) {
      const double v = vel[(int64_t)c * P + p];
      pa[1 + c] = vol * v;
      pa[4 + c] = mass[p] * v;
      pa[7 + c] = force[(int64_t)c * P + p];
    }
  }
#pragma unroll
  for (int c = 0; c < kStaticParticleK; ++c) {
    const double t = diag_block_sum(pa[c], sh);
    if (threadIdx.x == 0) ppartial[(int64_t)blockIdx.x * kStaticParticleK + c] = t;
  }
}

// out[20] as diag_final_kernel writes it; node partials summed exactly as there, particle partials in block order
template <int D>
__global__ void __launch_bounds__(kDiagThreads) diag_final_static_kernel(const double *__restrict__ partial, int nblocks,
                                                                         const double *__restrict__ ppartial, int npblocks,
                                                                         int64_t P, double *__restrict__ out) {
  __shared__ double sh[kDiagThreads / 32];
  __shared__ double tot[kDiagK + kStaticParticleK];
  for (int c = 0; c < kDiagK; ++c) {
    double v = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += kDiagThreads) v += partial[(int64_t)b * kDiagK + c];
    const double t = diag_block_sum(v, sh);
    if (threadIdx.x == 0) tot[c] = t;
  }
  for (int c = 0; c < kStaticParticleK; ++c) {
    double v = 0.0;
    for (int b = threadIdx.x; b < npblocks; b += kDiagThreads) v += ppartial[(int64_t)b * kStaticParticleK + c];
    const double t = diag_block_sum(v, sh);
    if (threadIdx.x == 0) tot[kDiagK + c] = t;
  }
  if (threadIdx.x == 0) {
    for (int c = 0; c < 20; ++c) out[c] = 0.0;
    out[0] = tot[0];
    out[1] = tot[1];
    for (int c = 0; c < D; ++c) {
      out[2 + c] = tot[2 + c] / tot[0];
      out[14 + c] = tot[5 + c];
      if (P > 0) {
        out[5 + c] = tot[9 + c] / tot[8];
        out[11 + c] = tot[15 + c] / (double)P;
        out[17 + c] = tot[12 + c];
      }
      out[8 + c] = out[2 + c] - out[5 + c];
    }
  }
}

int64_t diagnostics_static_max_particles() { return kStaticMaxParticles; }
int64_t diagnostics_static_scratch_bytes() { return (int64_t)kStaticDoubles * 8; }

// No cudaMalloc / cudaFree / allocating routine, no synchronisation: four launches on the handle's stream.
// The caller (api.cu) has made the handle's device current.
lbmimb_status launch_diagnostics_static(lbmimb_lattice *h, double eps_den, double *out_dev) {
  if (h->P > kStaticMaxParticles)
    return fail(LBMIMB_EINVAL, "lbmimb_diagnostics_static_dev: %lld particles exceed the static scratch (at most %lld); "
                               "use lbmimb_diagnostics", (long long)h->P, (long long)kStaticMaxParticles);
  const int dev = h->prm.device;
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(LBMIMB_EINVAL, "device ordinal %d beyond %d", dev, kStaticMaxDevices);
  if (!g_diag_static_ptr[dev]) {   // set-up, once per device, that device being current
    double *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_diag_static_scratch);
    if (e != cudaSuccess || !ptr) return cuda_fail(e, "cudaGetSymbolAddress(g_diag_static_scratch)");
    g_diag_static_ptr[dev] = ptr;
  }
  double *partial = g_diag_static_ptr[dev];
  double *ppartial = partial + (size_t)kStaticNodeRows * kDiagK;
  const int layout = h->aa ? (h->aa_swapped ? kLayoutSwapped : kLayoutNatural) : kLayoutPull;
  const int nb = grid_for(h->g.N, kDiagThreads, kStaticNodeRows);
  const int nbp = (int)((h->P + kDiagThreads - 1) / kDiagThreads);
  const double *fst = h->f[h->cur];
  const int hp = h->P > 0;
  if (h->g.dim == 2) {
    diag_nodes_kernel<2><<<nb, kDiagThreads, 0, h->stream>>>(fst, h->tag, h->g, h->sl, layout, hp, eps_den, partial);
    LBMIMB_LAUNCH_CHECK(h, "diag_nodes_kernel");
    if (nbp > 0) {
      diag_particles_static_kernel<2><<<nbp, kDiagThreads, 0, h->stream>>>(h->P, h->vel, h->radius, h->mass, h->force, ppartial);
      LBMIMB_LAUNCH_CHECK(h, "diag_particles_static_kernel");
    }
    diag_final_static_kernel<2><<<1, kDiagThreads, 0, h->stream>>>(partial, nb, ppartial, nbp, h->P, out_dev);
  } else {
    diag_nodes_kernel<3><<<nb, kDiagThreads, 0, h->stream>>>(fst, h->tag, h->g, h->sl, layout, hp, eps_den, partial);
    LBMIMB_LAUNCH_CHECK(h, "diag_nodes_kernel");
    if (nbp > 0) {
      diag_particles_static_kernel<3><<<nbp, kDiagThreads, 0, h->stream>>>(h->P, h->vel, h->radius, h->mass, h->force, ppartial);
      LBMIMB_LAUNCH_CHECK(h, "diag_particles_static_kernel");
    }
    diag_final_static_kernel<3><<<1, kDiagThreads, 0, h->stream>>>(partial, nb, ppartial, nbp, h->P, out_dev);
  }
  LBMIMB_LAUNCH_CHECK(h, "diag_final_static_kernel");
  return LBMIMB_OK;
}

}  // namespace lbmimb
