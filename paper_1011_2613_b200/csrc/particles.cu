// Particle-side kernels: packed records, cell list (counting sort), the particle ->
// lattice mapping (a1), the force/torque reduction (a3) and the soft-sphere DEM (a4).
#include <cmath>
#include <cstring>

#include "collide.cuh"
#include "lbmimb_internal.cuh"

namespace lbmimb {

// ---------------------------------------------------------------------------
// helpers
// ---------------------------------------------------------------------------
__device__ __forceinline__ double min_image_d(double d, int n) {
  const double hn = 0.5 * (double)n;
  if (d > hn) return d - (double)n;
  if (d < -hn) return d + (double)n;
  return d;
}

__device__ __forceinline__ int wrap_i(int i, int n) {
  i %= n;
  return i < 0 ? i + n : i;
}

// neighbour-cell offsets along one axis: periodic axes must not visit a cell twice
__device__ __forceinline__ int off_lo(int nc, int periodic) { return periodic ? (nc >= 3 ? -1 : 0) : -1; }
__device__ __forceinline__ int off_hi(int nc, int periodic) { return periodic ? (nc >= 2 ? 1 : 0) : 1; }

static int blocks_for(int64_t n, int threads) { return (int)((n + threads - 1) / threads > 0 ? (n + threads - 1) / threads : 1); }

// ---------------------------------------------------------------------------
// packed records for the fused step kernel
// ---------------------------------------------------------------------------
__global__ void pack_records_kernel(int dim, int64_t P, const double *__restrict__ pos, const double *__restrict__ vel,
                                    const double *__restrict__ omega, const double *__restrict__ radius,
                                    double *__restrict__ prec) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  if (dim == 2) {
    double *r = prec + p * 6;
    r[0] = pos[p];
    r[1] = pos[P + p];
    r[2] = vel[p];
    r[3] = vel[P + p];
    r[4] = omega[p];
    r[5] = radius[p];
  } else {
    double *r = prec + p * 10;
    r[0] = pos[p];
    r[1] = pos[P + p];
    r[2] = pos[2 * P + p];
    r[3] = vel[p];
    r[4] = vel[P + p];
    r[5] = vel[2 * P + p];
    r[6] = omega[p];
    r[7] = omega[P + p];
    r[8] = omega[2 * P + p];
    r[9] = radius[p];
  }
}

// ---------------------------------------------------------------------------
// set_particles_dev: the checks the host variant does on its host arrays, done on the device BEFORE anything
// is committed to the handle: radius and mass positive and finite, centres inside [-1/2, n) per axis;
// also the largest / smallest radius (the cell-list geometry needs them on the host).
// res: [0] number of bad particles, [1] lowest bad index + 1 (as a negative max), [2..3] rmax bits, [4..5] rmin bits
// ---------------------------------------------------------------------------
__global__ void validate_particles_kernel(int dim, int64_t P, int nx, int ny, int nz, const double *__restrict__ pos,
                                          const double *__restrict__ radius, const double *__restrict__ mass,
                                          int32_t *__restrict__ res) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const double R = radius[p], m = mass[p];
  bool ok = R > 0.0 && m > 0.0 && isfinite(R) && isfinite(m);
  const int n[3] = {nx, ny, nz};
  for (int a = 0; a < dim; ++a) {
    const double x = pos[(int64_t)a * P + p];
    ok = ok && x >= -0.5 && x < (double)n[a];
  }
  if (!ok) {
    atomicAdd(res, 1);
    atomicMax(res + 1, (int32_t)(0x7fffffff - (p > 0x7ffffffe ? 0x7ffffffe : p)));
    return;
  }
  // positive finite doubles order like their bit patterns
  atomicMax(reinterpret_cast<unsigned long long *>(res + 2), (unsigned long long)__double_as_longlong(R));
  atomicMin(reinterpret_cast<unsigned long long *>(res + 4), (unsigned long long)__double_as_longlong(R));
}

lbmimb_status validate_particles_dev(lbmimb_lattice *h, int64_t P, const double *pos_dev, const double *radius_dev,
                                     const double *mass_dev, double *rmax, double *rmin) {
  int32_t *res = h->counters + 8;   // words 8..13 of the 16-word counter block
  const unsigned long long init[3] = {0ull, 0ull, ~0ull};
  LBMIMB_CUDA(cudaMemcpyAsync(res, init, sizeof(init), cudaMemcpyHostToDevice, h->stream));
  validate_particles_kernel<<<blocks_for(P, 256), 256, 0, h->stream>>>(h->gp.dim, P, h->gp.nx, h->gp.ny, h->gp.nz, pos_dev,
                                                                       radius_dev, mass_dev, res);
  LBMIMB_LAUNCH_CHECK(h, "validate_particles_kernel");
  unsigned long long out[3];
  LBMIMB_CUDA(cudaMemcpyAsync(out, res, sizeof(out), cudaMemcpyDeviceToHost, h->stream));
  LBMIMB_CUDA(cudaStreamSynchronize(h->stream));
  const int32_t nbad = (int32_t)(out[0] & 0xffffffffu), enc = (int32_t)(out[0] >> 32);
  if (nbad != 0)
    return fail(LBMIMB_EINVAL, "%d particle(s) with a non-positive / non-finite radius or mass or a centre outside "
                               "[-1/2, n); the first is particle %d", nbad, 0x7fffffff - enc);
  long long b;
  b = (long long)out[1];
  memcpy(rmax, &b, 8);
  b = (long long)out[2];
  memcpy(rmin, &b, 8);
  return LBMIMB_OK;
}

lbmimb_status launch_pack_records(lbmimb_lattice *h) {
  pack_records_kernel<<<blocks_for(h->P, 256), 256, 0, h->stream>>>(h->g.dim, h->P, h->pos, h->vel, h->omega,
                                                                    h->radius, h->prec);
  LBMIMB_LAUNCH_CHECK(h, "pack_records_kernel");
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// cell list: counting sort of the particles into cells of edge >= max(2 R_max, R_max + 1, 2)
// ---------------------------------------------------------------------------
struct CellGeom {
  int dim;
  int nc[3];
  double inv_e[3];
  int periodic[3];
};

__device__ __forceinline__ int cell_coord(double x, const CellGeom &cg, int a) {
  int c = (int)floor((x + 0.5) * cg.inv_e[a]);
  if (cg.periodic[a]) {
    c = wrap_i(c, cg.nc[a]);
  } else {
    c = c < 0 ? 0 : (c >= cg.nc[a] ? cg.nc[a] - 1 : c);
  }
  return c;
}

#include "verlet.cuh"

__global__ void cl_count_kernel(CellGeom cg, int64_t P, const double *__restrict__ pos, int32_t *__restrict__ cell_of,
                                int32_t *__restrict__ count) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int cx = cell_coord(pos[p], cg, 0);
  const int cy = cell_coord(pos[P + p], cg, 1);
  const int cz = cg.dim == 3 ? cell_coord(pos[2 * P + p], cg, 2) : 0;
  const int c = (cz * cg.nc[1] + cy) * cg.nc[0] + cx;
  cell_of[p] = c;
  atomicAdd(count + c, 1);
}

constexpr int kScanChunk = 2048;  // elements per block (256 threads x 8)

__global__ void scan_reduce_kernel(const int32_t *__restrict__ in, int64_t n, int32_t *__restrict__ block_sums) {
  __shared__ int32_t sh[8];
  const int64_t base = (int64_t)blockIdx.x * kScanChunk;
  int32_t v = 0;
  for (int e = threadIdx.x; e < kScanChunk; e += 256) {
    const int64_t idx = base + e;
    if (idx < n) v += in[idx];
  }
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    int32_t t = 0;
    for (int w = 0; w < 8; ++w) t += sh[w];
    block_sums[blockIdx.x] = t;
  }
}

// exclusive scan of the block sums by one block (serial over chunks of 1024 with a carry)
__global__ void scan_block_sums_kernel(int32_t *__restrict__ block_sums, int nb) {
  __shared__ int32_t sh[1024];
  __shared__ int32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < nb; base += 1024) {
    const int idx = base + threadIdx.x;
    const int32_t v = idx < nb ? block_sums[idx] : 0;
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      int32_t t = threadIdx.x >= o ? sh[threadIdx.x - o] : 0;
      __syncthreads();
      sh[threadIdx.x] += t;
      __syncthreads();
    }
    const int32_t incl = sh[threadIdx.x];
    if (idx < nb) block_sums[idx] = carry + incl - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry += incl;
    __syncthreads();
  }
}

__global__ void scan_final_kernel(const int32_t *__restrict__ in, int64_t n, const int32_t *__restrict__ block_sums,
                                  int32_t *__restrict__ out) {
  // one thread scans 8 consecutive elements; warp/block scan of the per-thread sums
  __shared__ int32_t wsum[8];
  const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * 8;
  int32_t v[8], tot = 0;
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    v[e] = (base + e < n) ? in[base + e] : 0;
    tot += v[e];
  }
  int32_t incl = tot;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int o = 1; o < 32; o <<= 1) {
    int32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  int32_t woff = 0;
  for (int w = 0; w < wid; ++w) woff += wsum[w];
  int32_t run = block_sums[blockIdx.x] + woff + incl - tot;
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    if (base + e < n) out[base + e] = run;
    run += v[e];
  }
}

__global__ void cl_fill_kernel(int64_t P, const int32_t *__restrict__ cell_of, const int32_t *__restrict__ start,
                               int32_t *__restrict__ fill, int32_t *__restrict__ items) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int c = cell_of[p];
  const int slot = atomicAdd(fill + c, 1);
  items[start[c] + slot] = (int32_t)p;
}

// ascending particle index inside each cell: makes every later traversal order deterministic
__global__ void cl_sort_kernel(int64_t ncells, const int32_t *__restrict__ start, int32_t *__restrict__ items) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncells) return;
  const int b = start[c], e = start[c + 1];
  for (int a = b + 1; a < e; ++a) {
    const int32_t v = items[a];
    int q = a - 1;
    while (q >= b && items[q] > v) {
      items[q + 1] = items[q];
      --q;
    }
    items[q + 1] = v;
  }
}

static CellGeom cell_geom(const lbmimb_lattice *h) {
  CellGeom cg;
  cg.dim = h->g.dim;
  cg.nc[0] = h->cl.ncx;
  cg.nc[1] = h->cl.ncy;
  cg.nc[2] = h->cl.ncz;
  cg.inv_e[0] = h->cl.inv_ex;
  cg.inv_e[1] = h->cl.inv_ey;
  cg.inv_e[2] = h->cl.inv_ez;
  cg.periodic[0] = !h->gp.bcx;
  cg.periodic[1] = !h->gp.bcy;
  cg.periodic[2] = !h->gp.bcz;
  return cg;
}

lbmimb_status finish_cell_list(lbmimb_lattice *h);

lbmimb_status build_cell_list(lbmimb_lattice *h) {
  double edge = 2.0 * h->rmax;
  if (edge < h->rmax + 1.0) edge = h->rmax + 1.0;
  if (edge < 2.0) edge = 2.0;
  int n[3] = {h->gp.nx, h->gp.ny, h->gp.nz};
  int nc[3] = {1, 1, 1};
  double inv_e[3] = {1.0, 1.0, 1.0};
  for (int a = 0; a < h->g.dim; ++a) {
    nc[a] = (int)floor((double)n[a] / edge);
    if (nc[a] < 1) nc[a] = 1;
    inv_e[a] = (double)nc[a] / (double)n[a];
  }
  CellList &cl = h->cl;
  cl.ncx = nc[0];
  cl.ncy = nc[1];
  cl.ncz = nc[2];
  cl.inv_ex = inv_e[0];
  cl.inv_ey = inv_e[1];
  cl.inv_ez = inv_e[2];
  cl.ncells = (int64_t)nc[0] * nc[1] * nc[2];
  if (cl.ncells > cl.ncells_max) return fail(LBMIMB_EINVAL, "internal: cell list larger than planned");
  const int64_t n1 = cl.ncells + 1;
  LBMIMB_CUDA(cudaMemsetAsync(cl.count, 0, (size_t)n1 * 4, h->stream));
  LBMIMB_CUDA(cudaMemsetAsync(cl.fill, 0, (size_t)cl.ncells * 4, h->stream));
  CellGeom cg = cell_geom(h);
  cl_count_kernel<<<blocks_for(h->P, 256), 256, 0, h->stream>>>(cg, h->P, h->pos, cl.cell_of, cl.count);
  LBMIMB_LAUNCH_CHECK(h, "cl_count_kernel");
  return finish_cell_list(h);
}

// second part of the counting sort: count[] and cell_of[] are filled (fill[] zeroed) -> start[], items[]
lbmimb_status finish_cell_list(lbmimb_lattice *h) {
  CellList &cl = h->cl;
  const int64_t n1 = cl.ncells + 1;
  cl.count_clean = false;
  const int nb = (int)((n1 + kScanChunk - 1) / kScanChunk);
  scan_reduce_kernel<<<nb, 256, 0, h->stream>>>(cl.count, n1, cl.block_sums);
  LBMIMB_LAUNCH_CHECK(h, "scan_reduce_kernel");
  scan_block_sums_kernel<<<1, 1024, 0, h->stream>>>(cl.block_sums, nb);
  LBMIMB_LAUNCH_CHECK(h, "scan_block_sums_kernel");
  scan_final_kernel<<<nb, 256, 0, h->stream>>>(cl.count, n1, cl.block_sums, cl.start);
  LBMIMB_LAUNCH_CHECK(h, "scan_final_kernel");
  cl_fill_kernel<<<blocks_for(h->P, 256), 256, 0, h->stream>>>(h->P, cl.cell_of, cl.start, cl.fill, cl.items);
  LBMIMB_LAUNCH_CHECK(h, "cl_fill_kernel");
  cl_sort_kernel<<<blocks_for(cl.ncells, 256), 256, 0, h->stream>>>(cl.ncells, cl.start, cl.items);
  LBMIMB_LAUNCH_CHECK(h, "cl_sort_kernel");
  h->cl_valid = true;
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// a1: mapping.  The inside test of ONE sample point, rounded exactly like the
// definition (include/lbmimb.h a1): every operation is a separate IEEE op, no FMA.
// ---------------------------------------------------------------------------
struct MapArgs {
  Geom g;              // the GLOBAL lattice (particle coordinates are global)
  SlabRows sl;         // which of its rows this handle stores
  int S, SD;
  int64_t P;
  const double *pos;
  const double *radius;
  uint32_t *tag;       // [N] node tags, make_tag(covering particle, count)
  int64_t *contested;
  int64_t contested_cap;
  int32_t *counters;
  double h_in, h_out;  // radius of a node's sample cloud + safety margin
  double hs;           // half edge of the sample cloud, 1/2 - 1/(2S)
};

__device__ __forceinline__ double sub_offset(int a, int S) {
  return __dsub_rn(__ddiv_rn(__dadd_rn((double)a, 0.5), (double)S), 0.5);
}

// Per-CTA table of the sample offsets: sample b = (az*S + ay)*S + ax -> (sub[ax], sub[ay], sub[az]).
struct SampleTable {
  double sx[256], sy[256], sz[256];
};

__device__ __forceinline__ void fill_sample_table(SampleTable &t, int S, int SD, int dim) {
  for (int b = threadIdx.x; b < SD; b += blockDim.x) {
    const int ax = b % S, r = b / S;
    const int ay = r % S, az = r / S;
    t.sx[b] = sub_offset(ax, S);
    t.sy[b] = sub_offset(ay, S);
    t.sz[b] = dim == 3 ? sub_offset(az, S) : 0.0;
  }
}

template <int D>
__device__ __forceinline__ bool sample_inside(const Geom &g, double di, double dj, double dk, double sx, double sy,
                                              double sz, double cx, double cy, double cz, double R2) {
  double dx = __dsub_rn(__dadd_rn(di, sx), cx);
  double dy = __dsub_rn(__dadd_rn(dj, sy), cy);
  if (!g.bcx) dx = min_image_d(dx, g.nx);
  if (!g.bcy) dy = min_image_d(dy, g.ny);
  double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
  if (D == 3) {
    double dz = __dsub_rn(__dadd_rn(dk, sz), cz);
    if (!g.bcz) dz = min_image_d(dz, g.nz);
    d2 = __dadd_rn(d2, __dmul_rn(dz, dz));
  }
  return d2 <= R2;
}

// number of inside samples of node (i,j,k) for one particle, computed by one warp
// (lane l tests samples l, l+32, ...); also returns this lane's inside bits in `bits`.
template <int D>
__device__ __forceinline__ int warp_count_samples(const Geom &g, int SD, const SampleTable &tab, int i, int j, int k,
                                                  double cx, double cy, double cz, double R2, unsigned &bits) {
  const int lane = threadIdx.x & 31;
  const double di = (double)i, dj = (double)j, dk = (double)k;
  int cnt = 0;
  bits = 0;
  for (int m = 0, b = lane; m * 32 < SD; ++m, b += 32) {
    bool in = false;
    if (b < SD) in = sample_inside<D>(g, di, dj, dk, tab.sx[b], tab.sy[b], tab.sz[b], cx, cy, cz, R2);
    const unsigned bal = __ballot_sync(0xffffffffu, in);
    cnt += __popc(bal);
    if (in) bits |= 1u << m;
  }
  return cnt;
}

__device__ __forceinline__ void bbox_axis(double c, double R, int n, int bc, int &lo, int &ext) {
  int l = (int)floor(c - R) - 1;
  int hgh = (int)ceil(c + R) + 1;
  if (bc) {
    if (l < 0) l = 0;
    if (hgh > n - 1) hgh = n - 1;
  } else if (hgh - l + 1 > n) {  // box wider than the periodic axis: every node once
    l = 0;
    hgh = n - 1;
  }
  lo = l;
  ext = hgh - l + 1;
  if (ext < 0) ext = 0;
}

#include "map_pass1.cuh"

// pass 2: nodes reached by more than one particle are recomputed from the definition:
// union of the inside samples, covering particle = most samples, ties -> lowest index.
// One warp per node.  The 3^D neighbour cells are read by one lane each, their particles are
// gathered into a per-warp candidate list, the candidates are distance-tested one per lane,
// and only the survivors are sampled (by the whole warp, lane l tests samples l, l+32, ...).
constexpr int kContestedCand = 64;  // candidates staged per round

template <int D>
__global__ void __launch_bounds__(128) map_contested_kernel(const MapArgs a, const CellGeom cg,
                                                            const int32_t *__restrict__ start,
                                                            const int32_t *__restrict__ items) {
  __shared__ SampleTable tab;
  __shared__ int32_t cand[4][kContestedCand];
  fill_sample_table(tab, a.S, a.SD, D);
  __syncthreads();
  int total = a.counters[0];
  if (total > a.contested_cap) total = (int)a.contested_cap;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
  // this lane's neighbour-cell offset (lanes beyond the 3^D offsets idle)
  const int lo0 = off_lo(cg.nc[0], cg.periodic[0]), n0 = off_hi(cg.nc[0], cg.periodic[0]) - lo0 + 1;
  const int lo1 = off_lo(cg.nc[1], cg.periodic[1]), n1 = off_hi(cg.nc[1], cg.periodic[1]) - lo1 + 1;
  const int lo2 = D == 3 ? off_lo(cg.nc[2], cg.periodic[2]) : 0;
  const int n2 = D == 3 ? off_hi(cg.nc[2], cg.periodic[2]) - lo2 + 1 : 1;
  const bool cell_lane = lane < n0 * n1 * n2;
  const int ox = lo0 + lane % n0, oy = lo1 + (lane / n0) % n1, oz = lo2 + lane / (n0 * n1);
  const double ro_h = a.h_out;
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
    unsigned ubits = 0;
    int best_cnt = 0, best_p = -1;
    // rounds of at most kContestedCand candidates (one round unless cells are crowded)
    while (__any_sync(0xffffffffu, b < en)) {
      int mine = en - b;
      int incl = mine;
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      int excl = incl - mine;
      int take = mine;
      if (excl >= kContestedCand) take = 0;
      else if (excl + take > kContestedCand) take = kContestedCand - excl;
      for (int m = 0; m < take; ++m) cand[wl][excl + m] = __ldg(items + b + m);
      b += take;
      int T = __shfl_sync(0xffffffffu, incl, 31);
      if (T > kContestedCand) T = kContestedCand;
      __syncwarp();
      for (int t0 = 0; t0 < T; t0 += 32) {
        // one candidate per lane: cheap reject (no sample of this node can lie inside a particle that far away)
        int p = -1;
        double pcx = 0.0, pcy = 0.0, pcz = 0.0, R = 0.0;
        bool near = false;
        if (t0 + lane < T) {
          p = cand[wl][t0 + lane];
          pcx = a.pos[p];
          pcy = a.pos[a.P + p];
          pcz = D == 3 ? a.pos[2 * a.P + p] : 0.0;
          R = a.radius[p];
          double ex = (double)i - pcx, ey = (double)j - pcy, ez = D == 3 ? (double)k - pcz : 0.0;
          if (!a.g.bcx) ex = min_image_d(ex, a.g.nx);
          if (!a.g.bcy) ey = min_image_d(ey, a.g.ny);
          if (D == 3 && !a.g.bcz) ez = min_image_d(ez, a.g.nz);
          const double ro = R + ro_h;
          near = ex * ex + ey * ey + ez * ez <= ro * ro;
        }
        unsigned live = __ballot_sync(0xffffffffu, near);
        while (live) {
          const int src = __ffs(live) - 1;
          live &= live - 1;
          const int sp = __shfl_sync(0xffffffffu, p, src);
          const double sx = __shfl_sync(0xffffffffu, pcx, src), sy = __shfl_sync(0xffffffffu, pcy, src);
          const double sz = __shfl_sync(0xffffffffu, pcz, src), sR = __shfl_sync(0xffffffffu, R, src);
          unsigned bits;
          const int cnt = warp_count_samples<D>(a.g, a.SD, tab, i, j, k, sx, sy, sz, __dmul_rn(sR, sR), bits);
          ubits |= bits;
          if (cnt > best_cnt || (cnt == best_cnt && cnt > 0 && sp < best_p)) {
            best_cnt = cnt;
            best_p = sp;
          }
        }
      }
      __syncwarp();
    }
    int ucnt = 0;
    for (int m = 0; m * 32 < a.SD; ++m) ucnt += __popc(__ballot_sync(0xffffffffu, (ubits >> m) & 1u));
    if (lane == 0) a.tag[x] = make_tag(best_p, ucnt);
  }
}

#include "map_table.cuh"

// table geometry of DESIGN.md R17 for the handle's (single) particle radius
static TableGeom table_geom(const lbmimb_lattice *h) {
  TableGeom t;
  const int D = h->g.dim;
  t.Nd = D == 2 ? LBMIMB_TABLE_ND_2D : LBMIMB_TABLE_ND_3D;
  t.Nt = D == 2 ? LBMIMB_TABLE_NT_2D : LBMIMB_TABLE_NT_3D;
  t.St = D == 2 ? LBMIMB_TABLE_ST_2D : LBMIMB_TABLE_ST_3D;
  const double sqD = sqrt((double)D);
  t.R = h->rmax;
  t.d0 = h->rmax - 0.5 * sqD;
  t.inv_dd = (double)t.Nd / sqD;
  t.dd = sqD / (double)t.Nd;
  t.full2 = t.d0 > 1e-9 ? (t.d0 - 1e-9) * (t.d0 - 1e-9) : 0.0;
  t.none2 = (t.d0 + sqD + 1e-9) * (t.d0 + sqD + 1e-9);
  t.tab = h->eps_table;
  return t;
}

int64_t eps_table_entries(int dim) {
  return dim == 2 ? (int64_t)LBMIMB_TABLE_ND_2D * LBMIMB_TABLE_NT_2D
                  : (int64_t)LBMIMB_TABLE_ND_3D * LBMIMB_TABLE_NT_3D * LBMIMB_TABLE_NT_3D;
}

// (re)builds the table when the radius changed since the last build
lbmimb_status ensure_eps_table(lbmimb_lattice *h) {
  if (h->P > 0 && h->rmin != h->rmax)
    return fail(LBMIMB_ESTATE, "table mapping needs one particle radius (PAPER.md:73), got %g .. %g", h->rmin, h->rmax);
  if (!(h->rmax >= 1.0)) return fail(LBMIMB_ESTATE, "table mapping needs a radius >= 1 lattice spacing");
  if (h->table_R == h->rmax) return LBMIMB_OK;
  const TableGeom t = table_geom(h);
  const int entries = (int)eps_table_entries(h->g.dim);
  if (h->g.dim == 2) build_eps_table_kernel<2><<<entries, 256, 0, h->stream>>>(t, h->eps_table);
  else build_eps_table_kernel<3><<<entries, 256, 0, h->stream>>>(t, h->eps_table);
  LBMIMB_LAUNCH_CHECK(h, "build_eps_table_kernel");
  h->table_R = h->rmax;
  return LBMIMB_OK;
}

static lbmimb_status launch_map_table(lbmimb_lattice *h, const MapArgs &a) {
  lbmimb_status st = ensure_eps_table(h);
  if (st != LBMIMB_OK) return st;
  const TableGeom t = table_geom(h);
  const double edge = 2.0 * h->rmax + 3.0;
  if (h->g.dim == 2) {
    if (edge * edge <= 256.0) map_table_kernel<2, 16><<<blocks_for(h->P, 8), 128, 0, h->stream>>>(a, t);
    else map_table_kernel<2, 32><<<blocks_for(h->P, 4), 128, 0, h->stream>>>(a, t);
  } else {
    map_table_kernel<3, 128><<<blocks_for(h->P, 1), 128, 0, h->stream>>>(a, t);
  }
  LBMIMB_LAUNCH_CHECK(h, "map_table_kernel");
  CellGeom cg = cell_geom(h);
  if (h->g.dim == 2)
    map_table_contested_kernel<2><<<148 * 4, 128, 0, h->stream>>>(a, t, cg, h->cl.start, h->cl.items);
  else
    map_table_contested_kernel<3><<<148 * 4, 128, 0, h->stream>>>(a, t, cg, h->cl.start, h->cl.items);
  LBMIMB_LAUNCH_CHECK(h, "map_table_contested_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_map(lbmimb_lattice *h) {
  lbmimb_status st;
  if (!h->cl_valid && (st = build_cell_list(h)) != LBMIMB_OK) return st;
  // one memset: the tags and, directly behind them in the workspace, the shared-node count and its overflow flag
  LBMIMB_CUDA(cudaMemsetAsync(h->tag, 0, (size_t)((char *)(h->counters + 16) - (char *)h->tag), h->stream));
  MapArgs a;
  a.g = h->gp;
  a.sl = h->sl;
  a.S = h->prm.subsamples;
  a.SD = h->SD;
  a.P = h->P;
  a.pos = h->pos;
  a.radius = h->radius;
  a.tag = h->tag;
  a.contested = h->contested;
  a.contested_cap = h->contested_cap;
  a.counters = h->counters;
  const double hs = sqrt((double)h->g.dim) * (0.5 - 0.5 / (double)a.S);
  a.h_in = hs + 1e-6;
  a.h_out = hs + 1e-6;
  a.hs = 0.5 - 0.5 / (double)a.S;
  if (h->map_mode == LBMIMB_MAP_TABLE) return launch_map_table(h, a);
  // threads per particle: enough lanes for the boundary shell without leaving most of them idle
  const double edge = 2.0 * h->rmax + 3.0;
  if (h->g.dim == 2) {
    const bool small = edge * edge <= 256.0;
    if (a.S == 8 && small) map_particles_kernel<2, 16, 8><<<blocks_for(h->P, 8), 128, 0, h->stream>>>(a);
    else if (a.S == 8) map_particles_kernel<2, 32, 8><<<blocks_for(h->P, 4), 128, 0, h->stream>>>(a);
    else map_particles_kernel<2, 32, 0><<<blocks_for(h->P, 4), 128, 0, h->stream>>>(a);
  } else {
    if (a.S == 4) map_particles_kernel<3, 128, 4><<<blocks_for(h->P, 1), 128, 0, h->stream>>>(a);
    else map_particles_kernel<3, 128, 0><<<blocks_for(h->P, 1), 128, 0, h->stream>>>(a);
  }
  LBMIMB_LAUNCH_CHECK(h, "map_particles_kernel");
  CellGeom cg = cell_geom(h);
  if (h->g.dim == 2)
    map_contested_kernel<2><<<148 * 16, 128, 0, h->stream>>>(a, cg, h->cl.start, h->cl.items);
  else
    map_contested_kernel<3><<<148 * 16, 128, 0, h->stream>>>(a, cg, h->cl.start, h->cl.items);
  LBMIMB_LAUNCH_CHECK(h, "map_contested_kernel");
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// a3: the per-particle sums of eq. (3) are formed inside the fused step (collide.cuh: reduce_runs) as
// fixed-point integers; this kernel turns them into force / torque and clears the accumulators for the
// next emitting step.  (Round 1 wrote a 32-byte exchange record per covered node and gathered the records
// per particle in a second pass over the bounding boxes: C3 0.38 GB written + 0.72 GB read, 0.18 ms.)
// ---------------------------------------------------------------------------
template <int D>
__global__ void finish_forces_kernel(int64_t P, long long *__restrict__ facc, double *__restrict__ force,
                                     double *__restrict__ torque) {
  constexpr int NV = D == 2 ? 3 : 6;
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  longlong2 *acc = reinterpret_cast<longlong2 *>(facc + p * (2 * NV));
  double v[NV];
#pragma unroll
  for (int c = 0; c < NV; ++c) {
    const longlong2 w = acc[c];
    v[c] = fixed_value(w.x, w.y);
    acc[c] = make_longlong2(0, 0);
  }
#pragma unroll
  for (int c = 0; c < D; ++c) force[(int64_t)c * P + p] = v[c];
  if (D == 2) {
    torque[p] = v[2];
  } else {
#pragma unroll
    for (int c = 0; c < 3; ++c) torque[(int64_t)c * P + p] = v[3 + c];
  }
}

lbmimb_status launch_finish_forces(lbmimb_lattice *h) {
  if (h->g.dim == 2)
    finish_forces_kernel<2><<<blocks_for(h->P, 256), 256, 0, h->stream>>>(h->P, h->facc, h->force, h->torque);
  else
    finish_forces_kernel<3><<<blocks_for(h->P, 256), 256, 0, h->stream>>>(h->P, h->facc, h->force, h->torque);
  LBMIMB_LAUNCH_CHECK(h, "finish_forces_kernel");
  return LBMIMB_OK;
}

// ---------------------------------------------------------------------------
// a4: DEM, eq. (4)-(5) with the readings R8-R11.  Contact search: the cell list above, or the
// Verlet neighbour lists of verlet.cuh (R19).
// ---------------------------------------------------------------------------
struct DemArgs {
  Geom g;
  CellGeom cg;
  int64_t P;
  double *pos, *vel, *omega;
  const double *radius, *mass, *force, *torque;
  double *fc;
  const int32_t *start, *items;
  double kn, ce;  // eta = ce * sqrt(kn * m_eff), ce = -2 ln e / sqrt(pi^2 + ln^2 e)
  double gp[3];
  double dt;
  // Verlet mode only (else nl_state == nullptr)
  int32_t *nl_state;
  const int32_t *nl_items, *nl_count;
  const double *nl_xref;
  int64_t nl_Pcap;
  int nl_every;
  double nl_h2;   // (skin/2)^2
};

// force of particle j on particle i (R8): k_n delta n_ij - eta (v_ij . n_ij) n_ij, added to F
template <int D>
__device__ __forceinline__ void pair_force(const DemArgs &a, const int *n, const double *xi, const double *vi,
                                           double Ri, double mi, int j, double *F) {
  double d[3] = {0.0, 0.0, 0.0}, dist2 = 0.0;
  for (int q = 0; q < D; ++q) {
    d[q] = xi[q] - a.pos[(int64_t)q * a.P + j];
    const bool per = q == 0 ? !a.g.bcx : (q == 1 ? !a.g.bcy : !a.g.bcz);
    if (per) d[q] = min_image_d(d[q], n[q]);
    dist2 += d[q] * d[q];
  }
  const double Rs = Ri + a.radius[j];
  if (dist2 >= Rs * Rs) return;
  const double dist = sqrt(dist2);
  const double delta = Rs - dist;
  if (!(delta > 0.0)) return;
  const double mj = a.mass[j];
  const double meff = mi * mj / (mi + mj);
  const double eta = a.ce * sqrt(a.kn * meff);
  double nrm[3], vn = 0.0;
  for (int q = 0; q < D; ++q) {
    nrm[q] = d[q] / dist;
    vn += (vi[q] - a.vel[(int64_t)q * a.P + j]) * nrm[q];
  }
  const double mag = a.kn * delta - eta * vn;
  for (int q = 0; q < D; ++q) F[q] += mag * nrm[q];
}

// walls: planes at -1/2 and n-1/2 of a wall axis, m_eff = m_i (R10)
template <int D>
__device__ __forceinline__ void wall_force(const DemArgs &a, const int *n, const double *xi, const double *vi,
                                           double Ri, double mi, double *F) {
  for (int q = 0; q < D; ++q) {
    const bool wall = q == 0 ? a.g.bcx : (q == 1 ? a.g.bcy : a.g.bcz);
    if (!wall) continue;
    const double eta = a.ce * sqrt(a.kn * mi);
    double delta = Ri - (xi[q] + 0.5);
    if (delta > 0.0) F[q] += a.kn * delta - eta * vi[q];
    delta = Ri - (((double)n[q] - 0.5) - xi[q]);
    if (delta > 0.0) F[q] += -a.kn * delta - eta * vi[q];
  }
}

// Contact force on particle i by ONE WARP: lane t takes the t-th of the 3^D cells around the particle (lanes
// beyond 3^D idle), sums the pair forces of that cell's particles in ascending index, and the lanes' partial
// sums are added in a fixed butterfly, so the result is reproducible.  A thread per particle walks the 27
// cells one after the other and pays two dependent memory latencies per neighbour candidate, ~70 times in a
// row (C5: 55 us per contact evaluation for 4,096 spheres); a warp per particle pays them two or three times.
// Every lane returns the total (walls included).
template <int D>
__device__ __forceinline__ void dem_contact_sum(const DemArgs &a, int64_t i, double *F) {
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  const int t = threadIdx.x & 31;
  double xi[3], vi[3];
  F[0] = F[1] = F[2] = 0.0;
  for (int c = 0; c < D; ++c) {
    xi[c] = a.pos[(int64_t)c * a.P + i];
    vi[c] = a.vel[(int64_t)c * a.P + i];
  }
  const double Ri = a.radius[i], mi = a.mass[i];
  int cc[3] = {0, 0, 0};
  for (int c = 0; c < D; ++c) cc[c] = cell_coord(xi[c], a.cg, c);
  const int nc0 = a.cg.nc[0], nc1 = a.cg.nc[1], nc2 = D == 3 ? a.cg.nc[2] : 1;
  constexpr int NC = D == 3 ? 27 : 9;
  if (t < NC) {
    const int ox = t % 3 - 1, oy = (t / 3) % 3 - 1, oz = D == 3 ? t / 9 - 1 : 0;
    int ex = cc[0] + ox, ey = cc[1] + oy, ez = cc[2] + oz;
    bool ok = ox >= off_lo(nc0, a.cg.periodic[0]) && ox <= off_hi(nc0, a.cg.periodic[0]) &&
              oy >= off_lo(nc1, a.cg.periodic[1]) && oy <= off_hi(nc1, a.cg.periodic[1]);
    if (D == 3) ok = ok && oz >= off_lo(nc2, a.cg.periodic[2]) && oz <= off_hi(nc2, a.cg.periodic[2]);
    if (a.cg.periodic[0]) ex = wrap_i(ex, nc0);
    else ok = ok && ex >= 0 && ex < nc0;
    if (a.cg.periodic[1]) ey = wrap_i(ey, nc1);
    else ok = ok && ey >= 0 && ey < nc1;
    if (D == 3) {
      if (a.cg.periodic[2]) ez = wrap_i(ez, nc2);
      else ok = ok && ez >= 0 && ez < nc2;
    }
    if (ok) {
      const int c = (ez * nc1 + ey) * nc0 + ex;
      const int bg = a.start[c], en = a.start[c + 1];
      for (int it = bg; it < en; ++it) {
        const int j = a.items[it];
        if (j == (int)i) continue;
        pair_force<D>(a, n, xi, vi, Ri, mi, j, F);
      }
    }
  }
#pragma unroll
  for (int q = 0; q < D; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) F[q] += __shfl_xor_sync(0xffffffffu, F[q], o);
  wall_force<D>(a, n, xi, vi, Ri, mi, F);
}

// The same sum by ONE THREAD: the 3^D cells one after the other (oz, oy, ox ascending).  For large sets
// (P > kDemWarpMaxP) there are enough particles to hide the dependent latencies, and a warp per particle
// only multiplies the threads: P2D (1,166,400 disks) 2.14 ms per step with warps against 0.44 ms with threads.
template <int D>
__device__ __forceinline__ void dem_contact_sum_serial(const DemArgs &a, int64_t i, double *F) {
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  double xi[3], vi[3];
  F[0] = F[1] = F[2] = 0.0;
  for (int c = 0; c < D; ++c) {
    xi[c] = a.pos[(int64_t)c * a.P + i];
    vi[c] = a.vel[(int64_t)c * a.P + i];
  }
  const double Ri = a.radius[i], mi = a.mass[i];
  int cc[3] = {0, 0, 0};
  for (int c = 0; c < D; ++c) cc[c] = cell_coord(xi[c], a.cg, c);
  const int nc0 = a.cg.nc[0], nc1 = a.cg.nc[1], nc2 = D == 3 ? a.cg.nc[2] : 1;
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
        const int c = (ez * nc1 + ey) * nc0 + ex;
        for (int it = a.start[c]; it < a.start[c + 1]; ++it) {
          const int j = a.items[it];
          if (j == (int)i) continue;
          pair_force<D>(a, n, xi, vi, Ri, mi, j, F);
        }
      }
  wall_force<D>(a, n, xi, vi, Ri, mi, F);
}

constexpr int64_t kDemWarpMaxP = 16384;   // up to here one warp per particle, beyond one thread per particle

// the same sums over the neighbour lists (ascending j).  Runs right after the three predicated
// build kernels of this evaluation, so one thread commits their outcome to the list state.
template <int D>
__global__ void dem_contact_list_kernel(const DemArgs a) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && nl_need(a.nl_state, a.nl_every)) {
    a.nl_state[NL_VALID] = 1;
    a.nl_state[NL_AGE] = 0;
    a.nl_state[NL_BUILDS] += 1;
    a.nl_state[NL_DISP] = 0;
  }
  if (i >= a.P) return;
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  double xi[3], vi[3], F[3] = {0.0, 0.0, 0.0};
  for (int c = 0; c < D; ++c) {
    xi[c] = a.pos[(int64_t)c * a.P + i];
    vi[c] = a.vel[(int64_t)c * a.P + i];
  }
  const double Ri = a.radius[i], mi = a.mass[i];
  const int cnt = a.nl_count[i];
  for (int k = 0; k < cnt; ++k) {
    const int j = a.nl_items[(int64_t)k * a.nl_Pcap + i];
    pair_force<D>(a, n, xi, vi, Ri, mi, j, F);
  }
  wall_force<D>(a, n, xi, vi, Ri, mi, F);
  for (int q = 0; q < D; ++q) a.fc[(int64_t)q * a.P + i] = F[q];
}

// first half: v += dt/2 a0; x += dt v (wrapped into [0,n) on periodic axes).  Verlet mode: raises
// the displacement flag of the rebuild rule when this particle is now farther than skin/2 from
// where it was when the lists were built.
template <int D>
__device__ __forceinline__ void dem_kick_drift_one(const DemArgs &a, int64_t p) {
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  const bool per[3] = {!a.g.bcx, !a.g.bcy, !a.g.bcz};
  const double m = a.mass[p];
  double xn[3] = {0.0, 0.0, 0.0};
  for (int q = 0; q < D; ++q) {
    const int64_t id = (int64_t)q * a.P + p;
    const double a0 = (a.force[id] + a.fc[id]) / m + a.gp[q];
    const double v = a.vel[id] + 0.5 * a.dt * a0;
    a.vel[id] = v;
    double x = a.pos[id] + a.dt * v;
    if (per[q]) {
      if (x >= (double)n[q]) x -= (double)n[q];
      if (x < 0.0) x += (double)n[q];
    }
    a.pos[id] = x;
    xn[q] = x;
  }
  if (a.nl_state != nullptr && verlet_disp2<D>(xn, a.nl_xref, a.nl_Pcap, p, n, per) > a.nl_h2) a.nl_state[NL_DISP] = 1;
}

template <int D>
__global__ void dem_kick_drift_kernel(const DemArgs a) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < a.P) dem_kick_drift_one<D>(a, p);
}

// second half: v += dt/2 a1; omega += dt T_h / I.  Verlet mode: the lists age by one step.
template <int D>
__device__ __forceinline__ void dem_kick_one(const DemArgs &a, int64_t p) {
  const double m = a.mass[p], R = a.radius[p];
  for (int q = 0; q < D; ++q) {
    const int64_t id = (int64_t)q * a.P + p;
    const double a1 = (a.force[id] + a.fc[id]) / m + a.gp[q];
    a.vel[id] = a.vel[id] + 0.5 * a.dt * a1;
  }
  const double I = (D == 3 ? 0.4 : 0.5) * m * R * R;
  constexpr int nt = D == 2 ? 1 : 3;
  for (int q = 0; q < nt; ++q) {
    const int64_t id = (int64_t)q * a.P + p;
    a.omega[id] = a.omega[id] + a.dt * a.torque[id] / I;
  }
}

template <int D>
__global__ void dem_kick_kernel(const DemArgs a) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p == 0 && a.nl_state != nullptr) a.nl_state[NL_AGE] += 1;
  if (p < a.P) dem_kick_one<D>(a, p);
}

// ---------------------------------------------------------------------------
// Cell-list mode: the DEM step in two kernels around the rebuild of the cell list.  Positions and velocities
// are double-buffered (pos2 / vel2), so that a particle can take its half step while its neighbours' contact
// sums still read the old state: no kernel boundary is needed between the contact sum and the kick.
//   first half : [a3: fixed-point force sums -> force / torque]  F_c(x, v) -> v2 = v + dt/2 a0, x2 = x + dt v2
//                (wrapped), cell of x2 counted
//   cell list of x2 (one single-block kernel for small sets, else the counting sort of build_cell_list)
//   second half: F_c(x2, v2) -> v = v2 + dt/2 a1, x = x2, omega += dt T_h / I, packed record
// Same per-particle arithmetic and summation order as the one-kernel-per-phase sequence of round 1 (and as the
// neighbour-list path below): bit for bit the same trajectories.  C5: 10 launches + 2 memsets -> 3 launches.
// ---------------------------------------------------------------------------
struct DemCellArgs {
  double *pos2, *vel2;          // state after the first half step
  double *pos_out, *vel_out;    // final state (the handle's pos / vel)
  int32_t *count, *cell_of;     // cell list under construction
  long long *facc;
  double *force_w, *torque_w;   // writable views of force / torque (FINISH)
  double *prec;
};

template <int D, bool FINISH, bool WARP>
__global__ void __launch_bounds__(128) dem_first_half_kernel(const DemArgs a, const DemCellArgs b) {
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t p = WARP ? gid >> 5 : gid;   // one warp, or one thread, per particle
  if (p >= a.P) return;
  const int64_t P = a.P;
  double Fc[3];
  if (WARP) {
    dem_contact_sum<D>(a, p, Fc);
    if ((threadIdx.x & 31) != 0) return;
  } else {
    dem_contact_sum_serial<D>(a, p, Fc);
  }
  double Fh[3] = {0.0, 0.0, 0.0};
  if (FINISH) {
    constexpr int NV = D == 2 ? 3 : 6;
    longlong2 *acc = reinterpret_cast<longlong2 *>(b.facc + p * (2 * NV));
    double v[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) {
      const longlong2 w = acc[c];
      v[c] = fixed_value(w.x, w.y);
      acc[c] = make_longlong2(0, 0);
    }
#pragma unroll
    for (int c = 0; c < D; ++c) {
      b.force_w[(int64_t)c * P + p] = v[c];
      Fh[c] = v[c];
    }
    if (D == 2) {
      b.torque_w[p] = v[2];
    } else {
#pragma unroll
      for (int c = 0; c < 3; ++c) b.torque_w[(int64_t)c * P + p] = v[3 + c];
    }
  } else {
#pragma unroll
    for (int c = 0; c < D; ++c) Fh[c] = a.force[(int64_t)c * P + p];
  }
  const int n[3] = {a.g.nx, a.g.ny, a.g.nz};
  const bool per[3] = {!a.g.bcx, !a.g.bcy, !a.g.bcz};
  const double m = a.mass[p];
  double xn[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int q = 0; q < D; ++q) {
    const int64_t id = (int64_t)q * P + p;
    const double a0 = (Fh[q] + Fc[q]) / m + a.gp[q];
    const double v = a.vel[id] + 0.5 * a.dt * a0;
    b.vel2[id] = v;
    double x = a.pos[id] + a.dt * v;
    if (per[q]) {
      if (x >= (double)n[q]) x -= (double)n[q];
      if (x < 0.0) x += (double)n[q];
    }
    b.pos2[id] = x;
    xn[q] = x;
  }
  const int cx = cell_coord(xn[0], a.cg, 0), cy = cell_coord(xn[1], a.cg, 1);
  const int cz = D == 3 ? cell_coord(xn[2], a.cg, 2) : 0;
  const int c = (cz * a.cg.nc[1] + cy) * a.cg.nc[0] + cx;
  b.cell_of[p] = c;
  atomicAdd(b.count + c, 1);
}

// a.pos / a.vel = the half-step state (pos2 / vel2), a.start / a.items = the cell list of pos2
template <int D, bool WARP>
__global__ void __launch_bounds__(128) dem_second_half_kernel(const DemArgs a, const DemCellArgs b) {
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t p = WARP ? gid >> 5 : gid;
  if (p >= a.P) return;
  const int64_t P = a.P;
  double Fc[3];
  if (WARP) {
    dem_contact_sum<D>(a, p, Fc);
    if ((threadIdx.x & 31) != 0) return;
  } else {
    dem_contact_sum_serial<D>(a, p, Fc);
  }
  const double m = a.mass[p], R = a.radius[p];
  double x[3] = {0.0, 0.0, 0.0}, v[3] = {0.0, 0.0, 0.0}, w[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int q = 0; q < D; ++q) {
    const int64_t id = (int64_t)q * P + p;
    const double a1 = (a.force[id] + Fc[q]) / m + a.gp[q];
    v[q] = a.vel[id] + 0.5 * a.dt * a1;
    x[q] = a.pos[id];
    b.vel_out[id] = v[q];
    b.pos_out[id] = x[q];
  }
  const double I = (D == 3 ? 0.4 : 0.5) * m * R * R;
  constexpr int nt = D == 2 ? 1 : 3;
#pragma unroll
  for (int q = 0; q < nt; ++q) {
    const int64_t id = (int64_t)q * P + p;
    w[q] = a.omega[id] + a.dt * a.torque[id] / I;
    a.omega[id] = w[q];
  }
  double *r = b.prec + p * prec_stride(D);
  if (D == 2) {
    r[0] = x[0];
    r[1] = x[1];
    r[2] = v[0];
    r[3] = v[1];
    r[4] = w[0];
    r[5] = R;
  } else {
    r[0] = x[0];
    r[1] = x[1];
    r[2] = x[2];
    r[3] = v[0];
    r[4] = v[1];
    r[5] = v[2];
    r[6] = w[0];
    r[7] = w[1];
    r[8] = w[2];
    r[9] = R;
  }
}

// Cell list of a small set from the counts the first half left: exclusive scan, fill, sort -- one block, so
// that block barriers stand where the counting sort of build_cell_list has five kernel boundaries.  Leaves
// count and fill zeroed for the next step.
constexpr int kListSmallP = 65536;
constexpr int kListSmallCells = 1024 * 64;
constexpr int kListSmallThreads = 1024;

__global__ void __launch_bounds__(kListSmallThreads) cl_small_kernel(int64_t P, int64_t ncells, int32_t *__restrict__ count,
                                                                   int32_t *__restrict__ start,
                                                                   int32_t *__restrict__ fill,
                                                                   int32_t *__restrict__ items,
                                                                   const int32_t *__restrict__ cell_of) {
  __shared__ int32_t wsum[kListSmallThreads / 32];
  const int tid = threadIdx.x;
  const int64_t n1 = ncells + 1;
  const int per = (int)((n1 + kListSmallThreads - 1) / kListSmallThreads);
  const int64_t lo = (int64_t)tid * per;
  int32_t tot = 0;
  for (int e = 0; e < per; ++e)
    if (lo + e < ncells) tot += count[lo + e];
  int32_t incl = tot;
  const int lane = tid & 31, wid = tid >> 5;
  for (int o = 1; o < 32; o <<= 1) {
    const int32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  int32_t woff = 0;
  for (int w = 0; w < wid; ++w) woff += wsum[w];
  int32_t run = woff + incl - tot;
  for (int e = 0; e < per; ++e)
    if (lo + e < n1) {
      start[lo + e] = run;
      if (lo + e < ncells) {
        run += count[lo + e];
        count[lo + e] = 0;
        fill[lo + e] = 0;
      }
    }
  __syncthreads();
  for (int64_t p = tid; p < P; p += kListSmallThreads) {
    const int c = cell_of[p];
    const int slot = atomicAdd(fill + c, 1);
    items[start[c] + slot] = (int32_t)p;
  }
  __syncthreads();
#pragma unroll 4
  for (int64_t c = tid; c < ncells; c += kListSmallThreads) {
    const int bg = start[c], en = start[c + 1];
    for (int q0 = bg + 1; q0 < en; ++q0) {
      const int32_t v = items[q0];
      int q = q0 - 1;
      while (q >= bg && items[q] > v) {
        items[q + 1] = items[q];
        --q;
      }
      items[q + 1] = v;
    }
    fill[c] = 0;
  }
}

// ---- neighbour-list storage (library-allocated; sized from packing bounds on the radii) ----
void neighbor_list_release(lbmimb_lattice *h) {
  if (h->nl.mem) cudaFree(h->nl.mem);
  h->nl.mem = nullptr;
  h->nl.items = h->nl.count = h->nl.state = h->nl.gcount = h->nl.gitems = nullptr;
  h->nl.x_ref = nullptr;
}

// positions were replaced: no valid list, and the overflow flags of the old particle set are history
lbmimb_status neighbor_list_invalidate(lbmimb_lattice *h) {
  if (h->nl.mem) {
    LBMIMB_CUDA(cudaMemsetAsync(h->nl.state + NL_VALID, 0, 4, h->stream));
    LBMIMB_CUDA(cudaMemsetAsync(h->nl.state + NL_OVF_LIST, 0, 8, h->stream));
  }
  return LBMIMB_OK;
}

lbmimb_status neighbor_list_prepare(lbmimb_lattice *h) {
  NeighborList &nl = h->nl;
  if (nl.mem && nl.rmax == h->rmax && nl.rmin == h->rmin) return LBMIMB_OK;
  neighbor_list_release(h);
  const int D = h->g.dim;
  const int n[3] = {h->gp.nx, h->gp.ny, h->gp.nz};
  const double cutoff = (2.0 * h->rmax + nl.skin) * (1.0 + 1e-9);  // margin: cell binning is rounded
  const double dmin = 1.5 * h->rmin;  // closest centres the sizing allows for (soft spheres overlap)
  double edge_max = 0.0;
  nl.ncells = 1;
  for (int a = 0; a < 3; ++a) {
    nl.nc[a] = 1;
    nl.inv_e[a] = 1.0;
    if (a >= D) continue;
    nl.nc[a] = (int)floor((double)n[a] / cutoff);
    if (nl.nc[a] < 1) nl.nc[a] = 1;
    nl.inv_e[a] = (double)nl.nc[a] / (double)n[a];
    nl.ncells *= nl.nc[a];
    const double e = (double)n[a] / (double)nl.nc[a];
    if (nl.nc[a] > 1 && e > edge_max) edge_max = e;
  }
  if (edge_max == 0.0) edge_max = cutoff;
  const int64_t pm = h->Pmax > 0 ? h->Pmax : 1;
  double c = 2.0 * pow(edge_max / dmin + 1.0, (double)D);
  double k = pow(2.0 * cutoff / dmin + 1.0, (double)D);
  if (c > (double)pm) c = (double)pm;
  if (k > (double)(pm > 1 ? pm - 1 : 1)) k = (double)(pm > 1 ? pm - 1 : 1);
  nl.C = (int)ceil(c);
  nl.K = (int)ceil(k);
  nl.Pcap = pm;
  auto al = [](uint64_t v) { return (v + 255) & ~(uint64_t)255; };
  const uint64_t b_items = al((uint64_t)nl.K * pm * 4), b_count = al((uint64_t)pm * 4), b_state = 256;
  const uint64_t b_gcount = al((uint64_t)nl.ncells * 4), b_gitems = al((uint64_t)nl.ncells * nl.C * 4);
  const uint64_t b_xref = al((uint64_t)3 * pm * 8);
  const uint64_t total = b_items + b_count + b_state + b_gcount + b_gitems + b_xref;
  if (total > ((uint64_t)16 << 30))
    return fail(LBMIMB_ENOMEM, "neighbour lists would need %.1f GB (K = %d slots per particle, R_min = %g, R_max = %g)",
                (double)total / 1073741824.0, nl.K, h->rmin, h->rmax);
  void *mem = nullptr;
  cudaError_t e = cudaMalloc(&mem, total);
  if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(neighbour lists)");
  char *q = (char *)mem;
  nl.mem = mem;
  nl.items = (int32_t *)q;   q += b_items;
  nl.count = (int32_t *)q;   q += b_count;
  nl.state = (int32_t *)q;   q += b_state;
  nl.gcount = (int32_t *)q;  q += b_gcount;
  nl.gitems = (int32_t *)q;  q += b_gitems;
  nl.x_ref = (double *)q;
  nl.rmax = h->rmax;
  nl.rmin = h->rmin;
  LBMIMB_CUDA(cudaMemsetAsync(nl.state, 0, 256, h->stream));
  return LBMIMB_OK;
}

static VerletArgs verlet_args(const lbmimb_lattice *h) {
  const NeighborList &nl = h->nl;
  VerletArgs v;
  v.g = h->gp;
  v.cg.dim = h->g.dim;
  for (int a = 0; a < 3; ++a) {
    v.cg.nc[a] = nl.nc[a];
    v.cg.inv_e[a] = nl.inv_e[a];
  }
  v.cg.periodic[0] = !h->gp.bcx;
  v.cg.periodic[1] = !h->gp.bcy;
  v.cg.periodic[2] = !h->gp.bcz;
  v.P = h->P;
  v.Pcap = nl.Pcap;
  v.ncells = nl.ncells;
  v.pos = h->pos;
  v.radius = h->radius;
  v.skin = nl.skin;
  v.every = nl.every;
  v.K = nl.K;
  v.C = nl.C;
  v.items = nl.items;
  v.count = nl.count;
  v.state = nl.state;
  v.gcount = nl.gcount;
  v.gitems = nl.gitems;
  v.x_ref = nl.x_ref;
  return v;
}

// the three predicated build kernels in front of a contact evaluation (rebuild rule of R19)
template <int D>
static lbmimb_status verlet_ensure(lbmimb_lattice *h, const VerletArgs &v) {
  int nbc = blocks_for(v.ncells, 256);
  if (nbc > 148 * 8) nbc = 148 * 8;
  verlet_clear_kernel<<<nbc, 256, 0, h->stream>>>(v);
  LBMIMB_LAUNCH_CHECK(h, "verlet_clear_kernel");
  verlet_bin_kernel<D><<<blocks_for(h->P, 256), 256, 0, h->stream>>>(v);
  LBMIMB_LAUNCH_CHECK(h, "verlet_bin_kernel");
  verlet_list_kernel<D><<<blocks_for(h->P, 128), 128, 0, h->stream>>>(v);
  LBMIMB_LAUNCH_CHECK(h, "verlet_list_kernel");
  return LBMIMB_OK;
}

// In cell-list mode the first-half kernel can also convert the fixed-point force sums (a3's last part).
bool dem_can_finish(const lbmimb_lattice *h) { return h->nl.mode != LBMIMB_NEIGHBOR_VERLET; }

template <int D>
static lbmimb_status dem_impl(lbmimb_lattice *h, const lbmimb_dem_params *dem, bool finish) {
  lbmimb_status st;
  const bool verlet = h->nl.mode == LBMIMB_NEIGHBOR_VERLET;
  if (verlet) {
    if ((st = neighbor_list_prepare(h)) != LBMIMB_OK) return st;
  } else if (!h->cl_valid && (st = build_cell_list(h)) != LBMIMB_OK) {
    return st;
  }
  DemArgs a;
  a.g = h->gp;
  a.P = h->P;
  a.pos = h->pos;
  a.vel = h->vel;
  a.omega = h->omega;
  a.radius = h->radius;
  a.mass = h->mass;
  a.force = h->force;
  a.torque = h->torque;
  a.fc = h->fc;
  a.start = h->cl.start;
  a.items = h->cl.items;
  a.kn = dem->kn;
  const double le = log(dem->restitution);
  a.ce = -2.0 * le / sqrt(M_PI * M_PI + le * le);
  for (int c = 0; c < 3; ++c) a.gp[c] = dem->g_particle[c];
  a.dt = dem->dt;
  a.nl_state = nullptr;
  a.nl_items = a.nl_count = nullptr;
  a.nl_xref = nullptr;
  a.nl_Pcap = 0;
  a.nl_every = 0;
  a.nl_h2 = 0.0;
  const int nb = blocks_for(h->P, 128);
  a.cg = cell_geom(h);
  if (verlet) {
    const VerletArgs v = verlet_args(h);
    a.nl_state = h->nl.state;
    a.nl_items = h->nl.items;
    a.nl_count = h->nl.count;
    a.nl_xref = h->nl.x_ref;
    a.nl_Pcap = h->nl.Pcap;
    a.nl_every = h->nl.every;
    const double hs = 0.5 * h->nl.skin;
    a.nl_h2 = hs * hs;
    if ((st = verlet_ensure<D>(h, v)) != LBMIMB_OK) return st;
    dem_contact_list_kernel<D><<<nb, 128, 0, h->stream>>>(a);
    LBMIMB_LAUNCH_CHECK(h, "dem_contact_list_kernel");
    dem_kick_drift_kernel<D><<<nb, 128, 0, h->stream>>>(a);
    LBMIMB_LAUNCH_CHECK(h, "dem_kick_drift_kernel");
    if ((st = verlet_ensure<D>(h, v)) != LBMIMB_OK) return st;
    dem_contact_list_kernel<D><<<nb, 128, 0, h->stream>>>(a);
    LBMIMB_LAUNCH_CHECK(h, "dem_contact_list_kernel");
    dem_kick_kernel<D><<<nb, 128, 0, h->stream>>>(a);
    LBMIMB_LAUNCH_CHECK(h, "dem_kick_kernel");
    h->cl_valid = false;   // the particles moved and no cell list was built at the new positions
    return LBMIMB_OK;
  }
  // ---- cell-list mode: first half, cell list of the new positions, second half
  CellList &cl = h->cl;
  if (!cl.count_clean) {
    LBMIMB_CUDA(cudaMemsetAsync(cl.count, 0, (size_t)(cl.ncells + 1) * 4, h->stream));
    cl.count_clean = true;
  }
  DemCellArgs b;
  b.pos2 = h->pos2;
  b.vel2 = h->vel2;
  b.pos_out = h->pos;
  b.vel_out = h->vel;
  b.count = cl.count;
  b.cell_of = cl.cell_of;
  b.facc = h->facc;
  b.force_w = h->force;
  b.torque_w = h->torque;
  b.prec = h->prec;
  const bool warp = h->P <= kDemWarpMaxP;
  const int nbw = warp ? blocks_for(h->P, 4) : blocks_for(h->P, 128);   // a warp (four per block) or a thread per particle
  if (warp) {
    if (finish) dem_first_half_kernel<D, true, true><<<nbw, 128, 0, h->stream>>>(a, b);
    else dem_first_half_kernel<D, false, true><<<nbw, 128, 0, h->stream>>>(a, b);
  } else {
    if (finish) dem_first_half_kernel<D, true, false><<<nbw, 128, 0, h->stream>>>(a, b);
    else dem_first_half_kernel<D, false, false><<<nbw, 128, 0, h->stream>>>(a, b);
  }
  LBMIMB_LAUNCH_CHECK(h, "dem_first_half_kernel");
  if (h->P <= kListSmallP && cl.ncells + 1 <= kListSmallCells) {
    cl_small_kernel<<<1, kListSmallThreads, 0, h->stream>>>(h->P, cl.ncells, cl.count, cl.start, cl.fill, cl.items,
                                                           cl.cell_of);
    LBMIMB_LAUNCH_CHECK(h, "cl_small_kernel");
  } else {
    LBMIMB_CUDA(cudaMemsetAsync(cl.fill, 0, (size_t)cl.ncells * 4, h->stream));
    if ((st = finish_cell_list(h)) != LBMIMB_OK) return st;   // scan, fill, sort of build_cell_list (count stays dirty)
  }
  h->cl_valid = true;
  a.pos = h->pos2;
  a.vel = h->vel2;
  if (warp) dem_second_half_kernel<D, true><<<nbw, 128, 0, h->stream>>>(a, b);
  else dem_second_half_kernel<D, false><<<nbw, 128, 0, h->stream>>>(a, b);
  LBMIMB_LAUNCH_CHECK(h, "dem_second_half_kernel");
  return LBMIMB_OK;   // cell list of the new positions and packed records are in place
}

// finish: also convert the fixed-point force sums of the last step (cell-list mode only, dem_can_finish).
// On return the packed records are current in cell-list mode; in neighbour-list mode the caller packs them.
lbmimb_status launch_dem(lbmimb_lattice *h, const lbmimb_dem_params *dem, bool finish) {
  return h->g.dim == 2 ? dem_impl<2>(h, dem, finish) : dem_impl<3>(h, dem, finish);
}

}  // namespace lbmimb
