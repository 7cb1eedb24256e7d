// Lattice kernels: rest-state init (a0), the fused collide-and-stream step (a2),
// the stream/unstream permutations behind set_distributions / fetch_fields (a5).
//
// Scheme: "pull", two buffers (A-B).  The stored array is the post-collision state
// f*(x, t-1); one thread per node gathers f_i(x,t) = f*_i(x - c_i) (periodic wrap) or,
// when x - c_i lies behind a wall, f*_{-i}(x) (half-way bounce-back, R15),
// collides with eq. (1) of the paper and writes f*(x,t) to the other
// buffer at its own node: every store is aligned and coalesced, the x-shifted loads
// are misaligned by one element and served from L1/L2 sectors.
#include "lbmimb_internal.cuh"

namespace lbmimb {

struct StepArgs {
  const double *__restrict__ fin;
  double *__restrict__ fout;
  const uint8_t *__restrict__ eps_cnt;
  const int32_t *__restrict__ pid;
  const double *__restrict__ prec;
  const double *__restrict__ beta_tab;
  double *__restrict__ s;
  int64_t N;
  int nx, ny, nz;
  int bcx, bcy, bcz;
  unsigned tiles;      // blocks per lattice row
  double omega;        // 1/tau
  double gx, gy, gz;   // g_fluid
};

constexpr int kStepThreads = 128;

template <int D>
__device__ __forceinline__ double min_image(double d, int n) {
  double hn = 0.5 * (double)n;
  if (d > hn) return d - (double)n;
  if (d < -hn) return d + (double)n;
  return d;
}

// ---------------------------------------------------------------------------
// a2: fused collide-and-stream.  IMB = particles present, EMIT = also store the
// exchange vector s = beta*rho*(V_S - u) (= beta sum_i Omega_i c_i, P6).
// ---------------------------------------------------------------------------
template <int D, bool IMB, bool EMIT>
__global__ void __launch_bounds__(kStepThreads) collide_stream_kernel(const StepArgs a) {
  using L = Lat<D>;
  constexpr int Q = L::Q;
  const unsigned row = blockIdx.x / a.tiles;
  const unsigned tile = blockIdx.x - row * a.tiles;
  const int i = (int)(tile * kStepThreads + threadIdx.x);
  if (i >= a.nx) return;
  const int k = D == 3 ? (int)(row / (unsigned)a.ny) : 0;
  const int j = (int)(row - (unsigned)k * (unsigned)a.ny);
  const int64_t x = ((int64_t)k * a.ny + j) * a.nx + i;

  // ---- gather (streaming) ----
  double f[Q];
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    constexpr int dummy = 0;
    (void)dummy;
    const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
    bool bounce = false;
    int is = i - cx, js = j - cy, ks = k - cz;
    if (cx != 0) {
      if (is < 0 || is >= a.nx) {
        if (a.bcx) bounce = true;
        else is = is < 0 ? is + a.nx : is - a.nx;
      }
    }
    if (cy != 0) {
      if (js < 0 || js >= a.ny) {
        if (a.bcy) bounce = true;
        else js = js < 0 ? js + a.ny : js - a.ny;
      }
    }
    if (D == 3 && cz != 0) {
      if (ks < 0 || ks >= a.nz) {
        if (a.bcz) bounce = true;
        else ks = ks < 0 ? ks + a.nz : ks - a.nz;
      }
    }
    const int64_t src = bounce ? (int64_t)opposite(q) * a.N + x
                               : (int64_t)q * a.N + ((int64_t)ks * a.ny + js) * a.nx + is;
    f[q] = a.fin[src];
  }

  int cnt = 0;
  if (IMB) cnt = a.eps_cnt[x];

  // ---- moments ----
  double rho = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    rho += f[q];
    if (L::cx(q) == 1) mx += f[q];
    if (L::cx(q) == -1) mx -= f[q];
    if (L::cy(q) == 1) my += f[q];
    if (L::cy(q) == -1) my -= f[q];
    if (D == 3) {
      if (L::cz(q) == 1) mz += f[q];
      if (L::cz(q) == -1) mz -= f[q];
    }
  }
  const double inv = 1.0 / rho;
  const double ux = mx * inv, uy = my * inv, uz = D == 3 ? mz * inv : 0.0;
  const double om = a.omega;
  const double uu15 = 1.5 * (ux * ux + uy * uy + uz * uz);

  double fs[Q];
  if (!IMB || cnt == 0) {
    // pure LBGK + body force:  f* = f - (f - feq)/tau + F_i,  F_i = 3 w rho c.g  (R3)
    const double ev0 = rho * (1.0 - uu15);
    fs[0] = f[0] - om * (f[0] - L::w(0) * ev0);
#pragma unroll
    for (int q = 1; q < Q; q += 2) {
      const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
      const double cu = cx * ux + cy * uy + (D == 3 ? cz * uz : 0.0);
      const double cg = cx * a.gx + cy * a.gy + (D == 3 ? cz * a.gz : 0.0);
      const double wr = L::w(q) * rho;
      const double e = wr * (1.0 - uu15 + 4.5 * cu * cu);   // even part of feq
      const double o = wr * 3.0 * cu;                        // odd part of feq
      const double Fo = 3.0 * wr * cg;
      fs[q] = f[q] - om * (f[q] - (e + o)) + Fo;
      fs[q + 1] = f[q + 1] - om * (f[q + 1] - (e - o)) - Fo;
    }
  } else {
    // immersed moving boundary node, eq. (1)-(2)
    const int p = a.pid[x];
    const double beta = __ldg(a.beta_tab + cnt);
    const double *pr = a.prec + (int64_t)p * prec_stride(D);
    double vx, vy, vz = 0.0;
    if (D == 2) {
      double rx = (double)i - __ldg(pr + 0), ry = (double)j - __ldg(pr + 1);
      if (!a.bcx) rx = min_image<D>(rx, a.nx);
      if (!a.bcy) ry = min_image<D>(ry, a.ny);
      const double w = __ldg(pr + 4);
      vx = __ldg(pr + 2) - w * ry;
      vy = __ldg(pr + 3) + w * rx;
    } else {
      double rx = (double)i - __ldg(pr + 0), ry = (double)j - __ldg(pr + 1), rz = (double)k - __ldg(pr + 2);
      if (!a.bcx) rx = min_image<D>(rx, a.nx);
      if (!a.bcy) ry = min_image<D>(ry, a.ny);
      if (!a.bcz) rz = min_image<D>(rz, a.nz);
      const double wx = __ldg(pr + 6), wy = __ldg(pr + 7), wz = __ldg(pr + 8);
      vx = __ldg(pr + 3) + (wy * rz - wz * ry);
      vy = __ldg(pr + 4) + (wz * rx - wx * rz);
      vz = __ldg(pr + 5) + (wx * ry - wy * rx);
    }
    const double vv15 = 1.5 * (vx * vx + vy * vy + vz * vz);
    const double omb = (1.0 - beta) * om;
    {
      const double eu = L::w(0) * rho * (1.0 - uu15);
      const double ev = L::w(0) * rho * (1.0 - vv15);
      fs[0] = f[0] - omb * (f[0] - eu) + beta * (ev - eu);
    }
#pragma unroll
    for (int q = 1; q < Q; q += 2) {
      const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
      const double cu = cx * ux + cy * uy + (D == 3 ? cz * uz : 0.0);
      const double cv = cx * vx + cy * vy + (D == 3 ? cz * vz : 0.0);
      const double cg = cx * a.gx + cy * a.gy + (D == 3 ? cz * a.gz : 0.0);
      const double wr = L::w(q) * rho;
      const double eu = wr * (1.0 - uu15 + 4.5 * cu * cu), ou = wr * 3.0 * cu;
      const double ev = wr * (1.0 - vv15 + 4.5 * cv * cv), ov = wr * 3.0 * cv;
      const double Fo = 3.0 * wr * cg;
      // Omega_q = f_-q - f_q + feq_q(V) - feq_-q(u);  Omega_-q = f_q - f_-q + feq_-q(V) - feq_q(u)
      const double df = f[q + 1] - f[q];
      const double Op = df + (ev + ov) - (eu - ou);
      const double Om = -df + (ev - ov) - (eu + ou);
      fs[q] = f[q] - omb * (f[q] - (eu + ou)) + beta * Op + Fo;
      fs[q + 1] = f[q + 1] - omb * (f[q + 1] - (eu - ou)) + beta * Om - Fo;
    }
    if (EMIT) {
      const double br = beta * rho;
      a.s[x] = br * (vx - ux);
      a.s[a.N + x] = br * (vy - uy);
      if (D == 3) a.s[2 * a.N + x] = br * (vz - uz);
    }
  }

#pragma unroll
  for (int q = 0; q < Q; ++q) a.fout[(int64_t)q * a.N + x] = fs[q];
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
// Gather of the pre-collision state f_i(x,t) from the stored post-collision array
// (the same permutation the step kernel applies), for one node.
// ---------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void gather_node(const double *__restrict__ fpost, const Geom &g, int i, int j, int k,
                                            double *f) {
  using L = Lat<D>;
  const int64_t x = ((int64_t)k * g.ny + j) * g.nx + i;
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
      if (g.bcy) bounce = true;
      else js = js < 0 ? js + g.ny : js - g.ny;
    }
    if (D == 3 && (ks < 0 || ks >= g.nz)) {
      if (g.bcz) bounce = true;
      else ks = ks < 0 ? ks + g.nz : ks - g.nz;
    }
    const int64_t src = bounce ? (int64_t)opposite(q) * g.N + x
                               : (int64_t)q * g.N + ((int64_t)ks * g.ny + js) * g.nx + is;
    f[q] = fpost[src];
  }
}

// set_distributions: inverse permutation.  f*_q(x) = f_q(x + c_q), or f_{-q}(x) when x + c_q is behind a wall.
template <int D>
__global__ void unstream_kernel(const double *__restrict__ fpre, double *__restrict__ fpost, const Geom g) {
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
        if (g.bcy) bounce = true;
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
  const uint8_t *eps_cnt;
  const int32_t *pid;
  const double *s;
  void *dst;
  int lo[3], ext[3];
  int64_t box;
  int what;
  int have_particles;
};

template <int D>
__global__ void fetch_kernel(const FetchArgs a, const Geom g) {
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
      ((uint8_t *)a.dst)[b] = a.eps_cnt[x];
    } else if (a.what == LBMIMB_FIELD_PID) {
      ((int32_t *)a.dst)[b] = a.pid[x];
    } else if (a.what == LBMIMB_FIELD_S) {
      const bool cov = a.have_particles && a.eps_cnt[x] > 0;
      for (int c = 0; c < D; ++c) ((double *)a.dst)[(int64_t)c * a.box + b] = cov ? a.s[(int64_t)c * g.N + x] : 0.0;
    } else {
      double f[L::Q];
      gather_node<D>(a.fpost, g, i, j, k, f);
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

template <int D>
static void launch_cs(lbmimb_lattice *h, const StepArgs &a, unsigned blocks, bool imb, bool emit) {
  if (!imb)
    collide_stream_kernel<D, false, false><<<blocks, kStepThreads, 0, h->stream>>>(a);
  else if (!emit)
    collide_stream_kernel<D, true, false><<<blocks, kStepThreads, 0, h->stream>>>(a);
  else
    collide_stream_kernel<D, true, true><<<blocks, kStepThreads, 0, h->stream>>>(a);
}

lbmimb_status launch_collide_stream(lbmimb_lattice *h, bool emit) {
  StepArgs a;
  a.fin = h->f[h->cur];
  a.fout = h->f[h->cur ^ 1];
  a.eps_cnt = h->eps_cnt;
  a.pid = h->pid;
  a.prec = h->prec;
  a.beta_tab = h->beta_tab;
  a.s = h->s;
  a.N = h->g.N;
  a.nx = h->g.nx;
  a.ny = h->g.ny;
  a.nz = h->g.nz;
  a.bcx = h->g.bcx;
  a.bcy = h->g.bcy;
  a.bcz = h->g.bcz;
  a.tiles = (unsigned)((h->g.nx + kStepThreads - 1) / kStepThreads);
  a.omega = 1.0 / h->prm.tau;
  a.gx = h->prm.g_fluid[0];
  a.gy = h->prm.g_fluid[1];
  a.gz = h->g.dim == 3 ? h->prm.g_fluid[2] : 0.0;
  const int64_t blocks = (int64_t)a.tiles * h->g.ny * h->g.nz;
  if (blocks > 0x7fffffff) return fail(LBMIMB_EINVAL, "lattice needs more than 2^31 thread blocks");
  const bool imb = h->P > 0;
  if (h->g.dim == 2)
    launch_cs<2>(h, a, (unsigned)blocks, imb, emit);
  else
    launch_cs<3>(h, a, (unsigned)blocks, imb, emit);
  LBMIMB_LAUNCH_CHECK(h, "collide_stream_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_unstream(lbmimb_lattice *h, const double *f_pre, double *f_post) {
  if (h->g.dim == 2)
    unstream_kernel<2><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(f_pre, f_post, h->g);
  else
    unstream_kernel<3><<<grid_for(h->g.N, 256), 256, 0, h->stream>>>(f_pre, f_post, h->g);
  LBMIMB_LAUNCH_CHECK(h, "unstream_kernel");
  return LBMIMB_OK;
}

lbmimb_status launch_fetch(lbmimb_lattice *h, int what, const int64_t lo[3], const int64_t hi[3], void *dst_dev) {
  FetchArgs a;
  a.fpost = h->f[h->cur];
  a.eps_cnt = h->eps_cnt;
  a.pid = h->pid;
  a.s = h->s;
  a.dst = dst_dev;
  a.box = 1;
  for (int c = 0; c < 3; ++c) {
    a.lo[c] = (int)lo[c];
    a.ext[c] = (int)(hi[c] - lo[c]);
    a.box *= a.ext[c];
  }
  a.what = what;
  a.have_particles = h->P > 0;
  if (h->g.dim == 2)
    fetch_kernel<2><<<grid_for(a.box, 256), 256, 0, h->stream>>>(a, h->g);
  else
    fetch_kernel<3><<<grid_for(a.box, 256), 256, 0, h->stream>>>(a, h->g);
  LBMIMB_LAUNCH_CHECK(h, "fetch_kernel");
  return LBMIMB_OK;
}

}  // namespace lbmimb
