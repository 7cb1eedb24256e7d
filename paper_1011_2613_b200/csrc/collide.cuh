// Node-local collision of eq. (1) shared by the step kernels of lattice.cu (pull A-B and
// in-place AA), and the in-kernel force / torque sums of eq. (3).  In place on the gathered populations f[Q].
//
// Algebra (same real-number result as the paper's form, regrouped to cut fp64 work):
//   om = 1/tau, a = (1-beta) om.  With feq_q(u) = E_u + O_u, feq_-q(u) = E_u - O_u (even / odd part
//   in c_q), Omega_q = f_-q - f_q + feq_q(V) - feq_-q(u) (eq. (2)), F_q = 3 w rho c_q.g (R3):
//     f*_q  = (1-a-beta) f_q  + beta f_-q + w rho [K + 4.5((a-beta)(c.u)^2 + beta (c.V)^2)] + 3 w rho c.U
//     f*_-q = (1-a-beta) f_-q + beta f_q  + w rho [K + ...]                                 - 3 w rho c.U
//   K = (a-beta)(1 - 1.5 u.u) + beta (1 - 1.5 V.V),   U = (a+beta) u + beta V + g.
//   beta = 0 (no solid): f*_q = (1-om) f_q + w rho om [1 - 1.5u.u + 4.5 (c.u)^2 + 3 c.(u + tau g)].
// The exchange vector is emitted through the identity sum_{i>=1} Omega_i c_i = rho (V - u) (P6).
#pragma once
#include "lbmimb_internal.cuh"

namespace lbmimb {

struct CollideParams {
  double omega;          // 1/tau
  double gx, gy, gz;     // g_fluid
  double tgx, tgy, tgz;  // tau * g_fluid
};

inline CollideParams make_collide_params(const lbmimb_lattice *h) {
  CollideParams c;
  c.omega = 1.0 / h->prm.tau;
  c.gx = h->prm.g_fluid[0];
  c.gy = h->prm.g_fluid[1];
  c.gz = h->g.dim == 3 ? h->prm.g_fluid[2] : 0.0;
  c.tgx = h->prm.tau * c.gx;
  c.tgy = h->prm.tau * c.gy;
  c.tgz = h->prm.tau * c.gz;
  return c;
}

template <int D>
__device__ __forceinline__ void moments(const double (&f)[Lat<D>::Q], double &rho, double &ux, double &uy,
                                        double &uz) {
  using L = Lat<D>;
  double r = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
#pragma unroll
  for (int q = 0; q < L::Q; ++q) {
    r += f[q];
    if (L::cx(q) == 1) mx += f[q];
    if (L::cx(q) == -1) mx -= f[q];
    if (L::cy(q) == 1) my += f[q];
    if (L::cy(q) == -1) my -= f[q];
    if (D == 3) {
      if (L::cz(q) == 1) mz += f[q];
      if (L::cz(q) == -1) mz -= f[q];
    }
  }
  const double inv = 1.0 / r;
  rho = r;
  ux = mx * inv;
  uy = my * inv;
  uz = D == 3 ? mz * inv : 0.0;
}

template <int D>
__device__ __forceinline__ double cdot(int q, double x, double y, double z) {
  using L = Lat<D>;
  double r = 0.0;
  bool first = true;
  if (L::cx(q) != 0) {
    r = L::cx(q) == 1 ? x : -x;
    first = false;
  }
  if (L::cy(q) != 0) {
    r = first ? (L::cy(q) == 1 ? y : -y) : (L::cy(q) == 1 ? r + y : r - y);
    first = false;
  }
  if (D == 3 && L::cz(q) != 0) {
    r = first ? (L::cz(q) == 1 ? z : -z) : (L::cz(q) == 1 ? r + z : r - z);
  }
  return r;
}

// pure LBGK + body force
template <int D>
__device__ __forceinline__ void collide_fluid(double (&f)[Lat<D>::Q], const CollideParams &c, double rho, double ux,
                                              double uy, double uz) {
  using L = Lat<D>;
  const double om = c.omega, omc = 1.0 - om;
  const double base = 1.0 - 1.5 * (ux * ux + uy * uy + uz * uz);
  const double ro = rho * om;
  const double upx = ux + c.tgx, upy = uy + c.tgy, upz = uz + c.tgz;
  f[0] = omc * f[0] + (L::w(0) * ro) * base;
#pragma unroll
  for (int q = 1; q < L::Q; q += 2) {
    const double cu = cdot<D>(q, ux, uy, uz);
    const double cup = cdot<D>(q, upx, upy, upz);
    const double wro = L::w(q) * ro;
    const double A = wro * fma(4.5 * cu, cu, base);
    const double B = (3.0 * wro) * cup;
    f[q] = fma(omc, f[q], A + B);
    f[q + 1] = fma(omc, f[q + 1], A - B);
  }
}

// immersed-moving-boundary node (also exact for beta = 0)
template <int D>
__device__ __forceinline__ void collide_imb(double (&f)[Lat<D>::Q], const CollideParams &c, double rho, double ux,
                                            double uy, double uz, double beta, double vx, double vy, double vz) {
  using L = Lat<D>;
  const double a = (1.0 - beta) * c.omega;
  const double c1 = 1.0 - a - beta;
  const double amb = a - beta, apb = a + beta;
  const double K = amb * (1.0 - 1.5 * (ux * ux + uy * uy + uz * uz)) + beta * (1.0 - 1.5 * (vx * vx + vy * vy + vz * vz));
  const double Ux = apb * ux + beta * vx + c.gx, Uy = apb * uy + beta * vy + c.gy, Uz = apb * uz + beta * vz + c.gz;
  const double amb45 = 4.5 * amb, b45 = 4.5 * beta;
  f[0] = (1.0 - a) * f[0] + (L::w(0) * rho) * K;
#pragma unroll
  for (int q = 1; q < L::Q; q += 2) {
    const double cu = cdot<D>(q, ux, uy, uz);
    const double cv = cdot<D>(q, vx, vy, vz);
    const double cU = cdot<D>(q, Ux, Uy, Uz);
    const double wr = L::w(q) * rho;
    const double E = wr * fma(amb45 * cu, cu, fma(b45 * cv, cv, K));
    const double O = (3.0 * wr) * cU;
    const double fp = f[q], fm = f[q + 1];
    f[q] = fma(c1, fp, fma(beta, fm, E + O));
    f[q + 1] = fma(c1, fm, fma(beta, fp, E - O));
  }
}

// Exchange vector of a covered node: one aligned record per node (16 B in 2D, 32 B = one DRAM
// sector in 3D) so that the store and the later gather of a3 move whole sectors.
template <int D>
__device__ __forceinline__ void store_exchange(double *__restrict__ s, int64_t x, double sx, double sy, double sz) {
  if (D == 2) {
    reinterpret_cast<double2 *>(s)[x] = make_double2(sx, sy);
  } else {
    double2 *p = reinterpret_cast<double2 *>(s) + 2 * x;
    p[0] = make_double2(sx, sy);
    p[1] = make_double2(sz, 0.0);
  }
}

// V_S = v_p + omega_p x (x_node - x_p), minimum image on periodic axes (R5); also returns the lever
// arm r = x_node - x_p of eq. (3)
template <int D>
__device__ __forceinline__ void solid_velocity(const double *__restrict__ pr, int i, int j, int k, int nx, int ny,
                                               int nz, int bcx, int bcy, int bcz, double &vx, double &vy, double &vz,
                                               double &rx, double &ry, double &rz) {
  auto mi = [](double d, int n) {
    const double hn = 0.5 * (double)n;
    if (d > hn) return d - (double)n;
    if (d < -hn) return d + (double)n;
    return d;
  };
  if (D == 2) {
    rx = (double)i - __ldg(pr + 0);
    ry = (double)j - __ldg(pr + 1);
    rz = 0.0;
    if (!bcx) rx = mi(rx, nx);
    if (!bcy) ry = mi(ry, ny);
    const double w = __ldg(pr + 4);
    vx = __ldg(pr + 2) - w * ry;
    vy = __ldg(pr + 3) + w * rx;
    vz = 0.0;
  } else {
    rx = (double)i - __ldg(pr + 0);
    ry = (double)j - __ldg(pr + 1);
    rz = (double)k - __ldg(pr + 2);
    if (!bcx) rx = mi(rx, nx);
    if (!bcy) ry = mi(ry, ny);
    if (!bcz) rz = mi(rz, nz);
    const double wx = __ldg(pr + 6), wy = __ldg(pr + 7), wz = __ldg(pr + 8);
    vx = __ldg(pr + 3) + (wy * rz - wz * ry);
    vy = __ldg(pr + 4) + (wz * rx - wx * rz);
    vz = __ldg(pr + 5) + (wx * ry - wy * rx);
  }
}

// ---------------------------------------------------------------------------
// a3 inside a2: F_p = -sum s_n, T_p = -sum r_n x s_n (eq. (3), sign of R6) summed while
// the step runs.  The lanes of a warp are consecutive nodes of one lattice row, so the nodes of a particle
// form runs of equal `key` (covering particle, -1 = not covered / not a node).  Each run is summed by a
// segmented shuffle tree (fixed shape => the fp64 partial sum of a run is reproducible), and the head lane of
// the run adds the partial sum to the particle's accumulators as 64-bit FIXED-POINT integers: integer
// addition is associative, so the total does not depend on the order in which warps arrive, and the
// reduction is bitwise reproducible without a second pass over the lattice.
//   value = hi 2^-40 + lo 2^-91: hi = rint(v 2^40), lo = rint((v - hi 2^-40) 2^91); the remainder is exact
//   and |lo| <= 2^50, so thousands of runs add without overflow and a sum resolves 2^-91 ~ 4e-28 (|v| < 2^11).
// A run lies in one lattice row, so the lever arm components r_y, r_z are the same on all its nodes and
//   sum r x s = (r_y S_z - r_z S_y,  r_z S_x - sum r_x s_z,  sum r_x s_y - r_y S_x),  S = sum s:
// five sums per run in 3D (three in 2D) instead of six, combined by the head lane.
// ---------------------------------------------------------------------------
// double -> integer without the (slow) conversion unit: for |x| < 2^51, x + 1.5 2^52 has the integer nearest to x in
// its low mantissa bits, and subtracting the constant again gives that integer back as a double, exactly.
__device__ __forceinline__ long long round_to_ll(double x, double &rounded) {
  constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52
  const double t = x + kMagic;
  rounded = t - kMagic;
  return __double_as_longlong(t) - __double_as_longlong(kMagic);
}

__device__ __forceinline__ void fixed_add(long long *acc, double v) {
  constexpr double k40 = 1099511627776.0, k52 = 4503599627370496.0;
  double hi_d, lo_d;
  const long long hi = round_to_ll(v * k40, hi_d);          // |v| < 2^11 (a force in lattice units)
  const double rem = v - hi_d * (1.0 / k40);                // exact, |rem| <= 2^-41
  const long long lo = round_to_ll((rem * k40) * (k52 * 0.5), lo_d);   // rem 2^91: |.| <= 2^50
  atomicAdd(reinterpret_cast<unsigned long long *>(acc), (unsigned long long)hi);
  if (lo != 0) atomicAdd(reinterpret_cast<unsigned long long *>(acc) + 1, (unsigned long long)lo);
}

__host__ __device__ __forceinline__ double fixed_value(long long hi, long long lo) {
  return (double)hi * (1.0 / 1099511627776.0) + ((double)lo * (2.0 / 4503599627370496.0)) * (1.0 / 1099511627776.0);
}

// Whole warp must call.  key < 0: this lane contributes nothing.  On return the FIRST lane of every run of equal
// keys holds the run's sums in v[NV] and the function returns true there (false on all other lanes).
template <int NV>
__device__ __forceinline__ bool reduce_runs(int key, double (&v)[NV]) {
  const unsigned lane = threadIdx.x & 31u;
  const int prev = __shfl_up_sync(0xffffffffu, key, 1);
  const bool boundary = key < 0 || lane == 0 || prev != key;       // first lane of a run (or an idle lane)
  const unsigned bmask = __ballot_sync(0xffffffffu, boundary);
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    // lanes lane+1 .. lane+d all continue this lane's run?
    const unsigned between = ((1u << d) - 1u) << 1;
    const bool take = lane + d < 32u && ((bmask >> lane) & between) == 0u;
    if (!__any_sync(0xffffffffu, take)) break;   // no run is longer than d: the remaining steps add nothing
#pragma unroll
    for (int c = 0; c < NV; ++c) {
      const double o = __shfl_down_sync(0xffffffffu, v[c], d);
      if (take) v[c] += o;
    }
  }
  return boundary && key >= 0;
}

}  // namespace lbmimb
