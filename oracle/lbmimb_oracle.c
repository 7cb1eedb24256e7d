/*
 * oracle/lbmimb_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU restatement (fp64) of the hot path of
 * arxiv/paper_1011_2613 ("Large-Scale DNS of Gas-Solid Flow on Mole-8.5"):
 * LBGK D2Q9/D3Q19 collide-and-stream with the Noble-Torczynski immersed moving
 * boundary term (eq. (1), :41 beta, :43 eq. (2)), the hydrodynamic
 * force/torque sums (eq. (3)), sub-cell sampling of the solid
 * fraction (definition of eps) and the frictionless soft-sphere
 * DEM (eq. (4)-(5)).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference leg may build, load or call this file.  It shares no code, header,
 * table or helper with paper_1011_2613_b200/csrc (the CUDA product path) and
 * the product never calls it.
 *
 * Style: one node at a time, two buffers (read t, write t+1), literal sums in
 * the paper's order and notation, no blocking / fusion / reordering.  The only
 * parallelism is "#pragma omp parallel for" on an outermost loop whose
 * iterations write disjoint outputs.  Compile with -O2 -ffp-contract=off so
 * that no FMA contraction happens (the inside test of orc_map must round the
 * same way as the CUDA path's __dmul_rn/__dadd_rn chain: DESIGN.md R4).
 *
 * Readings of the paper where it is silent or garbled are those of DESIGN.md
 * section "Readings" (R1..R16 = SURVEY.md section 8(c) G1..G16).
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned by at
 * least one closed form / invariant / hand value, EXCEPT the convention
 *   - orc_map's choice of the covering particle when two particles share a node
 *     (R5: most samples, ties -> lowest index): "parity unpinned" (convention;
 *     brute-forced on tiny inputs only).
 * The wall contact of contact_forces (R10) is pinned by the static equilibrium of
 * a sphere resting on the lower / upper wall (x = R - 1/2 - m|g|/k_n and its
 * mirror) and by the first-contact law at all four walls of a 2D box
 * (test_R10_*); the order of a coupled step (R11: map -> step -> forces -> DEM,
 * load from the pre-collision state, held over the DEM step) lives in
 * oracle/__init__.py: coupled_step and is pinned by two hand-derived steps of a
 * light particle in a uniform stream (test_R11_*).
 * Precision: everything is fp64 except the exchange vector s of a node and the
 * per-particle sums of orc_forces, which are formed in long double and rounded
 * once (R12: the literal sum_i Omega_i c_i cancels f-sized terms; see
 * orc_collide_node).
 * The Verlet-list functions (orc_verlet_*, orc_dem_step_verlet, R19)
 * are pinned in tests/test_oracle_verlet_pins.py (hand lists, lattice shell
 * counts, bitwise equality with the all-pairs trajectory, rebuild counts).
 * The table look-up of the solid fraction (orc_eps_table, orc_map_table;
 * PAPER.md:71-77, R17) is pinned in tests/test_oracle_table_pins.py (quadrature
 * of the covered area / volume, symmetries, agreement with a fine sampled map).
 * The suspension diagnostics (orc_diagnostics, R18) are pinned in
 * tests/test_oracle_diag_pins.py (closed forms, exact rationals, momentum
 * conservation); the averaging convention itself (which weights define the
 * "area-averaged" velocities) is "parity unpinned": the paper prints no formula.
 * The whole IMB term is checked physically by the drag of a periodic array
 * against Hasimoto's series (test_P16_...).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------ */
/* Velocity sets (R1).  PAPER.md:35 names D2Q9 / D3Q19 and defers to a      */
/* reference; the standard sets are used, c_s^2 = 1/3.  Opposite of odd i   */
/* is i+1.                                                                   */
/* ------------------------------------------------------------------------ */
static const int C_D2Q9[9][3] = {
    {0, 0, 0},  {1, 0, 0},  {-1, 0, 0}, {0, 1, 0},  {0, -1, 0},
    {1, 1, 0},  {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0}};
static const double W_D2Q9[9] = {4.0 / 9.0,  1.0 / 9.0,  1.0 / 9.0,
                                 1.0 / 9.0,  1.0 / 9.0,  1.0 / 36.0,
                                 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};
static const int C_D3Q19[19][3] = {
    {0, 0, 0},  {1, 0, 0},   {-1, 0, 0}, {0, 1, 0},   {0, -1, 0},
    {0, 0, 1},  {0, 0, -1},  {1, 1, 0},  {-1, -1, 0}, {1, -1, 0},
    {-1, 1, 0}, {1, 0, 1},   {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
    {0, 1, 1},  {0, -1, -1}, {0, 1, -1}, {0, -1, 1}};
static const double W_D3Q19[19] = {
    1.0 / 3.0,  1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0,
    1.0 / 18.0, 1.0 / 18.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};

static int nq(int dim) { return dim == 2 ? 9 : 19; }
static const int *cvec(int dim, int i) {
  return dim == 2 ? C_D2Q9[i] : C_D3Q19[i];
}
static double wgt(int dim, int i) { return dim == 2 ? W_D2Q9[i] : W_D3Q19[i]; }
static int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }

/* Exposes the tables so that tests can check sum w = 1, sum w c c = I/3 ... */
void orc_velocity_set(int dim, int *c_out /*[Q][3]*/, double *w_out /*[Q]*/,
                      int *opp_out /*[Q]*/) {
  int Q = nq(dim);
  for (int i = 0; i < Q; ++i) {
    for (int a = 0; a < 3; ++a) c_out[3 * i + a] = cvec(dim, i)[a];
    w_out[i] = wgt(dim, i);
    opp_out[i] = opp(i);
  }
}

/* f_i^eq(rho,u) = w_i rho (1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u)   (R1) */
static double feq_i(int dim, int i, double rho, const double *u) {
  const int *c = cvec(dim, i);
  double cu = 0.0, uu = 0.0;
  for (int a = 0; a < dim; ++a) {
    cu += c[a] * u[a];
    uu += u[a] * u[a];
  }
  return wgt(dim, i) * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

/* the same expression in long double (used only for the exchange vector s of
 * orc_collide_node, see there) */
static long double wgt_ld(int dim, int i) { /* the weights of R1 as long double quotients */
  if (dim == 2) return i == 0 ? 4.0L / 9.0L : (i < 5 ? 1.0L / 9.0L : 1.0L / 36.0L);
  return i == 0 ? 1.0L / 3.0L : (i < 7 ? 1.0L / 18.0L : 1.0L / 36.0L);
}
static long double feq_i_ld(int dim, int i, long double rho, const long double *u) {
  const int *c = cvec(dim, i);
  long double cu = 0.0L, uu = 0.0L;
  for (int a = 0; a < dim; ++a) {
    cu += c[a] * u[a];
    uu += u[a] * u[a];
  }
  return wgt_ld(dim, i) * rho * (1.0L + 3.0L * cu + 4.5L * cu * cu - 1.5L * uu);
}

void orc_feq(int dim, double rho, const double *u, double *out /*[Q]*/) {
  int Q = nq(dim);
  for (int i = 0; i < Q; ++i) out[i] = feq_i(dim, i, rho, u);
}

/* beta = eps (tau - 1/2) / ((1 - eps) + (tau - 1/2)) */
double orc_beta(double eps, double tau) {
  return eps * (tau - 0.5) / ((1.0 - eps) + (tau - 0.5));
}

/*
 * One node of eq. (1), before streaming.
 *   rho = sum_i f_i, u = (sum_i f_i c_i)/rho                 (bare u: R2)
 *   Omega_i = f_{-i} - f_i + f_i^eq(rho,V_S) - f_{-i}^eq(rho,u)  eq. (2)
 *   F_i = 3 w_i rho (c_i . g)                                (R3)
 *   f*_i = f_i - (1-beta)(f_i - f_i^eq(rho,u))/tau + beta Omega_i + F_i
 *   s = beta sum_{i>=1} Omega_i c_i     (the bracket of eq. (3), R7)
 * beta = 0 => Omega and s are zero (eps = 0 nodes).
 */
void orc_collide_node(int dim, double tau, const double *g /*[3]*/,
                      const double *f /*[Q]*/, double beta,
                      const double *vs /*[3]*/, double *fstar /*[Q]*/,
                      double *s /*[3]*/, double *rho_out, double *u_out /*[3]*/) {
  int Q = nq(dim);
  double rho = 0.0, m[3] = {0.0, 0.0, 0.0}, u[3] = {0.0, 0.0, 0.0};
  for (int i = 0; i < Q; ++i) rho += f[i];
  for (int i = 0; i < Q; ++i)
    for (int a = 0; a < dim; ++a) m[a] += f[i] * cvec(dim, i)[a];
  for (int a = 0; a < dim; ++a) u[a] = m[a] / rho;

  double omega[19];
  for (int i = 0; i < Q; ++i) {
    if (beta != 0.0)
      omega[i] = f[opp(i)] - f[i] + feq_i(dim, i, rho, vs) -
                 feq_i(dim, opp(i), rho, u);
    else
      omega[i] = 0.0;
  }
  /* s = beta sum_{i>=1} Omega_i c_i, the literal sum, evaluated in long double:
   * the sum cancels f-sized terms (|f| <= 0.45) down to rho (V_S - u), so in
   * fp64 every node's s would carry an absolute rounding error of ~Q 2^-53 |f|
   * ~ 1e-15 however small s is, which is 1e-10 of s itself on slowly moving
   * nodes: not good enough to referee a 1e-10 relative force tolerance
   * (R12).  rho and u are re-formed in long double from the same fp64
   * f, Omega_i from them; the result is rounded once to fp64.  f* above/below
   * keeps the paper's double precision. */
  s[0] = s[1] = s[2] = 0.0;
  if (beta != 0.0) {
    long double rl = 0.0L, ml[3] = {0.0L, 0.0L, 0.0L}, ul[3] = {0.0L, 0.0L, 0.0L};
    long double vl[3] = {vs[0], vs[1], vs[2]}, sl[3] = {0.0L, 0.0L, 0.0L};
    for (int i = 0; i < Q; ++i) rl += (long double)f[i];
    for (int i = 0; i < Q; ++i)
      for (int a = 0; a < dim; ++a) ml[a] += (long double)f[i] * cvec(dim, i)[a];
    for (int a = 0; a < dim; ++a) ul[a] = ml[a] / rl;
    for (int i = 1; i < Q; ++i) {
      long double om = (long double)f[opp(i)] - (long double)f[i] +
                       feq_i_ld(dim, i, rl, vl) - feq_i_ld(dim, opp(i), rl, ul);
      for (int a = 0; a < dim; ++a) sl[a] += om * cvec(dim, i)[a];
    }
    for (int a = 0; a < dim; ++a) s[a] = (double)((long double)beta * sl[a]);
  }

  for (int i = 0; i < Q; ++i) {
    const int *c = cvec(dim, i);
    double cg = 0.0;
    for (int a = 0; a < dim; ++a) cg += c[a] * g[a];
    double Fi = 3.0 * wgt(dim, i) * rho * cg;
    fstar[i] = f[i] - (1.0 - beta) * (f[i] - feq_i(dim, i, rho, u)) / tau +
               beta * omega[i] + Fi;
  }
  *rho_out = rho;
  for (int a = 0; a < 3; ++a) u_out[a] = u[a];
}

/* a0: f_i = f_i^eq(rho=1,u=0) = w_i on every node; layout f[q][k][j][i]. */
void orc_init(int dim, int64_t N, double *f) {
  int Q = nq(dim);
  for (int i = 0; i < Q; ++i)
    for (int64_t x = 0; x < N; ++x) f[(int64_t)i * N + x] = wgt(dim, i);
}

/* rho and bare u of every node (R2), u layout [dim][N]. */
void orc_macros(int dim, int64_t N, const double *f, double *rho_out,
                double *u_out) {
  int Q = nq(dim);
#pragma omp parallel for
  for (int64_t x = 0; x < N; ++x) {
    double rho = 0.0, m[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < Q; ++i) rho += f[(int64_t)i * N + x];
    for (int i = 0; i < Q; ++i)
      for (int a = 0; a < dim; ++a)
        m[a] += f[(int64_t)i * N + x] * cvec(dim, i)[a];
    rho_out[x] = rho;
    for (int a = 0; a < dim; ++a) u_out[(int64_t)a * N + x] = m[a] / rho;
  }
}

/* minimum image of a separation along a periodic axis of n nodes */
static double min_image(double d, int64_t n) {
  if (d > 0.5 * (double)n) return d - (double)n;
  if (d < -0.5 * (double)n) return d + (double)n;
  return d;
}

static int64_t wrap(int64_t i, int64_t n) {
  i %= n;
  return i < 0 ? i + n : i;
}

/*
 * a1: sub-cell sampling of the solid fraction (eps = area/volume
 * of the cell covered by solid; R4).  For every particle, every node of its
 * bounding box [floor(c-R)-1, ceil(c+R)+1]^D (wrapped in periodic axes,
 * clipped at walls), every sample point p = x_node + ((a+1/2)/S - 1/2):
 *   inside <=> dx*dx + dy*dy (+ dz*dz) <= R*R   (left to right, no FMA),
 * d = p - c reduced by minimum image in periodic axes.  A sample inside
 * several particles counts once.  eps_cnt = number of inside samples,
 * pid = particle with most samples in that cell, ties -> lowest index (R5).
 * Returns 0, or -1 if S^D > 255 or out of memory.
 */
int orc_map(int dim, const int64_t *n, const int32_t *bc, int S, int64_t P,
            const double *pos /*[dim][P]*/, const double *radius,
            uint8_t *eps_cnt /*[N]*/, int32_t *pid /*[N]*/) {
  int64_t nx = n[0], ny = n[1], nz = dim == 3 ? n[2] : 1;
  int64_t N = nx * ny * nz;
  int SD = dim == 2 ? S * S : S * S * S;
  if (SD > 255) return -1;
  int words = (SD + 63) / 64;
  uint64_t *mask = (uint64_t *)calloc((size_t)N * words, sizeof(uint64_t));
  uint8_t *best = (uint8_t *)calloc((size_t)N, 1);
  if (!mask || !best) {
    free(mask);
    free(best);
    return -1;
  }
  for (int64_t x = 0; x < N; ++x) pid[x] = -1;

  for (int64_t p = 0; p < P; ++p) {
    double c[3] = {pos[p], pos[P + p], dim == 3 ? pos[2 * P + p] : 0.0};
    double R = radius[p];
    int64_t lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (int a = 0; a < dim; ++a) {
      lo[a] = (int64_t)floor(c[a] - R) - 1;
      hi[a] = (int64_t)ceil(c[a] + R) + 1;
      if (bc[a] != 0) {
        if (lo[a] < 0) lo[a] = 0;
        if (hi[a] > n[a] - 1) hi[a] = n[a] - 1;
      }
    }
    for (int64_t kk = lo[2]; kk <= hi[2]; ++kk)
      for (int64_t jj = lo[1]; jj <= hi[1]; ++jj)
        for (int64_t ii = lo[0]; ii <= hi[0]; ++ii) {
          int64_t i = bc[0] == 0 ? wrap(ii, nx) : ii;
          int64_t j = bc[1] == 0 ? wrap(jj, ny) : jj;
          int64_t k = dim == 3 ? (bc[2] == 0 ? wrap(kk, nz) : kk) : 0;
          int64_t node = (k * ny + j) * nx + i;
          uint64_t m[4] = {0, 0, 0, 0};
          int cnt = 0;
          int Sz = dim == 3 ? S : 1;
          for (int az = 0; az < Sz; ++az)
            for (int ay = 0; ay < S; ++ay)
              for (int ax = 0; ax < S; ++ax) {
                double px = (double)i + (((double)ax + 0.5) / (double)S - 0.5);
                double py = (double)j + (((double)ay + 0.5) / (double)S - 0.5);
                double dx = px - c[0];
                double dy = py - c[1];
                if (bc[0] == 0) dx = min_image(dx, nx);
                if (bc[1] == 0) dy = min_image(dy, ny);
                double d2 = dx * dx + dy * dy;
                if (dim == 3) {
                  double pz =
                      (double)k + (((double)az + 0.5) / (double)S - 0.5);
                  double dz = pz - c[2];
                  if (bc[2] == 0) dz = min_image(dz, nz);
                  d2 = d2 + dz * dz;
                }
                if (d2 <= R * R) {
                  int bit = (az * S + ay) * S + ax;
                  m[bit >> 6] |= (uint64_t)1 << (bit & 63);
                  ++cnt;
                }
              }
          if (cnt > 0) {
            for (int w = 0; w < words; ++w) mask[node * words + w] |= m[w];
            if (cnt > best[node]) { /* strict: ties keep the lower index */
              best[node] = (uint8_t)cnt;
              pid[node] = (int32_t)p;
            }
          }
        }
  }
  for (int64_t x = 0; x < N; ++x) {
    int cnt = 0;
    for (int w = 0; w < words; ++w)
      cnt += __builtin_popcountll(mask[x * words + w]);
    eps_cnt[x] = (uint8_t)cnt;
  }
  free(mask);
  free(best);
  return 0;
}

/* ------------------------------------------------------------------------ */
/* NEXT-1: the paper's own eps method, table look-up gamma = phi(d, theta)    */
/* (eq. (6); Fig. 1 is missing, so the discretisation is the  */
/* reading R17 of DESIGN.md).  "For a lattice and a solid particle with a     */
/* given radius, gamma can be determined by two factors: the distance between */
/* the lattice and the origin of the solid particle d, and the orientation of */
/* the lattice to the solid particle theta"; gamma "is pre-calculated".       */
/*                                                                            */
/* R17.  w = sqrt(D)/2 (half diagonal of a cell), d0 = R - w, dd = sqrt(D)/Nd.*/
/* The orientation is kept as the ratios of the sorted absolute components of */
/* the displacement, a >= b >= c: t1 = b/a (= tan theta in 2D), t2 = c/a, so  */
/* that no transcendental function enters an index.  Entry (k, m1[, m2]):     */
/*   d_k = d0 + (k + 1/2) dd,  t1 = (m1 + 1/2)/Nt,  t2 = (m2 + 1/2)/Nt,       */
/*   r = d_k (1, t1, t2)/sqrt(1 + t1^2 + t2^2)  (cell centre relative to the  */
/*   particle centre), n = number of the St^D sub-cell points of that cell    */
/*   inside the particle (same point set and inside test as R4),              */
/*   code = (255 n + St^D/2) / St^D  (integer; gamma = code/255).             */
/* Returns 0, -1 on bad arguments (R < 1, sizes).                             */
/* ------------------------------------------------------------------------ */
int orc_eps_table(int dim, double R, int Nd, int Nt, int St,
                  uint8_t *table /*[Nd][Nt] (2D) or [Nd][Nt][Nt] (3D)*/) {
  if (!(R >= 1.0) || Nd < 1 || Nt < 1 || St < 1 || (dim != 2 && dim != 3))
    return -1;
  double sqD = sqrt((double)dim);
  double d0 = R - 0.5 * sqD;
  double dd = sqD / (double)Nd;
  int64_t total = dim == 2 ? (int64_t)St * St : (int64_t)St * St * St;
  int Nt2 = dim == 3 ? Nt : 1;
#pragma omp parallel for
  for (int k = 0; k < Nd; ++k)
    for (int m1 = 0; m1 < Nt; ++m1)
      for (int m2 = 0; m2 < Nt2; ++m2) {
        double dk = d0 + ((double)k + 0.5) * dd;
        double t1 = ((double)m1 + 0.5) / (double)Nt;
        double t2 = dim == 3 ? ((double)m2 + 0.5) / (double)Nt : 0.0;
        double nrm = dim == 3 ? sqrt((1.0 + t1 * t1) + t2 * t2) : sqrt(1.0 + t1 * t1);
        double rx = dk / nrm;
        double ry = rx * t1;
        double rz = rx * t2;
        int64_t n = 0;
        int Sz = dim == 3 ? St : 1;
        for (int az = 0; az < Sz; ++az)
          for (int ay = 0; ay < St; ++ay)
            for (int ax = 0; ax < St; ++ax) {
              double px = rx + (((double)ax + 0.5) / (double)St - 0.5);
              double py = ry + (((double)ay + 0.5) / (double)St - 0.5);
              double d2 = px * px + py * py;
              if (dim == 3) {
                double pz = rz + (((double)az + 0.5) / (double)St - 0.5);
                d2 = d2 + pz * pz;
              }
              if (d2 <= R * R) ++n;
            }
        table[((int64_t)k * Nt + m1) * Nt2 + m2] =
            (uint8_t)((255 * n + total / 2) / total);
      }
  return 0;
}

/* Look-up of one node: displacement delta = x_node - c (already reduced by
 * minimum image).  d = sqrt(dx*dx + dy*dy (+ dz*dz)) left to right;
 * d < d0 -> 255; k = (int)((d - d0) * (Nd / sqrt(D))), k >= Nd -> 0;
 * m = min((int)(t * Nt), Nt - 1) with t1 = b/a, t2 = c/a of the sorted
 * absolute components a >= b >= c. */
static int table_lookup(int dim, double R, int Nd, int Nt, const uint8_t *table,
                        const double *delta) {
  double sqD = sqrt((double)dim);
  double d0 = R - 0.5 * sqD;
  double inv_dd = (double)Nd / sqD;
  double d2 = delta[0] * delta[0] + delta[1] * delta[1];
  if (dim == 3) d2 = d2 + delta[2] * delta[2];
  double d = sqrt(d2);
  if (d < d0) return 255;
  double u = (d - d0) * inv_dd;
  if (u >= (double)Nd) return 0;
  int k = (int)u;
  double a = fabs(delta[0]), b = fabs(delta[1]), c = dim == 3 ? fabs(delta[2]) : 0.0;
  double t;
  if (a < b) { t = a; a = b; b = t; }
  if (dim == 3) {
    if (b < c) { t = b; b = c; c = t; }
    if (a < b) { t = a; a = b; b = t; }
  }
  int m1 = (int)((b / a) * (double)Nt);
  if (m1 > Nt - 1) m1 = Nt - 1;
  int m2 = 0, Nt2 = 1;
  if (dim == 3) {
    Nt2 = Nt;
    m2 = (int)((c / a) * (double)Nt);
    if (m2 > Nt - 1) m2 = Nt - 1;
  }
  return table[((int64_t)k * Nt + m1) * Nt2 + m2];
}

/*
 * a1 in table mode: for every particle, every node of its bounding box (same
 * box as orc_map), code_p = look-up of the node's displacement.  Node result:
 * eps_code = min(255, sum_p code_p) (non-overlapping particles cover disjoint
 * parts of a cell, so their fractions add), pid = particle with the largest
 * code, ties -> lowest index (R5), -1 if the sum is 0.  All particles must
 * have the same radius ("a solid particle with a given radius").
 * Returns 0, -1 bad arguments / out of memory, -2 radii differ.
 */
int orc_map_table(int dim, const int64_t *n, const int32_t *bc, int Nd, int Nt,
                  const uint8_t *table /* orc_eps_table(dim, radius[0], Nd, Nt, .) */,
                  int64_t P, const double *pos, const double *radius,
                  uint8_t *eps_code /*[N]*/, int32_t *pid /*[N]*/) {
  int64_t nx = n[0], ny = n[1], nz = dim == 3 ? n[2] : 1;
  int64_t N = nx * ny * nz;
  for (int64_t x = 0; x < N; ++x) {
    eps_code[x] = 0;
    pid[x] = -1;
  }
  if (P == 0) return 0;
  double R = radius[0];
  for (int64_t p = 1; p < P; ++p)
    if (radius[p] != R) return -2;
  uint8_t *best = (uint8_t *)calloc((size_t)N, 1);
  int32_t *sum = (int32_t *)calloc((size_t)N, sizeof(int32_t));
  if (!best || !sum || !(R >= 1.0)) {
    free(best);
    free(sum);
    return -1;
  }
  for (int64_t p = 0; p < P; ++p) {
    double c[3] = {pos[p], pos[P + p], dim == 3 ? pos[2 * P + p] : 0.0};
    int64_t lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (int a = 0; a < dim; ++a) {
      lo[a] = (int64_t)floor(c[a] - R) - 1;
      hi[a] = (int64_t)ceil(c[a] + R) + 1;
      if (bc[a] != 0) {
        if (lo[a] < 0) lo[a] = 0;
        if (hi[a] > n[a] - 1) hi[a] = n[a] - 1;
      } else if (hi[a] - lo[a] + 1 > n[a]) { /* box wider than the axis: every node once */
        lo[a] = 0;
        hi[a] = n[a] - 1;
      }
    }
    for (int64_t kk = lo[2]; kk <= hi[2]; ++kk)
      for (int64_t jj = lo[1]; jj <= hi[1]; ++jj)
        for (int64_t ii = lo[0]; ii <= hi[0]; ++ii) {
          int64_t i = bc[0] == 0 ? wrap(ii, nx) : ii;
          int64_t j = bc[1] == 0 ? wrap(jj, ny) : jj;
          int64_t k = dim == 3 ? (bc[2] == 0 ? wrap(kk, nz) : kk) : 0;
          int64_t node = (k * ny + j) * nx + i;
          double delta[3] = {(double)i - c[0], (double)j - c[1],
                             dim == 3 ? (double)k - c[2] : 0.0};
          for (int a = 0; a < dim; ++a)
            if (bc[a] == 0) delta[a] = min_image(delta[a], n[a]);
          int code = table_lookup(dim, R, Nd, Nt, table, delta);
          if (code > 0) {
            sum[node] += code;
            if (code > best[node]) { /* strict: ties keep the lower index */
              best[node] = (uint8_t)code;
              pid[node] = (int32_t)p;
            }
          }
        }
  }
  for (int64_t x = 0; x < N; ++x) eps_code[x] = (uint8_t)(sum[x] > 255 ? 255 : sum[x]);
  free(best);
  free(sum);
  return 0;
}

/*
 * a2: one time step of eq. (1) on the whole lattice, f_in (time t) ->
 * f_out (time t+1).  Collision per node (orc_collide_node), then streaming:
 * target y = x + c_i; periodic axes wrap; if y leaves the domain through a
 * wall axis, half-way bounce-back: f_out[x][-i] = f*_i(x) (R15), else
 * f_out[y][i] = f*_i(x).  On eps>0 nodes V_S = v_p + omega_p x (x - x_p)
 * (minimum image; R5) with p = pid[x]; the node's exchange vector s is stored
 * to s_out[dim][N] when s_out != NULL (zero on eps = 0 nodes).  eps =
 * eps_cnt[x] / eps_den with eps_den = S^D for the sampled map (orc_map) and
 * 255 for the table map (orc_map_table).
 */
void orc_step(int dim, const int64_t *n, const int32_t *bc, double tau,
              const double *g, int eps_den, const double *f_in, double *f_out,
              const uint8_t *eps_cnt, const int32_t *pid, int64_t P,
              const double *pos, const double *vel, const double *omega,
              double *s_out) {
  int Q = nq(dim);
  int64_t nx = n[0], ny = n[1], nz = dim == 3 ? n[2] : 1;
  int64_t N = nx * ny * nz;
  double SD = (double)eps_den; /* eps = eps_cnt / eps_den: S^D (sampling, R4) or 255 (table, R17) */
#pragma omp parallel for
  for (int64_t k = 0; k < nz; ++k)
    for (int64_t j = 0; j < ny; ++j)
      for (int64_t i = 0; i < nx; ++i) {
        int64_t x = (k * ny + j) * nx + i;
        double f[19], fstar[19], s[3], rho, u[3];
        double vs[3] = {0.0, 0.0, 0.0}, beta = 0.0;
        for (int q = 0; q < Q; ++q) f[q] = f_in[(int64_t)q * N + x];
        if (eps_cnt != NULL && eps_cnt[x] > 0) {
          int64_t p = pid[x];
          double eps = (double)eps_cnt[x] / SD;
          beta = orc_beta(eps, tau);
          double r[3] = {0.0, 0.0, 0.0};
          r[0] = (double)i - pos[p];
          r[1] = (double)j - pos[P + p];
          if (dim == 3) r[2] = (double)k - pos[2 * P + p];
          for (int a = 0; a < dim; ++a)
            if (bc[a] == 0) r[a] = min_image(r[a], n[a]);
          if (dim == 2) {
            double w = omega[p];
            vs[0] = vel[p] - w * r[1];
            vs[1] = vel[P + p] + w * r[0];
          } else {
            double wx = omega[p], wy = omega[P + p], wz = omega[2 * P + p];
            vs[0] = vel[p] + (wy * r[2] - wz * r[1]);
            vs[1] = vel[P + p] + (wz * r[0] - wx * r[2]);
            vs[2] = vel[2 * P + p] + (wx * r[1] - wy * r[0]);
          }
        }
        orc_collide_node(dim, tau, g, f, beta, vs, fstar, s, &rho, u);
        if (s_out != NULL)
          for (int a = 0; a < dim; ++a) s_out[(int64_t)a * N + x] = s[a];
        for (int q = 0; q < Q; ++q) {
          const int *c = cvec(dim, q);
          int64_t t[3] = {i + c[0], j + c[1], k + c[2]};
          int bounced = 0;
          for (int a = 0; a < dim; ++a) {
            if (t[a] < 0 || t[a] >= n[a]) {
              if (bc[a] == 0)
                t[a] = wrap(t[a], n[a]);
              else
                bounced = 1;
            }
          }
          if (bounced)
            f_out[(int64_t)opp(q) * N + x] = fstar[q];
          else
            f_out[(int64_t)q * N + (t[2] * ny + t[1]) * nx + t[0]] = fstar[q];
        }
      }
}

/*
 * a3: literal eq. (3), over the nodes with pid = p, with the
 * sign of R6: the printed sum is the momentum the FLUID gains per step, the
 * force ON THE PARTICLE is its negative.  h^D/dt = 1 (R7).
 *   F_p = - sum_n s_n,   T_p = - sum_n (x_n - x_p) x s_n   (minimum image)
 * torque layout: [1][P] in 2D (z component), [3][P] in 3D.
 * abs_f[p] = sum_n |s_n|, abs_t[p] = sum_n |r_n x s_n| (tolerance scale, R12).
 */
void orc_forces(int dim, const int64_t *n, const int32_t *bc, const double *s,
                const int32_t *pid, int64_t P, const double *pos, double *force,
                double *torque, double *abs_f, double *abs_t) {
  int64_t nx = n[0], ny = n[1], nz = dim == 3 ? n[2] : 1;
  int64_t N = nx * ny * nz;
  int nt = dim == 2 ? 1 : 3;
  /* the per-particle sums are accumulated in long double and rounded once (R12: the
   * oracle must be well inside the 1e-10 relative tolerance it referees) */
  long double *Fl = (long double *)calloc((size_t)(P > 0 ? P : 1) * 6, sizeof(long double));
  long double *Tl = Fl + (size_t)(P > 0 ? P : 1) * 3;
  for (int64_t p = 0; p < P * dim; ++p) force[p] = 0.0;
  for (int64_t p = 0; p < P * nt; ++p) torque[p] = 0.0;
  for (int64_t p = 0; p < P; ++p) abs_f[p] = abs_t[p] = 0.0;
  if (!Fl) return;
  for (int64_t k = 0; k < nz; ++k)
    for (int64_t j = 0; j < ny; ++j)
      for (int64_t i = 0; i < nx; ++i) {
        int64_t x = (k * ny + j) * nx + i;
        int64_t p = pid[x];
        if (p < 0) continue;
        double sv[3] = {0.0, 0.0, 0.0}, r[3] = {0.0, 0.0, 0.0};
        for (int a = 0; a < dim; ++a) sv[a] = s[(int64_t)a * N + x];
        r[0] = (double)i - pos[p];
        r[1] = (double)j - pos[P + p];
        if (dim == 3) r[2] = (double)k - pos[2 * P + p];
        for (int a = 0; a < dim; ++a)
          if (bc[a] == 0) r[a] = min_image(r[a], n[a]);
        for (int a = 0; a < dim; ++a) Fl[(int64_t)a * P + p] -= (long double)sv[a];
        long double tl[3];
        tl[0] = (long double)r[1] * sv[2] - (long double)r[2] * sv[1];
        tl[1] = (long double)r[2] * sv[0] - (long double)r[0] * sv[2];
        tl[2] = (long double)r[0] * sv[1] - (long double)r[1] * sv[0];
        double t[3] = {(double)tl[0], (double)tl[1], (double)tl[2]};
        if (dim == 2) {
          Tl[p] -= tl[2];
          abs_t[p] += fabs(t[2]);
        } else {
          for (int a = 0; a < 3; ++a) Tl[(int64_t)a * P + p] -= tl[a];
          abs_t[p] += sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
        }
        abs_f[p] += sqrt(sv[0] * sv[0] + sv[1] * sv[1] + sv[2] * sv[2]);
      }
  for (int64_t p = 0; p < P * dim; ++p) force[p] = (double)Fl[p];
  for (int64_t p = 0; p < P * nt; ++p) torque[p] = (double)Tl[p];
  free(Fl);
}

/* ------------------------------------------------------------------------ */
/* DEM, eq. (4)-(5), readings R8-R11.                          */
/* ------------------------------------------------------------------------ */

/* The printed "eta_n" has units of time: it is the contact
 * duration t_c = sqrt((pi^2 + ln^2 e) m_eff / k_n) (R9). */
double orc_contact_duration(double kn, double e, double mi, double mj) {
  double meff = mi * mj / (mi + mj);
  double le = log(e);
  return sqrt((M_PI * M_PI + le * le) * meff / kn);
}

/* Damping coefficient of the linear spring-dashpot that gives restitution e:
 * eta_n = -2 ln(e) sqrt(k_n m_eff / (pi^2 + ln^2 e))  (R9). */
double orc_damping(double kn, double e, double meff) {
  double le = log(e);
  return -2.0 * le * sqrt(kn * meff / (M_PI * M_PI + le * le));
}

/*
 * Contact forces on every particle for positions x and velocities v (R8, R10):
 *   delta = (R_i + R_j) - |r_i - r_j|, contact iff delta > 0,
 *   F_ij = k_n delta n_ij - eta_n (v_ij . n_ij) n_ij, n_ij = (r_i - r_j)/|r_i - r_j|
 * (minimum image), v_ij = v_i - v_j, no clamp, no friction, no torque.
 * Walls of a wall axis are the planes at -1/2 and n-1/2: same law with
 * m_eff = m_i, R_j = 0, v_j = 0.
 * Brute force over all pairs j != i in ascending j (the definition).
 */
static void contact_forces(int dim, const int64_t *n, const int32_t *bc,
                           int64_t P, const double *x, const double *v,
                           const double *radius, const double *mass, double kn,
                           double e, double *fc /*[dim][P]*/) {
#pragma omp parallel for
  for (int64_t i = 0; i < P; ++i) {
    double F[3] = {0.0, 0.0, 0.0};
    for (int64_t j = 0; j < P; ++j) {
      if (j == i) continue;
      double d[3] = {0.0, 0.0, 0.0}, dist2 = 0.0;
      for (int a = 0; a < dim; ++a) {
        d[a] = x[(int64_t)a * P + i] - x[(int64_t)a * P + j];
        if (bc[a] == 0) d[a] = min_image(d[a], n[a]);
        dist2 += d[a] * d[a];
      }
      double Rs = radius[i] + radius[j];
      if (dist2 >= Rs * Rs) continue;
      double dist = sqrt(dist2);
      double delta = Rs - dist;
      if (!(delta > 0.0)) continue;
      double meff = mass[i] * mass[j] / (mass[i] + mass[j]);
      double eta = orc_damping(kn, e, meff);
      double nrm[3], vn = 0.0;
      for (int a = 0; a < dim; ++a) {
        nrm[a] = d[a] / dist;
        vn += (v[(int64_t)a * P + i] - v[(int64_t)a * P + j]) * nrm[a];
      }
      for (int a = 0; a < dim; ++a)
        F[a] += kn * delta * nrm[a] - eta * vn * nrm[a];
    }
    for (int a = 0; a < dim; ++a) {
      if (bc[a] == 0) continue;
      double eta = orc_damping(kn, e, mass[i]);
      double xa = x[(int64_t)a * P + i], va = v[(int64_t)a * P + i];
      /* lower wall, plane at -1/2, normal +1 */
      double delta = radius[i] - (xa + 0.5);
      if (delta > 0.0) F[a] += kn * delta * 1.0 - eta * (va * 1.0) * 1.0;
      /* upper wall, plane at n-1/2, normal -1 */
      delta = radius[i] - (((double)n[a] - 0.5) - xa);
      if (delta > 0.0) F[a] += kn * delta * (-1.0) - eta * (va * -1.0) * (-1.0);
    }
    for (int a = 0; a < dim; ++a) fc[(int64_t)a * P + i] = F[a];
  }
}

void orc_contact_forces(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                        const double *x, const double *v, const double *radius,
                        const double *mass, double kn, double e, double *fc) {
  contact_forces(dim, n, bc, P, x, v, radius, mass, kn, e, fc);
}

/*
 * a4: one DEM step of size dt with the hydrodynamic force/torque fh/th of the
 * last reduction held constant over the step (R11, velocity-Verlet):
 *   a0 = (F_h + F_c(x, v))/m + g_p;  v_half = v + dt/2 a0;  x' = x + dt v_half
 *   (wrap periodic axes into [0,n));  a1 = (F_h + F_c(x', v_half))/m + g_p;
 *   v' = v_half + dt/2 a1;  omega' = omega + dt T_h / I,
 *   I = 2/5 m R^2 (sphere) or 1/2 m R^2 (disk).
 * Updates pos, vel, omega in place.  Returns 0 or -1 (out of memory).
 */
int orc_dem_step(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                 double *pos, double *vel, double *omega, const double *radius,
                 const double *mass, const double *fh, const double *th,
                 double kn, double e, const double *gp, double dt) {
  double *fc = (double *)malloc(sizeof(double) * (size_t)(dim * P));
  if (!fc) return -1;
  contact_forces(dim, n, bc, P, pos, vel, radius, mass, kn, e, fc);
  for (int64_t p = 0; p < P; ++p)
    for (int a = 0; a < dim; ++a) {
      int64_t id = (int64_t)a * P + p;
      double a0 = (fh[id] + fc[id]) / mass[p] + gp[a];
      vel[id] = vel[id] + 0.5 * dt * a0;
      double xn = pos[id] + dt * vel[id];
      if (bc[a] == 0) {
        if (xn >= (double)n[a]) xn -= (double)n[a];
        if (xn < 0.0) xn += (double)n[a];
      }
      pos[id] = xn;
    }
  contact_forces(dim, n, bc, P, pos, vel, radius, mass, kn, e, fc);
  for (int64_t p = 0; p < P; ++p) {
    for (int a = 0; a < dim; ++a) {
      int64_t id = (int64_t)a * P + p;
      double a1 = (fh[id] + fc[id]) / mass[p] + gp[a];
      vel[id] = vel[id] + 0.5 * dt * a1;
    }
    double I = (dim == 3 ? 0.4 : 0.5) * mass[p] * radius[p] * radius[p];
    int nt = dim == 2 ? 1 : 3;
    for (int a = 0; a < nt; ++a) {
      int64_t id = (int64_t)a * P + p;
      omega[id] = omega[id] + dt * th[id] / I;
    }
  }
  free(fc);
  return 0;
}

/* ------------------------------------------------------------------------ */
/* Verlet neighbour list ("The neighbor-list of each solid      */
/* particle is established roughly every 100th time step"), reading R19.      */
/* ------------------------------------------------------------------------ */

/*
 * The list of particle i, by its definition (brute force over all j):
 *   L(i) = { j != i : |r_i - r_j|^2 < (R_i + R_j + skin)^2 }   (minimum image),
 * j ascending.  dist2 is summed left to right without FMA.  start[P+1] (CSR
 * offsets) and items[cap] are outputs.  Returns the number of entries, or
 * -(needed) when cap is too small (nothing useful written then).
 */
int64_t orc_verlet_build(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                         const double *x, const double *radius, double skin,
                         int64_t *start /*[P+1]*/, int32_t *items, int64_t cap) {
  int64_t total = 0;
  for (int64_t i = 0; i < P; ++i) {
    start[i] = total;
    for (int64_t j = 0; j < P; ++j) {
      if (j == i) continue;
      double dist2 = 0.0;
      for (int a = 0; a < dim; ++a) {
        double d = x[(int64_t)a * P + i] - x[(int64_t)a * P + j];
        if (bc[a] == 0) d = min_image(d, n[a]);
        dist2 += d * d;
      }
      double Rc = (radius[i] + radius[j]) + skin;
      if (dist2 < Rc * Rc) {
        if (total < cap) items[total] = (int32_t)j;
        ++total;
      }
    }
  }
  start[P] = total;
  return total <= cap ? total : -total;
}

/* Largest squared displacement (minimum image) of any particle from the
 * positions x_ref at which the list was built. */
double orc_verlet_max_disp2(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                            const double *x, const double *x_ref) {
  double m = 0.0;
  for (int64_t i = 0; i < P; ++i) {
    double d2 = 0.0;
    for (int a = 0; a < dim; ++a) {
      double d = x[(int64_t)a * P + i] - x_ref[(int64_t)a * P + i];
      if (bc[a] == 0) d = min_image(d, n[a]);
      d2 += d * d;
    }
    if (d2 > m) m = d2;
  }
  return m;
}

/* Contact forces as in contact_forces(), but particle i only looks at the
 * members of its list (in list order); walls as before. */
static void contact_forces_list(int dim, const int64_t *n, const int32_t *bc,
                                int64_t P, const double *x, const double *v,
                                const double *radius, const double *mass,
                                double kn, double e, const int64_t *start,
                                const int32_t *items, double *fc) {
  for (int64_t i = 0; i < P; ++i) {
    double F[3] = {0.0, 0.0, 0.0};
    for (int64_t t = start[i]; t < start[i + 1]; ++t) {
      int64_t j = items[t];
      double d[3] = {0.0, 0.0, 0.0}, dist2 = 0.0;
      for (int a = 0; a < dim; ++a) {
        d[a] = x[(int64_t)a * P + i] - x[(int64_t)a * P + j];
        if (bc[a] == 0) d[a] = min_image(d[a], n[a]);
        dist2 += d[a] * d[a];
      }
      double Rs = radius[i] + radius[j];
      if (dist2 >= Rs * Rs) continue;
      double dist = sqrt(dist2);
      double delta = Rs - dist;
      if (!(delta > 0.0)) continue;
      double meff = mass[i] * mass[j] / (mass[i] + mass[j]);
      double eta = orc_damping(kn, e, meff);
      double nrm[3], vn = 0.0;
      for (int a = 0; a < dim; ++a) {
        nrm[a] = d[a] / dist;
        vn += (v[(int64_t)a * P + i] - v[(int64_t)a * P + j]) * nrm[a];
      }
      for (int a = 0; a < dim; ++a)
        F[a] += kn * delta * nrm[a] - eta * vn * nrm[a];
    }
    for (int a = 0; a < dim; ++a) {
      if (bc[a] == 0) continue;
      double eta = orc_damping(kn, e, mass[i]);
      double xa = x[(int64_t)a * P + i], va = v[(int64_t)a * P + i];
      double delta = radius[i] - (xa + 0.5);
      if (delta > 0.0) F[a] += kn * delta * 1.0 - eta * (va * 1.0) * 1.0;
      delta = radius[i] - (((double)n[a] - 0.5) - xa);
      if (delta > 0.0) F[a] += kn * delta * (-1.0) - eta * (va * -1.0) * (-1.0);
    }
    for (int a = 0; a < dim; ++a) fc[(int64_t)a * P + i] = F[a];
  }
}

void orc_contact_forces_list(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                             const double *x, const double *v, const double *radius,
                             const double *mass, double kn, double e,
                             const int64_t *start, const int32_t *items, double *fc) {
  contact_forces_list(dim, n, bc, P, x, v, radius, mass, kn, e, start, items, fc);
}


/*
 * Rebuild rule (R19), applied before EVERY contact evaluation (two per step):
 * rebuild at the current positions when there is no list yet, or the list is
 * `every` or more steps old ("roughly every 100th time step"), or
 * some particle has moved farther than skin/2 from where it was when the list
 * was built (squared displacement > (skin/2)^2).  The last condition is what
 * makes the list exact: while it holds for nobody, two particles that touch
 * now (distance < R_i + R_j) were closer than R_i + R_j + skin at build time,
 * so they are in each other's lists and the forces equal the all-pairs sum.
 * state[0] = list valid, state[1] = age in steps, state[2] = number of builds.
 * Returns 0, or -1 when the list does not fit cap.
 */
static int verlet_ensure(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                         const double *x, const double *radius, double skin,
                         int64_t every, int64_t *state, double *x_ref,
                         int64_t *start, int32_t *items, int64_t cap) {
  int need = !state[0] || state[1] >= every;
  if (!need) {
    double h = 0.5 * skin;
    need = orc_verlet_max_disp2(dim, n, bc, P, x, x_ref) > h * h;
  }
  if (!need) return 0;
  if (orc_verlet_build(dim, n, bc, P, x, radius, skin, start, items, cap) < 0) return -1;
  memcpy(x_ref, x, sizeof(double) * (size_t)(dim * P));
  state[0] = 1;
  state[1] = 0;
  state[2] += 1;
  return 0;
}

/*
 * a4 with the neighbour list: the step of orc_dem_step (R11), with both contact
 * evaluations summing over the lists kept in (state, x_ref, start, items) and
 * the rebuild rule above in front of each.  The list ages by one per step.
 */
int orc_dem_step_verlet(int dim, const int64_t *n, const int32_t *bc, int64_t P,
                        double *pos, double *vel, double *omega, const double *radius,
                        const double *mass, const double *fh, const double *th,
                        double kn, double e, const double *gp, double dt,
                        double skin, int64_t every, int64_t *state, double *x_ref,
                        int64_t *start, int32_t *items, int64_t cap) {
  double *fc = (double *)malloc(sizeof(double) * (size_t)(dim * P));
  if (!fc) return -1;
  if (verlet_ensure(dim, n, bc, P, pos, radius, skin, every, state, x_ref, start, items, cap)) {
    free(fc);
    return -1;
  }
  contact_forces_list(dim, n, bc, P, pos, vel, radius, mass, kn, e, start, items, fc);
  for (int64_t p = 0; p < P; ++p)
    for (int a = 0; a < dim; ++a) {
      int64_t id = (int64_t)a * P + p;
      double a0 = (fh[id] + fc[id]) / mass[p] + gp[a];
      vel[id] = vel[id] + 0.5 * dt * a0;
      double xn = pos[id] + dt * vel[id];
      if (bc[a] == 0) {
        if (xn >= (double)n[a]) xn -= (double)n[a];
        if (xn < 0.0) xn += (double)n[a];
      }
      pos[id] = xn;
    }
  if (verlet_ensure(dim, n, bc, P, pos, radius, skin, every, state, x_ref, start, items, cap)) {
    free(fc);
    return -1;
  }
  contact_forces_list(dim, n, bc, P, pos, vel, radius, mass, kn, e, start, items, fc);
  for (int64_t p = 0; p < P; ++p) {
    for (int a = 0; a < dim; ++a) {
      int64_t id = (int64_t)a * P + p;
      double a1 = (fh[id] + fc[id]) / mass[p] + gp[a];
      vel[id] = vel[id] + 0.5 * dt * a1;
    }
    double I = (dim == 3 ? 0.4 : 0.5) * mass[p] * radius[p] * radius[p];
    int nt = dim == 2 ? 1 : 3;
    for (int a = 0; a < nt; ++a) {
      int64_t id = (int64_t)a * P + p;
      omega[id] = omega[id] + dt * th[id] / I;
    }
  }
  state[1] += 1;
  free(fc);
  return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
