/*
 * lbmimb.h -- C-ABI of the B200-native LBM-IMB-DEM hot path of arxiv/paper_1011_2613
 * ("Large-Scale DNS of Gas-Solid Flow on Mole-8.5").  Implemented by
 * paper_1011_2613_b200/csrc (hand-written CUDA, sm_100a), built into
 * paper_1011_2613_b200/liblbmimb.so.  No torch / C++ types cross this boundary.
 *
 * Citations are PAPER.md:<line> (the paper) and DESIGN.md R<k> (readings of the paper
 * where it is silent or garbled; R<k> = SURVEY.md 8(c) G<k>).
 *
 * ---------------------------------------------------------------------------------------
 * Conventions
 * ---------------------------------------------------------------------------------------
 * Lattice units h = dt = 1.  Node (i,j,k) sits at the integer position (i,j,k); its cell is
 * the unit square/cube centred on it, so the domain is [-1/2, n-1/2) per axis.
 * Node index  x = (k*ny + j)*nx + i  (x is the fastest-varying axis); nz = 1 in 2D.
 * Distributions f[q][k][j][i] (SoA, fp64), Q = 9 (dim 2) or 19 (dim 3).
 * Direction order (part of the ABI, R1); opposite of odd q is q+1:
 *   D2Q9 : 0:(0,0) 1:(1,0) 2:(-1,0) 3:(0,1) 4:(0,-1) 5:(1,1) 6:(-1,-1) 7:(1,-1) 8:(-1,1)
 *   D3Q19: 0 rest; 1..6 = +x,-x,+y,-y,+z,-z; 7:(1,1,0) 8:(-1,-1,0) 9:(1,-1,0) 10:(-1,1,0)
 *          11:(1,0,1) 12:(-1,0,-1) 13:(1,0,-1) 14:(-1,0,1) 15:(0,1,1) 16:(0,-1,-1)
 *          17:(0,1,-1) 18:(0,-1,1)
 *   weights 4/9, 1/9, 1/36 (D2Q9); 1/3, 1/18, 1/36 (D3Q19); c_s^2 = 1/3.
 * Particle arrays are SoA: pos[D][P], vel[D][P], omega[1][P] (2D, z component) or
 * omega[3][P] (3D), radius[P], mass[P], force[D][P], torque[1|3][P].
 *
 * Pointers: every pointer argument is a HOST pointer owned by the caller unless its name
 * ends in _dev (then it is a device pointer on the handle's device, e.g. a torch tensor's
 * data_ptr()).  The library never keeps a caller's host pointer after the call returns.
 * Device memory is owned by the handle, or by the caller when params.workspace is given.
 *
 * Errors: every call returns an lbmimb_status; nothing throws or aborts across the ABI.
 * On error the handle stays valid and, where possible, unchanged; lbmimb_last_error()
 * returns a thread-local description of the last failure on the calling thread.
 * Errors that only a kernel can detect (the list of nodes shared by several particles overflowed, a
 * neighbour list or a cell of its build grid overflowed: particle sets that overlap far more deeply than
 * soft spheres in contact do) are reported as ESTATE by the next call that synchronises: synchronize,
 * get_particles, fetch_fields, diagnostics, fetch_neighbor_list and reduce_particle_forces with host outputs.
 * The flags are cleared by the next map_particles / set_particles.
 *
 * Ordering: the set_, get_ and fetch_ calls and reduce_particle_forces with non-NULL host outputs are
 * complete when they return; map_particles, step, dem_step and the _dev variants are
 * asynchronous on the handle's stream.  One handle must not be used from two threads at
 * the same time.  There is no CPU fallback: without a CUDA device create_lattice fails.
 */
#ifndef LBMIMB_H
#define LBMIMB_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbmimb_lattice lbmimb_lattice; /* opaque; owns (or borrows) all device memory */

typedef enum {
  LBMIMB_OK = 0,
  LBMIMB_EINVAL = 1, /* bad argument */
  LBMIMB_ENOMEM = 2, /* device or host allocation failed / workspace too small */
  LBMIMB_ECUDA = 3,  /* a CUDA runtime call or kernel failed */
  LBMIMB_ESTATE = 4  /* call out of order (e.g. step with particles set but not mapped) */
} lbmimb_status;

typedef struct {
  int32_t dim;        /* 2 -> D2Q9, 3 -> D3Q19 */
  int32_t subsamples; /* S per axis for the solid-fraction sampling; 1 <= S, S^dim <= 255 */
  int64_t n[3];       /* nodes per axis, n[2] = 1 in 2D; each >= 1 */
  int32_t bc[3];      /* per axis: 0 periodic, 1 half-way bounce-back walls at both ends (R15) */
  int32_t device;     /* CUDA ordinal */
  double tau;         /* relaxation time of eq. (1), > 0.5 */
  double g_fluid[3];  /* acceleration g in F_i = 3 w_i rho (c_i . g)  (R3) */
  void *stream;       /* cudaStream_t to run on (e.g. torch.cuda.current_stream().cuda_stream), NULL = default */
  void *workspace_dev;      /* optional caller-owned device buffer, 256-byte aligned; NULL = library allocates */
  uint64_t workspace_bytes; /* size of workspace_dev; must be >= lbmimb_workspace_bytes() */
  int32_t streaming;  /* LBMIMB_STREAM_AB (0, default) or LBMIMB_STREAM_AA: how step() propagates, see below */
  int32_t flags;      /* 0, or LBMIMB_FLAG_EXCHANGE_FIELD */
  int64_t slab_y0;    /* slab lattices only: global index of this lattice's first owned row */
  int64_t slab_ny;    /* rows of the GLOBAL lattice; 0 (default) = this lattice is the whole one */
} lbmimb_params;

/*
 * Slabs: domain decomposition along y ("Parallel implementation", Fig. 2).
 * A lattice with slab_ny > 0 owns the rows [slab_y0, slab_y0 + n[1]) of a global lattice of slab_ny rows
 * (x and z whole).  bc[1] is the boundary of the GLOBAL lattice; an end of the slab that is not such a wall gets
 * one ghost row (lbmimb_slab_ghost_rows).  One time step of the decomposed lattice:
 *     every slab:  lbmimb_map_particles, lbmimb_step(h, 1)
 *     every slab, every end with a ghost row:  lbmimb_pack_halo(h, side, buf)  ->  transport to the neighbour
 *                  ->  lbmimb_unpack_halo(neighbour, 1 - side, buf)            (before the neighbour's next step)
 *     particles cut by a slab face: lbmimb_export_force_sums_dev on every slab, integer SUM over the slabs (any
 *                  order: the sums are fixed-point integers), lbmimb_import_force_sums_dev, then
 *                  lbmimb_reduce_particle_forces / lbmimb_dem_step on every slab (the particles are replicated).
 * What crosses a face per step: the 5 (D3Q19) / 3 (D2Q9) populations that stream through it, n[0]*n[2] nodes
 * each (lbmimb_halo_count doubles), and 12 (6) 64-bit words per particle.  The transport (peer copies, NCCL,
 * MPI) is the caller's: the library only packs and unpacks device buffers.
 * Particles keep GLOBAL coordinates and every slab is given ALL of them, so the map, V_S, the lever arms and the
 * DEM step are the same arithmetic as on the undivided lattice: maps and force sums agree with it bit for bit,
 * distributions to rounding order (none changes: bit for bit as well).  Ownership rule for a particle cut by a
 * face: every covered node adds to the sums of the slab that OWNS the node; ghost rows add nothing.
 * fetch_fields addresses the owned rows (row 0 = first owned row); set_distributions takes the STORED rows
 * (ghost rows included, i.e. global rows slab_y0 - ghost_lo ... , wrapped on a periodic axis).
 * lbmimb_diagnostics sums over the owned rows only.  Slab lattices stream with two arrays (LBMIMB_STREAM_AB);
 * lbmimb_run_coupled is not available on them (the force sums must cross slabs inside the step).
 */

/*
 * flags.  EXCHANGE_FIELD: keep the exchange vector s of every covered node of the last step in device memory
 * (2 or 4 doubles per node) so that lbmimb_fetch_fields(LBMIMB_FIELD_S) can return it -- a diagnostic / test
 * output.  The per-particle force and torque never need it: they are summed inside the fused step.
 */
#define LBMIMB_FLAG_EXCHANGE_FIELD 1

/*
 * Streaming schemes of a2 (same results up to rounding order; both are fused collide-and-stream kernels):
 *   AB: "pull" with two distribution arrays (2 x Q x N doubles); a step reads one and writes the other.
 *   AA: in-place AA-pattern on ONE array (Q x N doubles): even steps touch only the own node, odd steps
 *       gather from and scatter to the neighbours.  Halves the footprint, which is what lets the paper's
 *       512 x 2016 x 512 D3Q19 lattice (80.3 GB of distributions) fit one 180 GB B200.
 *       In AA mode fetch_fields stages through a grow-only device buffer of the largest box fetched so far,
 *       allocated by the library outside the workspace (ENOMEM if that fails: fetch sub-boxes of a large lattice).
 */
enum { LBMIMB_STREAM_AB = 0, LBMIMB_STREAM_AA = 1 };

typedef struct {
  double kn;            /* stiffness k_n of eq. (4) */
  double restitution;   /* e of eq. (5), 0 < e <= 1 */
  double g_particle[3]; /* gravitational acceleration on the particles */
  double dt;            /* DEM time step (1 = one LBM step, R11) */
} lbmimb_dem_params;

/* selectors of lbmimb_fetch_fields */
enum {
  LBMIMB_FIELD_F = 0,       /* double [Q][box]  distributions f_i(x, t) (post-streaming, pre-collision) */
  LBMIMB_FIELD_RHO = 1,     /* double [box]     rho = sum_i f_i */
  LBMIMB_FIELD_U = 2,       /* double [D][box]  bare u = sum_i f_i c_i / rho (no half-force shift, R2) */
  LBMIMB_FIELD_EPS_CNT = 3, /* uint8  [box]     inside-sample count n_s, eps = n_s / S^D */
  LBMIMB_FIELD_PID = 4,     /* int32  [box]     covering particle, -1 = none */
  LBMIMB_FIELD_S = 5        /* double [D][box]  exchange vector s of the last step (0 where eps = 0); needs
                               LBMIMB_FLAG_EXCHANGE_FIELD, else ESTATE */
};

/*
 * Mapping modes of a1 (lbmimb_set_mapping_mode).
 * SAMPLING (default): the S^D sub-cell points of lbmimb_map_particles below; eps = n_s / S^D.
 * TABLE: the paper's own method (eq. (6)): gamma = phi(d, theta) is pre-calculated for
 *   "a solid particle with a given radius" and looked up per node from the distance d between the cell
 *   centre and the particle centre and the orientation of the displacement.  Fig. 1 is not available, so
 *   the discretisation is DESIGN.md R17:  sqD = sqrt(D), d0 = R - sqD/2, dd = sqD/Nd;
 *     entry (k, m1[, m2]): d_k = d0 + (k+1/2) dd, t1 = (m1+1/2)/Nt, t2 = (m2+1/2)/Nt, cell centre
 *       r = d_k (1, t1, t2)/sqrt(1 + t1^2 + t2^2), n = number of the St^D sub-cell points
 *       r + ((a+1/2)/St - 1/2) inside the particle (|p|^2 <= R^2, fp64, no FMA, left to right),
 *       code = (255 n + St^D/2) / St^D (integer division), gamma = code/255;
 *     look-up of a node with displacement delta (minimum image): d = sqrt(dx^2 + dy^2 (+ dz^2));
 *       d < d0 -> 255;  k = (int)((d - d0) * (Nd/sqD)), k >= Nd -> 0;  a >= b >= c the sorted |delta|,
 *       m1 = min((int)((b/a) Nt), Nt-1), m2 = min((int)((c/a) Nt), Nt-1);
 *     a node reached by several particles: code = min(255, sum of their codes), covering particle =
 *       largest code, ties -> lowest index.
 *   eps_cnt then holds the code and eps = code/255.  All particles must have one radius >= 1 (else
 *   map_particles returns ESTATE).  Integer results, bit-exact against this definition.
 */
enum { LBMIMB_MAP_SAMPLING = 0, LBMIMB_MAP_TABLE = 1 };
#define LBMIMB_TABLE_ND_2D 128
#define LBMIMB_TABLE_NT_2D 32
#define LBMIMB_TABLE_ST_2D 256
#define LBMIMB_TABLE_ND_3D 128
#define LBMIMB_TABLE_NT_3D 16
#define LBMIMB_TABLE_ST_3D 64
#define LBMIMB_TABLE_DEN 255

/* Bytes of device memory a lattice of these parameters needs (0 on invalid parameters). */
uint64_t lbmimb_workspace_bytes(const lbmimb_params *params, int64_t max_particles);

/*
 * a0. Creates a lattice at rest: f_i = f_i^eq(rho=1, u=0) = w_i on every node, time t = 0, no
 * particles.  0 <= max_particles <= 2^24 bounds later set_particles calls (a node's tag word holds the
 * sample count in 8 bits and the covering particle in 24).  *out receives the handle.
 * EINVAL: bad dim / n / bc / tau <= 0.5 / S^dim > 255 / flags / max_particles; ENOMEM; ECUDA (no device, ...).
 */
lbmimb_status lbmimb_create_lattice(const lbmimb_params *params, int64_t max_particles,
                                    lbmimb_lattice **out);
lbmimb_status lbmimb_destroy_lattice(lbmimb_lattice *h); /* NULL is allowed */

/*
 * Replaces the particle set (P <= max_particles; P = 0 removes all particles).  omega may be
 * NULL (= 0).  radius > 0, mass > 0.  Centres must lie in [-1/2, n) per axis (the domain is
 * [-1/2, n-1/2); dem_step wraps periodic coordinates into [0, n)).
 * Invalidates the particle map: the next step needs map_particles first (else ESTATE).
 */
lbmimb_status lbmimb_set_particles(lbmimb_lattice *h, int64_t P, const double *pos, const double *vel,
                                   const double *omega, const double *radius, const double *mass);
/* Replaces velocities only (prescribed-velocity runs); keeps the map valid. */
lbmimb_status lbmimb_set_particle_velocities(lbmimb_lattice *h, const double *vel, const double *omega);
/* Reads the particle state back; any of the outputs may be NULL. */
lbmimb_status lbmimb_get_particles(lbmimb_lattice *h, double *pos, double *vel, double *omega);
int64_t lbmimb_num_particles(const lbmimb_lattice *h);

/*
 * a1. Particle -> lattice mapping (PAPER.md:46 definition of eps; :71-77 why it is hard; R4, R5).
 * For every node the number n_s of the S^D sub-cell sample points
 *   p = x_node + ((a + 1/2)/S - 1/2) per axis, a = 0..S-1,
 * that lie inside any particle (|p - c|^2 <= R^2, minimum image in periodic axes, evaluated in
 * fp64 without FMA contraction, left to right), and the covering particle: the one with most
 * samples in the cell, ties -> lowest index, -1 if none.  Integer results, bit-exact against
 * the definition.  Uses a cell list over the particles.  Asynchronous.
 */
lbmimb_status lbmimb_map_particles(lbmimb_lattice *h);

/* Selects the mapping mode (see above).  Invalidates the particle map.  EINVAL on an unknown mode. */
lbmimb_status lbmimb_set_mapping_mode(lbmimb_lattice *h, int32_t mode);
/*
 * Copies the look-up table of TABLE mode for the current particle radius into dst (uint8
 * [Nd][Nt] in 2D, [Nd][Nt][Nt] in 3D; capacity = bytes available at dst).  Synchronous.
 * ESTATE unless TABLE mode is selected and particles with one radius >= 1 are set.
 */
lbmimb_status lbmimb_fetch_eps_table(lbmimb_lattice *h, uint8_t *dst, int64_t capacity);

/*
 * a2. nsteps fused collide-and-stream steps of eq. (1) with beta,
 * Omega^S of eq. (2) driven by V_S = v_p + omega_p x (x_node - x_p), the body
 * force F_i (R3) and periodic / half-way bounce-back streaming.  Advances t by nsteps.
 * The LAST step of the call also forms, inside the same kernel, the per-particle sums of eq. (3) over the
 * exchange vectors s = beta sum_i Omega_i c_i = beta rho (V_S - u) of its covered nodes (and keeps s per node
 * if the lattice has LBMIMB_FLAG_EXCHANGE_FIELD).
 * ESTATE if particles are set but not mapped.  nsteps = 0 is a no-op.  Asynchronous.
 */
lbmimb_status lbmimb_step(lbmimb_lattice *h, int32_t nsteps);

/*
 * a3. Hydrodynamic force and torque on every particle from the last step's exchange vectors,
 * eq. (3) with the sign of R6 (force ON the particle):
 *   F_p = - sum_{n: pid=p} s_n,   T_p = - sum_n (x_n - x_p) x s_n   (minimum image), h^D/dt = 1.
 * The sums were formed by the last step (runs of a particle's nodes are pre-summed per warp in a fixed tree
 * and added as 64-bit fixed-point integers (resolution 2^-91; a run's partial sum must stay below 2^11 in
 * lattice units, which any stable simulation does by many orders of magnitude), so the result does not depend on the order
 * in which thread blocks ran: bitwise reproducible); this call converts them.  force / torque may be NULL:
 * results stay on the device for dem_step; otherwise they are copied to the host and the call is synchronous.
 * ESTATE if no step has run since the last map_particles.
 */
lbmimb_status lbmimb_reduce_particle_forces(lbmimb_lattice *h, double *force, double *torque);

/*
 * a4. One soft-sphere DEM step (eq. (4)-(5); R8-R11): linear spring-dashpot
 * normal contacts found with a cell list (or neighbour lists, see lbmimb_set_neighbor_mode), wall contacts on
 * wall axes, velocity-Verlet
 *   a0 = (F_h + F_c(x,v))/m + g_p; v' = v + dt/2 a0; x' = x + dt v' (wrapped into [0,n) on
 *   periodic axes); a1 = (F_h + F_c(x',v'))/m + g_p; v'' = v' + dt/2 a1; omega' = omega + dt T_h/I
 * with F_h, T_h of the last reduce_particle_forces (zero if none ran since set_particles).
 * Invalidates the particle map.  Asynchronous.
 */
lbmimb_status lbmimb_dem_step(lbmimb_lattice *h, const lbmimb_dem_params *dem);

/*
 * nsteps coupled steps of the paper's method, each = map_particles -> step(1) -> reduce_particle_forces
 * (results kept on the device) -> dem_step, the order of BASELINE.json configs[4].  Bit for bit
 * what calling the four entry points in a loop gives.  The first step is launched call by call; the launches of
 * the following steps are captured ONCE, two steps at a time (both parities of the distribution arrays), into a
 * CUDA graph and replayed, which removes the per-launch host cost of the ~25 small particle-side kernels of a
 * step (the neighbour-list rebuild rule is decided on the device, so the launch sequence never changes).  The
 * graph is re-captured when the number of particles, their radii, a mode or the DEM parameters change.
 * LBMIMB_NO_GRAPH=1 in the environment keeps to plain launches.  Asynchronous.  Errors as for the four calls.
 */
lbmimb_status lbmimb_run_coupled(lbmimb_lattice *h, const lbmimb_dem_params *dem, int32_t nsteps);

/*
 * Contact search of a4 (lbmimb_set_neighbor_mode).
 * CELLS (default): a cell list over the particles, rebuilt whenever positions change.
 * VERLET: the paper's scheme ("The neighbor-list of each solid particle is established
 *   roughly every 100th time step"; it "uses more memory to trade for less searching work").  The paper
 *   prints neither the list's cut-off nor what triggers a rebuild; R19:
 *     L(i) = { j != i : |r_i - r_j|^2 < ((R_i + R_j) + skin)^2 }  (minimum image; fp64, no FMA, the squared
 *     distance summed x, y, z left to right), j ascending;
 *     before EVERY contact evaluation (two per dem_step) the lists are rebuilt at the current positions
 *     if there is no valid list (first use, or set_particles since), or the list is `every` or more
 *     dem_steps old, or some particle's squared displacement (minimum image, same arithmetic) from its
 *     position at the last build exceeds (skin/2)^2.  While no displacement exceeds skin/2, every
 *     touching pair is in the lists, so the contact forces equal the all-pairs sum of R8 exactly.
 *   The decision is taken on the device (no host synchronisation); contact sums run over the lists in
 *   ascending j.  List storage is allocated by the library (cudaMalloc, outside the workspace) from
 *   packing bounds on the particles' radii: slots per particle K = (2 (2 R_max + skin)/(1.5 R_min) + 1)^D;
 *   particle sets that overlap so deeply that a list (or a cell of the build grid) overflows make
 *   lbmimb_synchronize / lbmimb_fetch_neighbor_list return ESTATE.
 * set_neighbor_mode: skin > 0 and every >= 1 for VERLET (ignored for CELLS); drops any existing list.
 * EINVAL on an unknown mode or bad skin / every.
 */
enum { LBMIMB_NEIGHBOR_CELLS = 0, LBMIMB_NEIGHBOR_VERLET = 1 };
lbmimb_status lbmimb_set_neighbor_mode(lbmimb_lattice *h, int32_t mode, double skin, int64_t every);
/*
 * Copies the current neighbour lists to the host as CSR: start[P+1] (int64 offsets), items[start[P]]
 * (int32, j ascending inside each list); capacity = entries available at items.  info[4] (may be NULL):
 * [0] 1 if a valid list exists (else start is all zero), [1] its age in dem_steps, [2] number of list
 * builds since set_neighbor_mode, [3] total entries start[P].  Synchronous.
 * ESTATE if VERLET mode is not selected or a list overflowed; EINVAL if capacity < info[3] (info is still
 * filled, nothing else is written).
 */
lbmimb_status lbmimb_fetch_neighbor_list(lbmimb_lattice *h, int64_t *start, int32_t *items, int64_t capacity,
                                         int64_t *info);

/*
 * a5. Copies a field of the sub-box [lo, hi) (node coordinates, x first; 2D: lo[2]=0, hi[2]=1)
 * into dst, laid out [component][k][j][i] over the box, x fastest.  `what` is one of
 * LBMIMB_FIELD_*.  Synchronous.  EPS_CNT / PID need a valid map, S needs a step after it.
 */
lbmimb_status lbmimb_fetch_fields(lbmimb_lattice *h, int32_t what, const int64_t lo[3],
                                  const int64_t hi[3], void *dst);

/*
 * Area/volume-averaged suspension diagnostics: the quantities of PAPER.md:154 and Figs. 5/7 ("area-averaged
 * inter-phase slip velocity V_ry and drag force F_dy").  The paper prints no formula; R18:
 *   eps_x = eps_cnt_x / S^D (code/255 in TABLE mode), u = bare velocity (R2) of the current distributions,
 *   A_g = sum_x (1 - eps_x);  U_g = sum_x (1 - eps_x) u_x / A_g;
 *   V_s = sum_p vol_p v_p / sum_p vol_p, vol_p = pi R^2 | 4/3 pi R^3;  V_r = U_g - V_s;
 *   F_d = sum_p F_p / P with F_p of the last reduce_particle_forces (0 if none ran since set_particles).
 * out[LBMIMB_DIAG_LEN] (host): [0] A_g  [1] sum_x rho  [2:5] U_g  [5:8] V_s  [8:11] V_r  [11:14] F_d
 *   [14:17] sum_x rho u  [17:20] sum_p m_p v_p   (unused z components and all particle entries with P = 0 are 0).
 * Two-stage device reduction in a fixed order (deterministic for a given lattice).  Synchronous.
 * ESTATE if particles are set but not mapped.
 */
#define LBMIMB_DIAG_LEN 20
lbmimb_status lbmimb_diagnostics(lbmimb_lattice *h, double *out);

/*
 * lbmimb_diagnostics for callers that cannot call cudaMalloc and must not synchronise (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation): the same 20 quantities, written to out_dev
 * (DEVICE pointer, LBMIMB_DIAG_LEN doubles), asynchronous on the handle's stream.  It allocates nothing, frees
 * nothing and calls no allocating routine: its scratch (the per-block partial sums of the two reduction stages) is
 * a static device array inside the library of lbmimb_diagnostics_static_scratch_bytes() = 403,456 bytes, which
 * every GPU that loads the library holds until the process exits.  The particle sums are formed by one block per
 * 256 particles, so the array bounds the particle count: more than
 * lbmimb_diagnostics_static_max_particles() = 1,048,576 particles -> EINVAL (use lbmimb_diagnostics).
 * Node sums are bit for bit those of lbmimb_diagnostics; particle sums (V_s, F_d, solid momentum) are added in
 * a different order and agree to rounding.  All calls on a device share the array, which keeps the last call's
 * contents; every call overwrites exactly the rows it reads back, so nothing has to be cleared.  Calls that overlap
 * on the GPU (two handles on two streams) race on it: serialise them.  The device-side error flags (see "Errors")
 * are not looked at, since that needs a synchronisation.
 * EINVAL: NULL argument, too many particles; ESTATE if particles are set but not mapped.
 */
int64_t lbmimb_diagnostics_static_max_particles(void);
int64_t lbmimb_diagnostics_static_scratch_bytes(void);
lbmimb_status lbmimb_diagnostics_static_dev(lbmimb_lattice *h, double *out_dev);

/* Replaces all distributions: f[Q][nz][ny][nx] = f_i(x, t) as LBMIMB_FIELD_F returns them. */
lbmimb_status lbmimb_set_distributions(lbmimb_lattice *h, const double *f);

/* Device-pointer variants (same layouts).  reduce_particle_forces_dev is asynchronous on the handle's stream;
 * set_particles_dev first checks the arrays with a kernel (same conditions as set_particles; one small
 * read-back, so it synchronises) and commits nothing on EINVAL. */
lbmimb_status lbmimb_set_particles_dev(lbmimb_lattice *h, int64_t P, const double *pos_dev,
                                       const double *vel_dev, const double *omega_dev,
                                       const double *radius_dev, const double *mass_dev);
lbmimb_status lbmimb_reduce_particle_forces_dev(lbmimb_lattice *h, double *force_dev, double *torque_dev);

/*
 * Slab lattices (see "Slabs" above).  side: 0 = lower (y-) end, 1 = upper (y+) end.
 * pack_halo copies the populations LEAVING through that end (c_y = -1 for side 0, +1 for side 1) of the
 * first / last owned row of the current (post-collision) state into dst_dev, laid out [slot][k][i] with the
 * slots in ascending direction index (D2Q9: 4,6,7 | 3,5,8; D3Q19: 4,8,9,16,18 | 3,7,10,15,17);
 * unpack_halo stores such a buffer, packed by the neighbour across that end with the opposite side, in the
 * ghost row of that end.  lbmimb_halo_count doubles per buffer.  Asynchronous on the handle's stream.
 * ESTATE: not a slab, or that end is a wall of the global lattice.
 */
int64_t lbmimb_halo_count(const lbmimb_lattice *h);
int32_t lbmimb_slab_ghost_rows(const lbmimb_lattice *h, int32_t side); /* 0 or 1; -1 on bad arguments */
lbmimb_status lbmimb_pack_halo(lbmimb_lattice *h, int32_t side, double *dst_dev);
lbmimb_status lbmimb_unpack_halo(lbmimb_lattice *h, int32_t side, const double *src_dev);
/*
 * The per-particle force / torque sums of the last step as the integers the fused kernel accumulated:
 * lbmimb_force_sums_count(h) = P * (3 | 6) * 2 int64 words ([P][value][hi, lo], value = hi 2^-40 + lo 2^-91).
 * Adding the arrays of all slabs word by word gives the sums of the undivided lattice exactly.  export copies
 * them out, import replaces them (both asynchronous).  ESTATE unless a step has run since the last map and
 * reduce_particle_forces has not consumed the sums yet.
 */
int64_t lbmimb_force_sums_count(const lbmimb_lattice *h);
lbmimb_status lbmimb_export_force_sums_dev(lbmimb_lattice *h, int64_t *dst_dev);
lbmimb_status lbmimb_import_force_sums_dev(lbmimb_lattice *h, const int64_t *src_dev);

/* Blocks until all work queued on the handle's stream has finished. */
lbmimb_status lbmimb_synchronize(lbmimb_lattice *h);
/* Number of steps taken since creation / set_distributions. */
int64_t lbmimb_time(const lbmimb_lattice *h);
/* Kernels launched by this handle so far (bench.py's gpu_launches). */
int64_t lbmimb_launch_count(const lbmimb_lattice *h);
const char *lbmimb_last_error(void); /* thread-local, never NULL */
const char *lbmimb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LBMIMB_H */
