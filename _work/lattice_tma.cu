// a2, B200 version: the fused collide-and-stream step as a persistent, warp-specialised
// kernel whose loads are TMA bulk copies (cp.async.bulk global -> shared, mbarrier
// complete_tx) staged through a ring of shared-memory tiles.
//
// Why: the one-thread-per-node kernel of lattice.cu keeps 19 fp64 loads per thread in
// registers, so bytes in flight are tied to register occupancy (~16 warps/SM, ncu
// profiles/r1a) and the kernel stalls at ~80 % of the copy bandwidth.  Here one producer
// lane per CTA streams whole row segments (Q rows x TX nodes) into NSTAGE shared-memory
// stages; the consumer warps copy their 19 values to registers, release the stage at once
// and collide while the next stages are already in flight.  Bytes in flight per SM =
// CTAs/SM x NSTAGE x Q x (TX+2) x 8 B (~170 KB), independent of registers.
//
// Same arithmetic, same pull/two-buffer scheme and same state layout as lattice.cu; the
// x-shifted rows are fetched as 16-byte-aligned supersets (TX+2 elements) and read from
// shared memory with a one-element offset, so every global access is aligned.
#include <cstdlib>

#include "collide.cuh"
#include "lbmimb_internal.cuh"

namespace lbmimb {

struct TmaStepArgs {
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
  unsigned tiles_per_row;
  unsigned num_tiles;
  CollideParams cp;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// TMA bulk copy global -> shared, completion signalled on an mbarrier (bytes % 16 == 0, both 16 B aligned)
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// source row of direction q for the lattice row (j,k): array index and row index, `bounce` when the
// source lies behind a y/z wall (then it is the node's own row of the opposite direction)
template <int D>
__device__ __forceinline__ void source_row(const TmaStepArgs &a, int q, int j, int k, int &qs, int64_t &row,
                                           bool &bounce) {
  using L = Lat<D>;
  int js = j - L::cy(q), ks = k - L::cz(q);
  bounce = false;
  if (js < 0 || js >= a.ny) {
    if (a.bcy) bounce = true;
    else js = js < 0 ? js + a.ny : js - a.ny;
  }
  if (D == 3 && (ks < 0 || ks >= a.nz)) {
    if (a.bcz) bounce = true;
    else ks = ks < 0 ? ks + a.nz : ks - a.nz;
  }
  if (bounce) {
    qs = opposite(q);
    row = (int64_t)k * a.ny + j;
  } else {
    qs = q;
    row = (int64_t)ks * a.ny + js;
  }
}

template <int D, int TX, int NSTAGE, bool IMB, bool EMIT, int MINB>
__global__ void __launch_bounds__(TX + 32, MINB) collide_stream_tma_kernel(const TmaStepArgs a) {
  using L = Lat<D>;
  constexpr int Q = L::Q;
  constexpr int RS = TX + 2;  // doubles per staged row
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *stage_base = reinterpret_cast<double *>(smem_raw);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)NSTAGE * Q * RS * sizeof(double));
  uint64_t *empty = full + NSTAGE;
  constexpr int kConsumerWarps = TX / 32;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, kConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int warp = threadIdx.x >> 5;
  if (warp == kConsumerWarps) {
    // ===================== producer: one lane issues the bulk copies =====================
    if ((threadIdx.x & 31) == 0) {
      unsigned it = 0;
      for (unsigned t = blockIdx.x; t < a.num_tiles; t += gridDim.x, ++it) {
        const int s = it % NSTAGE;
        const uint32_t ph = (it / NSTAGE) & 1u;
        mbar_wait(empty + s, ph ^ 1u);
        const unsigned row = t / a.tiles_per_row;
        const int x0 = (int)(t - row * a.tiles_per_row) * TX;
        const int txe = min(TX, a.nx - x0);
        const int k = D == 3 ? (int)(row / (unsigned)a.ny) : 0;
        const int j = (int)(row - (unsigned)k * (unsigned)a.ny);
        double *st = stage_base + (size_t)s * Q * RS;
        // bytes this stage will receive
        uint32_t bytes = 0;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          int qs;
          int64_t srow;
          bool bounce;
          source_row<D>(a, q, j, k, qs, srow, bounce);
          const int cx = bounce ? 0 : L::cx(q);
          uint32_t b = (uint32_t)txe * 8u;
          if (cx == 1 && (x0 > 0 || !a.bcx)) b += 16u;
          if (cx == -1 && (x0 + txe < a.nx || !a.bcx)) b += 16u;
          bytes += b;
        }
        mbar_expect_tx(full + s, bytes);
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          int qs;
          int64_t srow;
          bool bounce;
          source_row<D>(a, q, j, k, qs, srow, bounce);
          const int cx = bounce ? 0 : L::cx(q);
          const double *g = a.fin + (int64_t)qs * a.N + srow * a.nx;  // start of the source row
          double *d = st + q * RS;
          if (cx == 0) {
            bulk_g2s(d, g + x0, (uint32_t)txe * 8u, full + s);
          } else if (cx == 1) {
            // need elements x0-1 .. x0+txe-2; staged as [x0-2, x0+txe) at d[0..txe+2)
            if (x0 > 0) {
              bulk_g2s(d, g + x0 - 2, (uint32_t)(txe + 2) * 8u, full + s);
            } else {
              if (!a.bcx) bulk_g2s(d, g + a.nx - 2, 16u, full + s);
              bulk_g2s(d + 2, g, (uint32_t)txe * 8u, full + s);
            }
          } else {
            // need elements x0+1 .. x0+txe; staged as [x0, x0+txe+2) at d[0..txe+2)
            if (x0 + txe < a.nx) {
              bulk_g2s(d, g + x0, (uint32_t)(txe + 2) * 8u, full + s);
            } else {
              bulk_g2s(d, g + x0, (uint32_t)txe * 8u, full + s);
              if (!a.bcx) bulk_g2s(d + txe, g, 16u, full + s);
            }
          }
        }
      }
    }
    return;
  }

  // ===================== consumers: one thread per node of the tile =====================
  const int tl = threadIdx.x;  // 0 .. TX-1
  unsigned it = 0;
  for (unsigned t = blockIdx.x; t < a.num_tiles; t += gridDim.x, ++it) {
    const int s = it % NSTAGE;
    const uint32_t ph = (it / NSTAGE) & 1u;
    const unsigned row = t / a.tiles_per_row;
    const int x0 = (int)(t - row * a.tiles_per_row) * TX;
    const int txe = min(TX, a.nx - x0);
    const int k = D == 3 ? (int)(row / (unsigned)a.ny) : 0;
    const int j = (int)(row - (unsigned)k * (unsigned)a.ny);
    const int i = x0 + tl;
    const bool live = tl < txe;
    const int64_t x = ((int64_t)k * a.ny + j) * a.nx + i;
    int cnt = 0;
    if (IMB && live) cnt = a.eps_cnt[x];

    const double *st = stage_base + (size_t)s * Q * RS;
    mbar_wait(full + s, ph);
    double f[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      int qs;
      int64_t srow;
      bool bounce;
      source_row<D>(a, q, j, k, qs, srow, bounce);
      const int cx = bounce ? 0 : L::cx(q);
      // cx = +1: row staged from x0-2, wanted element x0+tl-1 -> index tl+1
      // cx = -1: row staged from x0,   wanted element x0+tl+1 -> index tl+1
      f[q] = st[q * RS + tl + (cx != 0 ? 1 : 0)];
    }
    __syncwarp();
    if ((tl & 31) == 0) mbar_arrive(empty + s);

    if (a.bcx && live && (i == 0 || i == a.nx - 1)) {
      // x walls: the two end nodes of a lattice row bounce their own opposite population back
#pragma unroll
      for (int q = 1; q < Q; ++q) {
        const int cx = L::cx(q);
        if ((cx == 1 && i == 0) || (cx == -1 && i == a.nx - 1)) f[q] = a.fin[(int64_t)opposite(q) * a.N + x];
      }
    }
    if (!live) {
#pragma unroll
      for (int q = 0; q < Q; ++q) f[q] = L::w(q);   // idle lanes of a ragged tile: harmless values
    }

    double rho, ux, uy, uz;
    moments<D>(f, rho, ux, uy, uz);
    if (!IMB || !__any_sync(0xffffffffu, cnt > 0)) {
      collide_fluid<D>(f, a.cp, rho, ux, uy, uz);
    } else {
      double beta = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
      if (cnt > 0) {
        const int p = a.pid[x];
        beta = __ldg(a.beta_tab + cnt);
        solid_velocity<D>(a.prec + (int64_t)p * prec_stride(D), i, j, k, a.nx, a.ny, a.nz, a.bcx, a.bcy, a.bcz, vx,
                          vy, vz);
      }
      collide_imb<D>(f, a.cp, rho, ux, uy, uz, beta, vx, vy, vz);
      if (EMIT && cnt > 0) {
        const double br = beta * rho;
        store_exchange<D>(a.s, x, br * (vx - ux), br * (vy - uy), br * (vz - uz));
      }
    }
    if (live) {
#pragma unroll
      for (int q = 0; q < Q; ++q) a.fout[(int64_t)q * a.N + x] = f[q];
    }
  }
}

template <int D, int TX, int NSTAGE, bool IMB, bool EMIT, int MINB>
static lbmimb_status launch_one(lbmimb_lattice *h, const TmaStepArgs &a) {
  constexpr int Q = Lat<D>::Q;
  const size_t smem = (size_t)NSTAGE * Q * (TX + 2) * sizeof(double) + 2 * NSTAGE * sizeof(uint64_t);
  auto kern = collide_stream_tma_kernel<D, TX, NSTAGE, IMB, EMIT, MINB>;
  static int ctas_per_sm = 0, num_sms = 0;
  if (ctas_per_sm == 0) {
    LBMIMB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int n = 0;
    LBMIMB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, TX + 32, smem));
    if (n < 1) return fail(LBMIMB_ECUDA, "TMA step kernel does not fit on an SM");
    int dev = 0;
    LBMIMB_CUDA(cudaGetDevice(&dev));
    LBMIMB_CUDA(cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev));
    ctas_per_sm = n;
  }
  unsigned grid = (unsigned)(ctas_per_sm * num_sms);
  if (grid > a.num_tiles) grid = a.num_tiles;
  kern<<<grid, TX + 32, smem, h->stream>>>(a);
  LBMIMB_LAUNCH_CHECK(h, "collide_stream_tma_kernel");
  return LBMIMB_OK;
}

template <int D, int TX, int NSTAGE, int MINB>
static lbmimb_status launch_sel(lbmimb_lattice *h, const TmaStepArgs &a, bool imb, bool emit) {
  if (!imb) return launch_one<D, TX, NSTAGE, false, false, MINB>(h, a);
  if (!emit) return launch_one<D, TX, NSTAGE, true, false, MINB>(h, a);
  return launch_one<D, TX, NSTAGE, true, true, MINB>(h, a);
}

// Returns LBMIMB_OK and sets *done = false when the lattice does not meet the alignment rule
// of the bulk copies (nx even); the caller then uses the plain kernel of lattice.cu.
lbmimb_status launch_collide_stream_tma(lbmimb_lattice *h, bool emit, int variant, bool *done) {
  *done = false;
  if (h->g.nx % 2 != 0 || h->g.nx < 4) return LBMIMB_OK;
  TmaStepArgs a;
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
  a.cp = make_collide_params(h);
  const bool imb = h->P > 0;
  lbmimb_status st;
  auto tiles = [&](int TX) -> bool {
    const int64_t tpr = (h->g.nx + TX - 1) / TX;
    const int64_t nt = tpr * h->g.ny * h->g.nz;
    if (nt > 0x7fffffff) return false;
    a.tiles_per_row = (unsigned)tpr;
    a.num_tiles = (unsigned)nt;
    return true;
  };
  if (h->g.dim == 3) {
    switch (variant) {
      case 11: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<3, 128, 2, 4>(h, a, imb, emit); break;
      case 12: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<3, 128, 4, 2>(h, a, imb, emit); break;
      case 13: if (!tiles(256)) return LBMIMB_OK; st = launch_sel<3, 256, 2, 2>(h, a, imb, emit); break;
      case 14: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<3, 128, 3, 2>(h, a, imb, emit); break;
      default: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<3, 128, 3, 3>(h, a, imb, emit); break;
    }
  } else {
    switch (variant) {
      case 11: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<2, 128, 4, 4>(h, a, imb, emit); break;
      case 12: if (!tiles(256)) return LBMIMB_OK; st = launch_sel<2, 256, 4, 3>(h, a, imb, emit); break;
      case 13: if (!tiles(256)) return LBMIMB_OK; st = launch_sel<2, 256, 3, 4>(h, a, imb, emit); break;
      case 14: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<2, 128, 8, 3>(h, a, imb, emit); break;
      default: if (!tiles(128)) return LBMIMB_OK; st = launch_sel<2, 128, 6, 4>(h, a, imb, emit); break;
    }
  }
  if (st != LBMIMB_OK) return st;
  *done = true;
  return LBMIMB_OK;
}

}  // namespace lbmimb
