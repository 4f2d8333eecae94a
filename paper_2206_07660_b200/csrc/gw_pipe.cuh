// gw_pipe.cuh — building blocks shared by the stage kernels: cp.async stage jobs, mbarrier rings, cluster helpers and the
// complex-tile DMMA passes (small-K GEMMs against an nao x nao matrix held in shared memory).
// Stage 4 runs 256 threads per CTA with a 3-deep cp.async ring (NTHR, NSTAGE below); stages 1 and 3 are warp specialised
// (gw_stage1.cu, gw_stage3.cu) and use the mbarrier ring / setmaxnreg helpers further down.  One CTA per SM everywhere.
#pragma once
#include <cuda.h>
#include "gw_common.cuh"

namespace gwp {

constexpr int NTHR = 256, NSTAGE = 3;
constexpr int PASS_ROWS = 64;   // rows per pass job: one 8-row m-tile per warp

// exact n / d for n*d < 2^32 (d >= 1), without an integer divide in the inner loops
struct FastDiv {
  unsigned d, m;
  __host__ __device__ FastDiv() : d(1), m(0) {}
  __host__ __device__ explicit FastDiv(unsigned dd) : d(dd), m(dd <= 1 ? 0u : (unsigned)((1ull << 32) / dd + 1)) {}
  __device__ __forceinline__ unsigned div(unsigned n) const { return m ? __umulhi(n, m) : n; }
};


__device__ __forceinline__ void cp_async16_zfill(void *smem, const void *gmem, bool ok) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  int n = ok ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(n));
}

// rows [row0, row0+64) of a dense (rows x nao) matrix -> stage[r][ldp]
__device__ __forceinline__ void issue_pass_job(c128 *stage, const c128 *src, int row0, int rows_total, int nao, int ldp) {
  const int nrow = min(PASS_ROWS, rows_total - row0);
  const int total = nrow * nao;
  const c128 *s = src + (size_t)row0 * nao;
  for (int i = threadIdx.x; i < total; i += NTHR) {
    const int r = i / nao, a = i - r * nao;
    cp_async16(stage + r * ldp + a, s + i);
  }
}

// One pass job: this warp's m-tile (8 rows of a flat (Q,x) row index) times the nao x nao matrix held in sG as
// [n][k] (K contiguous, zero padded):  out(row, n) = Σ_k stage[row][k] * sG[n][k].
//   TRANSPOSED = true : row = (Q,x) -> out[(Q*nao + n)*nao + x]   (per-Q transpose)
//   TRANSPOSED = false: out[row*nao + n]
template <int KSP_MAX, bool TRANSPOSED>
__device__ __forceinline__ void pass_compute(const c128 *sStage, const c128 *sG, c128 *out, int row0, int rows_total,
                                             int nao, int ldp, int ksp, int ndt, int w = -1) {
  if (w < 0) w = threadIdx.x >> 5;          // m-tile of this warp within the job
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  if (row0 + 8 * w >= rows_total) return;   // whole m-tile beyond the panel (warp-uniform)
  c128 a[KSP_MAX];
#pragma unroll
  for (int ks = 0; ks < KSP_MAX; ks++)
    if (ks < ksp) a[ks] = sStage[(8 * w + g) * ldp + 4 * ks + c];
  const int row = row0 + 8 * w + g;
  const bool rok = row < rows_total;
  int Q = 0, x = 0;
  if (TRANSPOSED) { Q = row / nao; x = row - Q * nao; }
  for (int nt = 0; nt < ndt; nt++) {
    double cr[2] = {0.0, 0.0}, ci[2] = {0.0, 0.0};
    const c128 *bp = sG + (8 * nt + g) * ldp + c;
#pragma unroll
    for (int ks = 0; ks < KSP_MAX; ks++)
      if (ks < ksp) cmma(cr, ci, a[ks], bp[4 * ks]);
    const int col = 8 * nt + 2 * c;
    if (rok) {
      if (TRANSPOSED) {
        if (col < nao) out[((size_t)Q * nao + col) * nao + x] = make_double2(cr[0], ci[0]);
        if (col + 1 < nao) out[((size_t)Q * nao + col + 1) * nao + x] = make_double2(cr[1], ci[1]);
      } else {
        if (col < nao) out[(size_t)row * nao + col] = make_double2(cr[0], ci[0]);
        if (col + 1 < nao) out[(size_t)row * nao + col + 1] = make_double2(cr[1], ci[1]);
      }
    }
  }
}

// the last n-tile of a pass GEMM is done with plain FMAs when it holds at most two valid columns
__host__ __device__ __forceinline__ bool pass_tail_fma(int nao, int ndt) { return ndt >= 2 && nao - 8 * (ndt - 1) <= 2; }
// executed flops of one 8-row m-tile of a pass GEMM (ndt n-tiles, ksp k-steps): DMMA tiles (4 x 512 flops per k-step) plus the FMA tail
static inline double pass_mtile_flops(int nao, int ndt, int ksp, bool exact_path) {
  if (exact_path && pass_tail_fma(nao, ndt)) return (double)(ndt - 1) * ksp * 2048.0 + 8.0 * (nao - 8 * (ndt - 1)) * 4.0 * ksp * 8.0;
  return (double)ndt * ksp * 2048.0;
}

// pass_compute for ksp == KSP known at compile time (the production shapes: nao = 26 -> 7, nao = 52 -> 13): no branch between
// the DMMAs of an n-tile, every B fragment loaded PF k-steps (4*PF DMMAs) before its use.  Same sums in the same order as
// pass_compute.
// Warp w owns the MT m-tiles 8*(MT*w + i) of a job; every B fragment is loaded once and used by all MT tiles
// (2*MT independent accumulator chains).
template <int KSP, bool TRANSPOSED, int MT>
__device__ __forceinline__ void pass_compute_exact_mt(const c128 *sStage, const c128 *sG, c128 *out, int row0, int rows_total,
                                                      int nao, int ldp, int w, FastDiv fd) {
  constexpr int NDT = (KSP + 1) / 2, PF = 3, NB = PF + 1;
  constexpr bool CACHE_A = KSP * MT <= 8;   // keep the A fragments of the m-tile(s) in registers, else stream them like B
  constexpr int NA = CACHE_A ? KSP : NB;
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  const int rbase = row0 + 8 * MT * w;
  if (rbase >= rows_total) return;          // all m-tiles of this warp beyond the panel (warp-uniform)
  c128 a[MT][NA];
  const c128 *ap[MT];
  c128 *o[MT];
  bool rok[MT];
  int ostride;
#pragma unroll
  for (int i = 0; i < MT; i++) {
    ap[i] = sStage + (8 * (MT * w + i) + g) * ldp + c;
    if (CACHE_A) {
#pragma unroll
      for (int ks = 0; ks < KSP; ks++) a[i][ks] = ap[i][4 * ks];
    }
    const int row = rbase + 8 * i + g;
    rok[i] = row < rows_total;
    if (TRANSPOSED) { const int Q = (int)fd.div((unsigned)row), x = row - Q * nao; o[i] = out + ((size_t)Q * nao + 2 * c) * nao + x; }
    else o[i] = out + (size_t)row * nao + 2 * c;
  }
  ostride = TRANSPOSED ? nao : 1;
  const c128 *bp = sG + g * ldp + c;
  // A last n-tile with only one or two valid columns (nao = 25, 26: two of eight) is not worth four DMMAs per k-step: those columns
  // are formed with plain FP64 FMAs from the same A fragments, each lane summing its own k's, the four lanes of a row then adding up
  const bool tail_fma = pass_tail_fma(nao, NDT);
  const int ndt_run = tail_fma ? NDT - 1 : NDT;
  double cr[MT][2], ci[MT][2];
  {
    // a real loop over the n-tiles (bounded register pressure); B fragments (and, for long K, A fragments) are streamed
    // PF k-steps ahead
#pragma unroll 1
    for (int nt = 0; nt < ndt_run; nt++) {
      const c128 *bq = bp + nt * 8 * ldp;
      c128 b[NB];
#pragma unroll
      for (int ks = 0; ks < PF && ks < KSP; ks++) {
        b[ks % NB] = bq[4 * ks];
        if (!CACHE_A) {
#pragma unroll
          for (int i = 0; i < MT; i++) a[i][ks % NB] = ap[i][4 * ks];
        }
      }
#pragma unroll
      for (int i = 0; i < MT; i++) { cr[i][0] = cr[i][1] = 0.0; ci[i][0] = ci[i][1] = 0.0; }
#pragma unroll
      for (int ks = 0; ks < KSP; ks++) {
        if (ks + PF < KSP) {
          b[(ks + PF) % NB] = bq[4 * (ks + PF)];
          if (!CACHE_A) {
#pragma unroll
            for (int i = 0; i < MT; i++) a[i][(ks + PF) % NB] = ap[i][4 * (ks + PF)];
          }
        }
#pragma unroll
        for (int i = 0; i < MT; i++) cmma(cr[i], ci[i], a[i][CACHE_A ? ks : ks % NB], b[ks % NB]);
      }
      const bool c0 = nt < NDT - 1 || 8 * nt + 2 * c < nao, c1 = nt < NDT - 1 || 8 * nt + 2 * c + 1 < nao;
#pragma unroll
      for (int i = 0; i < MT; i++) {
        if (rok[i] && c0) o[i][0] = make_double2(cr[i][0], ci[i][0]);
        if (rok[i] && c1) o[i][ostride] = make_double2(cr[i][1], ci[i][1]);
        o[i] += 8 * ostride;
      }
    }
    if (tail_fma) {
      const int n0 = 8 * (NDT - 1);
      const c128 *g0 = sG + n0 * ldp + c;                 // rows n0, n0 + 1 of the [n][k] matrix, this lane's k = 4 ks + c
      c128 t0[MT], t1[MT];
#pragma unroll
      for (int i = 0; i < MT; i++) { t0[i] = make_double2(0.0, 0.0); t1[i] = make_double2(0.0, 0.0); }
#pragma unroll
      for (int ks = 0; ks < KSP; ks++) {
        const c128 b0 = g0[4 * ks], b1 = g0[ldp + 4 * ks];
#pragma unroll
        for (int i = 0; i < MT; i++) {
          const c128 av = CACHE_A ? a[i][CACHE_A ? ks : 0] : ap[i][4 * ks];
          cfma(t0[i], av, b0);
          cfma(t1[i], av, b1);
        }
      }
#pragma unroll
      for (int i = 0; i < MT; i++) {
#pragma unroll
        for (int off = 1; off <= 2; off <<= 1) {
          t0[i].x += __shfl_xor_sync(0xffffffffu, t0[i].x, off); t0[i].y += __shfl_xor_sync(0xffffffffu, t0[i].y, off);
          t1[i].x += __shfl_xor_sync(0xffffffffu, t1[i].x, off); t1[i].y += __shfl_xor_sync(0xffffffffu, t1[i].y, off);
        }
        // o[i] points at column n0 + 2c of this lane's row: lane c = 0 stores column n0, lane c = 1 column n0 + 1
        if (rok[i] && c == 0) o[i][0] = t0[i];
        if (rok[i] && c == 1 && n0 + 1 < nao) o[i][-ostride] = t1[i];
      }
    }
  }
}

// "final" job for the K range [a0, a0 + 4*ksp) of one Q: A = Aq[i][a0..] (nao x nao, [i][a]) -> stage[i][ldp];
// B = Bq[a0..][j] (nao x nao, [a][j]) -> [a - a0][ldt]; K beyond nao is zero filled
__device__ __forceinline__ void issue_final_job(c128 *stage, const c128 *Aq, const c128 *Bq, int nao, int ldp, int ldt, int ksp, int naop, int a0) {
  const int kw = 4 * ksp;
  for (int i = threadIdx.x; i < nao * kw; i += NTHR) {
    const int r = i / kw, cc = i - r * kw;
    const bool ok = a0 + cc < nao;
    cp_async16_zfill(stage + r * ldp + cc, ok ? Aq + r * nao + a0 + cc : Aq, ok);
  }
  c128 *sB = stage + naop * ldp;
  for (int i = threadIdx.x; i < kw * nao; i += NTHR) {
    const int r = i / nao;
    const bool ok = a0 + r < nao;
    cp_async16_zfill(sB + r * ldt + (i - r * nao), ok ? Bq + (size_t)a0 * nao + i : Bq, ok);
  }
}

// acc[i][j] += Σ_a A[i][a] B[a][j] for the output tiles owned by this warp (tile = w + 8*ti over an ndt x ndt grid)
template <int NCT>
__device__ __forceinline__ void final_compute(const c128 *stage, double (&sgr)[NCT][2], double (&sgi)[NCT][2], int ldp, int ldt,
                                              int ksp, int ndt, int naop) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const c128 *sA = stage, *sB = stage + naop * ldp;
#pragma unroll
  for (int ti = 0; ti < NCT; ti++) {
    const int tile = w + 8 * ti;
    if (tile < ndt * ndt) {
      const int mi = tile / ndt, nj = tile - mi * ndt;
      const c128 *ap = sA + (8 * mi + g) * ldp + c;
      const c128 *bp = sB + c * ldt + 8 * nj + g;
      for (int ks = 0; ks < ksp; ks++) cmma(sgr[ti], sgi[ti], ap[4 * ks], bp[4 * ks * ldt]);
    }
  }
}

// Straight-line version of final_compute for KS k-steps and an NDT x NDT tile grid known at compile time: all fragments
// of a k-step group are loaded before the DMMAs that use them, the NCT tiles of the warp are interleaved (2*NCT
// independent chains).
template <int KS, int NDT, int NCT>
__device__ __forceinline__ void final_compute_exact(const c128 *stage, double (&sgr)[NCT][2], double (&sgi)[NCT][2], int ldp, int ldt,
                                                    int naop) {
  if (NCT * 8 < NDT * NDT) return;          // never launched with such a pair (the plan picks NCT from ndt)
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const c128 *sA = stage, *sB = stage + naop * ldp;
  const c128 *ap[NCT], *bp[NCT];
  bool on[NCT];
#pragma unroll
  for (int ti = 0; ti < NCT; ti++) {
    const int tile = w + 8 * ti;
    on[ti] = tile < NDT * NDT;
    const int mi = on[ti] ? tile / NDT : 0, nj = on[ti] ? tile - mi * NDT : 0;
    ap[ti] = sA + (8 * mi + g) * ldp + c;
    bp[ti] = sB + c * ldt + 8 * nj + g;
  }
  constexpr int GK = (NCT <= 2) ? 4 : 1;    // k-steps per load group
#pragma unroll
  for (int k0 = 0; k0 < KS; k0 += GK) {
    c128 a[NCT][GK], b[NCT][GK];
#pragma unroll
    for (int ti = 0; ti < NCT; ti++)
#pragma unroll
      for (int kk = 0; kk < GK; kk++)
        if (k0 + kk < KS && on[ti]) { a[ti][kk] = ap[ti][4 * (k0 + kk)]; b[ti][kk] = bp[ti][4 * (k0 + kk) * ldt]; }
#pragma unroll
    for (int kk = 0; kk < GK; kk++)
#pragma unroll
      for (int ti = 0; ti < NCT; ti++)
        if (k0 + kk < KS && on[ti]) cmma(sgr[ti], sgi[ti], a[ti][kk], b[ti][kk]);
  }
}

// store the warp-owned tiles of an nao x nao result, scaled
template <int NCT>
__device__ __forceinline__ void final_store(c128 *out, const double (&sgr)[NCT][2], const double (&sgi)[NCT][2], double pref, int nao, int ndt,
                                            bool conj = false) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const double prefi = conj ? -pref : pref;
#pragma unroll
  for (int ti = 0; ti < NCT; ti++) {
    const int tile = w + 8 * ti;
    if (tile < ndt * ndt) {
      const int mi = tile / ndt, nj = tile - mi * ndt;
      const int i = 8 * mi + g, j = 8 * nj + 2 * c;
      if (i < nao) {
        if (j < nao) out[i * nao + j] = make_double2(pref * sgr[ti][0], prefi * sgi[ti][0]);
        if (j + 1 < nao) out[i * nao + j + 1] = make_double2(pref * sgr[ti][1], prefi * sgi[ti][1]);
      }
    }
  }
}

// load the warp-owned tiles of an nao x nao array into the accumulators (the inverse of final_store with pref = 1)
template <int NCT>
__device__ __forceinline__ void final_load(const c128 *in, double (&sgr)[NCT][2], double (&sgi)[NCT][2], int nao, int ndt) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
#pragma unroll
  for (int ti = 0; ti < NCT; ti++) {
    const int tile = w + 8 * ti;
    if (tile < ndt * ndt) {
      const int mi = tile / ndt, nj = tile - mi * ndt;
      const int i = 8 * mi + g, j = 8 * nj + 2 * c;
      if (i < nao) {
        if (j < nao) { sgr[ti][0] = in[i * nao + j].x; sgi[ti][0] = in[i * nao + j].y; }
        if (j + 1 < nao) { sgr[ti][1] = in[i * nao + j + 1].x; sgi[ti][1] = in[i * nao + j + 1].y; }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Warp-specialised pipeline: one producer warp fills a ring of stage buffers with cp.async (completion tracked by an
// mbarrier per stage), NCONS consumer warps wait on "full", compute on FP64 tensor cores, and release "empty".
// No CTA-wide barrier in steady state.
// ---------------------------------------------------------------------------------------------------------------
constexpr int NCONS = 8;                 // consumer warps
constexpr int NPROD_THR = 128;           // producer threads (one warpgroup)
constexpr int NTHR_WS = 32 * (NCONS + 4);   // consumers = two warpgroups; producer = warp NCONS of a third warpgroup

// register rebalancing between the producer and consumer warpgroups (all warps of a warpgroup must execute it)
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(N)); }

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (count must be pre-accounted: .noinc)
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t *bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}

// ---- thread-block-cluster helpers (a kernel launched without cluster dimensions is a cluster of one) ----
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
// arrive (release at cluster scope) on the mbarrier at the same shared-memory offset in CTA `rank` of this cluster
__device__ __forceinline__ void mbar_arrive_cluster(uint64_t *bar, unsigned rank) {
  unsigned remote;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(remote) : "r"(smem_u32(bar)), "r"(rank));
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];\n" ::"r"(remote) : "memory");
}
// wait with acquire at cluster scope (the arrivals may come from the peer CTA)
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAITC:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONEC;\n"
      "bra LAB_WAITC;\n"
      "DONEC:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

struct Ring {
  uint64_t *full, *empty;   // [nstage] each
  int nstage;
  unsigned it = 0;          // stage index of the next job (same sequence on both sides)
  unsigned ph = 0;          // parity of the current round (no integer division per job)
  __device__ __forceinline__ int stage() const { return (int)it; }
  __device__ __forceinline__ void advance() { if (++it == (unsigned)nstage) { it = 0; ph ^= 1u; } }
  // producer side
  __device__ __forceinline__ int acquire() { const int s = stage(); mbar_wait(empty + s, ph ^ 1u); return s; }
  __device__ __forceinline__ void commit() { cp_async_arrive_noinc(full + stage()); advance(); }
  // consumer side
  __device__ __forceinline__ int wait() { const int s = stage(); mbar_wait(full + s, ph); return s; }
  __device__ __forceinline__ void release() { __syncwarp(); if ((threadIdx.x & 31) == 0) mbar_arrive(empty + stage()); advance(); }
};

// ---- TMA (cp.async.bulk.tensor) and L2 eviction policies, shared by stages 1 and 3 ----
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap *map, int x, int y, uint64_t *bar, uint64_t pol) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;\n"
               ::"r"(dst), "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// the slabs are read exactly once after they are written (evict first); the V blocks are shared by every CTA working on the same
// q / k (evict last)
__device__ __forceinline__ uint64_t policy_evict_first() { uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p)); return p; }
__device__ __forceinline__ uint64_t policy_evict_last() { uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p)); return p; }
__device__ __forceinline__ uint64_t policy_evict_normal() { uint64_t p; asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;\n" : "=l"(p)); return p; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda; the entry point's address is a
// process-wide constant, cached).  View: [rows][ncplx complex] row-major matrix of doubles, box = box_rows x 8 complex (128 bytes),
// 128-byte swizzle, zero fill outside the array.
static inline int make_tensor_map(CUtensorMap *map, const void *base, size_t rows, int ncplx, int box_rows) {
  typedef CUresult (*Fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                         const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static Fn fn = nullptr;
  if (!fn) {
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      return (int)cudaErrorNotSupported;
    }
    fn = (Fn)ptr;
  }
  const cuuint64_t gdim[2] = {(cuuint64_t)2 * ncplx, (cuuint64_t)rows};
  const cuuint64_t gstr[1] = {(cuuint64_t)ncplx * 16};
  const cuuint32_t box[2] = {16u, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
}

// producer-warpgroup versions of the job issue functions (128 threads: threadIdx.x - 32*NCONS)
__device__ __forceinline__ void ws_issue_rows(c128 *stage, const c128 *src, int row0, int rows_total, int nao, int ldp, FastDiv fd) {
  const int nrow = min(PASS_ROWS, rows_total - row0);
  const int total = nrow * nao;
  const c128 *s = src + (size_t)row0 * nao;
  for (int i = threadIdx.x - 32 * NCONS; i < total; i += NPROD_THR) {
    const int r = (int)fd.div((unsigned)i), a = i - r * nao;
    cp_async16(stage + r * ldp + a, s + i);
  }
}
// K range [a0, a0 + 4*ksp) of one Q: A = Aq[i][a0..] -> stage[i][ldp]; B = Bq[a0..][j] -> [a - a0][ldt]; K beyond nao is zero filled
__device__ __forceinline__ void ws_issue_final(c128 *stage, const c128 *Aq, const c128 *Bq, int nao, int ldp, int ldt, int ksp, int naop, FastDiv fd, FastDiv fk, int a0) {
  const int lane = threadIdx.x - 32 * NCONS;
  const int kw = 4 * ksp;
  for (int i = lane; i < nao * kw; i += NPROD_THR) {
    const int r = (int)fk.div((unsigned)i), cc = i - r * kw;
    const bool ok = a0 + cc < nao;
    cp_async16_zfill(stage + r * ldp + cc, ok ? Aq + r * nao + a0 + cc : Aq, ok);
  }
  c128 *sB = stage + naop * ldp;
  for (int i = lane; i < kw * nao; i += NPROD_THR) {
    const int r = (int)fd.div((unsigned)i);
    const bool ok = a0 + r < nao;
    cp_async16_zfill(sB + r * ldt + (i - r * nao), ok ? Bq + (size_t)a0 * nao + i : Bq, ok);
  }
}
// nao x nao matrix -> sG[r][ldp] (TRANSPOSE: sG[c][ldp + r])
template <bool TRANSPOSE>
__device__ __forceinline__ void ws_issue_matrix(c128 *sG, const c128 *src, int nao, int ldp, FastDiv fd) {
  const int n2 = nao * nao;
  for (int i = threadIdx.x - 32 * NCONS; i < n2; i += NPROD_THR) {
    const int r = (int)fd.div((unsigned)i), cc = i - r * nao;
    cp_async16(TRANSPOSE ? sG + cc * ldp + r : sG + r * ldp + cc, src + i);
  }
}

// consumer-side pass: like pass_compute but the warp index is the consumer warp index (0..7) and no early return
// before the ring release is needed (caller releases).
// pass-geometry shared by the stages
struct PassGeom { int ldp, ksp, ksp_max, ndt, naop, ldt, nct; bool ok; };
static inline PassGeom pass_geom(int nao) {
  PassGeom g;
  g.ksp = (nao + 3) / 4;
  g.ok = g.ksp <= 16;
  g.ksp_max = g.ksp <= 7 ? 7 : (g.ksp <= 13 ? 13 : 16);
  g.ndt = (nao + 7) / 8;
  g.naop = 8 * g.ndt;
  int r4 = g.ksp * 4; if (r4 % 8 == 0) r4 += 4;   // ≡ 4 (mod 8): conflict-free K-contiguous fragments
  g.ldp = r4;
  g.ldt = g.naop + 2;                              // ≡ 2 (mod 8): conflict-free K-major fragments
  g.nct = (g.ndt * g.ndt + 7) / 8 <= 2 ? 2 : 8;
  return g;
}
static inline int gw_num_sms() {
  int dev = 0, nsm = 148;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) { cudaGetLastError(); nsm = 148; }
  return nsm;
}

}  // namespace gwp
