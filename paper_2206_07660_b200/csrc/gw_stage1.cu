// gw_stage1.cu — stage 1, Eq. 28b (Algorithm 1 first k loop):
//
//   P0t[t][q][Q][Q'] = -(s/N_k) Σ_k Σ_abcd V[k][k+q][Q][d][a] G[t][k+q][a][b] V[k+q][k][Q'][b][c] G[tbar][k][c][d]
//
// Formulation used here (exact algebra, no input symmetry assumed):
//   Z_k[Q][(b,c)] = Σ_d Σ_a G[tbar][k][c][d] V[k][k+q][Q][d][a] G[t][k+q][a][b]        (two small GEMMs, K = nao)
//   P0t[Q][Q']    = -(s/N_k) Σ_k Σ_(b,c) Z_k[Q][(b,c)] · V[k+q][k][Q'][(b,c)]            (one GEMM,  K = N_k·nao²)
// so the second operand is the raw V block (rows Q', K contiguous), never transformed.
//
// Work decomposition: a work item is a row panel [TM = 32 Q-rows] x [all naux Q'] of one (t,q); it is owned by one CTA
// (naux <= 128) or by a cluster of two or four CTAs that split the Q' columns (naux <= 256 / 512), and its accumulators stay in
// registers over the whole k loop (the k-sum is inside the K loop; no cross-CTA reduction, deterministic).
// A CTA is warp specialised (16 warps, register budgets rebalanced with setmaxnreg):
//   main warps 0-7   : acc[Q][Q'] += Σ_K Z[Q][K] V[k+q][k][Q'][K] on FP64 tensor cores (DMMA.8x8x4), operands streamed through an
//                      mbarrier-tracked TMA ring.  Complex tile products use the 3M scheme: three real DMMAs per complex
//                      8x8x4 product, K1 += Ar·Br, K2 += Ai·Bi, K3 += (Ar+Ai)·(Br+Bi); Re = K1 − K2, Im = K3 − K1 − K2, with
//                      three real accumulator sets per tile (warp tile 2 x 4 tiles) and the operand sums formed in registers
//   pass warps 8-11  : produce Z for the NEXT k while the main warps consume the current one
//                        pass 1:  Xt[Q][b][d] = Σ_a V[k][k+q][Q][d][a] G[t][k+q][a][b]      rows (Q,d) flat
//                        pass 2:  Z [Q][b][c] = Σ_d Xt[Q][b][d] G[tbar][k][c][d]            rows (Q,b) flat; in place
//                      (in a cluster each CTA transforms half of the panel rows)
//   producer warps   : one thread of warp 12 feeds the main ring with TMA (cp.async.bulk.tensor.2d, 128-byte swizzle: one box
//                      of Z rows and one box of V[k+q][k] rows per job, completion by mbarrier expect-tx); warp 15 feeds the
//                      pass ring and the G matrices with cp.async (26-wide rows need padded destinations)
// Xt/Z live in two per-cluster slabs of the workspace (TM·nao² complex each, double buffered over k, written and
// re-read within ~100 µs, i.e. L2 resident); they never exist as a [t][q][k] tensor.
#include "gw_pipe.cuh"

namespace s1 {

using gwp::FastDiv;
constexpr int NMAINW = 8, NPASSW = 4;                 // main / pass warps; warps 12..15 are the producer warpgroup
constexpr int NTHR1 = 32 * 16;
constexpr int T_MPROD = 32 * 12, N_MPROD = 96;        // main-ring producer threads [384, 480)
constexpr int T_PPROD = 32 * 15, N_PPROD = 32;        // pass-ring producer threads [480, 512)
constexpr int NST_MAX = 8, PST_MAX = 4;
constexpr int KC = 8;           // complex K per main job (one 128-byte row per operand row)
constexpr int MT_W = 2;         // m-tiles per main warp
// n-tiles per main warp: 3M scheme 4 (three accumulator sets; 4 column groups x 4 = 16 n-tiles = 128 columns per CTA), 4-real-GEMM
// scheme 7 (two accumulator sets; 28 n-tiles = 224 columns per CTA)
constexpr int NJ_3M = 4, NJ_4M = 7;
constexpr int TM = 32;          // panel rows
constexpr int REG_MAIN = 176, REG_PASS = 120, REG_PROD = 40;   // 256*176 + 128*120 + 128*40 = 65536

struct Params {
  GwDims d;
  const c128 *V, *G;
  c128 *P0t, *scratch;
  int cs;                // CTAs per cluster = column splits of the panel
  int rsplit;            // cs == 2: panel rows transformed by CTA 0 (CTA 1 takes the other TM - rsplit): 16, or fewer when CTA 0 owns one more
                         // n-tile of the main GEMM than CTA 1, so that main + pass work of the two CTAs balance
  int ncp;               // column passes: an item covers cs*8*ntc columns of its Q panel (ncp > 1 only for naux > 448; Z is
                         // then produced once per pass)
  int nqt, nitems;       // Q tiles per (t,q); total work items
  int nteff;             // tau nodes evaluated: ntau, or ceil(ntau/2) under GW_SYM_TR (the rest is mirrored)
  int herm;              // GW_SYM_TR: P0t[t][q] is Hermitian, only the column tiles up to the panel's diagonal block are computed
  int nqeff;             // q points evaluated: nq, or the q <= -q half under GW_SYM_TR (P0[-q] = P0[q]^T is copied)
  short qirr[128];       // the evaluated q points when nqeff < nq
  __device__ __forceinline__ int qof(int i) const { return nqeff < d.nq ? (int)qirr[i] : i; }
  int ldp, ksp, ndt;     // pass smem row stride (complex), k-steps = ceil(nao/4), n-tiles over nao
  int nt, ntc;           // n-tiles over naux; n-tiles per CTA
  int main_units, pass_units;   // complex elements per main / pass stage buffer
  int main_off;                 // offset of the main ring in the (1024-byte aligned) dynamic shared memory, complex elements
  int prows;                    // rows per pass job: 8 * (m-tiles per pass warp) * 4 pass warps
  int nstage, pstage, ng;       // ring depths; number of G buffers (2: G[t] and G[tbar] side by side, 1: time shared)
  size_t slab_units;     // complex elements per slab (two slabs per cluster)
  FastDiv fd_nao;
};

using gwp::Ring; using gwp::tma_load_2d; using gwp::mbar_expect_tx; using gwp::policy_evict_first; using gwp::policy_evict_last;

// rows [row0, row0+prows) of a dense (rows x nao) matrix -> stage[r][ldp]   (pass-ring producer warp)
__device__ __forceinline__ void issue_rows(c128 *stage, const c128 *src, int row0, int rows_total, int nao, int ldp, FastDiv fd, int prows) {
  const int nrow = min(prows, rows_total - row0);
  const int total = nrow * nao;
  const c128 *s = src + (size_t)row0 * nao;
  for (int i = threadIdx.x - T_PPROD; i < total; i += N_PPROD) {
    const int r = (int)fd.div((unsigned)i), a = i - r * nao;
    cp_async16(stage + r * ldp + a, s + i);
  }
}
// nao x nao matrix -> sG[r][ldp] (TRANSPOSE: sG[c][ldp + r])
template <bool TRANSPOSE>
__device__ __forceinline__ void issue_matrix(c128 *sG, const c128 *src, int nao, int ldp, FastDiv fd) {
  const int n2 = nao * nao;
  for (int i = threadIdx.x - T_PPROD; i < n2; i += N_PPROD) {
    const int r = (int)fd.div((unsigned)i), cc = i - r * nao;
    cp_async16(TRANSPOSE ? sG + cc * ldp + r : sG + r * ldp + cc, src + i);
  }
}

// main warps: one main job (KC/4 k-steps) for this warp's MTW x NJM tiles (n-tiles NSTRIDE apart); all fragment loads
// hoisted per k-step.  S3M: acc[0] += Ar Br, acc[1] += Ai Bi, acc[2] += (Ar+Ai)(Br+Bi); else acc[0] / acc[1] = real / imaginary
// part by four real DMMAs.
template <bool S3M, int NJM, int NSTRIDE, int MTW, int NJ>
__device__ __forceinline__ void main_compute(const c128 *sAw, const c128 *sBw, double (&acc)[S3M ? 3 : 2][MT_W][NJ][2], int c, int sw) {
#pragma unroll
  for (int ks = 0; ks < KC / 4; ks++) {
    const int u = (4 * ks + c) ^ sw;
    c128 a[MTW], b[NJM];
#pragma unroll
    for (int i = 0; i < MTW; i++) a[i] = sAw[i * 8 * KC + u];
#pragma unroll
    for (int jn = 0; jn < NJM; jn++) b[jn] = sBw[jn * NSTRIDE * 8 * KC + u];
    if constexpr (S3M) {
      double as[MTW];
#pragma unroll
      for (int i = 0; i < MTW; i++) as[i] = a[i].x + a[i].y;
#pragma unroll
      for (int jn = 0; jn < NJM; jn++) {
        const double bs = b[jn].x + b[jn].y;
#pragma unroll
        for (int i = 0; i < MTW; i++) {
          dmma884(acc[0][i][jn][0], acc[0][i][jn][1], a[i].x, b[jn].x);
          dmma884(acc[1][i][jn][0], acc[1][i][jn][1], a[i].y, b[jn].y);
          dmma884(acc[2][i][jn][0], acc[2][i][jn][1], as[i], bs);
        }
      }
    } else {
#pragma unroll
      for (int jn = 0; jn < NJM; jn++)
#pragma unroll
        for (int i = 0; i < MTW; i++) cmma(acc[0][i][jn], acc[1][i][jn], a[i], b[jn]);
    }
  }
}

// njm (1..NJ) is warp-uniform: pick the straight-line instance
template <bool S3M, int NSTRIDE, int MTW, int NJ, int NJM = NJ>
__device__ __forceinline__ void main_dispatch(int njm, const c128 *sAw, const c128 *sBw, double (&acc)[S3M ? 3 : 2][MT_W][NJ][2], int c, int sw) {
  if (njm == NJM) main_compute<S3M, NJM, NSTRIDE, MTW, NJ>(sAw, sBw, acc, c, sw);
  else if constexpr (NJM > 1) main_dispatch<S3M, NSTRIDE, MTW, NJ, NJM - 1>(njm, sAw, sBw, acc, c, sw);
}

// decode a work item: Q-tile index fastest (a cluster's item sequence cycles through full and ragged panels, so the short,
// bandwidth-hungry ragged panels are spread over the whole run), then t, then q slowest (concurrent clusters share the V
// blocks of one q in L2)
struct Item { int t, ql, Q0, tm_rows, cbase; };   // cbase: first n-tile of the item's column pass (per cluster)
__device__ __forceinline__ Item decode_item(const Params &P, int item) {
  const GwDims &d = P.d;
  Item it;
  const int qt = item % P.nqt; int r = item / P.nqt;
  it.cbase = (r % P.ncp) * P.cs * P.ntc; r /= P.ncp;
  it.t = r % P.nteff; it.ql = P.qof(r / P.nteff); it.Q0 = qt * TM; it.tm_rows = min(TM, d.naux - it.Q0);
  return it;
}

template <int KSP_MAX, bool S3M>
__global__ void __launch_bounds__(NTHR1, 1) p0_kernel(const Params P, const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmZ) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // the TMA destinations (128-byte swizzle) need 1024-byte alignment: the launch asks for 1 KB of slack
  c128 *smem = reinterpret_cast<c128 *>(smem_raw + ((1024u - (gwp::smem_u32(smem_raw) & 1023u)) & 1023u));
  const GwDims d = P.d;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao, ldp = P.ldp, naop = 8 * P.ndt;
  c128 *sG0 = smem;                                       // pass 1: sG0[b][a] = G[t][k+q][a][b]
  c128 *sG1 = sG0 + (P.ng == 2 ? naop * ldp : 0);         // pass 2: sG1[c][d] = G[tbar][k][c][d]  (== sG0 when time shared)
  c128 *sPass = smem + P.ng * naop * ldp;                 // pstage x pass_units
  c128 *sMain = smem + P.main_off;                        // nstage x main_units (1024-byte aligned stages)
  __shared__ uint64_t bars[2 * NST_MAX + 2 * PST_MAX + 6];
  uint64_t *full_m = bars, *empty_m = bars + NST_MAX, *full_p = bars + 2 * NST_MAX, *empty_p = full_p + PST_MAX;
  uint64_t *bar_g = empty_p + PST_MAX, *bar_phase = bar_g + 1, *zready = bar_g + 2, *zfree = bar_g + 4;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int cs = P.cs;
  const unsigned rank = cs > 1 ? gwp::cluster_ctarank() : 0u;
  const int cid = blockIdx.x / cs, ncl = gridDim.x / cs;
  c128 *slab0 = P.scratch + (size_t)cid * 2 * P.slab_units;
  const size_t vb = (size_t)naux * n2;
  const int nmain = (n2 + KC - 1) / KC;
  const int nkk = d.nk * d.ns;                            // k loop of Eq. 28b with the spin sum inside
  // panel rows transformed by this CTA's pass warps
  const int rows_cta = cs == 2 ? (rank == 0 ? P.rsplit : TM - P.rsplit) : TM / cs;
  const int r0 = cs == 2 ? (rank == 0 ? 0 : P.rsplit) : (int)rank * rows_cta;

  // zero all dynamic smem once (pad rows/columns must hold finite values: they meet zero operands); init barriers
  {
    const int tot = P.main_off + P.nstage * P.main_units;
    for (int i = threadIdx.x; i < tot; i += NTHR1) smem[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
      for (int i = 0; i < P.nstage; i++) { gwp::mbar_init(full_m + i, 1); gwp::mbar_init(empty_m + i, NMAINW); }
      for (int i = 0; i < P.pstage; i++) { gwp::mbar_init(full_p + i, N_PPROD); gwp::mbar_init(empty_p + i, NPASSW); }
      gwp::mbar_init(bar_g, N_PPROD);
      gwp::mbar_init(bar_phase, NPASSW);
      for (int i = 0; i < 2; i++) { gwp::mbar_init(zready + i, NPASSW * cs); gwp::mbar_init(zfree + i, NMAINW * cs); }
      asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
  }
  __syncthreads();
  if (cs > 1) gwp::cluster_sync_all();

  if (w >= NMAINW + NPASSW) {
    // ====================================== producer warpgroup ======================================
    gwp::reg_dec<REG_PROD>();
    if (w < 15) {
      // ---- main-ring producer: ONE thread issues two TMA box loads per job (Z rows of the current k; raw V[k+q][k] rows of
      //      this CTA's columns) and arms the stage's mbarrier with the byte count ----
      if (w == NMAINW + NPASSW && lane == 0) {
        Ring rm; rm.full = full_m; rm.empty = empty_m; rm.nstage = P.nstage; rm.it = 0; rm.ph = 0;
        unsigned kit = 0;
        const uint64_t polA = policy_evict_first(), polB = policy_evict_last();
        const unsigned bytesA = TM * KC * 16u, bytesB = 8u * (unsigned)P.ntc * KC * 16u;
        for (int item = cid; item < P.nitems; item += ncl) {
          const Item it = decode_item(P, item);
          const int q = d.q0 + it.ql;
          for (int kk = 0; kk < nkk; kk++, kit++) {
            const int k = d.ns == 4 ? kk >> 2 : (d.ns == 2 ? kk >> 1 : kk);   // spin term innermost: the V blocks of (k, q) serve all of them
            const int kq = gw_kadd(d, k, q);
            const int yB = (int)gw_vbwd(d, it.ql, k, kq) * naux + 8 * (it.cbase + (int)rank * P.ntc);   // row of V viewed as [blocks*naux][nao²]
            const int yA = (cid * 2 + (int)(kit & 1u)) * TM;           // row of the slab area viewed as [2*nclusters*TM][nao²]
            if (cs > 1) gwp::mbar_wait_cluster(zready + (kit & 1u), (kit >> 1) & 1u);
            else gwp::mbar_wait(zready + (kit & 1u), (kit >> 1) & 1u);
            asm volatile("fence.proxy.async.global;\n" ::: "memory");   // Z was written through the generic proxy
            for (int j = 0; j < nmain; j++) {
              const int s = rm.acquire();
              const unsigned dst = gwp::smem_u32(sMain + s * P.main_units);
              mbar_expect_tx(full_m + s, bytesA + bytesB);
              tma_load_2d(dst, &tmZ, 2 * KC * j, yA, full_m + s, polA);
              tma_load_2d(dst + bytesA, &tmV, 2 * KC * j, yB, full_m + s, polB);
              rm.advance();
            }
          }
        }
      }
    } else {
      // ---- pass-ring producer (32 threads): G matrices, V[k][k+q] rows (pass 1), Xt rows from the slab (pass 2) ----
      Ring rp; rp.full = full_p; rp.empty = empty_p; rp.nstage = P.pstage; rp.it = 0; rp.ph = 0;
      unsigned kit = 0, ph = 0;
      for (int item = cid; item < P.nitems; item += ncl) {
        const Item it = decode_item(P, item);
        const int q = d.q0 + it.ql;
        const int my_rows = max(0, min(it.tm_rows, r0 + rows_cta) - r0) * nao, npass = (my_rows + P.prows - 1) / P.prows;
        for (int kk = 0; kk < nkk; kk++, kit++) {
          // spin term (sigma, sigma') of Eq. 28b: G^{sigma sigma'} at k+q (block b1) and G^{sigma' sigma} at k (block b2).  One block:
          // b1 = b2 = 0; collinear: b1 = b2 = sigma; two-component: b1 = 2 sigma + sigma', b2 = its spin transpose
          const int k = d.ns == 4 ? kk >> 2 : (d.ns == 2 ? kk >> 1 : kk);
          const int b1 = d.ns == 4 ? kk & 3 : (d.ns == 2 ? kk & 1 : 0), b2 = d.ns == 4 ? ((b1 & 1) << 1) | (b1 >> 1) : b1;
          const int kq = gw_kadd(d, k, q);
          const c128 *Vt = P.V + gw_vfwd(d, it.ql, k, kq) * vb + (size_t)(it.Q0 + r0) * n2;
          const c128 *Xs = slab0 + (size_t)(kit & 1u) * P.slab_units + (size_t)r0 * n2;
          const size_t gstride = (size_t)d.ntau * d.nk * n2;           // one spin block of G[t][k]
          const c128 *Gt = P.G + b1 * gstride + ((size_t)it.t * d.nk + kq) * n2, *Gm = P.G + b2 * gstride + ((size_t)(d.ntau - 1 - it.t) * d.nk + k) * n2;
          // pass 1 (its G buffer was last read two phases ago; a time-shared buffer must wait for the previous phase)
          if (P.ng == 2) issue_matrix<true>(sG0, Gt, nao, ldp, P.fd_nao);
          if (ph > 0) gwp::mbar_wait(bar_phase, (ph - 1) & 1u);
          if (P.ng == 1) issue_matrix<true>(sG0, Gt, nao, ldp, P.fd_nao);
          gwp::cp_async_arrive_noinc(bar_g);
          for (int j = 0; j < npass; j++) {
            const int s = rp.acquire();
            issue_rows(sPass + s * P.pass_units, Vt, j * P.prows, my_rows, nao, ldp, P.fd_nao, P.prows);
            rp.commit();
          }
          ph++;
          // pass 2: reads the Xt rows written by pass 1
          if (P.ng == 2) issue_matrix<false>(sG1, Gm, nao, ldp, P.fd_nao);
          gwp::mbar_wait(bar_phase, (ph - 1) & 1u);
          if (P.ng == 1) issue_matrix<false>(sG1, Gm, nao, ldp, P.fd_nao);
          gwp::cp_async_arrive_noinc(bar_g);
          for (int j = 0; j < npass; j++) {
            const int s = rp.acquire();
            issue_rows(sPass + s * P.pass_units, Xs, j * P.prows, my_rows, nao, ldp, P.fd_nao, P.prows);
            rp.commit();
          }
          ph++;
        }
      }
      asm volatile("cp.async.wait_all;\n" ::: "memory");
    }
  } else if (w >= NMAINW) {
    // ========================================= pass warps =========================================
    if constexpr (REG_PASS > 65536 / NTHR1) gwp::reg_inc<REG_PASS>(); else gwp::reg_dec<REG_PASS>();
    // m-tile slot of this warp in a pass job.  Pass warp 8 + s runs on SM sub-partition s (each has its own FP64 pipe,
    // profiles/r02_fp64_subcores.md); sub-partition 0 also carries the main-ring producer and, in CTA 0 of a cluster with an odd n-tile
    // count, a main warp with one more n-tile.  When a CTA's rows do not fill the last pass job, the last slots are the empty ones: the
    // warp of sub-partition 0 takes the last slot (measured on config P: stage 1 272.0 -> 266.6 ms).
    const int wp = (w - NMAINW + NPASSW - 1) & (NPASSW - 1);
    constexpr int PMT = KSP_MAX <= 8 ? 2 : 1;          // m-tiles per pass warp on the exact path (prows = 32*PMT there)
    Ring rp; rp.full = full_p; rp.empty = empty_p; rp.nstage = P.pstage; rp.it = 0; rp.ph = 0;
    unsigned kit = 0, ph = 0;
    for (int item = cid; item < P.nitems; item += ncl) {
      const Item it = decode_item(P, item);
      const int my_rows = max(0, min(it.tm_rows, r0 + rows_cta) - r0) * nao, npass = (my_rows + P.prows - 1) / P.prows;
      for (int kk = 0; kk < nkk; kk++, kit++) {
        c128 *Xs = slab0 + (size_t)(kit & 1u) * P.slab_units + (size_t)r0 * n2;
        // this slab was read by the main GEMM of iteration kit-2
        if (kit >= 2) {
          if (cs > 1) gwp::mbar_wait_cluster(zfree + (kit & 1u), ((kit >> 1) - 1u) & 1u);
          else gwp::mbar_wait(zfree + (kit & 1u), ((kit >> 1) - 1u) & 1u);
        }
        gwp::mbar_wait(bar_g, ph & 1u);
        for (int j = 0; j < npass; j++) {
          const int s = rp.wait();
          if (P.ksp == KSP_MAX) gwp::pass_compute_exact_mt<KSP_MAX, true, PMT>(sPass + s * P.pass_units, sG0, Xs, j * P.prows, my_rows, nao, ldp, wp, P.fd_nao);
          else gwp::pass_compute<KSP_MAX, true>(sPass + s * P.pass_units, sG0, Xs, j * P.prows, my_rows, nao, ldp, P.ksp, P.ndt, wp);
          rp.release();
        }
        __threadfence(); __syncwarp();
        if (lane == 0) gwp::mbar_arrive(bar_phase);
        ph++;
        gwp::mbar_wait(bar_g, ph & 1u);
        for (int j = 0; j < npass; j++) {
          const int s = rp.wait();
          if (P.ksp == KSP_MAX) gwp::pass_compute_exact_mt<KSP_MAX, false, PMT>(sPass + s * P.pass_units, sG1, Xs, j * P.prows, my_rows, nao, ldp, wp, P.fd_nao);
          else gwp::pass_compute<KSP_MAX, false>(sPass + s * P.pass_units, sG1, Xs, j * P.prows, my_rows, nao, ldp, P.ksp, P.ndt, wp);
          rp.release();
        }
        __threadfence(); __syncwarp();
        if (lane == 0) {
          gwp::mbar_arrive(bar_phase);
          if (cs > 1) { for (int r = 0; r < cs; r++) gwp::mbar_arrive_cluster(zready + (kit & 1u), (unsigned)r); }
          else gwp::mbar_arrive(zready + (kit & 1u));
        }
        ph++;
      }
    }
  } else {
    // ========================================= main warps =========================================
    gwp::reg_inc<REG_MAIN>();
    constexpr int NJ = S3M ? NJ_3M : NJ_4M, NACC = S3M ? 3 : 2;
    const int g = lane >> 2, c = lane & 3;
    // TMA 128-byte swizzle: 16-byte unit u of row r sits at u ^ (r & 7).  Fragment lane group g reads matrix row rho(g) of its
    // 8-row tile, so that the two rows of a quarter-warp differ in bit 2 (conflict-free); the accumulator rows / columns are
    // permuted accordingly in the epilogue.
    const int rho = (g >> 1) + 4 * (g & 1);
    const int sw = rho;
    Ring rm; rm.full = full_m; rm.empty = empty_m; rm.nstage = P.nstage; rm.it = 0; rm.ph = 0;
    unsigned kit = 0;
    for (int item = cid; item < P.nitems; item += ncl) {
      const Item it = decode_item(P, item);
      const int col0 = 8 * (it.cbase + (int)rank * P.ntc);    // first Q' column of this CTA in this item
      const int ncols = max(0, min(naux - col0, 8 * P.ntc));
      const int ntc_mine = (ncols + 7) / 8;
      const int mtc = (it.tm_rows + 7) / 8;
      // tile ownership.  Full panels: warp w owns m-tiles 2*mh, 2*mh+1 (mh = w >> 2) and every 4th n-tile, starting at column group
      // noff.  Group 0 is the one with an extra n-tile when the count is not a multiple of four; it goes to warps 1 and 6, i.e. to SM
      // sub-partitions 1 and 2, which carry no producer warp (sub-partition 0: the TMA issuer, 3: the cp.async producer).  Measured on
      // config Q: stage 1 4 221 -> 4 186 ms against group 0 on sub-partitions 0 and 1; level on config P.  Ragged last panel
      // (<= 16 rows): all eight warps share m-tiles 0 (and 1), every 8th n-tile each, so the panel costs time in proportion
      // to its rows instead of a full panel's.
      const bool narrow = mtc <= 2;
      const int mh = narrow ? 0 : (w >> 2);
      const int noff = narrow ? w : (((w & 3) - mh + 3) & 3);
      const int nstride = narrow ? 8 : 4;
      const int mtw = (narrow && mtc == 1) ? 1 : MT_W;
      // Hermitian mode: columns right of the panel's diagonal block come from the mirror writes of the later panels
      const int ntc_item = P.herm ? min(ntc_mine, max(0, it.Q0 + TM - col0 + 7) / 8) : ntc_mine;
      const int njm = (ntc_item > noff) ? (ntc_item - noff + nstride - 1) / nstride : 0;
      const bool active = (mh * MT_W < mtc) && njm > 0;
      double acc[NACC][MT_W][NJ][2];
#pragma unroll
      for (int x = 0; x < NACC; x++)
#pragma unroll
        for (int i = 0; i < MT_W; i++)
#pragma unroll
          for (int j = 0; j < NJ; j++) acc[x][i][j][0] = acc[x][i][j][1] = 0.0;

      for (int kk = 0; kk < nkk; kk++, kit++) {
        for (int j = 0; j < nmain; j++) {
          const int s = rm.wait();
          if (active) {
            const c128 *sAw = sMain + s * P.main_units + (8 * mh * MT_W + rho) * KC;
            const c128 *sBw = sMain + s * P.main_units + TM * KC + (8 * noff + rho) * KC;
            // narrow panels: njm <= ceil(4 NJ / 8)
            if (narrow) {
              if (mtw == 1) main_dispatch<S3M, 8, 1, NJ, (NJ + 1) / 2>(njm, sAw, sBw, acc, c, sw);
              else main_dispatch<S3M, 8, 2, NJ, (NJ + 1) / 2>(njm, sAw, sBw, acc, c, sw);
            } else main_dispatch<S3M, 4, MT_W, NJ>(njm, sAw, sBw, acc, c, sw);
          }
          rm.release();
        }
        // every cp.async read of this k's slab has landed: hand it back to the pass warps (of all CTAs in the cluster)
        if (lane == 0) {
          if (cs > 1) { for (int r = 0; r < cs; r++) gwp::mbar_arrive_cluster(zfree + (kit & 1u), (unsigned)r); }
          else gwp::mbar_arrive(zfree + (kit & 1u));
        }
      }
      // ---- epilogue: scale by -(s/N_k), store this CTA's columns of the panel ----
      const double pref = -(double)d.s / (double)d.nk;
      // under GW_SYM_TR the mirrored tau node receives a copy: P0^q(beta - tau) = P0^q(tau)
      // and (full q range) the partner q receives the transpose: P0^{-q}_{Q'Q}(tau) = P0^{q}_{QQ'}(beta - tau) = P0^{q}_{QQ'}(tau)
      const int tbar = d.ntau - 1 - it.t;
      const int nct = (P.nteff < d.ntau && tbar != it.t) ? 2 : 1;
      const int qn = (P.nqeff < d.nq) ? gw_ksub(d, 0, it.ql) : it.ql;
      const int ncq = (qn != it.ql) ? 2 : 1;
      for (int cp = 0; cp < nct * ncq; cp++) {
        const int tt = (cp & 1) && nct == 2 ? tbar : it.t;
        const bool tr = cp >= nct;
        c128 *out = P.P0t + ((size_t)tt * d.nq + (tr ? qn : it.ql)) * naux * naux;
#pragma unroll
        for (int i = 0; i < MT_W; i++) {
          const int Q = it.Q0 + 8 * (mh * MT_W + i) + rho;            // accumulator row g holds matrix row rho(g)
#pragma unroll
          for (int jn = 0; jn < NJ; jn++) {
            if (jn < njm && Q < naux) {
              // accumulator columns 2c, 2c+1 hold matrix columns rho(2c) = c and rho(2c+1) = c + 4 of the n-tile
              const int ca = 8 * (noff + nstride * jn) + c, cb = ca + 4;
              // 3M: Re = K1 - K2, Im = K3 - K1 - K2
              c128 v0, v1;
              if constexpr (S3M) {
                v0 = make_double2(pref * (acc[0][i][jn][0] - acc[1][i][jn][0]), pref * (acc[2][i][jn][0] - acc[0][i][jn][0] - acc[1][i][jn][0]));
                v1 = make_double2(pref * (acc[0][i][jn][1] - acc[1][i][jn][1]), pref * (acc[2][i][jn][1] - acc[0][i][jn][1] - acc[1][i][jn][1]));
              } else {
                v0 = make_double2(pref * acc[0][i][jn][0], pref * acc[1][i][jn][0]);
                v1 = make_double2(pref * acc[0][i][jn][1], pref * acc[1][i][jn][1]);
              }
              // element (Q, col) goes to [Q][col], or to [col][Q] in the transposed copy for -q; in Hermitian mode the elements
              // left of the diagonal block also fill their mirror image with the conjugate
#pragma unroll
              for (int e = 0; e < 2; e++) {
                const int cl = e ? cb : ca;
                if (cl < ncols) {
                  const c128 v = e ? v1 : v0;
                  const size_t col = (size_t)(col0 + cl);
                  const size_t direct = tr ? col * naux + Q : (size_t)Q * naux + col;
                  out[direct] = v;
                  if (P.herm && (int)col < it.Q0) out[tr ? (size_t)Q * naux + col : col * naux + Q] = make_double2(v.x, -v.y);
                }
              }
            }
          }
        }
      }
    }
  }
  // a CTA must not exit while its peer may still arrive on its barriers
  if (cs > 1) gwp::cluster_sync_all();
}

// GW_SYM_TR: the q <= -q half of the mesh (only for the full q range and nk <= 128)
static int fill_qirr(const GwDims &d, short *qirr) {
  if (!(d.sym & GW_SYM_TR) || d.nk > 128 || d.q0 != 0 || d.nq != d.nk) return d.nq;
  int n = 0;
  for (int q = 0; q < d.nk; q++) if (q <= gw_ksub(d, 0, q)) qirr[n++] = (short)q;
  return n;
}

struct Plan {
  int main_off;
  int rsplit;
  int s3m;               // 1: 3M scheme in the main GEMM (16 n-tiles per CTA), 0: 4-real-GEMM scheme (28 n-tiles per CTA)
  int cs, ncp, ksp_max, nqt, nitems, nteff, nqeff, ldp, ksp, ndt, nt, ntc, main_units, pass_units, prows, nstage, pstage, ng, nclusters;
  size_t smem, slab_units, work_bytes;
  bool ok;
};

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  pl.nt = (d.naux + 7) / 8;
  // scheme (measured, profiles/r02_3m_vs_4m.md): 3M while a panel fits one CTA or a 2-CTA cluster (naux <= 256); wider panels would need
  // a 4-CTA cluster under 3M, which measured slower than the 2-CTA cluster of the 4-real-GEMM scheme with its 224-column tile
  pl.s3m = pl.nt <= 8 * NJ_3M ? 1 : 0;
  const int NJ = pl.s3m ? NJ_3M : NJ_4M;
  pl.cs = pl.nt <= 4 * NJ ? 1 : 2;
  pl.ncp = (pl.nt + pl.cs * 4 * NJ - 1) / (pl.cs * 4 * NJ);
  pl.ntc = (pl.nt + pl.cs * pl.ncp - 1) / (pl.cs * pl.ncp);
  pl.ksp = (d.nao + 3) / 4;
  pl.ksp_max = pl.ksp <= 7 ? 7 : (pl.ksp <= 13 ? 13 : 16);
  if (pl.ksp > 16) { pl.ok = false; return pl; }
  pl.ndt = (d.nao + 7) / 8;
  // row split of the pass work in a 2-CTA cluster: when the n-tiles do not split evenly (naux = 200: 13 + 12) CTA 0 carries one more
  // n-tile of the main GEMM per job, so it transforms fewer panel rows; weights = tensor instructions per n-tile and per panel row and k
  pl.rsplit = TM / 2;
  if (pl.cs == 2 && pl.ncp == 1 && pl.nt > pl.ntc) {
    const int n0 = pl.ntc, n1 = pl.nt - pl.ntc;
    const double per_tile = 4.0 * ((d.nao * d.nao + 3) / 4) * (pl.s3m ? 3.0 : 4.0);
    const double per_row = 2.0 * (d.nao / 8.0) * (gwp::pass_mtile_flops(d.nao, pl.ndt, pl.ksp, pl.ksp == pl.ksp_max) / 512.0);
    int shift = (int)((n0 - n1) * per_tile / (2.0 * per_row) + 0.5);
    if (shift > TM / 4) shift = TM / 4;
    pl.rsplit = TM / 2 - shift;
  }
  int r4 = pl.ksp * 4; if (r4 % 8 == 0) r4 += 4;
  pl.ldp = r4;
  pl.nqt = (d.naux + TM - 1) / TM;
  pl.nteff = (d.sym & GW_SYM_TR) ? (d.ntau + 1) / 2 : d.ntau;
  { short tmp[128]; pl.nqeff = fill_qirr(d, tmp); }
  pl.nitems = pl.nqt * pl.ncp * pl.nteff * pl.nqeff;
  pl.main_units = (TM + 8 * pl.ntc) * KC;
  pl.prows = (pl.ksp == pl.ksp_max && pl.ksp_max <= 8) ? 64 : 32;
  pl.pass_units = pl.prows * pl.ldp;
  // shared memory: prefer both G matrices resident and a 3-deep pass ring; shrink them while the main ring has < 4 stages
  const size_t gsz = (size_t)8 * pl.ndt * pl.ldp * sizeof(c128), psz = (size_t)pl.pass_units * sizeof(c128), msz = (size_t)pl.main_units * sizeof(c128);
  const size_t cap = 225 * 1024;            // 1 KB of the 227 KB is alignment slack for the TMA destinations
  const int tryng[4] = {2, 2, 1, 1}, tryps[4] = {3, 2, 3, 2};
  for (int i = 0; i < 4; i++) {
    pl.ng = tryng[i]; pl.pstage = tryps[i];
    const size_t fixed = (pl.ng * gsz + pl.pstage * psz + 1023) / 1024 * 1024;      // main stages start 1024-byte aligned
    pl.main_off = (int)(fixed / sizeof(c128));
    pl.nstage = fixed < cap ? (int)((cap - fixed) / msz) : 0;
    if (pl.nstage > 6) pl.nstage = 6;
    pl.smem = fixed + (size_t)pl.nstage * msz + 1024;
    if (pl.nstage >= 4) break;
  }
  const int nsm = gwp::gw_num_sms();
  pl.nclusters = nsm / pl.cs;
  if (pl.nclusters > pl.nitems) pl.nclusters = pl.nitems;
  pl.slab_units = (((size_t)TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.work_bytes = 256 + (size_t)nsm * 2 * pl.slab_units * sizeof(c128);
  pl.ok = pl.nstage >= 2;
  return pl;
}

}  // namespace s1

size_t gw_stage1_workspace(const gw_problem *p) {
  s1::Plan pl = s1::make_plan(p);
  return pl.ok ? pl.work_bytes : 0;
}

// executed flops: a complex tile product is 4 DMMA.8x8x4 = 2048 flops in the two passes and 3 (1536 flops, 3M) in the main GEMM
double gw_stage1_flops(const gw_problem *p) {
  s1::Plan pl = s1::make_plan(p);
  if (!pl.ok) return 0.0;
  GwDims d = gw_dims(p);
  double tiles = 0.0;
  for (int qt = 0; qt < pl.nqt; qt++) {
    const int tm_rows = (d.naux - qt * s1::TM) < s1::TM ? (d.naux - qt * s1::TM) : s1::TM;
    double mt_pass = 0.0;                       // 8-row m-tiles of the two passes, per CTA of the cluster
    for (int r = 0; r < pl.cs; r++) {
      const int rc = pl.cs == 2 ? (r == 0 ? pl.rsplit : s1::TM - pl.rsplit) : s1::TM / pl.cs;
      const int r0 = pl.cs == 2 ? (r == 0 ? 0 : pl.rsplit) : r * rc;
      int rows = tm_rows < r0 + rc ? tm_rows - r0 : rc;
      if (rows < 0) rows = 0;
      mt_pass += (rows * d.nao + 7) / 8;
    }
    const double pass = 2.0 * mt_pass * pl.ncp * gwp::pass_mtile_flops(d.nao, pl.ndt, pl.ksp, pl.ksp == pl.ksp_max);
    const int mtc = (tm_rows + 7) / 8;
    // main: warps whose first m-tile is valid execute MT_W m-tiles x their n-tiles x 2 k-steps per job
    const double mtiles = mtc <= 2 ? (double)mtc : (double)((mtc + s1::MT_W - 1) / s1::MT_W) * s1::MT_W;   // ragged panel: narrow ownership
    const double nmain = (d.nao * d.nao + s1::KC - 1) / s1::KC;
    int nt_eff = pl.nt;                         // Hermitian mode: n-tiles up to the panel's diagonal block
    if ((d.sym & GW_SYM_TR) && nt_eff > (qt * s1::TM + s1::TM + 7) / 8) nt_eff = (qt * s1::TM + s1::TM + 7) / 8;
    const double mainv = mtiles * nt_eff * (s1::KC / 4) * nmain * (pl.s3m ? 1536.0 : 2048.0);
    tiles += pass + mainv;
  }
  return tiles * (double)d.nk * d.ns * pl.nteff * pl.nqeff;
}

template <int KSP_MAX, bool S3M>
static int launch_p0(const s1::Plan &pl, const s1::Params &P, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(s1::p0_kernel<KSP_MAX, S3M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return (int)e;
  const int n2 = P.d.nao * P.d.nao;
  CUtensorMap tmV, tmZ;
  int rc = gwp::make_tensor_map(&tmV, P.V, gw_vblocks(P.d) * P.d.naux, n2, 8 * pl.ntc);
  if (rc) return rc;
  rc = gwp::make_tensor_map(&tmZ, P.scratch, (size_t)gwp::gw_num_sms() * 2 * s1::TM, n2, s1::TM);
  if (rc) return rc;
  cudaLaunchConfig_t cfg; memset(&cfg, 0, sizeof(cfg));
  cudaLaunchAttribute attr[1];
  cfg.blockDim = dim3(s1::NTHR1, 1, 1);
  cfg.dynamicSmemBytes = pl.smem;
  cfg.stream = st;
  int ncl = pl.nclusters;
  if (pl.cs > 1) {
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = pl.cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // co-resident clusters (a GPC with an odd number of free SMs leaves one unpaired)
    cfg.gridDim = dim3(pl.cs * ncl, 1, 1);
    int maxcl = 0;
    if (cudaOccupancyMaxActiveClusters(&maxcl, s1::p0_kernel<KSP_MAX, S3M>, &cfg) == cudaSuccess && maxcl > 0 && maxcl < ncl) ncl = maxcl;
    else cudaGetLastError();
  }
  cfg.gridDim = dim3(pl.cs * ncl, 1, 1);
  e = cudaLaunchKernelEx(&cfg, s1::p0_kernel<KSP_MAX, S3M>, P, tmV, tmZ);
  return (int)e;
}

int gw_launch_stage1(const gw_problem *p, const c128 *G, c128 *P0t, cudaStream_t st) {
  s1::Plan pl = s1::make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  s1::Params P;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.G = G; P.P0t = P0t;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.cs = pl.cs; P.rsplit = pl.rsplit; P.ncp = pl.ncp; P.nqt = pl.nqt; P.nitems = pl.nitems; P.nteff = pl.nteff; P.herm = (P.d.sym & GW_SYM_TR) ? 1 : 0; P.nqeff = s1::fill_qirr(P.d, P.qirr); P.ldp = pl.ldp; P.ksp = pl.ksp; P.ndt = pl.ndt; P.nt = pl.nt; P.ntc = pl.ntc;
  P.main_units = pl.main_units; P.pass_units = pl.pass_units; P.main_off = pl.main_off; P.prows = pl.prows; P.nstage = pl.nstage; P.pstage = pl.pstage; P.ng = pl.ng;
  P.slab_units = pl.slab_units;
  P.fd_nao = gwp::FastDiv((unsigned)P.d.nao);
  if (pl.s3m) {
    if (pl.ksp_max == 7) return launch_p0<7, true>(pl, P, st);
    if (pl.ksp_max == 13) return launch_p0<13, true>(pl, P, st);
    return launch_p0<16, true>(pl, P, st);
  }
  if (pl.ksp_max == 7) return launch_p0<7, false>(pl, P, st);
  if (pl.ksp_max == 13) return launch_p0<13, false>(pl, P, st);
  return launch_p0<16, false>(pl, P, st);
}
