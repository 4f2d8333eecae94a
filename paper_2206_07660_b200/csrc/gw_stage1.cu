// gw_stage1.cu — stage 1, Eq. 28b (Algorithm 1 first k loop):
//
//   P0t[t][q][Q][Q'] = -(s/N_k) Σ_k Σ_abcd V[k][k+q][Q][d][a] G[t][k+q][a][b] V[k+q][k][Q'][b][c] G[tbar][k][c][d]
//
// Formulation used here (exact algebra, no input symmetry assumed):
//   Z_k[Q][(b,c)] = Σ_d Σ_a G[tbar][k][c][d] V[k][k+q][Q][d][a] G[t][k+q][a][b]        (two small GEMMs, K = nao)
//   P0t[Q][Q']    = -(s/N_k) Σ_k Σ_(b,c) Z_k[Q][(b,c)] · V[k+q][k][Q'][(b,c)]            (one GEMM,  K = N_k·nao²)
// so the second operand is the raw V block (rows Q', K contiguous), never transformed.
//
// Work decomposition: a persistent CTA owns a row panel [TM Q-rows] x [all naux Q'] of one (t,q) and keeps
// it in registers over the whole k loop (the k-sum is inside the K loop; no cross-CTA reduction).  Because the
// panel spans every Q', each Z row is produced exactly once (no recomputation of the V·G transforms across
// column tiles).  Per k the CTA runs three phases, all on FP64 tensor cores (DMMA.8x8x4, 4-real-GEMM complex
// scheme) fed by one cp.async stage pipeline:
//   pass 1:  Xt[Q][b][d] = Σ_a V[k][k+q][Q][d][a] G[t][k+q][a][b]       rows (Q,d) are one flat M dimension
//   pass 2:  Z [Q][b][c] = Σ_d Xt[Q][b][d] G[tbar][k][c][d]             rows (Q,b) flat; in place
//   main  :  acc[Q][Q'] += Σ_K Z[Q][K] V[k+q][k][Q'][K],  K = (b,c) = nao² contiguous
// Xt/Z live in a per-CTA slab of the workspace (TM·nao² complex, written and re-read within ~100 µs, i.e. L2
// resident); they never exist as a full [t][q][k] tensor.
#include "gw_pipe.cuh"

namespace s1 {

using gwp::NCONS; using gwp::NTHR_WS; using gwp::PASS_ROWS; using gwp::FastDiv; using gwp::Ring;
constexpr int NSTAGE_MAX = 8;
constexpr int KC = 8;           // complex K per main job (one 128-byte row per operand row)
constexpr int MT_W = 2;         // m-tiles per warp in the main GEMM

struct Params {
  GwDims d;
  const c128 *V, *G;
  c128 *P0t, *scratch;
  int nqt, nitems;       // Q tiles per (t,q); total work items
  int ldp, ksp, ndt;     // pass smem row stride (complex), k-steps = ceil(nao/4), n-tiles over nao
  int nt;                // n-tiles over naux
  int stage_units;       // complex elements per stage buffer
  int nstage;            // ring depth (fits shared memory)
  size_t scratch_stride; // complex elements per CTA slab
  FastDiv fd_nao;
};

// main job (producer warp): A = Z[tm rows][k0..k0+8), B = Vb[naux rows][k0..k0+8); 16-byte units swizzled by row parity
template <int TM>
__device__ __forceinline__ void ws_issue_main(c128 *stage, const c128 *Z, int tm_rows, const c128 *Vb, int naux, int brows, int n2, int k0) {
  const int pt = threadIdx.x - 32 * NCONS;
  const int u = pt & 7, rsub = pt >> 3;                // 16 rows x 8 units per pass of the producer warpgroup
  const bool kok = k0 + u < n2;
  for (int r = rsub; r < TM; r += 16) {
    const bool ok = kok && (r < tm_rows);
    gwp::cp_async16_zfill(stage + r * KC + (u ^ ((r & 1) << 2)), ok ? Z + (size_t)r * n2 + k0 + u : Z, ok);
  }
  c128 *sB = stage + TM * KC;
  for (int r = rsub; r < brows; r += 16) {
    const bool ok = kok && (r < naux);
    gwp::cp_async16_zfill(sB + r * KC + (u ^ ((r & 1) << 2)), ok ? Vb + (size_t)r * n2 + k0 + u : Vb, ok);
  }
}

// consumer: one main job (KC/4 k-steps) for this warp's MT_W x NJM tiles; all fragment loads hoisted per k-step
template <int NJ, int NJM, int NSTRIDE>
__device__ __forceinline__ void main_compute(const c128 *sAw, const c128 *sBw, double (&accr)[MT_W][NJ][2], double (&acci)[MT_W][NJ][2], int c, int sw) {
#pragma unroll
  for (int ks = 0; ks < KC / 4; ks++) {
    const int u = (4 * ks + c) ^ sw;
    c128 a[MT_W], b[NJM];
#pragma unroll
    for (int i = 0; i < MT_W; i++) a[i] = sAw[i * 8 * KC + u];
#pragma unroll
    for (int jn = 0; jn < NJM; jn++) b[jn] = sBw[jn * NSTRIDE * 8 * KC + u];
#pragma unroll
    for (int jn = 0; jn < NJM; jn++)
#pragma unroll
      for (int i = 0; i < MT_W; i++) cmma(accr[i][jn], acci[i][jn], a[i], b[jn]);
  }
}

template <int NJ, int MH, int KSP_MAX>
__global__ void __launch_bounds__(NTHR_WS, 1) p0_kernel(const Params P) {
  constexpr int TM = 8 * MT_W * MH;
  constexpr int NSTRIDE = 8 / MH;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *smem = reinterpret_cast<c128 *>(smem_raw);
  const GwDims d = P.d;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao, ldp = P.ldp, naop = 8 * P.ndt;
  c128 *sGt = smem;                       // [naop][ldp]: sGt[b][a] = G[t][k+q][a][b]
  c128 *sGm = sGt + naop * ldp;           // [naop][ldp]: sGm[c][d] = G[tbar][k][c][d]
  c128 *sStage = sGm + naop * ldp;        // nstage x stage_units
  const int NSTAGE = P.nstage;
  __shared__ uint64_t bars[2 * NSTAGE_MAX + 2];
  uint64_t *bar_full = bars, *bar_empty = bars + NSTAGE_MAX, *bar_g = bars + 2 * NSTAGE_MAX, *bar_phase = bars + 2 * NSTAGE_MAX + 1;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  c128 *slab = P.scratch + (size_t)blockIdx.x * P.scratch_stride;
  const size_t vb = (size_t)naux * n2;
  const int brows = 8 * P.nt;

  // zero all dynamic smem once (pad rows/columns must hold finite values: they meet zero operands); init barriers
  {
    const int tot = 2 * naop * ldp + NSTAGE * P.stage_units;
    for (int i = threadIdx.x; i < tot; i += NTHR_WS) smem[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
      for (int i = 0; i < NSTAGE; i++) { gwp::mbar_init(bar_full + i, gwp::NPROD_THR); gwp::mbar_init(bar_empty + i, NCONS); }
      gwp::mbar_init(bar_g, gwp::NPROD_THR);
      gwp::mbar_init(bar_phase, NCONS);
    }
  }
  __syncthreads();
  Ring ring; ring.full = bar_full; ring.empty = bar_empty; ring.nstage = NSTAGE; ring.it = 0;
  unsigned gpar = 0, ppar = 0;     // parities of bar_g / bar_phase (advance identically on both sides)
  const int nmain = (n2 + KC - 1) / KC;

  if (w >= NCONS) {
    // =============================== producer warp ===============================
    gwp::reg_dec<40>();
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      // item order: Q-tile index slowest (so the round-robin gives every CTA the same mix of full and ragged tiles),
      // then q, then t fastest (concurrent CTAs share the V blocks of one q in L2)
      const int qt = item / (d.ntau * d.nq), t = item % d.ntau, ql = (item / d.ntau) % d.nq;
      const int q = d.q0 + ql, Q0 = qt * TM;
      const int tm_rows = min(TM, naux - Q0), rows = tm_rows * nao, npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
      for (int k = 0; k < d.nk; k++) {
        const int kq = gw_kadd(d, k, q);
        const c128 *Vt = P.V + ((size_t)k * d.nk + kq) * vb + (size_t)Q0 * n2;
        const c128 *Vb = P.V + ((size_t)kq * d.nk + k) * vb;
        // G matrices of this k (consumers finished the passes of the previous k: see the phase wait below)
        gwp::ws_issue_matrix<true>(sGt, P.G + ((size_t)t * d.nk + kq) * n2, nao, ldp, P.fd_nao);
        gwp::ws_issue_matrix<false>(sGm, P.G + ((size_t)(d.ntau - 1 - t) * d.nk + k) * n2, nao, ldp, P.fd_nao);
        gwp::cp_async_arrive_noinc(bar_g);
        for (int j = 0; j < npass; j++) {
          const int s = ring.acquire();
          gwp::ws_issue_rows(sStage + s * P.stage_units, Vt, j * PASS_ROWS, rows, nao, ldp, P.fd_nao);
          ring.commit();
        }
        gwp::mbar_wait(bar_phase, ppar); ppar ^= 1u;          // all Xt rows are in the slab
        for (int j = 0; j < npass; j++) {
          const int s = ring.acquire();
          gwp::ws_issue_rows(sStage + s * P.stage_units, slab, j * PASS_ROWS, rows, nao, ldp, P.fd_nao);
          ring.commit();
        }
        gwp::mbar_wait(bar_phase, ppar); ppar ^= 1u;          // Z complete; sGt/sGm free for the next k
        for (int j = 0; j < nmain; j++) {
          const int s = ring.acquire();
          ws_issue_main<TM>(sStage + s * P.stage_units, slab, tm_rows, Vb, naux, brows, n2, j * KC);
          ring.commit();
        }
      }
    }
    asm volatile("cp.async.wait_all;\n" ::: "memory");
  } else {
    // =============================== consumer warps ===============================
    gwp::reg_inc<232>();
    const int g = lane >> 2, c = lane & 3;
    const int mh = (MH == 2) ? (w >> 2) : 0;
    const int noff = (MH == 2) ? (((w & 3) - mh + 4) & 3) : w;
    const int njm = (P.nt > noff) ? (P.nt - noff + NSTRIDE - 1) / NSTRIDE : 0;   // n-tiles owned by this warp
    const int sw = (g & 1) << 2;
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      // item order: Q-tile index slowest (so the round-robin gives every CTA the same mix of full and ragged tiles),
      // then q, then t fastest (concurrent CTAs share the V blocks of one q in L2)
      const int qt = item / (d.ntau * d.nq), t = item % d.ntau, ql = (item / d.ntau) % d.nq;
      const int Q0 = qt * TM;
      const int tm_rows = min(TM, naux - Q0), rows = tm_rows * nao, npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
      const int mtc = (tm_rows + 7) / 8;
      double accr[MT_W][NJ][2], acci[MT_W][NJ][2];
#pragma unroll
      for (int i = 0; i < MT_W; i++)
#pragma unroll
        for (int j = 0; j < NJ; j++) { accr[i][j][0] = accr[i][j][1] = 0.0; acci[i][j][0] = acci[i][j][1] = 0.0; }

      for (int k = 0; k < d.nk; k++) {
        gwp::mbar_wait(bar_g, gpar); gpar ^= 1u;
        for (int j = 0; j < npass; j++) {
          const int s = ring.wait();
          if (P.ksp == KSP_MAX) gwp::pass_compute_exact<KSP_MAX, true>(sStage + s * P.stage_units, sGt, slab, j * PASS_ROWS, rows, nao, ldp);
          else gwp::pass_compute<KSP_MAX, true>(sStage + s * P.stage_units, sGt, slab, j * PASS_ROWS, rows, nao, ldp, P.ksp, P.ndt);
          ring.release();
        }
        __threadfence(); __syncwarp();
        if (lane == 0) gwp::mbar_arrive(bar_phase);
        for (int j = 0; j < npass; j++) {
          const int s = ring.wait();
          if (P.ksp == KSP_MAX) gwp::pass_compute_exact<KSP_MAX, false>(sStage + s * P.stage_units, sGm, slab, j * PASS_ROWS, rows, nao, ldp);
          else gwp::pass_compute<KSP_MAX, false>(sStage + s * P.stage_units, sGm, slab, j * PASS_ROWS, rows, nao, ldp, P.ksp, P.ndt);
          ring.release();
        }
        __threadfence(); __syncwarp();
        if (lane == 0) gwp::mbar_arrive(bar_phase);
        const bool active = (mh * MT_W < mtc) && njm > 0;
        for (int j = 0; j < nmain; j++) {
          const int s = ring.wait();
          if (active) {
            const c128 *sAw = sStage + s * P.stage_units + (8 * mh * MT_W + g) * KC;
            const c128 *sBw = sStage + s * P.stage_units + TM * KC + (8 * noff + g) * KC;
            if (njm == NJ) main_compute<NJ, NJ, NSTRIDE>(sAw, sBw, accr, acci, c, sw);
            else if (njm == NJ - 1) main_compute<NJ, NJ - 1, NSTRIDE>(sAw, sBw, accr, acci, c, sw);
            else {
#pragma unroll
              for (int ks = 0; ks < KC / 4; ks++) {
                const int u = (4 * ks + c) ^ sw;
                c128 a[MT_W];
#pragma unroll
                for (int i = 0; i < MT_W; i++) a[i] = sAw[i * 8 * KC + u];
#pragma unroll
                for (int jn = 0; jn < NJ; jn++) {
                  if (jn < njm) {
                    const c128 b = sBw[jn * NSTRIDE * 8 * KC + u];
#pragma unroll
                    for (int i = 0; i < MT_W; i++) cmma(accr[i][jn], acci[i][jn], a[i], b);
                  }
                }
              }
            }
          }
          ring.release();
        }
      }
      // ---- epilogue: scale by -(s/N_k), store the panel ----
      const double pref = -(double)d.s / (double)d.nk;
      c128 *out = P.P0t + ((size_t)t * d.nq + ql) * naux * naux;
#pragma unroll
      for (int i = 0; i < MT_W; i++) {
        const int Q = Q0 + 8 * (mh * MT_W + i) + g;
#pragma unroll
        for (int jn = 0; jn < NJ; jn++) {
          if (jn < njm && Q < naux) {
            const int col = 8 * (noff + NSTRIDE * jn) + 2 * c;
            if (col < naux) out[(size_t)Q * naux + col] = make_double2(pref * accr[i][jn][0], pref * acci[i][jn][0]);
            if (col + 1 < naux) out[(size_t)Q * naux + col + 1] = make_double2(pref * accr[i][jn][1], pref * acci[i][jn][1]);
          }
        }
      }
    }
  }
}

struct Plan {
  int mh, ksp_max, TM, nqt, nitems, ldp, ksp, ndt, nt, stage_units, grid, nstage;
  size_t smem, scratch_stride, work_bytes;
  bool ok;
};

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  pl.nt = (d.naux + 7) / 8;
  if (pl.nt <= 28) pl.mh = 2; else if (pl.nt <= 56) pl.mh = 1; else { pl.ok = false; return pl; }
  pl.TM = 8 * MT_W * pl.mh;
  pl.ksp = (d.nao + 3) / 4;
  pl.ksp_max = pl.ksp <= 7 ? 7 : (pl.ksp <= 13 ? 13 : 16);
  if (pl.ksp > 16) { pl.ok = false; return pl; }
  pl.ndt = (d.nao + 7) / 8;
  int r4 = pl.ksp * 4; if (r4 % 8 == 0) r4 += 4;
  pl.ldp = r4;
  pl.nqt = (d.naux + pl.TM - 1) / pl.TM;
  pl.nitems = pl.nqt * d.ntau * d.nq;
  int s_pass = PASS_ROWS * pl.ldp, s_main = (pl.TM + 8 * pl.nt) * KC;
  pl.stage_units = s_pass > s_main ? s_pass : s_main;
  const size_t fixed = (size_t)2 * 8 * pl.ndt * pl.ldp * sizeof(c128), per = (size_t)pl.stage_units * sizeof(c128);
  pl.nstage = (int)((225 * 1024 - fixed) / per);
  if (pl.nstage > 6) pl.nstage = 6;
  pl.smem = fixed + (size_t)pl.nstage * per;
  int dev = 0, nsm = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if (nsm <= 0) nsm = 148;
  pl.grid = pl.nitems < nsm ? pl.nitems : nsm;
  pl.scratch_stride = (((size_t)pl.TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.work_bytes = 256 + (size_t)nsm * pl.scratch_stride * sizeof(c128);
  pl.ok = pl.nstage >= 2;
  return pl;
}

}  // namespace s1

size_t gw_stage1_workspace(const gw_problem *p) {
  s1::Plan pl = s1::make_plan(p);
  return pl.ok ? pl.work_bytes : 0;
}

// executed flops: every complex tile MMA is 4 DMMA.8x8x4 = 2048 flops
double gw_stage1_flops(const gw_problem *p) {
  s1::Plan pl = s1::make_plan(p);
  if (!pl.ok) return 0.0;
  GwDims d = gw_dims(p);
  double tiles = 0.0;
  for (int qt = 0; qt < pl.nqt; qt++) {
    const int tm_rows = (d.naux - qt * pl.TM) < pl.TM ? (d.naux - qt * pl.TM) : pl.TM;
    const int rows = tm_rows * d.nao;
    const double mt_pass = (rows + 7) / 8;
    const double pass = 2.0 * mt_pass * pl.ndt * pl.ksp;
    const int mtc = (tm_rows + 7) / 8;
    // main: warps whose first m-tile is valid execute MT_W m-tiles x their n-tiles x 2 k-steps per job
    const double mtiles = (double)((mtc + s1::MT_W - 1) / s1::MT_W) * s1::MT_W;
    const double nmain = (d.nao * d.nao + s1::KC - 1) / s1::KC;
    const double mainv = mtiles * pl.nt * (s1::KC / 4) * nmain;
    tiles += pass + mainv;
  }
  return tiles * (double)d.nk * d.ntau * d.nq * 2048.0;
}

template <int NJ, int MH, int KSP_MAX>
static int launch_p0(const s1::Plan &pl, const s1::Params &P, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(s1::p0_kernel<NJ, MH, KSP_MAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return (int)e;
  s1::p0_kernel<NJ, MH, KSP_MAX><<<pl.grid, s1::NTHR_WS, pl.smem, st>>>(P);
  return (int)cudaGetLastError();
}

int gw_launch_stage1(const gw_problem *p, const c128 *G, c128 *P0t, cudaStream_t st) {
  s1::Plan pl = s1::make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  s1::Params P;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.G = G; P.P0t = P0t;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.nqt = pl.nqt; P.nitems = pl.nitems; P.ldp = pl.ldp; P.ksp = pl.ksp; P.ndt = pl.ndt; P.nt = pl.nt;
  P.stage_units = pl.stage_units; P.nstage = pl.nstage; P.scratch_stride = pl.scratch_stride;
  P.fd_nao = gwp::FastDiv((unsigned)P.d.nao);
  if (pl.mh == 2) {
    if (pl.ksp_max == 7) return launch_p0<7, 2, 7>(pl, P, st);
    if (pl.ksp_max == 13) return launch_p0<7, 2, 13>(pl, P, st);
    return launch_p0<7, 2, 16>(pl, P, st);
  } else {
    if (pl.ksp_max == 7) return launch_p0<7, 1, 7>(pl, P, st);
    if (pl.ksp_max == 13) return launch_p0<7, 1, 13>(pl, P, st);
    return launch_p0<7, 1, 16>(pl, P, st);
  }
}
