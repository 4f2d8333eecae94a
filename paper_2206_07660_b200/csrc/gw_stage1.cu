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
#include "gw_common.cuh"

namespace s1 {

constexpr int NWARP = 8, NTHR = 256, NSTAGE = 3;
constexpr int PASS_ROWS = 64;   // rows per pass job: one 8-row m-tile per warp
constexpr int KC = 8;           // complex K per main job (one 128-byte row per operand row)
constexpr int MT_W = 2;         // m-tiles per warp in the main GEMM

struct Params {
  GwDims d;
  const c128 *V, *G;
  c128 *P0t, *scratch;
  unsigned *counter;
  int nqt, nitems;       // Q tiles per (t,q); total work items
  int ldp, ksp, ndt;     // pass smem row stride (complex), k-steps = ceil(nao/4), n-tiles over nao
  int nt;                // n-tiles over naux
  int stage_units;       // complex elements per stage buffer
  size_t scratch_stride; // complex elements per CTA slab
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

// main job: A = Z[tm rows][k0..k0+8), B = Vb[naux rows][k0..k0+8); 16-byte units swizzled by row parity
template <int TM>
__device__ __forceinline__ void issue_main_job(c128 *stage, const c128 *Z, int tm_rows, const c128 *Vb, int naux, int brows,
                                               int n2, int k0) {
  for (int i = threadIdx.x; i < TM * KC; i += NTHR) {
    const int r = i >> 3, u = i & 7;
    const bool ok = (r < tm_rows) && (k0 + u < n2);
    cp_async16_zfill(stage + r * KC + (u ^ ((r & 1) << 2)), ok ? Z + (size_t)r * n2 + k0 + u : Z, ok);
  }
  c128 *sB = stage + TM * KC;
  for (int i = threadIdx.x; i < brows * KC; i += NTHR) {
    const int r = i >> 3, u = i & 7;
    const bool ok = (r < naux) && (k0 + u < n2);
    cp_async16_zfill(sB + r * KC + (u ^ ((r & 1) << 2)), ok ? Vb + (size_t)r * n2 + k0 + u : Vb, ok);
  }
}

// One pass job: this warp's m-tile (8 rows) times the nao x nao matrix held in sG as [n][k] (K contiguous).
// PASS = 1: out Xt[(Q*nao + b)*nao + d] for row (Q,d), column b.   PASS = 2: out Z[row*nao + c], in place.
template <int KSP_MAX, int PASS>
__device__ __forceinline__ void pass_compute(const c128 *sStage, const c128 *sG, c128 *slab, int row0, int rows_total,
                                             int nao, int ldp, int ksp, int ndt) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  if (row0 + 8 * w >= rows_total) return;   // whole m-tile beyond the panel (warp-uniform)
  c128 a[KSP_MAX];
#pragma unroll
  for (int ks = 0; ks < KSP_MAX; ks++)
    if (ks < ksp) a[ks] = sStage[(8 * w + g) * ldp + 4 * ks + c];
  const int row = row0 + 8 * w + g;
  const bool rok = row < rows_total;
  int Q = 0, dd = 0;
  if (PASS == 1) { Q = row / nao; dd = row - Q * nao; }
  for (int nt = 0; nt < ndt; nt++) {
    double cr[2] = {0.0, 0.0}, ci[2] = {0.0, 0.0};
    const c128 *bp = sG + (8 * nt + g) * ldp + c;
#pragma unroll
    for (int ks = 0; ks < KSP_MAX; ks++)
      if (ks < ksp) cmma(cr, ci, a[ks], bp[4 * ks]);
    const int col = 8 * nt + 2 * c;
    if (rok) {
      if (PASS == 1) {
        if (col < nao) slab[((size_t)Q * nao + col) * nao + dd] = make_double2(cr[0], ci[0]);
        if (col + 1 < nao) slab[((size_t)Q * nao + col + 1) * nao + dd] = make_double2(cr[1], ci[1]);
      } else {
        if (col < nao) slab[(size_t)row * nao + col] = make_double2(cr[0], ci[0]);
        if (col + 1 < nao) slab[(size_t)row * nao + col + 1] = make_double2(cr[1], ci[1]);
      }
    }
  }
}

template <int NJ, int MH, int KSP_MAX>
__global__ void __launch_bounds__(NTHR, 1) p0_kernel(const Params P) {
  constexpr int TM = 8 * MT_W * MH;
  constexpr int NSTRIDE = 8 / MH;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *smem = reinterpret_cast<c128 *>(smem_raw);
  const GwDims d = P.d;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao, ldp = P.ldp, naop = 8 * P.ndt;
  c128 *sGt = smem;                       // [naop][ldp]: sGt[b][a] = G[t][k+q][a][b]
  c128 *sGm = sGt + naop * ldp;           // [naop][ldp]: sGm[c][d] = G[tbar][k][c][d]
  c128 *sStage = sGm + naop * ldp;        // NSTAGE x stage_units
  __shared__ int s_item;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const int mh = (MH == 2) ? (w >> 2) : 0;
  const int noff = (MH == 2) ? (((w & 3) - mh + 4) & 3) : w;
  const int njm = (P.nt > noff) ? (P.nt - noff + NSTRIDE - 1) / NSTRIDE : 0;   // n-tiles owned by this warp
  c128 *slab = P.scratch + (size_t)blockIdx.x * P.scratch_stride;
  const size_t vb = (size_t)naux * n2;
  const int brows = 8 * P.nt;
  const int sw = (g & 1) << 2;

  // zero all dynamic smem once: pad rows/columns must hold finite values (they meet zero operands)
  {
    const int tot = 2 * naop * ldp + NSTAGE * P.stage_units;
    for (int i = threadIdx.x; i < tot; i += NTHR) smem[i] = make_double2(0.0, 0.0);
  }
  __syncthreads();

  for (;;) {
    if (threadIdx.x == 0) s_item = (int)atomicAdd(P.counter, 1u);
    __syncthreads();
    const int item = s_item;
    __syncthreads();
    if (item >= P.nitems) break;
    const int qt = item % P.nqt, t = (item / P.nqt) % d.ntau, ql = item / (P.nqt * d.ntau);
    const int q = d.q0 + ql, Q0 = qt * TM;
    const int tm_rows = min(TM, naux - Q0);
    const int rows = tm_rows * nao;                       // flat (Q,d) / (Q,b) rows of the passes
    const int npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
    const int nmain = (n2 + KC - 1) / KC;
    const int mtc = (tm_rows + 7) / 8;                    // valid m-tiles in this panel

    double accr[MT_W][NJ][2], acci[MT_W][NJ][2];
#pragma unroll
    for (int i = 0; i < MT_W; i++)
#pragma unroll
      for (int j = 0; j < NJ; j++) { accr[i][j][0] = accr[i][j][1] = 0.0; acci[i][j][0] = acci[i][j][1] = 0.0; }

    for (int k = 0; k < d.nk; k++) {
      const int kq = gw_kadd(d, k, q);
      const c128 *Vt = P.V + ((size_t)k * d.nk + kq) * vb + (size_t)Q0 * n2;   // V[k][k+q][Q0..]: rows (Q,d) x nao
      const c128 *Vb = P.V + ((size_t)kq * d.nk + k) * vb;                     // V[k+q][k]: rows Q' x nao²
      const c128 *G1 = P.G + ((size_t)t * d.nk + kq) * n2;
      const c128 *G2 = P.G + ((size_t)(d.ntau - 1 - t) * d.nk + k) * n2;
      // prefetch the first pass-1 jobs while the G matrices are loaded
      int issued = 0;
      for (; issued < NSTAGE - 1; issued++) {
        if (issued < npass) issue_pass_job(sStage + (issued % NSTAGE) * P.stage_units, Vt, issued * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
      }
      for (int i = threadIdx.x; i < n2; i += NTHR) {
        const int r = i / nao, cc = i - r * nao;
        sGt[cc * ldp + r] = G1[i];     // transposed: [b][a]
        sGm[r * ldp + cc] = G2[i];     // [c][d]
      }
      // ---- pass 1 ----
      for (int j = 0; j < npass; j++) {
        cp_async_wait<NSTAGE - 2>();
        __syncthreads();
        const int nx = j + NSTAGE - 1;
        if (nx < npass) issue_pass_job(sStage + (nx % NSTAGE) * P.stage_units, Vt, nx * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
        pass_compute<KSP_MAX, 1>(sStage + (j % NSTAGE) * P.stage_units, sGt, slab, j * PASS_ROWS, rows, nao, ldp, P.ksp, P.ndt);
      }
      cp_async_wait<0>();
      __syncthreads();    // all Xt rows written (CTA scope) before pass 2 streams them back
      // ---- pass 2 (in place on the slab) ----
      for (issued = 0; issued < NSTAGE - 1; issued++) {
        if (issued < npass) issue_pass_job(sStage + (issued % NSTAGE) * P.stage_units, slab, issued * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
      }
      for (int j = 0; j < npass; j++) {
        cp_async_wait<NSTAGE - 2>();
        __syncthreads();
        const int nx = j + NSTAGE - 1;
        if (nx < npass) issue_pass_job(sStage + (nx % NSTAGE) * P.stage_units, slab, nx * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
        pass_compute<KSP_MAX, 2>(sStage + (j % NSTAGE) * P.stage_units, sGm, slab, j * PASS_ROWS, rows, nao, ldp, P.ksp, P.ndt);
      }
      cp_async_wait<0>();
      __syncthreads();    // Z complete
      // ---- main GEMM over K = nao² ----
      for (issued = 0; issued < NSTAGE - 1; issued++) {
        if (issued < nmain) issue_main_job<TM>(sStage + (issued % NSTAGE) * P.stage_units, slab, tm_rows, Vb, naux, brows, n2, issued * KC);
        cp_async_commit();
      }
      for (int j = 0; j < nmain; j++) {
        cp_async_wait<NSTAGE - 2>();
        __syncthreads();
        const int nx = j + NSTAGE - 1;
        if (nx < nmain) issue_main_job<TM>(sStage + (nx % NSTAGE) * P.stage_units, slab, tm_rows, Vb, naux, brows, n2, nx * KC);
        cp_async_commit();
        const c128 *sA = sStage + (j % NSTAGE) * P.stage_units;
        const c128 *sB = sA + TM * KC;
        if (mh * MT_W < mtc) {
#pragma unroll
          for (int ks = 0; ks < KC / 4; ks++) {
            const int u = (4 * ks + c) ^ sw;
            c128 a[MT_W];
#pragma unroll
            for (int i = 0; i < MT_W; i++) a[i] = sA[(8 * (mh * MT_W + i) + g) * KC + u];
#pragma unroll
            for (int jn = 0; jn < NJ; jn++) {
              if (jn < njm) {
                const c128 b = sB[(8 * (noff + NSTRIDE * jn) + g) * KC + u];
#pragma unroll
                for (int i = 0; i < MT_W; i++) cmma(accr[i][jn], acci[i][jn], a[i], b);
              }
            }
          }
        }
      }
      cp_async_wait<0>();
      __syncthreads();
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

struct Plan {
  int mh, ksp_max, TM, nqt, nitems, ldp, ksp, ndt, nt, stage_units, grid;
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
  pl.smem = ((size_t)2 * 8 * pl.ndt * pl.ldp + (size_t)NSTAGE * pl.stage_units) * sizeof(c128);
  int dev = 0, nsm = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if (nsm <= 0) nsm = 148;
  pl.grid = pl.nitems < nsm ? pl.nitems : nsm;
  pl.scratch_stride = (((size_t)pl.TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.work_bytes = 256 + (size_t)nsm * pl.scratch_stride * sizeof(c128);
  pl.ok = pl.smem <= 227 * 1024;
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
  s1::p0_kernel<NJ, MH, KSP_MAX><<<pl.grid, s1::NTHR, pl.smem, st>>>(P);
  return (int)cudaGetLastError();
}

int gw_launch_stage1(const gw_problem *p, const c128 *G, c128 *P0t, cudaStream_t st) {
  s1::Plan pl = s1::make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  s1::Params P;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.G = G; P.P0t = P0t;
  P.counter = (unsigned *)p->work;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.nqt = pl.nqt; P.nitems = pl.nitems; P.ldp = pl.ldp; P.ksp = pl.ksp; P.ndt = pl.ndt; P.nt = pl.nt;
  P.stage_units = pl.stage_units; P.scratch_stride = pl.scratch_stride;
  cudaError_t e = cudaMemsetAsync(p->work, 0, 256, st);
  if (e != cudaSuccess) return (int)e;
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
