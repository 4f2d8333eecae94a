// gw_stage3.cu — stage 3, Eq. 31 (Algorithm 1 second k loop):
//
//   Sigma[t][k][i][j] = -(1/N_k) Σ_q Σ_QQ' Σ_ab V[k][k-q][Q][i][a] G[t][k-q][a][b] Wt[t][q][Q][Q'] V[k-q][k][Q'][b][j]
//
// Formulation (exact algebra, mirror image of stage 1; V1 = V[k][k-q], V2 = V[k-q][k]):
//   main  :  U[Q][(b,j)]  = Σ_Q' Wt[Q][Q'] V2[Q'][(b,j)]              GEMM, M = Q panel, N = nao², K = naux
//   pass A:  T[Q][a][j]   = Σ_b G[a][b] U[Q][b][j]                     rows (Q,j) flat, K = nao
//   final :  Sigma[i][j] += Σ_(Q,a) V1[Q][i][a] T[Q][a][j]             K = (Q,a)
// A persistent CTA owns one (t,k): it loops over q and over Q panels, and keeps the nao x nao Sigma accumulator in
// registers for the whole item, so the q-sum needs no cross-CTA reduction and the result is deterministic.
// U and T live in two per-CTA slabs of the workspace (L2 resident); the raw V2 block is the only big stream.
#include "gw_pipe.cuh"

// GW_SYM_TR bookkeeping shared by both stage-3 kernels: the k <= -k half of the mesh (only for the full q range, nk <= 128)
static int fill_kirr(const GwDims &d, short *kirr) {
  if (!(d.sym & GW_SYM_TR) || d.nk > 128 || d.q0 != 0 || d.nq != d.nk) return d.nk;
  int n = 0;
  for (int k = 0; k < d.nk; k++) if (k <= gw_ksub(d, 0, k)) kirr[n++] = (short)k;
  return n;
}

namespace s3 {

using gwp::NCONS; using gwp::NTHR_WS; using gwp::PASS_ROWS; using gwp::FastDiv; using gwp::Ring;
constexpr int NSTAGE_MAX = 8;
constexpr int KC = 8, MT_W = 2, NJ = 7, TM = 32;

struct Params {
  GwDims d;
  const c128 *V, *G, *Wt;
  c128 *Sigma, *scratch;
  int nqt, nitems;
  int ldp, ksp, ndt;      // pass / G smem row stride, k-steps over nao, tiles over nao
  int ldt;                // row stride of the T block in the final jobs
  int kh, kspf, ldpf;     // final jobs: K splits per Q, k-steps per split, row stride of the V1 part
  FastDiv fd_kw;          // divide by 4*kspf
  int nnt, nchunk, cht;   // n-tiles over nao², N chunks, n-tiles per chunk
  int ldb;                // row stride of the main-job B part
  int stage_units, nstage;
  int stage_off;          // offset of the ring in the 1024-byte aligned dynamic shared memory (complex elements)
  size_t slab_units;      // complex elements per slab (two slabs per CTA)
  int nkeff;              // k points evaluated: nk, or the k <= -k half under GW_SYM_TR (Sigma[-k] = conj Sigma[k] is copied)
  short kirr[128];        // the evaluated k points when nkeff < nk
  __device__ __forceinline__ int kof(int i) const { return nkeff < d.nk ? (int)kirr[i] : i; }
  int acc_mode;           // GW_ACC_CONTINUE / GW_ACC_PARTIAL (gw_common.cuh)
  FastDiv fd_nao;
};

// Main jobs are written by TMA with the 128-byte swizzle (16-byte unit u of row r sits at u ^ (r & 7)):
//   A = W[TM rows][8 K]: 32 rows x 128 B;   B = one 1 KB box per n-tile of the chunk: [8 K rows][8 columns of V2].
// Lane group g reads row / column rho(g) = (g >> 1) + 4 (g & 1) of its tile, so a quarter-warp touches eight different units.
using gwp::tma_load_2d; using gwp::mbar_expect_tx;

template <int NJM>
__device__ __forceinline__ void main_compute(const c128 *sAw, const c128 *sBw, double (&accr)[MT_W][NJ][2], double (&acci)[MT_W][NJ][2], int c, int rho) {
#pragma unroll
  for (int ks = 0; ks < KC / 4; ks++) {
    const int kr = 4 * ks + c;
    const int u = kr ^ rho;
    c128 a[MT_W], b[NJM];
#pragma unroll
    for (int i = 0; i < MT_W; i++) a[i] = sAw[i * 8 * KC + u];
    const c128 *bk = sBw + kr * 8 + u;
#pragma unroll
    for (int jn = 0; jn < NJM; jn++) b[jn] = bk[256 * jn];      // n-tiles 4 apart, 64 units per n-tile box
#pragma unroll
    for (int jn = 0; jn < NJM; jn++)
#pragma unroll
      for (int i = 0; i < MT_W; i++) cmma(accr[i][jn], acci[i][jn], a[i], b[jn]);
  }
}

template <int KSP_MAX, int NCT>
__global__ void __launch_bounds__(NTHR_WS, 1) sigma_kernel(const Params P, const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmV) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // the TMA destinations (128-byte swizzle) need 1024-byte alignment: the launch asks for 1 KB of slack
  c128 *smem = reinterpret_cast<c128 *>(smem_raw + ((1024u - (gwp::smem_u32(smem_raw) & 1023u)) & 1023u));
  const GwDims d = P.d;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao, ldp = P.ldp, naop = 8 * P.ndt, ndt = P.ndt;
  c128 *sG = smem;                    // [naop][ldp]: sG[a][b] = G[t][k-q][a][b]  (operand [n=a][k=b] of pass A)
  c128 *sStage = smem + P.stage_off;   // ring of 1024-byte aligned stage buffers
  const int NSTAGE = P.nstage;
  __shared__ uint64_t bars[2 * NSTAGE_MAX + 2];
  uint64_t *bar_full = bars, *bar_empty = bars + NSTAGE_MAX, *bar_g = bars + 2 * NSTAGE_MAX, *bar_phase = bars + 2 * NSTAGE_MAX + 1;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  c128 *slabU = P.scratch + (size_t)blockIdx.x * 2 * P.slab_units;
  c128 *slabT = slabU + P.slab_units;
  const size_t vb = (size_t)naux * n2;
  {
    const int tot = P.stage_off + NSTAGE * P.stage_units;
    for (int i = threadIdx.x; i < tot; i += NTHR_WS) smem[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
      for (int i = 0; i < NSTAGE; i++) { gwp::mbar_init(bar_full + i, gwp::NPROD_THR); gwp::mbar_init(bar_empty + i, NCONS); }
      gwp::mbar_init(bar_g, gwp::NPROD_THR);
      gwp::mbar_init(bar_phase, NCONS);
    }
  }
  __syncthreads();
  Ring ring; ring.full = bar_full; ring.empty = bar_empty; ring.nstage = NSTAGE; ring.it = 0;
  unsigned gpar = 0, ppar = 0;
  const int nmain = (naux + KC - 1) / KC;

  if (w >= NCONS) {
    // =============================== producer warpgroup ===============================
    gwp::reg_dec<40>();
    uint64_t polA, polB;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;\n" : "=l"(polA));
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(polB));
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      const int t = item % d.ntau, ik = item / d.ntau, k = P.kof(ik % P.nkeff), sg = ik / P.nkeff;
      const c128 *Gs = P.G + (size_t)sg * d.ntau * d.nk * n2;     // spin channel sg
      for (int ql = 0; ql < d.nq; ql++) {
        const int q = d.q0 + ql, kp = gw_ksub(d, k, q);
        const c128 *V1 = P.V + gw_vbwd(d, ql, kp, k) * vb;        // V[k][k-q][Q][i][a]
        const int yV = (int)gw_vfwd(d, ql, kp, k) * naux, yW = (t * d.nq + ql) * naux;   // first rows of V[k-q][k] and Wt[t][q] in the TMA views
        gwp::ws_issue_matrix<false>(sG, Gs + ((size_t)t * d.nk + kp) * n2, nao, ldp, P.fd_nao);
        gwp::cp_async_arrive_noinc(bar_g);
        for (int qt = 0; qt < P.nqt; qt++) {
          const int Q0 = qt * TM, tm_rows = min(TM, naux - Q0);
          for (int ch = 0; ch < P.nchunk; ch++) {
            const int nt0 = ch * P.cht, ntc = min(P.cht, P.nnt - nt0);
            for (int j = 0; j < nmain; j++) {
              const int s = ring.acquire();
              // main jobs come by TMA: one thread arms the barrier with the byte count and issues the boxes, the other
              // producer threads only arrive (the ring's full barriers count all 128 producer threads for every job type)
              if (w == NCONS) {                                  // first producer warp: its 32 lanes issue the boxes in one go
                const unsigned dst = gwp::smem_u32(sStage + s * P.stage_units);
                if (lane == 0) mbar_expect_tx(bar_full + s, (unsigned)(TM * KC * 16 + ntc * 1024));
                __syncwarp();
                if (lane == 31) tma_load_2d(dst, &tmW, 2 * KC * j, yW + Q0, bar_full + s, polA);
                if (lane < ntc) tma_load_2d(dst + TM * KC * 16 + 1024u * (unsigned)lane, &tmV, 16 * (nt0 + lane), yV + KC * j, bar_full + s, polB);
                if (lane != 0) gwp::mbar_arrive(bar_full + s);
              } else {
                gwp::mbar_arrive(bar_full + s);
              }
              ring.advance();
            }
          }
          const int rows = tm_rows * nao, npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
          gwp::mbar_wait(bar_phase, ppar); ppar ^= 1u;          // U^T of this panel is in slabU
          for (int j = 0; j < npass; j++) {
            const int s = ring.acquire();
            gwp::ws_issue_rows(sStage + s * P.stage_units, slabU, j * PASS_ROWS, rows, nao, ldp, P.fd_nao);
            ring.commit();
          }
          gwp::mbar_wait(bar_phase, ppar); ppar ^= 1u;          // T of this panel is in slabT
          const c128 *V1t = V1 + (size_t)Q0 * n2;
          for (int j = 0; j < tm_rows * P.kh; j++) {
            const int s = ring.acquire();
            const int jq = j / P.kh, h = j - jq * P.kh;
            gwp::ws_issue_final(sStage + s * P.stage_units, V1t + (size_t)jq * n2, slabT + (size_t)jq * n2, nao, P.ldpf, P.ldt, P.kspf, naop,
                                P.fd_nao, P.fd_kw, 4 * P.kspf * h);
            ring.commit();
          }
        }
      }
    }
    asm volatile("cp.async.wait_all;\n" ::: "memory");
  } else {
    // =============================== consumer warps ===============================
    gwp::reg_inc<232>();
    const int g = lane >> 2, c = lane & 3;
    const int rho = (g >> 1) + 4 * (g & 1);            // fragment row / column of this lane group in the TMA-swizzled main jobs
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      const int t = item % d.ntau, ik = item / d.ntau, k = P.kof(ik % P.nkeff), sg = ik / P.nkeff;
      c128 *Sout = P.Sigma + (((size_t)sg * d.ntau + t) * d.nk + k) * n2;
      double sgr[NCT][2], sgi[NCT][2];
#pragma unroll
      for (int i = 0; i < NCT; i++) { sgr[i][0] = sgr[i][1] = 0.0; sgi[i][0] = sgi[i][1] = 0.0; }
      if (P.acc_mode & GW_ACC_CONTINUE) gwp::final_load<NCT>(Sout, sgr, sgi, nao, ndt);
      for (int ql = 0; ql < d.nq; ql++) {
        gwp::mbar_wait(bar_g, gpar); gpar ^= 1u;
        for (int qt = 0; qt < P.nqt; qt++) {
          const int Q0 = qt * TM, tm_rows = min(TM, naux - Q0), mtc = (tm_rows + 7) / 8;
          // tile ownership: warp w owns m-tiles 2*mh, 2*mh+1 (mh = w >> 2) and every 4th n-tile; the ragged last panel
          // (<= 16 rows) is shared by all eight warps (m-tiles 0, 1, every 8th n-tile each)
          const bool narrow = mtc <= 2;
          const int mh = narrow ? 0 : (w >> 2);
          const int noff = narrow ? w : (((w & 3) - mh + 4) & 3);
          const int nstride = narrow ? 8 : 4;
          // ---- main GEMM, N chunk by N chunk; U^T written to slabU as [(Q,j)][b] ----
          for (int ch = 0; ch < P.nchunk; ch++) {
            const int nt0 = ch * P.cht, ntc = min(P.cht, P.nnt - nt0);
            const int n0 = nt0 * 8;
            const int njm = (ntc > noff) ? (ntc - noff + nstride - 1) / nstride : 0;
            const bool active = (mh * MT_W < mtc) && njm > 0;
            double accr[MT_W][NJ][2], acci[MT_W][NJ][2];
#pragma unroll
            for (int i = 0; i < MT_W; i++)
#pragma unroll
              for (int j = 0; j < NJ; j++) { accr[i][j][0] = accr[i][j][1] = 0.0; acci[i][j][0] = acci[i][j][1] = 0.0; }
            for (int jb = 0; jb < nmain; jb++) {
              const int s = ring.wait();
              if (active) {
                const c128 *sAw = sStage + s * P.stage_units + (8 * mh * MT_W + rho) * KC;
                const c128 *sBw = sStage + s * P.stage_units + TM * KC + 64 * noff;
                if (!narrow && njm == 7) main_compute<7>(sAw, sBw, accr, acci, c, rho);
                else if (!narrow && njm == 6) main_compute<6>(sAw, sBw, accr, acci, c, rho);
                else if (!narrow && njm == 5) main_compute<5>(sAw, sBw, accr, acci, c, rho);
                else {
#pragma unroll
                  for (int ks = 0; ks < KC / 4; ks++) {
                    const int kr = 4 * ks + c, u = kr ^ rho;
                    c128 a[MT_W];
#pragma unroll
                    for (int i = 0; i < MT_W; i++) a[i] = sAw[i * 8 * KC + u];
                    const c128 *bk = sBw + kr * 8 + u;
#pragma unroll
                    for (int jn = 0; jn < NJ; jn++) {
                      if (jn < njm) {
                        const c128 b = bk[64 * nstride * jn];
#pragma unroll
                        for (int i = 0; i < MT_W; i++) cmma(accr[i][jn], acci[i][jn], a[i], b);
                      }
                    }
                  }
                }
              }
              ring.release();
            }
            // store U^T: element (Q, n=(b,j)) -> slabU[(Q*nao + j)*nao + b]
#pragma unroll
            for (int i = 0; i < MT_W; i++) {
              const int Ql = 8 * (mh * MT_W + i) + rho;            // accumulator row g holds panel row rho(g)
#pragma unroll
              for (int jn = 0; jn < NJ; jn++) {
                if (jn < njm && Ql < tm_rows) {
#pragma unroll
                  for (int e = 0; e < 2; e++) {
                    const int n = n0 + 8 * (noff + nstride * jn) + c + 4 * e;   // accumulator columns 2c, 2c+1 hold columns c, c+4
                    if (n < n2) {
                      const int b = (int)P.fd_nao.div((unsigned)n), j = n - b * nao;
                      slabU[((size_t)Ql * nao + j) * nao + b] = make_double2(accr[i][jn][e], acci[i][jn][e]);
                    }
                  }
                }
              }
            }
          }
          __threadfence(); __syncwarp();
          if (lane == 0) gwp::mbar_arrive(bar_phase);
          // ---- pass A: T[Q][a][j] = Σ_b G[a][b] U[Q][b][j] ----
          const int rows = tm_rows * nao, npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
          for (int jb = 0; jb < npass; jb++) {
            const int s = ring.wait();
            if (P.ksp == KSP_MAX) gwp::pass_compute_exact_mt<KSP_MAX, true, 1>(sStage + s * P.stage_units, sG, slabT, jb * PASS_ROWS, rows, nao, ldp, w, P.fd_nao);
            else gwp::pass_compute<KSP_MAX, true>(sStage + s * P.stage_units, sG, slabT, jb * PASS_ROWS, rows, nao, ldp, P.ksp, ndt);
            ring.release();
          }
          __threadfence(); __syncwarp();
          if (lane == 0) gwp::mbar_arrive(bar_phase);
          // ---- final: Sigma[i][j] += Σ_(Q,a) V1[Q][i][a] T[Q][a][j]; one job per Q ----
          for (int jb = 0; jb < tm_rows * P.kh; jb++) {
            const int s = ring.wait();
            if (P.ksp == KSP_MAX && P.kh == 1) gwp::final_compute_exact<KSP_MAX, (KSP_MAX + 1) / 2, NCT>(sStage + s * P.stage_units, sgr, sgi, P.ldpf, P.ldt, naop);
            else if (P.ksp == KSP_MAX && P.kh == 2) gwp::final_compute_exact<(KSP_MAX + 1) / 2, (KSP_MAX + 1) / 2, NCT>(sStage + s * P.stage_units, sgr, sgi, P.ldpf, P.ldt, naop);
            else gwp::final_compute<NCT>(sStage + s * P.stage_units, sgr, sgi, P.ldpf, P.ldt, P.kspf, ndt, naop);
            ring.release();
          }
        }
      }
      const bool partial = (P.acc_mode & GW_ACC_PARTIAL) != 0;
      gwp::final_store<NCT>(Sout, sgr, sgi, partial ? 1.0 : -1.0 / (double)d.nk, nao, ndt);
      if (P.nkeff < d.nk && !partial) {                       // GW_SYM_TR: Sigma[t][-k] = conj(Sigma[t][k])
        const int kn = gw_ksub(d, 0, k);
        if (kn != k) gwp::final_store<NCT>(P.Sigma + (((size_t)sg * d.ntau + t) * d.nk + kn) * n2, sgr, sgi, -1.0 / (double)d.nk, nao, ndt, true);
      }
    }
  }
}

struct Plan {
  int stage_off;
  int ksp_max, nct, nqt, nitems, ldp, ksp, ndt, ldt, kh, kspf, ldpf, nnt, nchunk, cht, ldb, stage_units, grid, nstage;
  size_t smem, slab_units, work_bytes;
  bool ok;
};

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  pl.ksp = (d.nao + 3) / 4;
  if (pl.ksp > 16) { pl.ok = false; return pl; }
  pl.ksp_max = pl.ksp <= 7 ? 7 : (pl.ksp <= 13 ? 13 : 16);
  pl.ndt = (d.nao + 7) / 8;
  pl.nct = (pl.ndt * pl.ndt + 7) / 8 <= 2 ? 2 : 8;
  int r4 = pl.ksp * 4; if (r4 % 8 == 0) r4 += 4;
  pl.ldp = r4;
  int naop = 8 * pl.ndt;
  pl.ldt = naop + 2;                       // ≡ 2 (mod 8): conflict-free K-major B fragments
  pl.nnt = (d.nao * d.nao + 7) / 8;
  pl.nchunk = (pl.nnt + 4 * NJ - 1) / (4 * NJ);
  pl.cht = (pl.nnt + pl.nchunk - 1) / pl.nchunk;
  pl.ldb = pl.cht * 8 + 2;
  pl.nqt = (d.naux + TM - 1) / TM;
  { short tmp[128]; pl.nitems = d.ntau * fill_kirr(d, tmp) * d.ns; }
  const int s_pass = PASS_ROWS * pl.ldp, s_main = TM * KC + 64 * pl.cht;   // main: A 32 rows x 128 B + one 1 KB box per n-tile
  // the ring starts 1024-byte aligned and every stage is a multiple of 1024 bytes (TMA destinations, 128-byte swizzle)
  const size_t fixed = ((size_t)naop * pl.ldp * sizeof(c128) + 1023) / 1024 * 1024;
  pl.stage_off = (int)(fixed / sizeof(c128));
  // final jobs cover one Q, or half of its K range when a whole Q would leave fewer than 3 ring stages
  for (pl.kh = 1; pl.kh <= 2; pl.kh++) {
    pl.kspf = (pl.ksp + pl.kh - 1) / pl.kh;
    int f4 = pl.kspf * 4; if (f4 % 8 == 0) f4 += 4;
    pl.ldpf = f4;
    const int s_fin = naop * pl.ldpf + 4 * pl.kspf * pl.ldt + 8;
    pl.stage_units = s_pass;
    if (s_main > pl.stage_units) pl.stage_units = s_main;
    if (s_fin > pl.stage_units) pl.stage_units = s_fin;
    pl.stage_units = (pl.stage_units + 63) / 64 * 64;
    const size_t per = (size_t)pl.stage_units * sizeof(c128);
    pl.nstage = (int)((225 * 1024 - fixed) / per);
    if (pl.nstage > 6) pl.nstage = 6;
    pl.smem = fixed + (size_t)pl.nstage * per + 1024;
    if (pl.nstage >= 3) break;
  }
  if (pl.kh > 2) pl.kh = 2;
  const int nsm = gwp::gw_num_sms();
  pl.grid = pl.nitems < nsm ? pl.nitems : nsm;
  pl.slab_units = (((size_t)TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.work_bytes = 256 + (size_t)nsm * 2 * pl.slab_units * sizeof(c128);
  pl.ok = pl.nstage >= 2;
  return pl;
}

}  // namespace s3


static double s3_generic_flops(const gw_problem *p) {
  s3::Plan pl = s3::make_plan(p);
  if (!pl.ok) return 0.0;
  GwDims d = gw_dims(p);
  double tiles = 0.0;
  const double nmain = (d.naux + s3::KC - 1) / s3::KC;
  for (int qt = 0; qt < pl.nqt; qt++) {
    const int tm_rows = (d.naux - qt * s3::TM) < s3::TM ? (d.naux - qt * s3::TM) : s3::TM;
    const int mtc = (tm_rows + 7) / 8;
    const double mtiles = (mtc <= 2) ? (((d.nao + 3) / 4 == 7) ? (double)mtc : 2.0) /* ragged panel shared by all warps; s3 always runs 2 m-tiles */ : (double)((mtc + s3::MT_W - 1) / s3::MT_W) * s3::MT_W;
    tiles += mtiles * pl.nnt * (s3::KC / 4) * nmain;                         // main
    tiles += (double)((tm_rows * d.nao + 7) / 8) * gwp::pass_mtile_flops(d.nao, pl.ndt, pl.ksp, pl.ksp == pl.ksp_max) / 2048.0;   // pass A
    tiles += (double)tm_rows * pl.ndt * pl.ndt * pl.kspf * pl.kh;             // final
  }
  short tmp[128];
  return tiles * (double)d.nq * fill_kirr(d, tmp) * d.ntau * d.ns * 2048.0;
}

template <int KSP_MAX, int NCT>
static int launch_sigma(const s3::Plan &pl, const s3::Params &P, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(s3::sigma_kernel<KSP_MAX, NCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return (int)e;
  // tensor maps of the main jobs: Wt as [ntau*nq*naux rows][naux complex] (box 32 x 8), V as [nk*nk*naux rows][nao² complex] (box 8 x 8)
  CUtensorMap tmW, tmV;
  int rc = gwp::make_tensor_map(&tmW, P.Wt, (size_t)P.d.ntau * P.d.nq * P.d.naux, P.d.naux, s3::TM);
  if (rc) return rc;
  rc = gwp::make_tensor_map(&tmV, P.V, gw_vblocks(P.d) * P.d.naux, P.d.nao * P.d.nao, s3::KC);
  if (rc) return rc;
  s3::sigma_kernel<KSP_MAX, NCT><<<pl.grid, s3::NTHR_WS, pl.smem, st>>>(P, tmW, tmV);
  return (int)cudaGetLastError();
}

namespace s3 {
static int launch(const gw_problem *p, const c128 *G, const c128 *Wt, c128 *Sigma, cudaStream_t st, int acc_mode) {
  Plan pl = make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  s3::Params P;
  P.acc_mode = acc_mode;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.G = G; P.Wt = Wt; P.Sigma = Sigma;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.nqt = pl.nqt; P.nitems = pl.nitems; P.ldp = pl.ldp; P.ksp = pl.ksp; P.ndt = pl.ndt; P.ldt = pl.ldt; P.kh = pl.kh; P.kspf = pl.kspf; P.ldpf = pl.ldpf; P.fd_kw = gwp::FastDiv((unsigned)(4 * pl.kspf));
  P.nnt = pl.nnt; P.nchunk = pl.nchunk; P.cht = pl.cht; P.ldb = pl.ldb; P.stage_units = pl.stage_units; P.nstage = pl.nstage; P.stage_off = pl.stage_off; P.slab_units = pl.slab_units;
  P.fd_nao = gwp::FastDiv((unsigned)P.d.nao);
  P.nkeff = fill_kirr(P.d, P.kirr);
  if (pl.nct == 2) {
    if (pl.ksp_max == 7) return launch_sigma<7, 2>(pl, P, st);
    if (pl.ksp_max == 13) return launch_sigma<13, 2>(pl, P, st);
    return launch_sigma<16, 2>(pl, P, st);
  } else {
    if (pl.ksp_max == 7) return launch_sigma<7, 8>(pl, P, st);
    if (pl.ksp_max == 13) return launch_sigma<13, 8>(pl, P, st);
    return launch_sigma<16, 8>(pl, P, st);
  }
}
}  // namespace s3

// =====================================================================================================================
// s3w — warp-specialised stage-3 kernel for the production basis classes nao = 25..28 (KSP = 7 k-steps over nao, 4 x 4 Sigma
// tiles) and nao = 49..52 (KSP = 13, 7 x 7 tiles).  Same algebra as s3::sigma_kernel; the work of one (q, Q-panel) unit is
// split between warp roles that run concurrently:
//   main warps 0-7  : U = W·V2 (N chunk by N chunk, accumulators in registers), U^T stored to slabU[unit & 1].
//                     Complex tile products use the 3M scheme (three real DMMAs per complex 8x8x4 product instead of four):
//                       K1 += Ar·Br,  K2 += Ai·Bi,  K3 += (Ar+Ai)·(Br+Bi);   Re U = K1 − K2,  Im U = K3 − K1 − K2
//                     with three real accumulator sets per tile (warp tile 2 x 4 tiles = 96 registers) and the two operand sums
//                     formed in registers after the fragment loads (one DADD per fragment) (measured against the 4-real-GEMM scheme in
//                     profiles/r02_3m_vs_4m.md).
//   aux warps 8-11  : for the PREVIOUS unit: pass A (T = G·U, slabU -> slabT) and the final contraction
//                     Sigma += Σ_(Q,a) V1[Q][i][a] T[Q][a][j] (4-real-GEMM scheme); the nao x nao Sigma accumulator of the item
//                     lives in their registers (Sigma tile w + 4 i belongs to aux warp w)
//   producer warps  : one thread of warp 12 feeds the main ring by TMA (W panel + V2 chunk), warp 15 feeds the aux ring
//                     (G, slabU rows, V1 + slabT) with cp.async
// so the DMMA pipe never drains at a phase change and the small-K phases run beside the big GEMM.
// =====================================================================================================================
namespace s3w {

using gwp::FastDiv;
constexpr int NMAINW = 8, NAUXW = 4, NTHR = 512;
// aux-ring producer threads: the last NAP threads of the CTA (Geo<KSP>::NAP)
constexpr int KC = 8, MT_W = 2, NJ = 4, TM = 32;
constexpr int AROWS = 32;                     // pass A: rows per job (one m-tile per aux warp)
constexpr int NST_MAX = 8, AST_MAX = 4;
constexpr int REG_MAIN = 152, REG_AUX = 168, REG_PROD = 40;   // 256*152 + 128*168 + 128*40 = 65536

// compile-time geometry of a basis class: KSP = ceil(nao/4)
template <int KSP> struct Geo {
  static constexpr int NDT = (KSP + 1) / 2;                       // 8-wide tiles over nao
  static constexpr int NTA = (NDT * NDT + NAUXW - 1) / NAUXW;     // Sigma tiles per aux warp
  // aux-ring producer threads: warp 15, or warps 13-15 for the wide basis class (1 664-2 080 cp.async per aux job there).  Measured on
  // config Q, stage 3: 4 440 ms with 32 threads, 4 358 with 64, 4 346 with 96; at nao = 26 more producer threads cost (config P 296 -> 301 ms with 64)
  static constexpr int NAP = KSP <= 8 ? 32 : 96;
  static constexpr int KH = KSP <= 8 ? 1 : 3;                     // K pieces of one Q's final contraction (shared-memory budget)
  static constexpr int KSPF = (KSP + KH - 1) / KH;                // k-steps per piece (the last piece may have fewer)
  static constexpr int LDP = (4 * KSP) % 8 == 0 ? 4 * KSP + 4 : 4 * KSP;       // ≡ 4 (mod 8): conflict-free K-contiguous fragments
  static constexpr int LDPF = (4 * KSPF) % 8 == 0 ? 4 * KSPF + 4 : 4 * KSPF;
  static constexpr int LDT = 8 * NDT + 2;                         // ≡ 2 (mod 8): conflict-free K-major fragments
  static constexpr int AUX_UNITS = (AROWS * LDP > 8 * NDT * LDPF + 4 * KSPF * LDT + 8) ? AROWS * LDP : 8 * NDT * LDPF + 4 * KSPF * LDT + 8;
};

struct Params {
  GwDims d;
  const c128 *V, *G, *Wt;
  c128 *Sigma, *scratch;
  int nqt, nitems;
  int nnt, nchunk, cht;   // n-tiles over nao², N chunks, n-tiles per chunk
  int main_units, nstage, astage;
  int main_off;           // offset of the main ring in the 1024-byte aligned dynamic shared memory (complex elements)
  size_t slab_units;      // complex elements per slab (three slabs per CTA: U0, U1, T)
  int nkeff;              // k points evaluated: nk, or the k <= -k half under GW_SYM_TR (Sigma[-k] = conj Sigma[k] is copied)
  short kirr[128];        // the evaluated k points when nkeff < nk
  __device__ __forceinline__ int kof(int i) const { return nkeff < d.nk ? (int)kirr[i] : i; }
  int acc_mode;           // GW_ACC_CONTINUE / GW_ACC_PARTIAL (gw_common.cuh)
  FastDiv fd_nao;
};

using gwp::Ring;

// main job in shared memory (both parts written by TMA with the 128-byte swizzle: 16-byte unit u of row r sits at u ^ (r & 7)):
//   A = W[TM rows][8 K]                    32 rows x 128 B
//   B = one 1 KB box per n-tile: [8 K rows][8 columns]
// Lane group g reads row / column rho(g) = (g >> 1) + 4 (g & 1) of its tile, so a quarter-warp touches eight different units.
// 3M: k1 += Ar Br, k2 += Ai Bi, k3 += (Ar+Ai)(Br+Bi).
template <int NJM, int NSTRIDE = 4, int MTW = MT_W>
__device__ __forceinline__ void main_compute(const c128 *sAw, const c128 *sBw, double (&k1)[MT_W][NJ][2], double (&k2)[MT_W][NJ][2],
                                             double (&k3)[MT_W][NJ][2], int c, int rho) {
#pragma unroll
  for (int ks = 0; ks < KC / 4; ks++) {
    const int kr = 4 * ks + c;
    const int u = kr ^ rho;
    c128 a[MTW], b[NJM];
    double as[MTW];
#pragma unroll
    for (int i = 0; i < MTW; i++) a[i] = sAw[i * 8 * KC + u];
    const c128 *bk = sBw + kr * 8 + u;                  // row kr of the box, column rho swizzled by the row
#pragma unroll
    for (int jn = 0; jn < NJM; jn++) b[jn] = bk[64 * NSTRIDE * jn];
#pragma unroll
    for (int i = 0; i < MTW; i++) as[i] = a[i].x + a[i].y;
#pragma unroll
    for (int jn = 0; jn < NJM; jn++) {
      const double bs = b[jn].x + b[jn].y;
#pragma unroll
      for (int i = 0; i < MTW; i++) {
        dmma884(k1[i][jn][0], k1[i][jn][1], a[i].x, b[jn].x);
        dmma884(k2[i][jn][0], k2[i][jn][1], a[i].y, b[jn].y);
        dmma884(k3[i][jn][0], k3[i][jn][1], as[i], bs);
      }
    }
  }
}

// aux ring jobs (producer warp 15)
template <int NAP>
__device__ __forceinline__ void issue_rows(c128 *stage, const c128 *src, int row0, int rows_total, int nao, int ldp, FastDiv fd) {
  constexpr int T_APROD = NTHR - NAP, N_APROD = NAP;
  const int nrow = min(AROWS, rows_total - row0);
  const int total = nrow * nao;
  const c128 *s = src + (size_t)row0 * nao;
  for (int i = threadIdx.x - T_APROD; i < total; i += N_APROD) {
    const int r = (int)fd.div((unsigned)i), a = i - r * nao;
    cp_async16(stage + r * ldp + a, s + i);
  }
}
// final job for the K range [a0, a0 + 4 ksn) of one Q: A = V1[Q][i][a0..] -> stage[i][ldpf]; B = T[Q][a0..][j] -> [a - a0][ldt];
// K beyond nao is zero filled
template <int NDT, int NAP>
__device__ __forceinline__ void issue_final(c128 *stage, const c128 *Aq, const c128 *Bq, int nao, int ldpf, int ldt, int a0, int ksn, FastDiv fd) {
  constexpr int T_APROD = NTHR - NAP, N_APROD = NAP;
  const int lane = threadIdx.x - T_APROD, kw = 4 * ksn;
  if (a0 == 0 && kw >= nao) {                            // whole rows (one piece per Q)
    for (int i = lane; i < nao * nao; i += N_APROD) {
      const int r = (int)fd.div((unsigned)i), a = i - r * nao;
      cp_async16(stage + r * ldpf + a, Aq + i);
    }
  } else {
    const FastDiv fk((unsigned)kw);
    for (int i = lane; i < nao * kw; i += N_APROD) {
      const int r = (int)fk.div((unsigned)i), cc = i - r * kw;
      const bool ok = a0 + cc < nao;
      gwp::cp_async16_zfill(stage + r * ldpf + cc, ok ? Aq + r * nao + a0 + cc : Aq, ok);
    }
  }
  c128 *sB = stage + 8 * NDT * ldpf;
  for (int i = lane; i < kw * nao; i += N_APROD) {
    const int r = (int)fd.div((unsigned)i);
    const bool ok = a0 + r < nao;
    gwp::cp_async16_zfill(sB + r * ldt + (i - r * nao), ok ? Bq + (size_t)a0 * nao + i : Bq, ok);
  }
}
template <int NAP>
__device__ __forceinline__ void issue_matrix(c128 *sG, const c128 *src, int nao, int ldp, FastDiv fd) {
  constexpr int T_APROD = NTHR - NAP, N_APROD = NAP;
  for (int i = threadIdx.x - T_APROD; i < nao * nao; i += N_APROD) {
    const int r = (int)fd.div((unsigned)i), cc = i - r * nao;
    cp_async16(sG + r * ldp + cc, src + i);
  }
}

// aux warps: Sigma tiles t = w + 4 i (row tile t / NDT, column tile t % NDT):  acc[i] += A[row tile][K] · B[K][column tile] over
// the ksn k-steps of the job.  For NDT = 4 the warp's tiles share one column tile: one B fragment per k-step feeds four tiles.
// NMT < NDT (edge mode, NDT = 4): only the row tiles 0 .. NMT-1 of the warp's column tile; the rest is final_edge_fma's.
template <int KSP, int NMT = Geo<KSP>::NDT>
__device__ __forceinline__ void final_compute(const c128 *stage, double (&sgr)[Geo<KSP>::NTA][2], double (&sgi)[Geo<KSP>::NTA][2], int w, int ksn) {
  using Gm = Geo<KSP>;
  constexpr int NDT = Gm::NDT, NTA = Gm::NTA, ldpf = Gm::LDPF, ldt = Gm::LDT;
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  const c128 *ap = stage + g * ldpf + c;
  const c128 *bp = stage + 8 * NDT * ldpf + c * ldt + g;
  if constexpr (NDT == 4) {
#pragma unroll
    for (int ks = 0; ks < Gm::KSPF; ks++) {
      const c128 b = bp[4 * ks * ldt + 8 * w];
      c128 a[NMT];
#pragma unroll
      for (int mi = 0; mi < NMT; mi++) a[mi] = ap[8 * mi * ldpf + 4 * ks];
#pragma unroll
      for (int mi = 0; mi < NMT; mi++) cmma(sgr[mi], sgi[mi], a[mi], b);
    }
  } else {
    int aoff[NTA], boff[NTA];
#pragma unroll
    for (int i = 0; i < NTA; i++) {
      const int t = min(w + NAUXW * i, NDT * NDT - 1), mi = t / NDT, nj = t - mi * NDT;
      aoff[i] = 8 * mi * ldpf; boff[i] = 8 * nj;
    }
#pragma unroll
    for (int ks = 0; ks < Gm::KSPF; ks++) {
      if (ks < ksn) {
#pragma unroll
        for (int i = 0; i < NTA; i++) {
          if (w + NAUXW * i < NDT * NDT) cmma(sgr[i], sgi[i], ap[aoff[i] + 4 * ks], bp[4 * ks * ldt + boff[i]]);
        }
      }
    }
  }
}

// Edge mode (nao = 25, 26: gwp::pass_tail_fma; NDT = 4, one K piece).  The 26 x 26 Sigma block is a 3 x 3 grid of full 8 x 8 tiles
// plus a column strip (rows 0..nao-1 x columns 24, 25) and a row strip (rows 24, 25 x columns 0..23).  Seven of the sixteen tiles of
// the padded 4 x 4 grid hold those strips with two valid lines of eight; in edge mode aux warps 0..2 run the full tiles of their
// column tile on the tensor cores and aux warp 3 forms both strips with plain FP64 FMAs from the same fragments: lane (g, c) sums
// its own k = 4 ks + c,
//   tc[mi][e] += A[8 mi + g][k] B[k][24 + e]        (column strip; the 2 x 2 corner is its mi = 3, g < 2)
//   tr[nj][e] += A[24 + e][k]   B[k][8 nj + g]      (row strip)
// and the four lanes of a group add up once per unit (edge_reduce), so that the sum of a unit does not depend on where a V slab ends
// (GW_ACC_PARTIAL / GW_ACC_CONTINUE stay bit-identical to the resident call).
template <int KSP>
__device__ __forceinline__ void final_edge_fma(const c128 *stage, c128 (&tc)[4][2], c128 (&tr)[3][2]) {
  using Gm = Geo<KSP>;
  constexpr int NDT = Gm::NDT, ldpf = Gm::LDPF, ldt = Gm::LDT, N0 = 8 * (NDT - 1);
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  const c128 *ap = stage + g * ldpf + c;
  const c128 *ae = stage + N0 * ldpf + c;                       // rows 24, 25 of A (the same address in every lane group)
  const c128 *bp = stage + 8 * NDT * ldpf + c * ldt + g;
  const c128 *be = stage + 8 * NDT * ldpf + c * ldt + N0;       // columns 24, 25 of B
#pragma unroll
  for (int ks = 0; ks < Gm::KSPF; ks++) {
    const c128 b0 = be[4 * ks * ldt], b1 = be[4 * ks * ldt + 1];
    const c128 a0 = ae[4 * ks], a1 = ae[ldpf + 4 * ks];
    c128 a[NDT], b[NDT - 1];
#pragma unroll
    for (int mi = 0; mi < NDT; mi++) a[mi] = ap[8 * mi * ldpf + 4 * ks];
#pragma unroll
    for (int nj = 0; nj < NDT - 1; nj++) b[nj] = bp[4 * ks * ldt + 8 * nj];
#pragma unroll
    for (int mi = 0; mi < NDT; mi++) { cfma(tc[mi][0], a[mi], b0); cfma(tc[mi][1], a[mi], b1); }
#pragma unroll
    for (int nj = 0; nj < NDT - 1; nj++) { cfma(tr[nj][0], a0, b[nj]); cfma(tr[nj][1], a1, b[nj]); }
  }
}
// (pr, pi) += sum of t over the four lanes of a group
__device__ __forceinline__ void edge_reduce(double &pr, double &pi, c128 t) {
#pragma unroll
  for (int off = 1; off <= 2; off <<= 1) {
    t.x += __shfl_xor_sync(0xffffffffu, t.x, off);
    t.y += __shfl_xor_sync(0xffffffffu, t.y, off);
  }
  pr += t.x; pi += t.y;
}

template <int KSP>
__global__ void __launch_bounds__(NTHR, 1) sigma_ws_kernel(const Params P, const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmV) {
  using Gm = Geo<KSP>;
  constexpr int NDT = Gm::NDT, NTA = Gm::NTA, ldp = Gm::LDP, ldpf = Gm::LDPF, ldt = Gm::LDT, AUXU = Gm::AUX_UNITS, N_APROD = Gm::NAP;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // the TMA destinations (128-byte swizzle) need 1024-byte alignment: the launch asks for 1 KB of slack
  c128 *smem = reinterpret_cast<c128 *>(smem_raw + ((1024u - (gwp::smem_u32(smem_raw) & 1023u)) & 1023u));
  const GwDims d = P.d;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao;
  c128 *sG = smem;                                   // [8 NDT][ldp]: sG[a][b] = G[t][k-q][a][b]
  c128 *sAux = sG + 8 * NDT * ldp;                   // astage x AUXU
  c128 *sMain = smem + P.main_off;                   // nstage x main_units, 1024-byte aligned stages
  __shared__ uint64_t bars[2 * NST_MAX + 2 * AST_MAX + 6];
  uint64_t *full_m = bars, *empty_m = bars + NST_MAX, *full_a = bars + 2 * NST_MAX, *empty_a = full_a + AST_MAX;
  uint64_t *bar_g = empty_a + AST_MAX, *bar_phase = bar_g + 1, *uready = bar_g + 2, *ufree = bar_g + 4;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  c128 *slabU = P.scratch + (size_t)blockIdx.x * 3 * P.slab_units;
  c128 *slabT = slabU + 2 * P.slab_units;
  const size_t vb = (size_t)naux * n2;
  const int nmain = (naux + KC - 1) / KC;
  {
    const int tot = P.main_off + P.nstage * P.main_units;
    for (int i = threadIdx.x; i < tot; i += NTHR) smem[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
      for (int i = 0; i < P.nstage; i++) { gwp::mbar_init(full_m + i, 1); gwp::mbar_init(empty_m + i, NMAINW); }
      for (int i = 0; i < P.astage; i++) { gwp::mbar_init(full_a + i, N_APROD); gwp::mbar_init(empty_a + i, NAUXW); }
      gwp::mbar_init(bar_g, N_APROD);
      gwp::mbar_init(bar_phase, NAUXW);
      for (int i = 0; i < 2; i++) { gwp::mbar_init(uready + i, NMAINW); gwp::mbar_init(ufree + i, NAUXW); }
    }
  }
  __syncthreads();

  if (w >= NMAINW + NAUXW) {
    gwp::reg_dec<REG_PROD>();
    if (w < 16 - N_APROD / 32) {
      // ---- main-ring producer: the 32 lanes of warp 12 issue the TMA box loads of a job in one go (lane 0 arms the stage's
      //      mbarrier with the byte count, lanes < ntc load one 8 x 8 box of V2 each, lane 31 loads the W panel K slice) ----
      if (w == NMAINW + NAUXW) {
        Ring rm; rm.full = full_m; rm.empty = empty_m; rm.nstage = P.nstage; rm.it = 0; rm.ph = 0;
        const uint64_t polA = gwp::policy_evict_normal(), polB = gwp::policy_evict_last();
        for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
          const int t = item % d.ntau, k = P.kof((item / d.ntau) % P.nkeff);
          for (int ql = 0; ql < d.nq; ql++) {
            const int kp = gw_ksub(d, k, d.q0 + ql);
            const int yV = (int)gw_vfwd(d, ql, kp, k) * naux;         // V[k-q][k] rows of V viewed as [blocks*naux][nao²]
            const int yW = (t * d.nq + ql) * naux;                    // Wt[t][q] rows of Wt viewed as [ntau*nq*naux][naux]
            for (int qt = 0; qt < P.nqt; qt++) {
              for (int ch = 0; ch < P.nchunk; ch++) {
                const int nt0 = ch * P.cht, ntc = min(P.cht, P.nnt - nt0);
                for (int j = 0; j < nmain; j++) {
                  const int s = rm.acquire();
                  const unsigned dst = gwp::smem_u32(sMain + s * P.main_units);
                  if (lane == 0) gwp::mbar_expect_tx(full_m + s, (unsigned)(TM * KC * 16 + ntc * 1024));
                  __syncwarp();
                  if (lane == 31) gwp::tma_load_2d(dst, &tmW, 2 * KC * j, yW + qt * TM, full_m + s, polA);
                  if (lane < ntc) gwp::tma_load_2d(dst + TM * KC * 16 + 1024u * (unsigned)lane, &tmV, 16 * (nt0 + lane), yV + KC * j, full_m + s, polB);
                  rm.advance();
                }
              }
            }
          }
        }
      }
    } else {
      // ---- aux-ring producer: G per q, U^T rows of the finished unit (pass A), then V1[Q] + T[Q] per Q and K piece (final) ----
      Ring ra; ra.full = full_a; ra.empty = empty_a; ra.nstage = P.astage; ra.it = 0; ra.ph = 0;
      unsigned un = 0;
      for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
        const int t = item % d.ntau, ik = item / d.ntau, k = P.kof(ik % P.nkeff), sg = ik / P.nkeff;
        const c128 *Gs = P.G + (size_t)sg * d.ntau * d.nk * n2;   // spin channel sg
        for (int ql = 0; ql < d.nq; ql++) {
          const int kp = gw_ksub(d, k, d.q0 + ql);
          const c128 *V1 = P.V + gw_vbwd(d, ql, kp, k) * vb;      // V[k][k-q][Q][i][a]
          for (int qt = 0; qt < P.nqt; qt++, un++) {
            const int Q0 = qt * TM, tm_rows = min(TM, naux - Q0), rows = tm_rows * nao, npass = (rows + AROWS - 1) / AROWS;
            const c128 *U = slabU + (size_t)(un & 1u) * P.slab_units;
            // sG is free: pass A of the previous unit completed before its final jobs were issued
            if (qt == 0) issue_matrix<N_APROD>(sG, Gs + ((size_t)t * d.nk + kp) * n2, nao, ldp, P.fd_nao);
            gwp::cp_async_arrive_noinc(bar_g);
            gwp::mbar_wait(uready + (un & 1u), (un >> 1) & 1u);
            for (int j = 0; j < npass; j++) {
              const int s = ra.acquire();
              issue_rows<N_APROD>(sAux + s * AUXU, U, j * AROWS, rows, nao, ldp, P.fd_nao);
              ra.commit();
            }
            gwp::mbar_wait(bar_phase, un & 1u);                     // T of this unit is in slabT
            const c128 *V1t = V1 + (size_t)Q0 * n2;
            for (int j = 0; j < tm_rows; j++) {
#pragma unroll
              for (int h = 0; h < Gm::KH; h++) {
                const int s = ra.acquire();
                issue_final<NDT, N_APROD>(sAux + s * AUXU, V1t + (size_t)j * n2, slabT + (size_t)j * n2, nao, ldpf, ldt, 4 * Gm::KSPF * h,
                                 min(Gm::KSPF, KSP - Gm::KSPF * h), P.fd_nao);
                ra.commit();
              }
            }
          }
        }
      }
      asm volatile("cp.async.wait_all;\n" ::: "memory");
    }
  } else if (w >= NMAINW) {
    // ============================================ aux warps ============================================
    gwp::reg_inc<REG_AUX>();
    const int wa = w - NMAINW, g = lane >> 2, c = lane & 3;
    constexpr int EN0 = 8 * (NDT - 1);
    const bool edge = NDT == 4 && gwp::pass_tail_fma(nao, NDT);     // nao = 25, 26 (final_edge_fma)
    const bool ew = edge && wa == NAUXW - 1;                         // this warp forms the two strips
    Ring ra; ra.full = full_a; ra.empty = empty_a; ra.nstage = P.astage; ra.it = 0; ra.ph = 0;
    unsigned un = 0;
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      const int t = item % d.ntau, ik = item / d.ntau, k = P.kof(ik % P.nkeff), sg = ik / P.nkeff;
      c128 *Sst = P.Sigma + ((size_t)sg * d.ntau + t) * d.nk * n2;       // Sigma[sg][t]
      double sgr[NTA][2], sgi[NTA][2];
      // edge mode, aux warp 3: sgr / sgi[mi] hold the column strip (rows 8 mi + g, columns 24, 25: the places they have in the
      // accumulator of tile (mi, 3) in lane c = 0), pr the row strip (rows 24, 25, column 8 nj + g)
      c128 pr[3][2];
#pragma unroll
      for (int i = 0; i < NTA; i++) { sgr[i][0] = sgr[i][1] = 0.0; sgi[i][0] = sgi[i][1] = 0.0; }
#pragma unroll
      for (int i = 0; i < 3; i++) pr[i][0] = pr[i][1] = make_double2(0.0, 0.0);
      if (P.acc_mode & GW_ACC_CONTINUE) {                     // continue the q sum from the unscaled partial sums of the previous V slab
        const c128 *in = Sst + (size_t)k * n2;
#pragma unroll
        for (int ti = 0; ti < NTA; ti++) {
          const int tile = wa + NAUXW * ti;
          if (tile < NDT * NDT) {
            const int mi = tile / NDT, nj = tile - mi * NDT;
            const int i = 8 * mi + g, j0 = 8 * nj + 2 * c;
            if (i < nao && !(edge && !ew && mi == NDT - 1)) {
              if (j0 < nao) { sgr[ti][0] = in[i * nao + j0].x; sgi[ti][0] = in[i * nao + j0].y; }
              if (j0 + 1 < nao) { sgr[ti][1] = in[i * nao + j0 + 1].x; sgi[ti][1] = in[i * nao + j0 + 1].y; }
            }
          }
        }
        if (ew) {
#pragma unroll
          for (int e = 0; e < 2; e++) {
            if (EN0 + e < nao) {
#pragma unroll
              for (int nj = 0; nj < 3; nj++) pr[nj][e] = in[(EN0 + e) * nao + 8 * nj + g];
            }
          }
        }
      }
      for (int ql = 0; ql < d.nq; ql++) {
        for (int qt = 0; qt < P.nqt; qt++, un++) {
          const int Q0 = qt * TM, tm_rows = min(TM, naux - Q0), rows = tm_rows * nao, npass = (rows + AROWS - 1) / AROWS;
          gwp::mbar_wait(bar_g, un & 1u);
          for (int j = 0; j < npass; j++) {
            const int s = ra.wait();
            gwp::pass_compute_exact_mt<KSP, true, 1>(sAux + s * AUXU, sG, slabT, j * AROWS, rows, nao, ldp, wa, P.fd_nao);
            ra.release();
          }
          __threadfence(); __syncwarp();
          if (lane == 0) { gwp::mbar_arrive(bar_phase); gwp::mbar_arrive(ufree + (un & 1u)); }
          c128 tc[4][2], tr[3][2];                              // edge mode: the strips' sums over this unit, per k class
#pragma unroll
          for (int e = 0; e < 2; e++) {
#pragma unroll
            for (int i = 0; i < 4; i++) tc[i][e] = make_double2(0.0, 0.0);
#pragma unroll
            for (int i = 0; i < 3; i++) tr[i][e] = make_double2(0.0, 0.0);
          }
          for (int j = 0; j < tm_rows; j++) {
#pragma unroll
            for (int h = 0; h < Gm::KH; h++) {
              const int s = ra.wait();
              if constexpr (NDT == 4) {
                if (ew) final_edge_fma<KSP>(sAux + s * AUXU, tc, tr);
                else if (edge) final_compute<KSP, NDT - 1>(sAux + s * AUXU, sgr, sgi, wa, Gm::KSPF);
                else final_compute<KSP>(sAux + s * AUXU, sgr, sgi, wa, Gm::KSPF);
              } else {
                final_compute<KSP>(sAux + s * AUXU, sgr, sgi, wa, min(Gm::KSPF, KSP - Gm::KSPF * h));
              }
              ra.release();
            }
          }
          if (ew) {                                             // the strips of this unit: add the four k classes up
#pragma unroll
            for (int e = 0; e < 2; e++) {
#pragma unroll
              for (int i = 0; i < 4; i++) edge_reduce(sgr[i][e], sgi[i][e], tc[i][e]);
#pragma unroll
              for (int i = 0; i < 3; i++) edge_reduce(pr[i][e].x, pr[i][e].y, tr[i][e]);
            }
          }
        }
      }
      // Sigma[t][k] = -(1/N_k) acc: this warp's tiles
      const bool partial = (P.acc_mode & GW_ACC_PARTIAL) != 0;
      const double pref = partial ? 1.0 : -1.0 / (double)d.nk;
      const int kn = gw_ksub(d, 0, k);
      const int ncopy = (P.nkeff < d.nk && kn != k && !partial) ? 2 : 1;  // GW_SYM_TR: Sigma[t][-k] = conj(Sigma[t][k])
      for (int cp = 0; cp < ncopy; cp++) {
        c128 *out = Sst + (size_t)(cp ? kn : k) * n2;
        const double prefi = cp ? -pref : pref;
#pragma unroll
        for (int ti = 0; ti < NTA; ti++) {
          const int tile = wa + NAUXW * ti;
          if (tile < NDT * NDT) {
            const int mi = tile / NDT, nj = tile - mi * NDT;
            const int i = 8 * mi + g, j0 = 8 * nj + 2 * c;
            if (i < nao && !(edge && !ew && mi == NDT - 1)) {
              if (j0 < nao) out[i * nao + j0] = make_double2(pref * sgr[ti][0], prefi * sgi[ti][0]);
              if (j0 + 1 < nao) out[i * nao + j0 + 1] = make_double2(pref * sgr[ti][1], prefi * sgi[ti][1]);
            }
          }
        }
        if (ew && c == 0) {
#pragma unroll
          for (int e = 0; e < 2; e++) {
            if (EN0 + e < nao) {
#pragma unroll
              for (int nj = 0; nj < 3; nj++) out[(EN0 + e) * nao + 8 * nj + g] = make_double2(pref * pr[nj][e].x, prefi * pr[nj][e].y);
            }
          }
        }
      }
    }
  } else {
    // ============================================ main warps ============================================
    gwp::reg_inc<REG_MAIN>();
    const int g = lane >> 2, c = lane & 3;
    const int rho = (g >> 1) + 4 * (g & 1);           // fragment row / column of this lane group (see main_compute)
    Ring rm; rm.full = full_m; rm.empty = empty_m; rm.nstage = P.nstage; rm.it = 0; rm.ph = 0;
    unsigned un = 0;
    for (int item = blockIdx.x; item < P.nitems; item += gridDim.x) {
      for (int ql = 0; ql < d.nq; ql++) {
        for (int qt = 0; qt < P.nqt; qt++, un++) {
          const int Q0 = qt * TM, tm_rows = min(TM, naux - Q0), mtc = (tm_rows + 7) / 8;
          c128 *U = slabU + (size_t)(un & 1u) * P.slab_units;
          // tile ownership.  Full panels: warp w owns m-tiles 2*mh, 2*mh+1 (mh = w >> 2) and every 4th n-tile of the chunk (the column
          // group is rotated by mh, so the two main warps of a scheduler carry different groups).  The ragged last panel (<= 16 rows)
          // is shared by all eight warps (m-tiles 0 (and 1), every 8th n-tile each): it costs time in proportion to its rows.
          const bool narrow = mtc <= 2;
          const int mh = narrow ? 0 : (w >> 2);
          const int noff = narrow ? w : (((w & 3) - mh + 4) & 3);
          const int nstride = narrow ? 8 : 4;
          const int mtw = (narrow && mtc == 1) ? 1 : MT_W;
          for (int ch = 0; ch < P.nchunk; ch++) {
            const int nt0 = ch * P.cht, ntc = min(P.cht, P.nnt - nt0), n0 = nt0 * 8;
            const int njm = (ntc > noff) ? (ntc - noff + nstride - 1) / nstride : 0;
            const bool active = (mh * MT_W < mtc) && njm > 0;
            double k1[MT_W][NJ][2], k2[MT_W][NJ][2], k3[MT_W][NJ][2];
#pragma unroll
            for (int i = 0; i < MT_W; i++)
#pragma unroll
              for (int j = 0; j < NJ; j++) { k1[i][j][0] = k1[i][j][1] = 0.0; k2[i][j][0] = k2[i][j][1] = 0.0; k3[i][j][0] = k3[i][j][1] = 0.0; }
            for (int jb = 0; jb < nmain; jb++) {
              const int s = rm.wait();
              if (active) {
                const c128 *sAw = sMain + s * P.main_units + (8 * mh * MT_W + rho) * KC;
                const c128 *sBw = sMain + s * P.main_units + TM * KC + 64 * noff;
                if (narrow) {
                  if (mtw == 1 && njm == 2) main_compute<2, 8, 1>(sAw, sBw, k1, k2, k3, c, rho);
                  else if (mtw == 1) main_compute<1, 8, 1>(sAw, sBw, k1, k2, k3, c, rho);
                  else if (njm == 2) main_compute<2, 8, 2>(sAw, sBw, k1, k2, k3, c, rho);
                  else main_compute<1, 8, 2>(sAw, sBw, k1, k2, k3, c, rho);
                }
                else if (njm == 4) main_compute<4>(sAw, sBw, k1, k2, k3, c, rho);
                else if (njm == 3) main_compute<3>(sAw, sBw, k1, k2, k3, c, rho);
                else if (njm == 2) main_compute<2>(sAw, sBw, k1, k2, k3, c, rho);
                else main_compute<1>(sAw, sBw, k1, k2, k3, c, rho);
              }
              rm.release();
            }
            // slabU[un & 1] was read by pass A of unit un-2
            if (ch == 0 && un >= 2) gwp::mbar_wait(ufree + (un & 1u), ((un >> 1) - 1u) & 1u);
            // store U^T: element (Q, n=(b,j)) -> U[(Q*nao + j)*nao + b];  Re U = K1 - K2, Im U = K3 - K1 - K2
#pragma unroll
            for (int i = 0; i < MT_W; i++) {
              const int Ql = 8 * (mh * MT_W + i) + rho;            // accumulator row g holds panel row rho(g)
#pragma unroll
              for (int jn = 0; jn < NJ; jn++) {
                if (jn < njm && Ql < tm_rows) {
#pragma unroll
                  for (int e = 0; e < 2; e++) {
                    const int n = n0 + 8 * (noff + nstride * jn) + c + 4 * e;   // accumulator columns 2c, 2c+1 hold columns c, c+4
                    if (n < n2) {
                      const int b = (int)P.fd_nao.div((unsigned)n), j = n - b * nao;
                      U[((size_t)Ql * nao + j) * nao + b] = make_double2(k1[i][jn][e] - k2[i][jn][e], k3[i][jn][e] - k1[i][jn][e] - k2[i][jn][e]);
                    }
                  }
                }
              }
            }
          }
          __threadfence(); __syncwarp();
          if (lane == 0) gwp::mbar_arrive(uready + (un & 1u));
        }
      }
    }
  }
}

struct Plan { int ksp, nqt, nitems, nnt, nchunk, cht, main_units, nstage, astage, main_off, grid; size_t smem, slab_units, work_bytes; bool ok; };

template <int KSP>
static void plan_smem(Plan &pl) {
  using Gm = Geo<KSP>;
  pl.astage = 2;
  // 1 KB of the 227 KB is alignment slack: the main stages (TMA destinations, 128-byte swizzle) start 1024-byte aligned
  const size_t cap = 225 * 1024;
  const size_t fixed = (((size_t)8 * Gm::NDT * Gm::LDP + (size_t)pl.astage * Gm::AUX_UNITS) * sizeof(c128) + 1023) / 1024 * 1024;
  pl.main_off = (int)(fixed / sizeof(c128));
  pl.nstage = (int)((cap - fixed) / ((size_t)pl.main_units * sizeof(c128)));
  if (pl.nstage > 6) pl.nstage = 6;
  pl.smem = fixed + (size_t)pl.nstage * pl.main_units * sizeof(c128) + 1024;
}

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  pl.ksp = (d.nao + 3) / 4;
  if (pl.ksp != 7 && pl.ksp != 13) { pl.ok = false; return pl; }
  pl.nnt = (d.nao * d.nao + 7) / 8;
  pl.nchunk = (pl.nnt + 4 * NJ - 1) / (4 * NJ);
  pl.cht = (pl.nnt + pl.nchunk - 1) / pl.nchunk;
  pl.nqt = (d.naux + TM - 1) / TM;
  { short tmp[128]; pl.nitems = d.ntau * fill_kirr(d, tmp) * d.ns; }
  pl.main_units = TM * KC + 64 * pl.cht;      // A: 32 rows x 128 B; B: one 1 KB box per n-tile of the chunk
  if (pl.ksp == 7) plan_smem<7>(pl); else plan_smem<13>(pl);
  const int nsm = gwp::gw_num_sms();
  pl.grid = pl.nitems < nsm ? pl.nitems : nsm;
  pl.slab_units = (((size_t)TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.work_bytes = 256 + (size_t)nsm * 3 * pl.slab_units * sizeof(c128);
  pl.ok = pl.nstage >= 3;
  return pl;
}

// executed flops: a 3M tile product of the main GEMM is 3 DMMA.8x8x4 (1536 flops), a 4M one (pass A, final) 4 (2048)
static double flops(const gw_problem *p, const Plan &pl) {
  GwDims d = gw_dims(p);
  const int ndt = (pl.ksp + 1) / 2;
  const double nmain = (d.naux + KC - 1) / KC;
  double fl = 0.0;
  for (int qt = 0; qt < pl.nqt; qt++) {
    const int tm_rows = (d.naux - qt * TM) < TM ? (d.naux - qt * TM) : TM;
    const int mtc = (tm_rows + 7) / 8;
    const double mtiles = (mtc <= 2) ? (double)mtc : (double)((mtc + MT_W - 1) / MT_W) * MT_W;
    fl += mtiles * pl.nnt * (KC / 4) * nmain * 1536.0;                          // main (3M)
    fl += (double)((tm_rows * d.nao + 7) / 8) * gwp::pass_mtile_flops(d.nao, ndt, pl.ksp, true);   // pass A
    if (ndt == 4 && gwp::pass_tail_fma(d.nao, ndt))                               // final, edge mode: 3 x 3 DMMA tiles + 56 FMAs per lane and k-step
      fl += (double)tm_rows * pl.ksp * ((ndt - 1) * (ndt - 1) * 2048.0 + 56.0 * 32.0 * 2.0);
    else fl += (double)tm_rows * ndt * ndt * pl.ksp * 2048.0;                    // final
  }
  short tmp[128];
  return fl * (double)d.nq * fill_kirr(d, tmp) * d.ntau * d.ns;
}

template <int KSP>
static int launch_k(const Plan &pl, const Params &P, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(sigma_ws_kernel<KSP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return (int)e;
  // tensor maps: Wt as [ntau*nq*naux rows][naux complex], box 32 rows x 8 complex; V as [nk*nk*naux rows][nao² complex],
  // box 8 rows x 8 complex; 128-byte swizzle, zero fill outside the arrays
  CUtensorMap tmW, tmV;
  int rc = gwp::make_tensor_map(&tmW, P.Wt, (size_t)P.d.ntau * P.d.nq * P.d.naux, P.d.naux, TM);
  if (rc) return rc;
  rc = gwp::make_tensor_map(&tmV, P.V, gw_vblocks(P.d) * P.d.naux, P.d.nao * P.d.nao, KC);
  if (rc) return rc;
  sigma_ws_kernel<KSP><<<pl.grid, NTHR, pl.smem, st>>>(P, tmW, tmV);
  return (int)cudaGetLastError();
}

static int launch(const gw_problem *p, const c128 *G, const c128 *Wt, c128 *Sigma, cudaStream_t st, int acc_mode) {
  Plan pl = make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  Params P;
  P.acc_mode = acc_mode;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.G = G; P.Wt = Wt; P.Sigma = Sigma;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.nqt = pl.nqt; P.nitems = pl.nitems; P.nnt = pl.nnt; P.nchunk = pl.nchunk; P.cht = pl.cht;
  P.main_units = pl.main_units; P.nstage = pl.nstage; P.astage = pl.astage; P.slab_units = pl.slab_units;
  P.fd_nao = FastDiv((unsigned)P.d.nao);
  P.nkeff = fill_kirr(P.d, P.kirr);
  P.main_off = pl.main_off;
  return pl.ksp == 7 ? launch_k<7>(pl, P, st) : launch_k<13>(pl, P, st);
}

}  // namespace s3w

double gw_stage3_flops(const gw_problem *p) {
  s3w::Plan pw = s3w::make_plan(p);
  return pw.ok ? s3w::flops(p, pw) : s3_generic_flops(p);
}

size_t gw_stage3_workspace(const gw_problem *p) {
  s3w::Plan pw = s3w::make_plan(p);
  if (pw.ok) return pw.work_bytes;
  s3::Plan pl = s3::make_plan(p);
  return pl.ok ? pl.work_bytes : 0;
}

int gw_launch_stage3(const gw_problem *p, const c128 *G, const c128 *Wt, c128 *Sigma, cudaStream_t st, int acc_mode) {
  if (s3w::make_plan(p).ok) return s3w::launch(p, G, Wt, Sigma, st, acc_mode);
  return s3::launch(p, G, Wt, Sigma, st, acc_mode);
}
