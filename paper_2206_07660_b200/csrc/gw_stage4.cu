// gw_stage4.cu — stage 4, static exchange, Eq. 22:
//
//   K[k][i][j] = -(1/N_k) Σ_k' Σ_Q Σ_ab V[k][k'][Q][i][a] gamma[k'][a][b] V[k'][k][Q][b][j]
//
// Per (k,k') pair, with V1 = V[k][k'], V2 = V[k'][k] (each V block is read exactly once per call):
//   pass :  X[Q][i][b]  = Σ_a V1[Q][i][a] gamma[k'][a][b]          rows (Q,i) flat, K = nao
//   final:  part[i][j] += Σ_(Q,b) X[Q][i][b] V2[Q][b][j]            K = (Q,b)
// One persistent CTA per (k, q = k-k') item keeps the nao x nao partial in registers over all Q, writes it to the
// workspace, and a second kernel sums the partials over q in a fixed order (deterministic, no atomics).
#include "gw_pipe.cuh"

namespace s4 {

using gwp::NTHR; using gwp::PASS_ROWS;
constexpr int TM = 32;

struct Params {
  GwDims d;
  const c128 *V, *gamma;
  c128 *part, *scratch;
  unsigned *counter;
  int nitems, ldp, ksp, ndt, ldt, stage_units;
  int nstage;             // cp.async ring depth: 3, or 2 when three stages of the widest job do not fit (nao > 52)
  int kh, kspf, ldpf;     // final jobs: K splits per Q, k-steps per split, row stride of the X part
  size_t slab_units;
};

template <int KSP_MAX, int NCT>
__global__ void __launch_bounds__(NTHR, 1) exchange_kernel(const Params P) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *smem = reinterpret_cast<c128 *>(smem_raw);
  const GwDims d = P.d;
  const int NSTAGE = P.nstage;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao, ldp = P.ldp, ndt = P.ndt, naop = 8 * ndt;
  c128 *sGt = smem;                   // [naop][ldp]: sGt[b][a] = gamma[k'][a][b]
  c128 *sStage = sGt + naop * ldp;
  __shared__ int s_item;
  c128 *slab = P.scratch + (size_t)blockIdx.x * P.slab_units;
  const size_t vb = (size_t)naux * n2;
  {
    const int tot = naop * ldp + NSTAGE * P.stage_units;
    for (int i = threadIdx.x; i < tot; i += NTHR) smem[i] = make_double2(0.0, 0.0);
  }
  __syncthreads();
  for (;;) {
    if (threadIdx.x == 0) s_item = (int)atomicAdd(P.counter, 1u);
    __syncthreads();
    const int item = s_item;
    __syncthreads();
    if (item >= P.nitems) break;
    const int ql = item % d.nq, ik = item / d.nq, k = ik % d.nk, sg = ik / d.nk;      // sg: spin channel
    const int kp = gw_ksub(d, k, d.q0 + ql);
    const c128 *V1 = P.V + gw_vbwd(d, ql, kp, k) * vb, *V2 = P.V + gw_vfwd(d, ql, kp, k) * vb;   // V[k][k-q], V[k-q][k]
    const c128 *gm = P.gamma + ((size_t)sg * d.nk + kp) * n2;
    for (int i = threadIdx.x; i < n2; i += NTHR) { const int r = i / nao, cc = i - r * nao; sGt[cc * ldp + r] = gm[i]; }
    double sgr[NCT][2], sgi[NCT][2];
#pragma unroll
    for (int i = 0; i < NCT; i++) { sgr[i][0] = sgr[i][1] = 0.0; sgi[i][0] = sgi[i][1] = 0.0; }
    for (int Q0 = 0; Q0 < naux; Q0 += TM) {
      const int tm_rows = min(TM, naux - Q0), rows = tm_rows * nao, npass = (rows + PASS_ROWS - 1) / PASS_ROWS;
      const c128 *V1t = V1 + (size_t)Q0 * n2, *V2t = V2 + (size_t)Q0 * n2;
      int issued = 0;
      for (; issued < NSTAGE - 1; issued++) {
        if (issued < npass) gwp::issue_pass_job(sStage + (issued % NSTAGE) * P.stage_units, V1t, issued * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
      }
      for (int jb = 0; jb < npass; jb++) {
        if (NSTAGE == 3) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();
        const int nx = jb + NSTAGE - 1;
        if (nx < npass) gwp::issue_pass_job(sStage + (nx % NSTAGE) * P.stage_units, V1t, nx * PASS_ROWS, rows, nao, ldp);
        cp_async_commit();
        gwp::pass_compute<KSP_MAX, false>(sStage + (jb % NSTAGE) * P.stage_units, sGt, slab, jb * PASS_ROWS, rows, nao, ldp, P.ksp, ndt);
      }
      cp_async_wait<0>();
      __syncthreads();
      const int nfin = tm_rows * P.kh;
      auto issue_fin = [&](int j) {
        const int jq = j / P.kh, h = j - jq * P.kh;
        gwp::issue_final_job(sStage + (j % NSTAGE) * P.stage_units, slab + (size_t)jq * n2, V2t + (size_t)jq * n2, nao, P.ldpf, P.ldt, P.kspf, naop, 4 * P.kspf * h);
      };
      for (issued = 0; issued < NSTAGE - 1; issued++) {
        if (issued < nfin) issue_fin(issued);
        cp_async_commit();
      }
      for (int jb = 0; jb < nfin; jb++) {
        if (NSTAGE == 3) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();
        const int nx = jb + NSTAGE - 1;
        if (nx < nfin) issue_fin(nx);
        cp_async_commit();
        gwp::final_compute<NCT>(sStage + (jb % NSTAGE) * P.stage_units, sgr, sgi, P.ldpf, P.ldt, P.kspf, ndt, naop);
      }
      cp_async_wait<0>();
      __syncthreads();
    }
    gwp::final_store<NCT>(P.part + (((size_t)sg * d.nq + ql) * d.nk + k) * n2, sgr, sgi, 1.0, nao, ndt);
  }
}

// K[sg][k] = -(1/N_k) Σ_ql part[sg][ql][k]   (fixed summation order).  acc_mode: GW_ACC_CONTINUE starts from the unscaled sums in K,
// GW_ACC_PARTIAL stores unscaled sums (out-of-core V: the q sum continues across slabs in the resident order).
__global__ void exchange_reduce_kernel(GwDims d, const c128 *__restrict__ part, c128 *__restrict__ K, int acc_mode) {
  const size_t n = (size_t)d.nk * d.nao * d.nao;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * d.ns) return;
  const size_t sg = i / n, e = i - sg * n;
  double re = 0.0, im = 0.0;
  if (acc_mode & GW_ACC_CONTINUE) { re = K[i].x; im = K[i].y; }
  for (int ql = 0; ql < d.nq; ql++) { const c128 v = part[(sg * d.nq + ql) * n + e]; re += v.x; im += v.y; }
  const double pref = (acc_mode & GW_ACC_PARTIAL) ? 1.0 : -1.0 / (double)d.nk;
  K[i] = make_double2(pref * re, pref * im);
}

struct Plan { gwp::PassGeom g; int nitems, stage_units, nstage, grid, kh, kspf, ldpf; size_t smem, slab_units, part_units, work_bytes; bool ok; };

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  pl.g = gwp::pass_geom(d.nao);
  if (!pl.g.ok) { pl.ok = false; return pl; }
  pl.nitems = d.nk * d.nq * d.ns;
  const int s_pass = PASS_ROWS * pl.g.ldp;
  // a final job covers one Q, or 1/kh of its K range if a whole Q does not fit; the ring is 3 deep, or 2 for the widest bases
  pl.ok = false;
  for (pl.nstage = 3; pl.nstage >= 2 && !pl.ok; pl.nstage--) {
    for (pl.kh = 1; pl.kh <= 2; pl.kh++) {
      pl.kspf = (pl.g.ksp + pl.kh - 1) / pl.kh;
      int f4 = pl.kspf * 4; if (f4 % 8 == 0) f4 += 4;
      pl.ldpf = f4;
      const int s_fin = pl.g.naop * pl.ldpf + 4 * pl.kspf * pl.g.ldt + 8;
      pl.stage_units = s_pass > s_fin ? s_pass : s_fin;
      pl.smem = ((size_t)pl.g.naop * pl.g.ldp + (size_t)pl.nstage * pl.stage_units) * sizeof(c128);
      if (pl.smem <= 227 * 1024) { pl.ok = true; break; }
    }
    if (pl.ok) break;
  }
  const int nsm = gwp::gw_num_sms();
  pl.grid = pl.nitems < nsm ? pl.nitems : nsm;
  pl.slab_units = (((size_t)TM * d.nao * d.nao) + 15) / 16 * 16;
  pl.part_units = (size_t)d.ns * d.nq * d.nk * d.nao * d.nao;
  pl.work_bytes = 256 + ((size_t)nsm * pl.slab_units + pl.part_units) * sizeof(c128);
  return pl;
}

}  // namespace s4

size_t gw_stage4_workspace(const gw_problem *p) {
  s4::Plan pl = s4::make_plan(p);
  return pl.ok ? pl.work_bytes : 0;
}

double gw_stage4_flops(const gw_problem *p) {
  s4::Plan pl = s4::make_plan(p);
  if (!pl.ok) return 0.0;
  GwDims d = gw_dims(p);
  double tiles = 0.0;
  for (int Q0 = 0; Q0 < d.naux; Q0 += s4::TM) {
    const int tm_rows = (d.naux - Q0) < s4::TM ? (d.naux - Q0) : s4::TM;
    tiles += (double)((tm_rows * d.nao + 7) / 8) * pl.g.ndt * pl.g.ksp + (double)tm_rows * pl.g.ndt * pl.g.ndt * pl.kspf * pl.kh;
  }
  return tiles * (double)d.nk * d.nq * d.ns * 2048.0;
}

template <int KSP_MAX, int NCT>
static int launch_exchange(const s4::Plan &pl, const s4::Params &P, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(s4::exchange_kernel<KSP_MAX, NCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return (int)e;
  s4::exchange_kernel<KSP_MAX, NCT><<<pl.grid, s4::NTHR, pl.smem, st>>>(P);
  return (int)cudaGetLastError();
}

int gw_launch_stage4(const gw_problem *p, const c128 *gamma, c128 *K, cudaStream_t st, int acc_mode) {
  s4::Plan pl = s4::make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  s4::Params P;
  P.d = gw_dims(p); P.V = (const c128 *)p->V; P.gamma = gamma;
  P.counter = (unsigned *)p->work;
  P.scratch = (c128 *)((char *)p->work + 256);
  P.part = P.scratch + (size_t)gwp::gw_num_sms() * pl.slab_units;
  P.nitems = pl.nitems; P.ldp = pl.g.ldp; P.ksp = pl.g.ksp; P.ndt = pl.g.ndt; P.ldt = pl.g.ldt; P.kh = pl.kh; P.kspf = pl.kspf; P.ldpf = pl.ldpf;
  P.stage_units = pl.stage_units; P.nstage = pl.nstage; P.slab_units = pl.slab_units;
  cudaError_t e = cudaMemsetAsync(p->work, 0, 256, st);
  if (e != cudaSuccess) return (int)e;
  int rc;
  if (pl.g.nct == 2) {
    if (pl.g.ksp_max == 7) rc = launch_exchange<7, 2>(pl, P, st);
    else if (pl.g.ksp_max == 13) rc = launch_exchange<13, 2>(pl, P, st);
    else rc = launch_exchange<16, 2>(pl, P, st);
  } else {
    if (pl.g.ksp_max == 7) rc = launch_exchange<7, 8>(pl, P, st);
    else if (pl.g.ksp_max == 13) rc = launch_exchange<13, 8>(pl, P, st);
    else rc = launch_exchange<16, 8>(pl, P, st);
  }
  if (rc) return rc;
  const size_t n = (size_t)P.d.ns * P.d.nk * P.d.nao * P.d.nao;
  s4::exchange_reduce_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(P.d, P.part, K, acc_mode);
  return (int)cudaGetLastError();
}
