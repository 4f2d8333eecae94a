// gw_api.cu — the C ABI of include/gw.h: argument validation, dispatch, the host-buffer iteration and the
// FP64 peak probe.  No torch types, no exceptions across the boundary.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "gw_common.cuh"

// the current device must be sm_100; queried on every call (microseconds against kernels that run for seconds), so the
// verdict follows cudaSetDevice
static int check_arch() {
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return GW_EARCH; }
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return GW_EARCH; }
  return major == 10 ? GW_OK : GW_EARCH;
}

static int gw_sm_count() {
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) { cudaGetLastError(); nsm = 148; }
  return nsm;
}

static bool aligned16(const void *p) { return p && (((uintptr_t)p) & 15) == 0; }

static int check_problem(const gw_problem *p, bool need_T) {
  if (!p) return GW_EINVAL;
  if (p->nk1 <= 0 || p->nk2 <= 0 || p->nk3 <= 0 || p->nao <= 0 || p->naux <= 0 || p->ntau <= 0 || p->nw <= 0) return GW_EINVAL;
  if (p->spin_deg != 1 && p->spin_deg != 2) return GW_EINVAL;
  if ((p->symmetry & ~GW_SYM_TR) || p->reserved || (p->ns != 0 && p->ns != 1 && p->ns != 2 && p->ns != 4) || (p->v_layout != GW_V_FULL && p->v_layout != GW_V_QSLAB)) return GW_EINVAL;
  if (p->ns == 4 && (p->symmetry & GW_SYM_TR)) return GW_EINVAL;     // the time-reversal relations of GW_SYM_TR are those of spin-diagonal G
  const int64_t nk = (int64_t)p->nk1 * p->nk2 * p->nk3;
  if (nk > (1 << 20)) return GW_EINVAL;
  if (p->q_begin < 0 || p->q_end > nk || p->q_begin >= p->q_end) return GW_EINVAL;
  if (!aligned16(p->V)) return GW_EINVAL;
  if (need_T && (!aligned16(p->T_wt) || !aligned16(p->T_tw))) return GW_EINVAL;
  if (p->nao > GW_MAX_NAO || p->ntau > GW_MAX_NTAU || p->nw > GW_MAX_NTAU || p->nw > p->ntau || p->naux > GW_MAX_NAUX) return GW_ESHAPE;
  return GW_OK;
}

extern "C" int gw_polarization(const gw_problem *p, const gw_c128 *G, gw_c128 *P0t, void *stream) {
  int rc = check_problem(p, false); if (rc) return rc;
  if (!aligned16(G) || !aligned16(P0t)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  return gw_launch_stage1(p, (const c128 *)G, (c128 *)P0t, st);
}

extern "C" size_t gw_workspace_bytes(const gw_problem *p) {
  if (check_problem(p, false) != GW_OK) return 0;
  // a stage whose planner cannot place the problem answers 0: then the whole problem is refused (never a partial yes)
  const size_t s[4] = {gw_stage1_workspace(p), gw_stage2_workspace(p), gw_stage3_workspace(p), gw_stage4_workspace(p)};
  size_t m = 0;
  for (int i = 0; i < 4; i++) { if (s[i] == 0) return 0; if (s[i] > m) m = s[i]; }
  return (m + 255) / 256 * 256;
}

extern "C" int gw_screened_interaction(const gw_problem *p, const gw_c128 *P0t, gw_c128 *Wt, int32_t *info, void *stream) {
  int rc = check_problem(p, true); if (rc) return rc;
  if (!aligned16(P0t) || !aligned16(Wt) || (((uintptr_t)info) & 7)) return GW_EINVAL;
  if (!p->work || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  return gw_launch_stage2(p, (const c128 *)P0t, (c128 *)Wt, info, NULL, st);
}

extern "C" int gw_screened_interaction_phi(const gw_problem *p, const gw_c128 *P0t, gw_c128 *Wt, int32_t *info, double *phi, void *stream) {
  int rc = check_problem(p, true); if (rc) return rc;
  if (!aligned16(P0t) || !aligned16(Wt) || !phi || (((uintptr_t)phi) & 7) || (((uintptr_t)info) & 7)) return GW_EINVAL;
  if (!p->work || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  if ((rc = check_arch())) return rc;
  return gw_launch_stage2(p, (const c128 *)P0t, (c128 *)Wt, info, phi, (cudaStream_t)stream);
}

extern "C" int gw_transform(int32_t n_out, int32_t n_in, const gw_c128 *T, const gw_c128 *X, gw_c128 *Y, size_t len, void *stream) {
  if (!aligned16(T) || !aligned16(X) || !aligned16(Y) || n_out <= 0 || n_in <= 0) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  return gw_launch_transform(n_out, n_in, (const c128 *)T, (const c128 *)X, (c128 *)Y, len, (cudaStream_t)stream);
}

extern "C" int gw_selfenergy(const gw_problem *p, const gw_c128 *G, const gw_c128 *Wt, gw_c128 *Sigma, void *stream) {
  int rc = check_problem(p, false); if (rc) return rc;
  if (!aligned16(G) || !aligned16(Wt) || !aligned16(Sigma)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  return gw_launch_stage3(p, (const c128 *)G, (const c128 *)Wt, (c128 *)Sigma, st);
}

extern "C" int gw_exchange(const gw_problem *p, const gw_c128 *gamma, gw_c128 *K, void *stream) {
  int rc = check_problem(p, false); if (rc) return rc;
  if (!aligned16(gamma) || !aligned16(K)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  return gw_launch_stage4(p, (const c128 *)gamma, (c128 *)K, st);
}

extern "C" int gw_executed_flops(const gw_problem *p, double *out) {
  int rc = check_problem(p, false); if (rc) return rc;
  if (!out) return GW_EINVAL;
  gw_stage_flops(p, out);
  return GW_OK;
}

extern "C" int gw_launch_count(const gw_problem *p) {
  if (check_problem(p, false) != GW_OK) return 0;
  return gw_stage_launches(p);
}

#define CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { rc = (int)e_; goto done; } } while (0)

extern "C" int gw_sigma_iteration_host(const gw_problem *p, const gw_c128 *G, const gw_c128 *gamma, gw_c128 *Sigma, gw_c128 *K,
                                       gw_c128 *P0t_out, gw_c128 *Wt_out, float *stage_ms, void *stream) {
  int rc = check_problem(p, true); if (rc) return rc;
  if (!G || !gamma || !Sigma || !K) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  GwDims d = gw_dims(p);
  const size_t n2 = (size_t)d.nao * d.nao, a2 = (size_t)d.naux * d.naux;
  const size_t bV = gw_vblocks(d) * d.naux * n2 * 16, bG = (size_t)d.ns * d.ntau * d.nk * n2 * 16, bg = (size_t)d.ns * d.nk * n2 * 16;
  const size_t bP = (size_t)d.ntau * d.nq * a2 * 16, bT = (size_t)d.nw * d.ntau * 16;
  c128 *dV = 0, *dG = 0, *dg = 0, *dP = 0, *dS = 0, *dK = 0, *dTwt = 0, *dTtw = 0; void *dW = 0; int32_t *dinfo = 0;
  cudaEvent_t ev[7]; for (int i = 0; i < 7; i++) ev[i] = 0;
  int32_t hinfo[2] = {-1, -1};
  gw_problem dp = *p;
  size_t wb = 0;
  for (int i = 0; i < 7; i++) CU(cudaEventCreate(&ev[i]));
  CU(cudaMalloc(&dV, bV)); CU(cudaMalloc(&dG, bG)); CU(cudaMalloc(&dg, bg)); CU(cudaMalloc(&dP, bP));
  CU(cudaMalloc(&dS, bG)); CU(cudaMalloc(&dK, bg)); CU(cudaMalloc(&dTwt, bT)); CU(cudaMalloc(&dTtw, bT));
  CU(cudaMalloc(&dinfo, 8));
  dp.V = (const gw_c128 *)dV; dp.T_wt = (const gw_c128 *)dTwt; dp.T_tw = (const gw_c128 *)dTtw;
  wb = gw_workspace_bytes(&dp);
  CU(cudaMalloc(&dW, wb));
  dp.work = dW; dp.work_bytes = wb;
  CU(cudaEventRecord(ev[0], st));
  CU(cudaMemcpyAsync(dV, p->V, bV, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dG, G, bG, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dg, gamma, bg, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dTwt, p->T_wt, bT, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dTtw, p->T_tw, bT, cudaMemcpyHostToDevice, st));
  CU(cudaEventRecord(ev[1], st));
  if ((rc = gw_polarization(&dp, (gw_c128 *)dG, (gw_c128 *)dP, st))) goto done;
  if (P0t_out) CU(cudaMemcpyAsync(P0t_out, dP, bP, cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(ev[2], st));
  if ((rc = gw_screened_interaction(&dp, (gw_c128 *)dP, (gw_c128 *)dP, dinfo, st))) goto done;
  CU(cudaEventRecord(ev[3], st));
  if ((rc = gw_selfenergy(&dp, (gw_c128 *)dG, (gw_c128 *)dP, (gw_c128 *)dS, st))) goto done;
  CU(cudaEventRecord(ev[4], st));
  if ((rc = gw_exchange(&dp, (gw_c128 *)dg, (gw_c128 *)dK, st))) goto done;
  CU(cudaEventRecord(ev[5], st));
  if (Wt_out) CU(cudaMemcpyAsync(Wt_out, dP, bP, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(Sigma, dS, bG, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(K, dK, bg, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(hinfo, dinfo, 8, cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(ev[6], st));
  CU(cudaStreamSynchronize(st));
  if (stage_ms) for (int i = 0; i < 6; i++) CU(cudaEventElapsedTime(&stage_ms[i], ev[i], ev[i + 1]));
  if (hinfo[0] != -1 || hinfo[1] != -1) rc = GW_ENOTPD;
done:
  cudaFree(dV); cudaFree(dG); cudaFree(dg); cudaFree(dP); cudaFree(dS); cudaFree(dK); cudaFree(dTwt); cudaFree(dTtw); cudaFree(dW); cudaFree(dinfo);
  for (int i = 0; i < 7; i++) if (ev[i]) cudaEventDestroy(ev[i]);
  return rc;
}


// Out-of-core V: q-slabs of V are gathered from host memory into two device buffers on a copy stream while the previous slab
// computes; Sigma and K continue their q sums across slabs (GW_ACC_CONTINUE / GW_ACC_PARTIAL), so the result is the resident one.
extern "C" int gw_sigma_iteration_stream(const gw_problem *p, const gw_c128 *G, const gw_c128 *gamma, gw_c128 *Sigma, gw_c128 *K,
                                         size_t v_budget_bytes, float *stats, void *stream) {
  int rc = check_problem(p, true); if (rc) return rc;
  if (!G || !gamma || !Sigma || !K || p->v_layout != GW_V_FULL) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream, cs = 0;
  const GwDims d = gw_dims(p);
  const size_t n2 = (size_t)d.nao * d.nao, a2 = (size_t)d.naux * d.naux;
  const size_t blk = (size_t)d.naux * n2 * 16, perq = 2 * (size_t)d.nk * blk;          // one V block; the 2 nk blocks of one q
  int nqs = (int)((v_budget_bytes / 2) / perq);
  if (nqs < 1) return GW_ENOMEM;
  if (nqs > d.nq) nqs = d.nq;
  const int nslab = (d.nq + nqs - 1) / nqs;
  const size_t bG = (size_t)d.ns * d.ntau * d.nk * n2 * 16, bg = (size_t)d.ns * d.nk * n2 * 16;
  const size_t bP = (size_t)d.ntau * nqs * a2 * 16, bT = (size_t)d.nw * d.ntau * 16;
  c128 *dV[2] = {0, 0}, *dG = 0, *dg = 0, *dP = 0, *dS = 0, *dK = 0, *dTwt = 0, *dTtw = 0; void *dW = 0; int32_t *dinfo = 0, *hinfo = 0;
  cudaEvent_t ready[2] = {0, 0}, freed[2] = {0, 0}, e0 = 0, e1 = 0;
  gw_problem sp = *p;
  size_t wb = 0; double copied = 0.0; float ms = 0.f;
  const char *hV = (const char *)p->V;
  hinfo = (int32_t *)malloc(sizeof(int32_t) * 2 * nslab);
  if (!hinfo) return GW_ENOMEM;
  CU(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
  for (int i = 0; i < 2; i++) { CU(cudaEventCreateWithFlags(&ready[i], cudaEventDisableTiming)); CU(cudaEventCreateWithFlags(&freed[i], cudaEventDisableTiming)); }
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  for (int i = 0; i < 2; i++) CU(cudaMalloc(&dV[i], (size_t)nqs * perq));
  CU(cudaMalloc(&dG, bG)); CU(cudaMalloc(&dg, bg)); CU(cudaMalloc(&dP, bP)); CU(cudaMalloc(&dS, bG)); CU(cudaMalloc(&dK, bg));
  CU(cudaMalloc(&dTwt, bT)); CU(cudaMalloc(&dTtw, bT)); CU(cudaMalloc(&dinfo, 8 * (size_t)nslab));
  sp.T_wt = (const gw_c128 *)dTwt; sp.T_tw = (const gw_c128 *)dTtw; sp.v_layout = GW_V_QSLAB; sp.V = (const gw_c128 *)dV[0];
  sp.q_begin = p->q_begin; sp.q_end = p->q_begin + nqs;
  wb = gw_workspace_bytes(&sp);
  if (!wb) { rc = GW_ESHAPE; goto done; }
  CU(cudaMalloc(&dW, wb));
  sp.work = dW; sp.work_bytes = wb;
  CU(cudaEventRecord(e0, st));
  CU(cudaMemcpyAsync(dG, G, bG, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dg, gamma, bg, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dTwt, p->T_wt, bT, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(dTtw, p->T_tw, bT, cudaMemcpyHostToDevice, st));
  for (int s = 0; s < nslab; s++) {
    const int b = s & 1, q0 = p->q_begin + s * nqs, q1 = (q0 + nqs < p->q_end) ? q0 + nqs : p->q_end;
    // gather the slab: slot (ql, k, 0) = V[k][k+q], slot (ql, k, 1) = V[k+q][k]; the buffer was last read by slab s-2
    if (s >= 2) CU(cudaStreamWaitEvent(cs, freed[b], 0));
    for (int q = q0; q < q1; q++)
      for (int k = 0; k < d.nk; k++) {
        const int kq = gw_kadd(d, k, q);
        char *dst = (char *)dV[b] + (((size_t)(q - q0) * d.nk + k) * 2) * blk;
        CU(cudaMemcpyAsync(dst, hV + ((size_t)k * d.nk + kq) * blk, blk, cudaMemcpyHostToDevice, cs));
        CU(cudaMemcpyAsync(dst + blk, hV + ((size_t)kq * d.nk + k) * blk, blk, cudaMemcpyHostToDevice, cs));
        copied += 2.0 * (double)blk;
      }
    CU(cudaEventRecord(ready[b], cs));
    CU(cudaStreamWaitEvent(st, ready[b], 0));
    sp.V = (const gw_c128 *)dV[b]; sp.q_begin = q0; sp.q_end = q1;
    const int acc = (s > 0 ? GW_ACC_CONTINUE : 0) | (s < nslab - 1 ? GW_ACC_PARTIAL : 0);
    if ((rc = gw_polarization(&sp, (gw_c128 *)dG, (gw_c128 *)dP, st))) goto done;
    if ((rc = gw_screened_interaction(&sp, (gw_c128 *)dP, (gw_c128 *)dP, dinfo + 2 * s, st))) goto done;
    if ((rc = gw_launch_stage3(&sp, dG, dP, dS, st, acc))) goto done;
    if ((rc = gw_launch_stage4(&sp, dg, dK, st, acc))) goto done;
    CU(cudaEventRecord(freed[b], st));
  }
  CU(cudaMemcpyAsync(Sigma, dS, bG, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(K, dK, bg, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(hinfo, dinfo, 8 * (size_t)nslab, cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(e1, st));
  CU(cudaStreamSynchronize(st));
  CU(cudaEventElapsedTime(&ms, e0, e1));
  for (int s = 0; s < 2 * nslab; s++) if (hinfo[s] != -1) rc = GW_ENOTPD;
  if (stats) { stats[0] = ms; stats[1] = (float)(copied * 1e-9); stats[2] = (float)nslab; stats[3] = (float)nqs; }
done:
  if (cs) { cudaStreamSynchronize(cs); cudaStreamDestroy(cs); }
  cudaFree(dV[0]); cudaFree(dV[1]); cudaFree(dG); cudaFree(dg); cudaFree(dP); cudaFree(dS); cudaFree(dK); cudaFree(dTwt); cudaFree(dTtw); cudaFree(dW); cudaFree(dinfo);
  for (int i = 0; i < 2; i++) { if (ready[i]) cudaEventDestroy(ready[i]); if (freed[i]) cudaEventDestroy(freed[i]); }
  if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1);
  free(hinfo);
  return rc;
}

// ---- loop closure (gw_loop.cu) ----
extern "C" int gw_hartree(const gw_problem *p, const gw_c128 *gamma, gw_c128 *J, void *stream) {
  int rc = check_problem(p, false); if (rc) return rc;
  if (!aligned16(gamma) || !aligned16(J)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  return gw_launch_hartree(p, (const c128 *)gamma, (c128 *)J, (cudaStream_t)stream);
}

static int check_loop_args(int nk, int nao, int nwf, const void *omega, const void *S, const void *F, const void *G_w) {
  if (nk <= 0 || nao <= 0 || nwf <= 0 || nk > (1 << 20) || nwf > (1 << 20)) return GW_EINVAL;
  if (!omega || (((uintptr_t)omega) & 7) || !aligned16(S) || !aligned16(F) || !aligned16(G_w)) return GW_EINVAL;
  if (nao > GW_MAX_NAO) return GW_ESHAPE;
  return GW_OK;
}

extern "C" int gw_dyson_update(int32_t nk, int32_t nao, int32_t nwf, const double *omega, double mu, const gw_c128 *S, const gw_c128 *F,
                               const gw_c128 *Sigma_w, gw_c128 *G_w, int32_t *info, void *stream) {
  int rc = check_loop_args(nk, nao, nwf, omega, S, F, G_w); if (rc) return rc;
  if ((Sigma_w && !aligned16(Sigma_w)) || (((uintptr_t)info) & 7)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  return gw_launch_dyson_update(nk, nao, nwf, omega, mu, (const c128 *)S, (const c128 *)F, (const c128 *)Sigma_w, (c128 *)G_w, info, (cudaStream_t)stream);
}

extern "C" int gw_electron_count(int32_t nk, int32_t nao, int32_t nwf, int32_t spin_deg, const gw_c128 *t_beta, const gw_c128 *S,
                                 const gw_c128 *G_w, gw_c128 *partial, double *ne, void *stream) {
  if (nk <= 0 || nao <= 0 || nwf <= 0 || (spin_deg != 1 && spin_deg != 2)) return GW_EINVAL;
  if (!aligned16(t_beta) || !aligned16(S) || !aligned16(G_w) || !aligned16(partial) || !ne || (((uintptr_t)ne) & 7)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  return gw_launch_electron_count(nk, nao, nwf, spin_deg, (const c128 *)t_beta, (const c128 *)S, (const c128 *)G_w, (c128 *)partial, ne, (cudaStream_t)stream);
}

extern "C" int gw_find_mu(int32_t nk, int32_t nao, int32_t nwf, int32_t spin_deg, const double *omega, const gw_c128 *t_beta, const gw_c128 *S,
                          const gw_c128 *F, const gw_c128 *Sigma_w, double n_target, double mu_lo, double mu_hi, double mu_tol, gw_c128 *G_w,
                          gw_c128 *partial, double *ne_dev, double *mu_out, double *ne_out, int32_t *n_eval, void *stream) {
  int rc = check_loop_args(nk, nao, nwf, omega, S, F, G_w); if (rc) return rc;
  if ((spin_deg != 1 && spin_deg != 2) || !aligned16(t_beta) || !aligned16(partial) || !ne_dev || (((uintptr_t)ne_dev) & 7) || !mu_out || !ne_out) return GW_EINVAL;
  if ((Sigma_w && !aligned16(Sigma_w)) || !(mu_hi > mu_lo) || !(mu_tol > 0)) return GW_EINVAL;
  if ((rc = check_arch())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t *dinfo = 0; int32_t hinfo[2] = {-1, -1};
  int evals = 0; bool singular = false;
  CU(cudaMalloc(&dinfo, 8));
  {
    // N_e(mu): Eq. 16 for all (n, k), then Eq. 15; the value is read back (8 bytes) with the factorisation status
    auto NE = [&](double mu, double *val) -> int {
      int r = gw_launch_dyson_update(nk, nao, nwf, omega, mu, (const c128 *)S, (const c128 *)F, (const c128 *)Sigma_w, (c128 *)G_w, dinfo, st);
      if (r) return r;
      r = gw_launch_electron_count(nk, nao, nwf, spin_deg, (const c128 *)t_beta, (const c128 *)S, (const c128 *)G_w, (c128 *)partial, ne_dev, st);
      if (r) return r;
      cudaError_t e = cudaMemcpyAsync(val, ne_dev, 8, cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaMemcpyAsync(hinfo, dinfo, 8, cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      if (e != cudaSuccess) return (int)e;
      if (hinfo[0] != -1 || hinfo[1] != -1) singular = true;
      evals++;
      return 0;
    };
    double lo = mu_lo, hi = mu_hi, nlo = 0, nhi = 0, nmid = 0;
    if ((rc = NE(lo, &nlo)) || (rc = NE(hi, &nhi))) goto done;
    int it = 0;
    while ((nlo > n_target || nhi < n_target) && it < 60) {
      const double w = hi - lo;
      if (nlo > n_target) { lo -= w; if ((rc = NE(lo, &nlo))) goto done; }
      else { hi += w; if ((rc = NE(hi, &nhi))) goto done; }
      it++;
    }
    if (nlo > n_target || nhi < n_target) { rc = GW_ENOBRACKET; goto done; }
    for (it = 0; it < 200 && hi - lo > mu_tol; it++) {
      const double mid = 0.5 * (lo + hi);
      if ((rc = NE(mid, &nmid))) goto done;
      if (nmid < n_target) lo = mid; else hi = mid;
    }
    *mu_out = 0.5 * (lo + hi);
    if ((rc = NE(*mu_out, ne_out))) goto done;
    if (singular) rc = GW_ENOTPD;
  }
done:
  if (n_eval) *n_eval = evals;
  cudaFree(dinfo);
  return rc;
}

extern "C" int gw_phi_gw(int32_t nk, int32_t nq, int32_t nw, double beta, const double *w, const double *phi, double *out, void *stream) {
  if (nk <= 0 || nq <= 0 || nw <= 0 || !(beta > 0) || !w || !phi || !out || (((uintptr_t)w | (uintptr_t)phi | (uintptr_t)out) & 7)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  return gw_launch_phi_gw(nk, nq, nw, beta, w, phi, out, (cudaStream_t)stream);
}

extern "C" int gw_axpby(size_t n, double a_re, double a_im, const gw_c128 *X, double b_re, double b_im, gw_c128 *Y, void *stream) {
  if (!aligned16(X) || !aligned16(Y)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  return gw_launch_axpby(n, make_double2(a_re, a_im), (const c128 *)X, make_double2(b_re, b_im), (c128 *)Y, (cudaStream_t)stream);
}

// ---- FP64 peak probe: register-resident DMMA.8x8x4 loop, 8 independent accumulators per warp ----
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *out, int iters) {
  double acc[8][2];
#pragma unroll
  for (int i = 0; i < 8; i++) { acc[i][0] = threadIdx.x * 1e-3 + i; acc[i][1] = i; }
  double a = 1e-3 + threadIdx.x * 1e-9, b = 1e-3;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++) dmma884(acc[i][0], acc[i][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += acc[i][0] + acc[i][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int gw_fp64_peak(double ms, double *tflops, void *stream) {
  if (!tflops || !(ms > 0)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int nsm = gw_sm_count();
  double *out = 0; cudaEvent_t e0 = 0, e1 = 0; float t = 0;
  const int iters = 20000, grid = nsm * 2;
  const double fl = 2.0 * 256 * 8 * (double)iters * 8 * grid;   // per launch
  int reps = 1;
  CU(cudaMalloc(&out, sizeof(double) * grid * 256));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  fp64_peak_kernel<<<grid, 256, 0, st>>>(out, iters);            // warm-up, ~2.6 ms
  reps = (int)(ms / 2.6) + 1;
  CU(cudaEventRecord(e0, st));
  for (int r = 0; r < reps; r++) fp64_peak_kernel<<<grid, 256, 0, st>>>(out, iters);
  CU(cudaEventRecord(e1, st));
  CU(cudaEventSynchronize(e1));
  CU(cudaEventElapsedTime(&t, e0, e1));
  *tflops = fl * reps / (t * 1e-3) * 1e-12;
done:
  cudaFree(out); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1);
  return rc;
}

// ---- which warps share an FP64 pipe: the DMMA loop on the warps of warp_mask only (one 16-warp CTA per SM) ----
__global__ void __launch_bounds__(512, 1) fp64_subcore_kernel(unsigned mask, int iters, double *out) {
  const int w = threadIdx.x >> 5;
  if (!((mask >> w) & 1u)) return;
  double acc[12][2];
#pragma unroll
  for (int i = 0; i < 12; i++) { acc[i][0] = threadIdx.x * 1e-3 + i; acc[i][1] = i; }
  const double a = 1e-3 + threadIdx.x * 1e-9, b = 1e-3;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 12; i++) dmma884(acc[i][0], acc[i][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 12; i++) s += acc[i][0] + acc[i][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int gw_fp64_subcore_probe(uint32_t warp_mask, double *tflops, void *stream) {
  if (!tflops || !warp_mask || (warp_mask >> 16)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int nsm = gw_sm_count();
  double *out = 0; cudaEvent_t e0 = 0, e1 = 0; float t = 0;
  const int iters = 50000;
  int nw = 0;
  for (int i = 0; i < 16; i++) nw += (warp_mask >> i) & 1u;
  const double fl = 512.0 * 12 * (double)iters * nw * nsm;       // 512 flops per DMMA.8x8x4
  CU(cudaMalloc(&out, sizeof(double) * nsm * 512));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  fp64_subcore_kernel<<<nsm, 512, 0, st>>>(warp_mask, 1000, out);   // warm-up
  CU(cudaEventRecord(e0, st));
  fp64_subcore_kernel<<<nsm, 512, 0, st>>>(warp_mask, iters, out);
  CU(cudaEventRecord(e1, st));
  CU(cudaEventSynchronize(e1));
  CU(cudaEventElapsedTime(&t, e0, e1));
  *tflops = fl / (t * 1e-3) * 1e-12;
done:
  cudaFree(out); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1);
  return rc;
}

// ---- the same probe with plain DFMA (no tensor-core instruction): 16 independent chains per thread ----
__global__ void __launch_bounds__(256) fp64_dfma_kernel(double *out, int iters) {
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = threadIdx.x * 1e-3 + i;
  const double a = 1.0 - 1e-9 * threadIdx.x, b = 1e-6;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int gw_fp64_peak_dfma(double ms, double *tflops, void *stream) {
  if (!tflops || !(ms > 0)) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int nsm = gw_sm_count();
  double *out = 0; cudaEvent_t e0 = 0, e1 = 0; float t = 0;
  const int iters = 20000, grid = nsm * 4;
  const double fl = 2.0 * 256 * 16 * (double)iters * grid;      // per launch
  int reps = 1;
  CU(cudaMalloc(&out, sizeof(double) * grid * 256));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  fp64_dfma_kernel<<<grid, 256, 0, st>>>(out, iters);            // warm-up, ~2.6 ms
  reps = (int)(ms / 2.6) + 1;
  CU(cudaEventRecord(e0, st));
  for (int r = 0; r < reps; r++) fp64_dfma_kernel<<<grid, 256, 0, st>>>(out, iters);
  CU(cudaEventRecord(e1, st));
  CU(cudaEventSynchronize(e1));
  CU(cudaEventElapsedTime(&t, e0, e1));
  *tflops = fl * reps / (t * 1e-3) * 1e-12;
done:
  cudaFree(out); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1);
  return rc;
}


// ---- complex tile-product probe: the inner loop of the main GEMMs alone (operands resident in shared memory, 8 warps per CTA, one CTA
//      per SM), for the three ways of forming a complex 8x8x4 product on DMMA (profiles/r02_3m_vs_4m.md):
//        mode 0: 4M (four real DMMAs, warp tile 2 x 7);  mode 1: 3M Karatsuba, operand sums by DADD in registers (warp tile 2 x 4);
//        mode 2: 3M with the B sums pre-formed as a third plane in shared memory
template <int MODE, int MT, int NJ>
__global__ void __launch_bounds__(256, 1) cmma_probe_kernel(double *out, int iters) {
  constexpr int KC = 8, TM = 32, NCG = 8 / (TM / (8 * MT)), NCOLS = 8 * NCG * NJ, NACC = MODE == 0 ? 2 : 3;
  extern __shared__ __align__(128) unsigned char raw[];
  c128 *sA = reinterpret_cast<c128 *>(raw), *sB = sA + TM * KC;
  double *sB3 = reinterpret_cast<double *>(sB + NCOLS * KC);
  for (int i = threadIdx.x; i < TM * KC; i += blockDim.x) sA[i] = make_double2(1e-3 * (i % 7), -1e-3 * (i % 5));
  for (int i = threadIdx.x; i < NCOLS * KC; i += blockDim.x) { sB[i] = make_double2(1e-3 * (i % 3), 1e-3 * (i % 11)); sB3[i] = 1e-3; }
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3, rho = (g >> 1) + 4 * (g & 1);
  double acc[MT][NJ][NACC][2];
#pragma unroll
  for (int i = 0; i < MT; i++)
#pragma unroll
    for (int j = 0; j < NJ; j++)
#pragma unroll
      for (int x = 0; x < NACC; x++) acc[i][j][x][0] = acc[i][j][x][1] = 0.0;
  constexpr int MG = TM / (8 * MT);
  const c128 *sAw = sA + (8 * (w % MG) * MT + rho) * KC, *sBw = sB + (8 * (w / MG) + rho) * KC;
  const double *sB3w = sB3 + (8 * (w / MG) + rho) * KC;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int ks = 0; ks < KC / 4; ks++) {
      const int u = (4 * ks + c) ^ rho;
      c128 a[MT], b[NJ];
      double b3[NJ];
#pragma unroll
      for (int i = 0; i < MT; i++) a[i] = sAw[i * 8 * KC + u];
#pragma unroll
      for (int j = 0; j < NJ; j++) { b[j] = sBw[j * NCG * 8 * KC + u]; if (MODE == 2) b3[j] = sB3w[j * NCG * 8 * KC + u]; }
      if (MODE == 0) {
#pragma unroll
        for (int j = 0; j < NJ; j++)
#pragma unroll
          for (int i = 0; i < MT; i++) cmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
      } else {
        double as[MT];
#pragma unroll
        for (int i = 0; i < MT; i++) as[i] = a[i].x + a[i].y;
#pragma unroll
        for (int j = 0; j < NJ; j++) {
          const double bs = MODE == 1 ? b[j].x + b[j].y : b3[j];
#pragma unroll
          for (int i = 0; i < MT; i++) {
            dmma884(acc[i][j][0][0], acc[i][j][0][1], a[i].x, b[j].x);
            dmma884(acc[i][j][1][0], acc[i][j][1][1], a[i].y, b[j].y);
            dmma884(acc[i][j][2][0], acc[i][j][2][1], as[i], bs);
          }
        }
      }
    }
    __syncwarp();
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < MT; i++)
#pragma unroll
    for (int j = 0; j < NJ; j++)
#pragma unroll
      for (int x = 0; x < NACC; x++) s += acc[i][j][x][0] + acc[i][j][x][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int MODE, int MT, int NJ>
static int run_cmma_probe(double ms, double *tflops, cudaStream_t st) {
  constexpr int NCOLS = 8 * (8 / (32 / (8 * MT))) * NJ;
  const size_t smem = (size_t)(32 * 8 + NCOLS * 8) * 16 + (size_t)NCOLS * 8 * 8;
  int rc = 0;
  const int nsm = gw_sm_count(), iters = 4000;
  double *out = 0; cudaEvent_t e0 = 0, e1 = 0; float t = 0; int reps = 1;
  CU(cudaFuncSetAttribute(cmma_probe_kernel<MODE, MT, NJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  CU(cudaMalloc(&out, sizeof(double) * nsm * 256));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  cmma_probe_kernel<MODE, MT, NJ><<<nsm, 256, smem, st>>>(out, iters);
  CU(cudaEventRecord(e0, st));
  cmma_probe_kernel<MODE, MT, NJ><<<nsm, 256, smem, st>>>(out, iters);
  CU(cudaEventRecord(e1, st));
  CU(cudaEventSynchronize(e1));
  CU(cudaEventElapsedTime(&t, e0, e1));
  reps = (int)(ms / (t > 0.01f ? t : 0.01f)) + 1;
  CU(cudaEventRecord(e0, st));
  for (int r = 0; r < reps; r++) cmma_probe_kernel<MODE, MT, NJ><<<nsm, 256, smem, st>>>(out, iters);
  CU(cudaEventRecord(e1, st));
  CU(cudaEventSynchronize(e1));
  CU(cudaEventElapsedTime(&t, e0, e1));
  *tflops = 8.0 * 32.0 * NCOLS * 8.0 * iters * nsm * reps / (t * 1e-3) * 1e-12;   // 8 flops per complex multiply-add
done:
  cudaFree(out); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1);
  return rc;
}

extern "C" int gw_complex_mma_probe(int32_t mode, double ms, double *tflops, void *stream) {
  if (!tflops || !(ms > 0) || mode < 0 || mode > 2) return GW_EINVAL;
  int rc = check_arch(); if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  if (mode == 0) return run_cmma_probe<0, 2, 7>(ms, tflops, st);
  if (mode == 1) return run_cmma_probe<1, 2, 4>(ms, tflops, st);
  return run_cmma_probe<2, 2, 4>(ms, tflops, st);
}

extern "C" const char *gw_strerror(int code) {
  switch (code) {
    case GW_OK: return "ok";
    case GW_EINVAL: return "invalid argument (null/misaligned pointer, non-positive size or bad q range)";
    case GW_ENOMEM: return "workspace too small";
    case GW_EARCH: return "current device is not sm_100 (B200)";
    case GW_ESHAPE: return "size not supported by the kernels (nao > 64, ntau or nw > 200, nw > ntau, naux > 896)";
    case GW_ENOBRACKET: return "chemical-potential search: N_e(mu) does not bracket the target";
    case GW_ESTATIC: return "problem too large for the static scratch of gw_hartree_static (naux > 512): use gw_hartree with a workspace";
    case GW_ENOTPD: return "I - P0(q, iOmega) is not positive definite (non-positive Cholesky pivot in stage 2)";
    default: return code > 0 ? cudaGetErrorString((cudaError_t)code) : "unknown error";
  }
}
extern "C" int gw_version(void) { return 100; }
