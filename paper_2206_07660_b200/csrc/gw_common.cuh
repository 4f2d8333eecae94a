// gw_common.cuh — shared device/host helpers of libgw_b200 (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include "../../include/gw.h"

typedef double2 c128;   // (re, im); layout-compatible with gw_c128

// shape limits of the kernels (GW_ESHAPE, documented in gw.h)
#define GW_MAX_NAO 64
#define GW_MAX_NTAU 200
#define GW_MAX_NAUX 896

struct GwDims {
  int nk1, nk2, nk3, nk;
  int nao, naux, ntau, nw;
  int s;            // spin_deg
  int q0, nq;       // q shard
  int sym;          // gw_problem.symmetry
  int ns;           // spin blocks of G: 1, 2 (collinear: uu, dd) or 4 (two-component: uu, ud, du, dd)
  int vq;           // 1: p->V is a q-slab (GW_V_QSLAB), 0: the full tensor
};

static inline GwDims gw_dims(const gw_problem *p) {
  GwDims d;
  d.nk1 = p->nk1; d.nk2 = p->nk2; d.nk3 = p->nk3; d.nk = p->nk1 * p->nk2 * p->nk3;
  d.nao = p->nao; d.naux = p->naux; d.ntau = p->ntau; d.nw = p->nw; d.s = p->spin_deg;
  d.q0 = p->q_begin; d.nq = p->q_end - p->q_begin; d.sym = p->symmetry;
  d.ns = p->ns == 2 ? 2 : (p->ns == 4 ? 4 : 1); d.vq = p->v_layout == GW_V_QSLAB ? 1 : 0;
  return d;
}

// Γ-centred mesh arithmetic: k = (i1*nk2+i2)*nk3+i3, component-wise modulo
__host__ __device__ __forceinline__ int gw_kcombine(const GwDims &d, int k, int q, int sign) {
  int n23 = d.nk2 * d.nk3;
  int k1 = k / n23, k2 = (k / d.nk3) % d.nk2, k3 = k % d.nk3;
  int q1 = q / n23, q2 = (q / d.nk3) % d.nk2, q3 = q % d.nk3;
  int r1 = k1 + sign * q1; r1 = (r1 % d.nk1 + d.nk1) % d.nk1;
  int r2 = k2 + sign * q2; r2 = (r2 % d.nk2 + d.nk2) % d.nk2;
  int r3 = k3 + sign * q3; r3 = (r3 % d.nk3 + d.nk3) % d.nk3;
  return (r1 * d.nk2 + r2) * d.nk3 + r3;
}
__host__ __device__ __forceinline__ int gw_kadd(const GwDims &d, int k, int q) { return gw_kcombine(d, k, q, +1); }
__host__ __device__ __forceinline__ int gw_ksub(const GwDims &d, int k, int q) { return gw_kcombine(d, k, q, -1); }

// V block index (in blocks of naux*nao² elements) for the shard-local q index ql, with kq = k + q:
//   gw_vfwd = V[k][k+q],  gw_vbwd = V[k+q][k]   (gw.h "V layouts").  Stages 3/4 use them with k := k-q, kq := k.
__host__ __device__ __forceinline__ size_t gw_vfwd(const GwDims &d, int ql, int k, int kq) {
  return d.vq ? ((size_t)ql * d.nk + k) * 2 : (size_t)k * d.nk + kq;
}
__host__ __device__ __forceinline__ size_t gw_vbwd(const GwDims &d, int ql, int k, int kq) {
  return d.vq ? ((size_t)ql * d.nk + k) * 2 + 1 : (size_t)kq * d.nk + k;
}
// number of V blocks behind p->V
__host__ __device__ __forceinline__ size_t gw_vblocks(const GwDims &d) { return d.vq ? (size_t)d.nq * d.nk * 2 : (size_t)d.nk * d.nk; }

__device__ __forceinline__ c128 cmul(c128 a, c128 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ void cfma(c128 &acc, c128 a, c128 b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}

// FP64 tensor-core MMA, D(8x8) += A(8x4, row) * B(4x8, col).  On sm_100a this is one DMMA.8x8x4.
// Fragment layout (lane = 4*g + c): A[g][c], B[c][g], C[g][2c], C[g][2c+1].
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// complex 8x8 (+)= complex 8x4 * complex 4x8 as four real DMMAs (the "4-real-GEMM" scheme).
// cr/ci: real/imag accumulator fragments; a, b: this lane's complex A[g][c] and B[c][g] elements.
__device__ __forceinline__ void cmma(double (&cr)[2], double (&ci)[2], c128 a, c128 b) {
  // real and imaginary chains alternate, so consecutive DMMAs of one warp never depend on each other
  dmma884(cr[0], cr[1], a.x, b.x);
  dmma884(ci[0], ci[1], a.x, b.y);
  dmma884(cr[0], cr[1], -a.y, b.y);
  dmma884(ci[0], ci[1], a.y, b.x);
}

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// kernel launchers implemented per stage
int gw_launch_stage1(const gw_problem *p, const c128 *G, c128 *P0t, cudaStream_t st);
int gw_launch_stage2(const gw_problem *p, const c128 *P0t, c128 *Wt, int32_t *info, double *phi, cudaStream_t st);
int gw_launch_transform(int n_out, int n_in, const c128 *T, const c128 *X, c128 *Y, size_t len, cudaStream_t st);
// acc_mode (stages 3 and 4; used by the out-of-core driver to continue the q sum across V slabs in the resident order):
//   GW_ACC_CONTINUE : the accumulators start from the UNSCALED partial sums found in the output array
//   GW_ACC_PARTIAL  : the output array receives UNSCALED partial sums (no -(1/N_k), no symmetry mirror copies)
enum { GW_ACC_CONTINUE = 1, GW_ACC_PARTIAL = 2 };
int gw_launch_stage3(const gw_problem *p, const c128 *G, const c128 *Wt, c128 *Sigma, cudaStream_t st, int acc_mode = 0);
int gw_launch_stage4(const gw_problem *p, const c128 *gamma, c128 *K, cudaStream_t st, int acc_mode = 0);
int gw_launch_hartree(const gw_problem *p, const c128 *gamma, c128 *J, cudaStream_t st);
int gw_launch_dyson_update(int nk, int nao, int nwf, const double *omega, double mu, const c128 *S, const c128 *F, const c128 *Sigma_w, c128 *G_w,
                           int32_t *info, cudaStream_t st);
int gw_launch_electron_count(int nk, int nao, int nwf, int spin_deg, const c128 *t_beta, const c128 *S, const c128 *G_w, c128 *partial, double *ne,
                             cudaStream_t st);
int gw_launch_phi_gw(int nk, int nq, int nw, double beta, const double *w, const double *phi, double *out, cudaStream_t st);
int gw_launch_axpby(size_t n, c128 a, const c128 *X, c128 b, c128 *Y, cudaStream_t st);
size_t gw_stage1_workspace(const gw_problem *p);
size_t gw_stage2_workspace(const gw_problem *p);
size_t gw_stage3_workspace(const gw_problem *p);
size_t gw_stage4_workspace(const gw_problem *p);
double gw_stage1_flops(const gw_problem *p);
double gw_stage3_flops(const gw_problem *p);
double gw_stage4_flops(const gw_problem *p);
void gw_stage_flops(const gw_problem *p, double *out4);
int gw_stage_launches(const gw_problem *p);
