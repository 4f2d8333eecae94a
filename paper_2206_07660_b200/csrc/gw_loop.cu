// gw_loop.cu — loop closure of one scGW iteration (Fig. 4 steps 1, 3, 4):
//   Hartree term J (Eq. 20), Dyson equation G = [(iω_n + μ)S − F − Σ̃(iω_n)]^-1 (Eq. 16),
//   electron count N_e = (1/N_k) Σ_k tr[γ^k S^k] (Eq. 15), the chemical-potential search
//   ("threshold value of 1e-9") and the damping Y = aX + bY.
// The τ <-> iω_n transforms of the loop (Eq. 13, 14) are gw_transform (gw_stage2.cu) with the fermionic matrices.
// All of it is small batched FP64 work (nao x nao matrices, a few ms per iteration against seconds for stages 1 and 3),
// written for determinism: every reduction runs in a fixed order.
#include <math.h>
#include "gw_common.cuh"

namespace lp {

constexpr int NT = 256;

// fixed-order tree reduction of one complex value per thread over the CTA (NT threads); result valid in thread 0
__device__ __forceinline__ c128 block_sum(c128 v, c128 *red) {
  red[threadIdx.x] = v;
  __syncthreads();
  for (int s = NT / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) { red[threadIdx.x].x += red[threadIdx.x + s].x; red[threadIdx.x].y += red[threadIdx.x + s].y; }
    __syncthreads();
  }
  return red[0];
}

// ---- Hartree, Eq. 20:  rho[Q] = Σ_k' Σ_ab γ[k'][a][b] V[k'][k'][Q][b][a];   J[k][i][j] = (s/N_k) Σ_Q V[k][k][Q][i][j] rho[Q]
__global__ void __launch_bounds__(NT) hartree_rho_kernel(const GwDims d, int ql0, const c128 *__restrict__ V, const c128 *__restrict__ gamma, c128 *__restrict__ rho) {
  __shared__ c128 red[NT];
  const int Q = blockIdx.x, nao = d.nao, n2 = nao * nao;
  c128 acc = make_double2(0.0, 0.0);
  for (int sg = 0; sg < d.ns; sg++) {                      // Σ_sigma1 of Eq. 20: the spin-diagonal blocks
    if (d.ns == 4 && (sg == 1 || sg == 2)) continue;
    for (int kp = 0; kp < d.nk; kp++) {
      const c128 *Vq = V + (gw_vfwd(d, ql0, kp, kp) * d.naux + Q) * n2, *g = gamma + ((size_t)sg * d.nk + kp) * n2;
      for (int e = threadIdx.x; e < n2; e += NT) {
        const int b = e / nao, a = e - b * nao;
        cfma(acc, g[a * nao + b], Vq[e]);
      }
    }
  }
  const c128 tot = block_sum(acc, red);
  if (threadIdx.x == 0) rho[Q] = tot;
}

__global__ void __launch_bounds__(NT) hartree_j_kernel(const GwDims d, int ql0, const c128 *__restrict__ V, const c128 *__restrict__ rho, c128 *__restrict__ J) {
  const int k = blockIdx.y, n2 = d.nao * d.nao, e = blockIdx.x * NT + threadIdx.x;
  if (e >= n2) return;
  const c128 *Vk = V + gw_vfwd(d, ql0, k, k) * d.naux * n2 + e;
  c128 acc = make_double2(0.0, 0.0);
  for (int Q = 0; Q < d.naux; Q++) cfma(acc, Vk[(size_t)Q * n2], rho[Q]);
  const double pref = (double)d.s / (double)d.nk;
  J[(size_t)k * n2 + e] = make_double2(pref * acc.x, pref * acc.y);
}

// ---- Dyson equation, Eq. 16: one CTA per (n, k) inverts A = (μ + iω_n) S[k] − F[k] − Σ_w[n][k] in shared memory by Gauss-Jordan
// elimination with partial (row) pivoting, in place; the row swaps are undone as column swaps of the inverse at the end.
// A zero pivot column is reported through info = {n, k} (one 64-bit atomic minimum, as in stage 2).
__global__ void __launch_bounds__(NT) dyson_update_kernel(int nk, int nao, const double *__restrict__ omega, double mu, const c128 *__restrict__ S,
                                                          const c128 *__restrict__ F, const c128 *__restrict__ Sigma_w, c128 *__restrict__ G_w, int32_t *info) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128 *A = reinterpret_cast<c128 *>(smem_raw);       // [nao][ld]
  const int ld = nao + 1;
  c128 *col = A + (size_t)nao * ld;                    // [nao] column c before the elimination step
  int *piv = reinterpret_cast<int *>(col + nao);      // [nao]
  __shared__ int s_p;
  __shared__ double s_best;
  const int m = blockIdx.x, n = m / nk, k = m - n * nk, n2 = nao * nao;
  const c128 z = make_double2(mu, omega[n]);
  const c128 *Sk = S + (size_t)k * n2, *Fk = F + (size_t)k * n2, *Sw = Sigma_w ? Sigma_w + (size_t)m * n2 : nullptr;
  for (int e = threadIdx.x; e < n2; e += NT) {
    const int i = e / nao, j = e - i * nao;
    c128 a = cmul(z, Sk[e]);
    a.x -= Fk[e].x; a.y -= Fk[e].y;
    if (Sw) { a.x -= Sw[e].x; a.y -= Sw[e].y; }
    A[i * ld + j] = a;
  }
  __syncthreads();
  bool fail = false;
  for (int c = 0; c < nao; c++) {
    // pivot: the first row r >= c with the largest |A[r][c]| (warp 0; ties go to the smaller row index)
    if (threadIdx.x < 32) {
      double best = -1.0; int bp = c;
      for (int r = c + (int)threadIdx.x; r < nao; r += 32) {
        const double v = hypot(A[r * ld + c].x, A[r * ld + c].y);
        if (v > best) { best = v; bp = r; }
      }
      for (int off = 16; off > 0; off >>= 1) {
        const double ob = __shfl_down_sync(0xffffffffu, best, off);
        const int op = __shfl_down_sync(0xffffffffu, bp, off);
        if (ob > best || (ob == best && op < bp)) { best = ob; bp = op; }
      }
      if (threadIdx.x == 0) { s_p = bp; s_best = best; piv[c] = bp; }
    }
    __syncthreads();
    const int p = s_p;
    if (!(s_best > 0.0)) { fail = true; break; }        // uniform over the CTA
    if (p != c)
      for (int j = threadIdx.x; j < nao; j += NT) { const c128 t = A[c * ld + j]; A[c * ld + j] = A[p * ld + j]; A[p * ld + j] = t; }
    __syncthreads();
    const c128 pv = A[c * ld + c];
    const double den = pv.x * pv.x + pv.y * pv.y;
    const c128 pinv = make_double2(pv.x / den, -pv.y / den);
    for (int r = threadIdx.x; r < nao; r += NT) col[r] = A[r * ld + c];
    __syncthreads();
    for (int j = threadIdx.x; j < nao; j += NT) A[c * ld + j] = (j == c) ? pinv : cmul(A[c * ld + j], pinv);
    __syncthreads();
    for (int e = threadIdx.x; e < n2; e += NT) {
      const int r = e / nao, j = e - r * nao;
      if (r == c) continue;
      const c128 f = col[r], row = A[c * ld + j];
      c128 a = (j == c) ? make_double2(0.0, 0.0) : A[r * ld + j];
      a.x -= f.x * row.x - f.y * row.y;
      a.y -= f.x * row.y + f.y * row.x;
      A[r * ld + j] = a;
    }
    __syncthreads();
  }
  if (fail) {
    if (threadIdx.x == 0 && info) atomicMin(reinterpret_cast<unsigned long long *>(info), ((unsigned long long)(unsigned)k << 32) | (unsigned)n);
    return;
  }
  for (int c = nao - 1; c >= 0; c--) {
    const int p = piv[c];
    if (p != c)
      for (int r = threadIdx.x; r < nao; r += NT) { const c128 t = A[r * ld + c]; A[r * ld + c] = A[r * ld + p]; A[r * ld + p] = t; }
    __syncthreads();
  }
  c128 *out = G_w + (size_t)m * n2;
  for (int e = threadIdx.x; e < n2; e += NT) { const int i = e / nao, j = e - i * nao; out[e] = A[i * ld + j]; }
}

__global__ void set_info_kernel(int32_t *info) { info[0] = -1; info[1] = -1; }

// ---- Electron count, Eq. 15: partial[k] = Σ_ij −(Σ_n t_beta[n] G_w[n][k][i][j]) S[k][j][i];  N_e = (s/N_k) Re Σ_k partial[k]
__global__ void __launch_bounds__(NT) count_partial_kernel(int nk, int nao, int nwf, const c128 *__restrict__ t_beta, const c128 *__restrict__ S,
                                                           const c128 *__restrict__ G_w, c128 *__restrict__ partial) {
  __shared__ c128 red[NT];
  const int k = blockIdx.x, n2 = nao * nao;
  c128 acc = make_double2(0.0, 0.0);
  for (int e = threadIdx.x; e < n2; e += NT) {
    const int i = e / nao, j = e - i * nao;
    c128 gb = make_double2(0.0, 0.0);
    for (int n = 0; n < nwf; n++) cfma(gb, t_beta[n], G_w[((size_t)n * nk + k) * n2 + e]);
    cfma(acc, make_double2(-gb.x, -gb.y), S[(size_t)k * n2 + j * nao + i]);
  }
  const c128 tot = block_sum(acc, red);
  if (threadIdx.x == 0) partial[k] = tot;
}
__global__ void count_final_kernel(int nk, int spin_deg, const c128 *__restrict__ partial, double *__restrict__ ne) {
  double tot = 0.0;
  for (int k = 0; k < nk; k++) tot += partial[k].x;
  *ne = (double)spin_deg / (double)nk * tot;
}

__global__ void __launch_bounds__(NT) axpby_kernel(size_t n, c128 a, const c128 *__restrict__ X, c128 b, c128 *Y, bool use_y) {
  for (size_t i = (size_t)blockIdx.x * NT + threadIdx.x; i < n; i += (size_t)gridDim.x * NT) {
    c128 r = cmul(a, X[i]);
    if (use_y) { const c128 y = cmul(b, Y[i]); r.x += y.x; r.y += y.y; }
    Y[i] = r;
  }
}

// ---- Eq. 37 with quadrature weights: out = (1/(2 N_k beta)) Σ_q Σ_n w[n] phi[n][q]; one CTA, fixed order
__global__ void __launch_bounds__(NT) phi_gw_kernel(int nk, int nq, int nw, double beta, const double *__restrict__ w, const double *__restrict__ phi,
                                                    double *__restrict__ out) {
  __shared__ c128 red[NT];
  double acc = 0.0;
  for (int q = threadIdx.x; q < nq; q += NT)
    for (int n = 0; n < nw; n++) acc = fma(w[n], phi[(size_t)n * nq + q], acc);
  const c128 tot = block_sum(make_double2(acc, 0.0), red);
  if (threadIdx.x == 0) *out = tot.x / (2.0 * (double)nk * beta);
}

static size_t dyson_smem(int nao) { return ((size_t)nao * (nao + 1) + nao) * sizeof(c128) + (size_t)nao * sizeof(int); }

}  // namespace lp

int gw_launch_hartree(const gw_problem *p, const c128 *gamma, c128 *J, cudaStream_t st) {
  const GwDims d = gw_dims(p);
  if (!p->work || p->work_bytes < 256 + (size_t)d.naux * sizeof(c128) || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  c128 *rho = (c128 *)((char *)p->work + 256);
  // the diagonal blocks V[k][k] = V[k][k+0]: in the q-slab layout they are slot (0 - q_begin, k, 0), present iff the shard holds q = 0
  if (d.vq && !(d.q0 <= 0 && 0 < d.q0 + d.nq)) return GW_EINVAL;
  const int ql0 = -d.q0;
  lp::hartree_rho_kernel<<<d.naux, lp::NT, 0, st>>>(d, ql0, (const c128 *)p->V, gamma, rho);
  const int n2 = d.nao * d.nao;
  lp::hartree_j_kernel<<<dim3((n2 + lp::NT - 1) / lp::NT, d.nk), lp::NT, 0, st>>>(d, ql0, (const c128 *)p->V, rho, J);
  return (int)cudaGetLastError();
}

int gw_launch_dyson_update(int nk, int nao, int nwf, const double *omega, double mu, const c128 *S, const c128 *F, const c128 *Sigma_w, c128 *G_w,
                           int32_t *info, cudaStream_t st) {
  const size_t smem = lp::dyson_smem(nao);
  cudaError_t e = cudaFuncSetAttribute(lp::dyson_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  if (info) lp::set_info_kernel<<<1, 1, 0, st>>>(info);
  lp::dyson_update_kernel<<<nwf * nk, lp::NT, smem, st>>>(nk, nao, omega, mu, S, F, Sigma_w, G_w, info);
  return (int)cudaGetLastError();
}

int gw_launch_electron_count(int nk, int nao, int nwf, int spin_deg, const c128 *t_beta, const c128 *S, const c128 *G_w, c128 *partial, double *ne,
                             cudaStream_t st) {
  lp::count_partial_kernel<<<nk, lp::NT, 0, st>>>(nk, nao, nwf, t_beta, S, G_w, partial);
  lp::count_final_kernel<<<1, 1, 0, st>>>(nk, spin_deg, partial, ne);
  return (int)cudaGetLastError();
}

int gw_launch_axpby(size_t n, c128 a, const c128 *X, c128 b, c128 *Y, cudaStream_t st) {
  if (n == 0) return 0;
  size_t blocks = (n + lp::NT - 1) / lp::NT;
  if (blocks > 148 * 16) blocks = 148 * 16;
  lp::axpby_kernel<<<(unsigned)blocks, lp::NT, 0, st>>>(n, a, X, b, Y, !(b.x == 0.0 && b.y == 0.0));
  return (int)cudaGetLastError();
}

int gw_launch_phi_gw(int nk, int nq, int nw, double beta, const double *w, const double *phi, double *out, cudaStream_t st) {
  lp::phi_gw_kernel<<<1, lp::NT, 0, st>>>(nk, nq, nw, beta, w, phi, out);
  return (int)cudaGetLastError();
}
