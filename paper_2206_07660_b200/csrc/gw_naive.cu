// gw_naive.cu — one-thread-per-output debug kernels (GW_DEBUG_NAIVE=1 or gw_debug_set_naive(1)).
// They exist to cross-check the optimised kernels on the device at tiny sizes; never on the product path.
#include "gw_common.cuh"

__global__ void naive_p0_kernel(GwDims d, const c128 *__restrict__ V, const c128 *__restrict__ G, c128 *__restrict__ P0t) {
  const int t = blockIdx.x / d.nq, ql = blockIdx.x % d.nq, q = d.q0 + ql;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao;
  const size_t vb = (size_t)naux * n2;
  for (int o = threadIdx.x; o < naux * naux; o += blockDim.x) {
    const int Q = o / naux, Qp = o % naux;
    c128 acc = make_double2(0, 0);
    for (int k = 0; k < d.nk; k++) {
      const int kq = gw_kadd(d, k, q);
      const c128 *V1 = V + ((size_t)k * d.nk + kq) * vb + (size_t)Q * n2;
      const c128 *V2 = V + ((size_t)kq * d.nk + k) * vb + (size_t)Qp * n2;
      const c128 *G1 = G + ((size_t)t * d.nk + kq) * n2;
      const c128 *G2 = G + ((size_t)(d.ntau - 1 - t) * d.nk + k) * n2;
      for (int b = 0; b < nao; b++)
        for (int dd = 0; dd < nao; dd++) {
          c128 x = make_double2(0, 0), y = make_double2(0, 0);
          for (int a = 0; a < nao; a++) cfma(x, V1[dd * nao + a], G1[a * nao + b]);
          for (int c = 0; c < nao; c++) cfma(y, V2[b * nao + c], G2[c * nao + dd]);
          cfma(acc, x, y);
        }
    }
    const double pref = -(double)d.s / d.nk;
    P0t[((size_t)t * d.nq + ql) * naux * naux + o] = make_double2(pref * acc.x, pref * acc.y);
  }
}

// Y[o][m] = sum_i T[o][i] X[i][m], m over len
__global__ void naive_transform_kernel(int n_out, int n_in, const c128 *__restrict__ T, const c128 *__restrict__ X, c128 *__restrict__ Y, size_t len) {
  size_t m = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= len) return;
  for (int o = 0; o < n_out; o++) {
    c128 acc = make_double2(0, 0);
    for (int i = 0; i < n_in; i++) cfma(acc, T[(size_t)o * n_in + i], X[(size_t)i * len + m]);
    Y[(size_t)o * len + m] = acc;
  }
}

// one block per matrix: A = I - P (in `work`), Cholesky A = L L^H, X = L^-H L^-1 P in place on P.
__global__ void naive_dyson_kernel(int n, int nq, int q0, c128 *__restrict__ PW, c128 *__restrict__ work, int32_t *info) {
  c128 *P = PW + (size_t)blockIdx.x * n * n;
  c128 *A = work + (size_t)blockIdx.x * n * n;
  __shared__ int bad;
  if (threadIdx.x == 0) bad = 0;
  for (int o = threadIdx.x; o < n * n; o += blockDim.x) {
    int i = o / n, j = o % n;
    c128 v = P[o];
    A[o] = make_double2((i == j ? 1.0 : 0.0) - v.x, -v.y);
  }
  __syncthreads();
  for (int j = 0; j < n; j++) {
    // right-looking: scale column j, then update the trailing lower triangle
    double djj = A[(size_t)j * n + j].x;
    if (!(djj > 0.0)) { if (threadIdx.x == 0) bad = 1; djj = 1.0; }
    __syncthreads();
    const double r = sqrt(djj);
    if (threadIdx.x == 0) A[(size_t)j * n + j] = make_double2(r, 0.0);
    for (int i = j + 1 + threadIdx.x; i < n; i += blockDim.x) {
      c128 v = A[(size_t)i * n + j];
      A[(size_t)i * n + j] = make_double2(v.x / r, v.y / r);
    }
    __syncthreads();
    const int m = n - j - 1;
    for (int o = threadIdx.x; o < m * m; o += blockDim.x) {
      int i = j + 1 + o / m, c = j + 1 + o % m;
      if (c > i) continue;
      c128 li = A[(size_t)i * n + j], lc = A[(size_t)c * n + j];
      c128 &a = A[(size_t)i * n + c];      // a -= li * conj(lc)
      a.x -= li.x * lc.x + li.y * lc.y;
      a.y -= li.y * lc.x - li.x * lc.y;
    }
    __syncthreads();
  }
  // forward: L Y = P (each thread owns columns)
  for (int c = threadIdx.x; c < n; c += blockDim.x) {
    for (int i = 0; i < n; i++) {
      c128 s = P[(size_t)i * n + c];
      for (int k = 0; k < i; k++) { c128 l = A[(size_t)i * n + k], y = P[(size_t)k * n + c]; s.x -= l.x * y.x - l.y * y.y; s.y -= l.x * y.y + l.y * y.x; }
      double r = A[(size_t)i * n + i].x;
      P[(size_t)i * n + c] = make_double2(s.x / r, s.y / r);
    }
    // backward: L^H X = Y
    for (int i = n - 1; i >= 0; i--) {
      c128 s = P[(size_t)i * n + c];
      for (int k = i + 1; k < n; k++) { c128 l = A[(size_t)k * n + i], y = P[(size_t)k * n + c]; /* conj(l) * y */ s.x -= l.x * y.x + l.y * y.y; s.y -= l.x * y.y - l.y * y.x; }
      double r = A[(size_t)i * n + i].x;
      P[(size_t)i * n + c] = make_double2(s.x / r, s.y / r);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0 && bad && info) { info[0] = q0 + blockIdx.x % nq; info[1] = blockIdx.x / nq; }
}

__global__ void naive_sigma_kernel(GwDims d, const c128 *__restrict__ V, const c128 *__restrict__ G, const c128 *__restrict__ Wt, c128 *__restrict__ Sigma) {
  const int t = blockIdx.x / d.nk, k = blockIdx.x % d.nk;
  const int nao = d.nao, naux = d.naux, n2 = nao * nao;
  const size_t vb = (size_t)naux * n2;
  extern __shared__ c128 sh[];   // X[Q][b] for fixed i : naux*nao, then Y[Q'][b]
  c128 *X = sh, *Y = sh + naux * nao;
  for (int i = 0; i < nao; i++) {
    c128 acc = make_double2(0, 0);   // thread j < nao accumulates Sigma[i][j]
    for (int ql = 0; ql < d.nq; ql++) {
      const int q = d.q0 + ql, kp = gw_ksub(d, k, q);
      const c128 *V1 = V + ((size_t)k * d.nk + kp) * vb, *V2 = V + ((size_t)kp * d.nk + k) * vb;
      const c128 *Gp = G + ((size_t)t * d.nk + kp) * n2;
      const c128 *W = Wt + ((size_t)t * d.nq + ql) * naux * naux;
      __syncthreads();
      for (int o = threadIdx.x; o < naux * nao; o += blockDim.x) {
        int Q = o / nao, b = o % nao;
        c128 s = make_double2(0, 0);
        for (int a = 0; a < nao; a++) cfma(s, V1[(size_t)Q * n2 + i * nao + a], Gp[a * nao + b]);
        X[o] = s;
      }
      __syncthreads();
      for (int o = threadIdx.x; o < naux * nao; o += blockDim.x) {
        int Qp = o / nao, b = o % nao;
        c128 s = make_double2(0, 0);
        for (int Q = 0; Q < naux; Q++) cfma(s, X[Q * nao + b], W[(size_t)Q * naux + Qp]);
        Y[o] = s;
      }
      __syncthreads();
      if (threadIdx.x < nao) {
        int j = threadIdx.x;
        for (int Qp = 0; Qp < naux; Qp++)
          for (int b = 0; b < nao; b++) cfma(acc, Y[Qp * nao + b], V2[(size_t)Qp * n2 + b * nao + j]);
      }
    }
    if (threadIdx.x < nao) {
      const double pref = -1.0 / d.nk;
      Sigma[((size_t)t * d.nk + k) * n2 + i * nao + threadIdx.x] = make_double2(pref * acc.x, pref * acc.y);
    }
  }
}

__global__ void naive_exchange_kernel(GwDims d, const c128 *__restrict__ V, const c128 *__restrict__ gamma, c128 *__restrict__ K) {
  const int k = blockIdx.x, nao = d.nao, naux = d.naux, n2 = nao * nao;
  const size_t vb = (size_t)naux * n2;
  for (int o = threadIdx.x; o < n2; o += blockDim.x) {
    int i = o / nao, j = o % nao;
    c128 acc = make_double2(0, 0);
    for (int ql = 0; ql < d.nq; ql++) {
      const int kp = gw_ksub(d, k, d.q0 + ql);
      const c128 *V1 = V + ((size_t)k * d.nk + kp) * vb, *V2 = V + ((size_t)kp * d.nk + k) * vb;
      const c128 *g = gamma + (size_t)kp * n2;
      for (int Q = 0; Q < naux; Q++)
        for (int b = 0; b < nao; b++) {
          c128 tmp = make_double2(0, 0);
          for (int a = 0; a < nao; a++) cfma(tmp, V1[(size_t)Q * n2 + i * nao + a], g[a * nao + b]);
          cfma(acc, tmp, V2[(size_t)Q * n2 + b * nao + j]);
        }
    }
    const double pref = -1.0 / d.nk;
    K[(size_t)k * n2 + o] = make_double2(pref * acc.x, pref * acc.y);
  }
}

__global__ void set_info_kernel(int32_t *info) { info[0] = -1; info[1] = -1; }

int gw_naive_stage1(const gw_problem *p, const c128 *G, c128 *P0t, cudaStream_t st) {
  GwDims d = gw_dims(p);
  naive_p0_kernel<<<d.ntau * d.nq, 256, 0, st>>>(d, (const c128 *)p->V, G, P0t);
  return (int)cudaGetLastError();
}
int gw_naive_stage2(const gw_problem *p, const c128 *P0t, c128 *Wt, void *work, size_t work_bytes, int32_t *info, cudaStream_t st) {
  GwDims d = gw_dims(p);
  const size_t len = (size_t)d.nq * d.naux * d.naux;
  if (work_bytes < 2 * (size_t)d.nw * len * sizeof(c128)) return GW_ENOMEM;
  c128 *Pw = (c128 *)work, *A = Pw + (size_t)d.nw * len;
  if (info) set_info_kernel<<<1, 1, 0, st>>>(info);
  naive_transform_kernel<<<(unsigned)((len + 127) / 128), 128, 0, st>>>(d.nw, d.ntau, (const c128 *)p->T_wt, P0t, Pw, len);
  naive_dyson_kernel<<<d.nw * d.nq, 256, 0, st>>>(d.naux, d.nq, d.q0, Pw, A, info);
  naive_transform_kernel<<<(unsigned)((len + 127) / 128), 128, 0, st>>>(d.ntau, d.nw, (const c128 *)p->T_tw, Pw, Wt, len);
  return (int)cudaGetLastError();
}
int gw_naive_stage3(const gw_problem *p, const c128 *G, const c128 *Wt, c128 *Sigma, cudaStream_t st) {
  GwDims d = gw_dims(p);
  size_t sh = 2 * (size_t)d.naux * d.nao * sizeof(c128);
  if (sh > 48 * 1024) cudaFuncSetAttribute(naive_sigma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
  naive_sigma_kernel<<<d.ntau * d.nk, 128, sh, st>>>(d, (const c128 *)p->V, G, Wt, Sigma);
  return (int)cudaGetLastError();
}
int gw_naive_stage4(const gw_problem *p, const c128 *gamma, c128 *K, cudaStream_t st) {
  GwDims d = gw_dims(p);
  naive_exchange_kernel<<<d.nk, 256, 0, st>>>(d, (const c128 *)p->V, gamma, K);
  return (int)cudaGetLastError();
}
