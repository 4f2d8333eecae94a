// gw_stage2.cu — stage 2: Eq. 28a, Eq. 29, Eq. 30 (Algorithm 1 middle part).
//
//   P0w[n][q] = Σ_t T_wt[n][t] P0t[t][q]                  transform_kernel (GEMM with K = ntau, in place per column block)
//   Ww[n][q]  = (I − P0w[n][q])^-1 P0w[n][q]                dyson_kernel: one CTA per (n,q) matrix, blocked right-looking
//                                                           Cholesky A = I − P = L L^H, then L Y = P, L^H X = Y in place
//   Wt[t][q]  = Σ_n T_tw[t][n] Ww[n][q]                     transform_kernel again
//
// The paper solves Eq. 29 with a batched Cholesky solver; I − P0(iΩ) is Hermitian positive definite
// for time-reversal symmetric inputs (reading R5).  A non-positive pivot is reported through `info`.
// All rank-nb updates run on FP64 tensor cores (DMMA) with both operands in shared memory; the small triangular
// pieces (nb x nb Cholesky, substitutions) are done by threads in shared memory.
#include "gw_pipe.cuh"

namespace s2 {

constexpr int NTHR = 256;
constexpr int NTHR_D = 512;   // Dyson kernel: 16 warps (four per SM sub-partition) hide the latency of its global-memory updates
constexpr int NC = 64;   // columns per transform block

// ---------------- Eq. 28a / Eq. 30:  Y[o][m] = Σ_i T[o][i] X[i][m],  m over `len` ----------------
// In-place safe (X == Y): a CTA reads its whole [n_in][NC] column block into shared memory before it writes.
__global__ void __launch_bounds__(NTHR, 1) transform_kernel(int n_out, int n_in, const c128 *__restrict__ T, const c128 *X, c128 *Y,
                                                            size_t len, int nblocks) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *sX = reinterpret_cast<c128 *>(smem_raw);
  constexpr int LDX = NC + 2;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const int ksteps = (n_in + 3) / 4, rows_pad = ksteps * 4;
  for (int blk = blockIdx.x; blk < nblocks; blk += gridDim.x) {
    const size_t m0 = (size_t)blk * NC;
    const int ncol = (int)((len - m0) < (size_t)NC ? (len - m0) : (size_t)NC);
    __syncthreads();
    for (int i = threadIdx.x; i < rows_pad * NC; i += NTHR) {
      const int r = i / NC, cc = i - r * NC;
      const bool ok = r < n_in && cc < ncol;
      gwp::cp_async16_zfill(sX + r * LDX + cc, ok ? X + (size_t)r * len + m0 + cc : X, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();
    // output rows in chunks of 128 (two 8-row m-tiles per warp); the column block stays in shared memory
    for (int oc = 0; oc < n_out; oc += 128) {
      double accr[2][8][2], acci[2][8][2];
#pragma unroll
      for (int i = 0; i < 2; i++)
#pragma unroll
        for (int j = 0; j < 8; j++) { accr[i][j][0] = accr[i][j][1] = 0.0; acci[i][j][0] = acci[i][j][1] = 0.0; }
      const int o0 = oc + 8 * w + g, o1 = oc + 8 * (w + 8) + g;
      const bool act0 = oc + 8 * w < n_out, act1 = oc + 8 * (w + 8) < n_out;
      if (act0) {
        for (int ks = 0; ks < ksteps; ks++) {
          const int i = 4 * ks + c;
          c128 a0 = make_double2(0.0, 0.0), a1 = a0;
          if (i < n_in) {
            if (o0 < n_out) a0 = __ldg(T + (size_t)o0 * n_in + i);
            if (act1 && o1 < n_out) a1 = __ldg(T + (size_t)o1 * n_in + i);
          }
          const c128 *brow = sX + i * LDX + g;
#pragma unroll
          for (int nt = 0; nt < 8; nt++) {
            const c128 b = brow[8 * nt];
            cmma(accr[0][nt], acci[0][nt], a0, b);
            if (act1) cmma(accr[1][nt], acci[1][nt], a1, b);
          }
        }
      }
      // X may alias Y: the whole column block was read into shared memory before the first store of this block
#pragma unroll
      for (int h = 0; h < 2; h++) {
        const int o = h == 0 ? o0 : o1;
        if ((h == 0 ? act0 : act1) && o < n_out) {
#pragma unroll
          for (int nt = 0; nt < 8; nt++) {
            const int col = 8 * nt + 2 * c;
            if (col < ncol) Y[(size_t)o * len + m0 + col] = make_double2(accr[h][nt][0], acci[h][nt][0]);
            if (col + 1 < ncol) Y[(size_t)o * len + m0 + col + 1] = make_double2(accr[h][nt][1], acci[h][nt][1]);
          }
        }
      }
    }
  }
}

// ---------------- Eq. 29 ----------------
struct DysonParams {
  int n, nb, batch, nq, q0;
  int ldpan, ldn;          // smem strides: panel [row][ldpan]; block rows [k][ldn]
  int prow;                // rows of the panel buffer: every row an 8-row tile of an update can touch
  c128 *PW;                // batch matrices, n*n each (index = freq*nq + ql); overwritten by the solution
  c128 *slabs;             // per-CTA copy for A / L
  int32_t *info;
  double *phi;        // optional [batch]: tr{ln[I - P0w] + P0w} (summand of Eq. 37), or NULL
};

// C[r][col] -= Σ_k Aop(r,k) * Bop(k,col) over a tile range; operands in shared memory.
//  A element (r,k): AK_MAJOR ? conj(sA[k*lda + r]) : sA[r*lda + k]
//  B element (k,col): B_NMAJOR_CONJ ? conj(sB[col*ldb + k]) : sB[k*ldb + col]
//  rows r in [0,M), cols in [0,N); C element at Cg[(size_t)r*ldc + col]; LOWER: only tiles with col0 <= row0+7.
template <bool AK_MAJOR, bool B_NMAJOR_CONJ, bool LOWER>
__device__ __forceinline__ void update_tiles(c128 *Cg, int ldc, int M, int N, const c128 *sA, int lda, const c128 *sB, int ldb, int ksteps) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const int mtiles = (M + 7) / 8, ngroups = (N + 31) / 32;    // a work unit = one m-tile x four n-tiles
  for (int unit = w; unit < mtiles * ngroups; unit += NTHR_D / 32) {
    const int mt = unit / ngroups, ng = unit - mt * ngroups;
    const int r0 = 8 * mt, c0 = 32 * ng;
    if (LOWER && c0 > r0 + 7) continue;
    double cr[4][2], ci[4][2];
#pragma unroll
    for (int j = 0; j < 4; j++) { cr[j][0] = cr[j][1] = 0.0; ci[j][0] = ci[j][1] = 0.0; }
    const int r = r0 + g;
    // the C elements of this unit are loaded before the K loop, so that the global-memory latency runs under the DMMAs
    c128 cv[4][2];
#pragma unroll
    for (int j = 0; j < 4; j++)
#pragma unroll
      for (int e = 0; e < 2; e++) {
        const int col = c0 + 8 * j + 2 * c + e;
        const bool on = r < M && c0 + 8 * j < N && !(LOWER && c0 + 8 * j > r0 + 7) && col < N;
        cv[j][e] = on ? Cg[(size_t)r * ldc + col] : make_double2(0.0, 0.0);
      }
    for (int ks = 0; ks < ksteps; ks++) {
      const int k = 4 * ks + c;
      c128 a;
      if (AK_MAJOR) { a = sA[k * lda + r]; a.y = -a.y; } else { a = sA[r * lda + k]; }
#pragma unroll
      for (int j = 0; j < 4; j++) {
        const int col = c0 + 8 * j + g;
        if (c0 + 8 * j < N && !(LOWER && c0 + 8 * j > r0 + 7)) {
          c128 b;
          if (B_NMAJOR_CONJ) { b = sB[col * ldb + k]; b.y = -b.y; } else { b = sB[k * ldb + col]; }
          cmma(cr[j], ci[j], a, b);
        }
      }
    }
    if (r < M) {
#pragma unroll
      for (int j = 0; j < 4; j++) {
        if (c0 + 8 * j < N && !(LOWER && c0 + 8 * j > r0 + 7)) {
#pragma unroll
          for (int e = 0; e < 2; e++) {
            const int col = c0 + 8 * j + 2 * c + e;
            if (col < N) Cg[(size_t)r * ldc + col] = make_double2(cv[j][e].x - cr[j][e], cv[j][e].y - ci[j][e]);
          }
        }
      }
    }
  }
}

__global__ void __launch_bounds__(NTHR_D, 1) dyson_kernel(const DysonParams P) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *smem = reinterpret_cast<c128 *>(smem_raw);
  const int n = P.n, nb = P.nb, ldpan = P.ldpan, ldn = P.ldn;
  const int npad = (n + 7) / 8 * 8;
  c128 *sPan = smem;                          // [npad][ldpan]  (also reused as [nb][ldn] block row of L in the back solve)
  const int kst4 = 4 * ((nb + 3) / 4);
  const int pan_units = P.prow * ldpan > kst4 * ldn ? P.prow * ldpan : kst4 * ldn;
  c128 *sBlk = smem + pan_units;              // [nb][ldn]
  __shared__ int s_bad;
  __shared__ double s_piv;
  double *s_red = reinterpret_cast<double *>(smem);    // the panel buffer is free when the reduction runs (>= NTHR_D doubles)
  c128 *A = P.slabs + (size_t)blockIdx.x * n * n;
  const int kst = (nb + 3) / 4;

  for (int mi = blockIdx.x; mi < P.batch; mi += gridDim.x) {
    c128 *Pm = P.PW + (size_t)mi * n * n;
    if (threadIdx.x == 0) s_bad = 0;
    double trp = 0.0;                                  // this thread's share of Re tr P0w (fixed order: deterministic)
    for (int e = threadIdx.x; e < n * n; e += NTHR_D) {
      const int i = e / n, j = e - i * n;
      const c128 v = Pm[e];
      if (i == j) trp += v.x;
      A[e] = make_double2((i == j ? 1.0 : 0.0) - v.x, -v.y);
    }
    __syncthreads();
    // ---------- blocked right-looking Cholesky of A (lower) ----------
    for (int j0 = 0; j0 < n; j0 += nb) {
      const int jb = min(nb, n - j0), m = n - j0;
      for (int e = threadIdx.x; e < P.prow * 4 * kst; e += NTHR_D) { // panel rows r < m, cols < 4*kst (zero padded)
        const int r = e / (4 * kst), cc = e - r * (4 * kst);
        sPan[r * ldpan + cc] = (r < m && cc < jb) ? A[(size_t)(j0 + r) * n + j0 + cc] : make_double2(0.0, 0.0);
      }
      __syncthreads();
      for (int cc = 0; cc < jb; cc++) {                               // unblocked Cholesky of the jb x jb diagonal block
        if (threadIdx.x == 0) {
          double dd = sPan[cc * ldpan + cc].x;
          if (!(dd > 0.0)) { s_bad = 1; dd = 1.0; }
          s_piv = sqrt(dd);
          sPan[cc * ldpan + cc] = make_double2(s_piv, 0.0);
        }
        __syncthreads();
        const double inv = 1.0 / s_piv;
        for (int i = cc + 1 + threadIdx.x; i < jb; i += NTHR_D) { c128 v = sPan[i * ldpan + cc]; sPan[i * ldpan + cc] = make_double2(v.x * inv, v.y * inv); }
        __syncthreads();
        const int rem = jb - cc - 1;
        for (int e = threadIdx.x; e < rem * rem; e += NTHR_D) {
          const int i = cc + 1 + e / rem, c2 = cc + 1 + e % rem;
          if (c2 <= i) {
            const c128 li = sPan[i * ldpan + cc], lc = sPan[c2 * ldpan + cc];
            c128 &a = sPan[i * ldpan + c2];
            a.x -= li.x * lc.x + li.y * lc.y;
            a.y -= li.y * lc.x - li.x * lc.y;
          }
        }
        __syncthreads();
      }
      // panel rows below the block: L_i = A_i L_jj^{-H}  (one thread per row)
      for (int i = jb + threadIdx.x; i < m; i += NTHR_D) {
        c128 *row = sPan + i * ldpan;
        for (int cc = 0; cc < jb; cc++) {
          c128 s = row[cc];
          const c128 *lj = sPan + cc * ldpan;
          for (int k = 0; k < cc; k++) { const c128 l = row[k], d = lj[k]; s.x -= l.x * d.x + l.y * d.y; s.y -= l.y * d.x - l.x * d.y; }
          const double inv = 1.0 / lj[cc].x;
          row[cc] = make_double2(s.x * inv, s.y * inv);
        }
      }
      __syncthreads();
      for (int e = threadIdx.x; e < m * jb; e += NTHR_D) {              // write the factored panel back (lower part)
        const int r = e / jb, cc = e - r * jb;
        A[(size_t)(j0 + r) * n + j0 + cc] = (r >= cc) ? sPan[r * ldpan + cc] : make_double2(0.0, 0.0);
      }
      // trailing update A22 -= L21 L21^H (lower tiles)
      if (m > jb)
        update_tiles<false, true, true>(A + (size_t)(j0 + jb) * n + j0 + jb, n, m - jb, m - jb, sPan + jb * ldpan, ldpan, sPan + jb * ldpan, ldpan, kst);
      __syncthreads();
    }
    if (P.phi) {
      // Eq. 37 summand: tr ln[I - P0w] + tr P0w = 2 Σ_i ln L_ii + tr P0w  (tree reduction in a fixed order)
      double v = trp;
      for (int i = threadIdx.x; i < n; i += NTHR_D) v += 2.0 * log(A[(size_t)i * n + i].x);
      s_red[threadIdx.x] = v;
      __syncthreads();
      for (int h = NTHR_D / 2; h > 0; h >>= 1) {
        if (threadIdx.x < h) s_red[threadIdx.x] += s_red[threadIdx.x + h];
        __syncthreads();
      }
      if (threadIdx.x == 0) P.phi[mi] = s_red[0];
      __syncthreads();                                  // s_red lives in the panel buffer, which the forward solve fills next
    }
    // ---------- forward solve L Y = P (in place on Pm) ----------
    for (int j0 = 0; j0 < n; j0 += nb) {
      const int jb = min(nb, n - j0), m = n - j0;
      for (int e = threadIdx.x; e < P.prow * 4 * kst; e += NTHR_D) {
        const int r = e / (4 * kst), cc = e - r * (4 * kst);
        sPan[r * ldpan + cc] = (r < m && cc < jb) ? A[(size_t)(j0 + r) * n + j0 + cc] : make_double2(0.0, 0.0);
      }
      for (int e = threadIdx.x; e < 4 * kst * npad; e += NTHR_D) {
        const int r = e / npad, col = e - r * npad;
        sBlk[r * ldn + col] = (r < jb && col < n) ? Pm[(size_t)(j0 + r) * n + col] : make_double2(0.0, 0.0);
      }
      __syncthreads();
      for (int col = threadIdx.x; col < n; col += NTHR_D) {
        for (int r = 0; r < jb; r++) {
          c128 s = sBlk[r * ldn + col];
          const c128 *lr = sPan + r * ldpan;
          for (int k = 0; k < r; k++) { const c128 l = lr[k], y = sBlk[k * ldn + col]; s.x -= l.x * y.x - l.y * y.y; s.y -= l.x * y.y + l.y * y.x; }
          const double inv = 1.0 / lr[r].x;
          s.x *= inv; s.y *= inv;
          sBlk[r * ldn + col] = s;
          Pm[(size_t)(j0 + r) * n + col] = s;
        }
      }
      __syncthreads();
      if (m > jb)
        update_tiles<false, false, false>(Pm + (size_t)(j0 + jb) * n, n, m - jb, n, sPan + jb * ldpan, ldpan, sBlk, ldn, kst);
      __syncthreads();
    }
    // ---------- backward solve L^H X = Y (in place on Pm) ----------
    const int nblk = (n + nb - 1) / nb;
    for (int bj = nblk - 1; bj >= 0; bj--) {
      const int j0 = bj * nb, jb = min(nb, n - j0);
      c128 *sRow = sPan;    // block row of L: sRow[k][i] = L[j0+k][i], i < j0 + jb
      for (int e = threadIdx.x; e < 4 * kst * npad; e += NTHR_D) {
        const int r = e / npad, col = e - r * npad;
        sRow[r * ldn + col] = (r < jb && col < j0 + jb) ? A[(size_t)(j0 + r) * n + col] : make_double2(0.0, 0.0);
        sBlk[r * ldn + col] = (r < jb && col < n) ? Pm[(size_t)(j0 + r) * n + col] : make_double2(0.0, 0.0);
      }
      __syncthreads();
      for (int col = threadIdx.x; col < n; col += NTHR_D) {
        for (int r = jb - 1; r >= 0; r--) {
          c128 s = sBlk[r * ldn + col];
          for (int k = r + 1; k < jb; k++) { const c128 l = sRow[k * ldn + j0 + r], x = sBlk[k * ldn + col]; s.x -= l.x * x.x + l.y * x.y; s.y -= l.x * x.y - l.y * x.x; }
          const double inv = 1.0 / sRow[r * ldn + j0 + r].x;
          s.x *= inv; s.y *= inv;
          sBlk[r * ldn + col] = s;
          Pm[(size_t)(j0 + r) * n + col] = s;
        }
      }
      __syncthreads();
      if (j0 > 0)
        update_tiles<true, false, false>(Pm, n, j0, n, sRow, ldn, sBlk, ldn, kst);
      __syncthreads();
    }
    // one 64-bit atomic minimum over (n, q): info[0] = q is the low word, info[1] = n the high word; {-1,-1} = all ones
    if (threadIdx.x == 0 && s_bad && P.info)
      atomicMin(reinterpret_cast<unsigned long long *>(P.info), ((unsigned long long)(unsigned)(mi / P.nq) << 32) | (unsigned)(P.q0 + mi % P.nq));
    __syncthreads();
  }
}

__global__ void set_info_kernel2(int32_t *info) { info[0] = -1; info[1] = -1; }

struct Plan { int nb, ldpan, ldn, prow, grid_d, grid_t, nblocks; size_t smem_d, smem_t, work_bytes; bool ok; };

static Plan make_plan(const gw_problem *p) {
  Plan pl; memset(&pl, 0, sizeof(pl));
  GwDims d = gw_dims(p);
  const int n = d.naux, npad = (n + 7) / 8 * 8;
  pl.ldn = npad + 2;
  pl.ok = false;
  for (int nb = 32; nb >= 4; nb /= 2) {
    const int kst4 = (nb + 3) / 4 * 4;
    const int ldpan = kst4 + 4;
    int prow = n > nb ? nb + (n - nb + 7) / 8 * 8 : npad;
    if (prow < npad) prow = npad;
    size_t pan = (size_t)prow * ldpan; const size_t alt = (size_t)kst4 * pl.ldn;
    if (alt > pan) pan = alt;
    const size_t bytes = (pan + (size_t)kst4 * pl.ldn) * sizeof(c128);
    if (bytes <= 226 * 1024 && bytes >= NTHR_D * sizeof(double)) { pl.nb = nb; pl.ldpan = ldpan; pl.prow = prow; pl.smem_d = bytes; pl.ok = true; break; }
  }
  const int nsm = gwp::gw_num_sms();
  const int batch = d.nw * d.nq;
  pl.grid_d = batch < nsm ? batch : nsm;
  const size_t len = (size_t)d.nq * n * n;
  pl.nblocks = (int)((len + NC - 1) / NC);
  pl.grid_t = pl.nblocks < nsm ? pl.nblocks : nsm;
  const int kin = d.ntau > d.nw ? d.ntau : d.nw;
  pl.smem_t = (size_t)((kin + 3) / 4 * 4) * (NC + 2) * sizeof(c128);
  pl.work_bytes = 256 + (size_t)nsm * n * n * sizeof(c128);
  if (pl.smem_t > 227 * 1024) pl.ok = false;
  return pl;
}

}  // namespace s2

size_t gw_stage2_workspace(const gw_problem *p) {
  s2::Plan pl = s2::make_plan(p);
  return pl.ok ? pl.work_bytes : 0;
}

int gw_launch_stage2(const gw_problem *p, const c128 *P0t, c128 *Wt, int32_t *info, double *phi, cudaStream_t st) {
  s2::Plan pl = s2::make_plan(p);
  if (!pl.ok) return GW_ESHAPE;
  if (!p->work || p->work_bytes < pl.work_bytes || (((uintptr_t)p->work) & 255)) return GW_ENOMEM;
  GwDims d = gw_dims(p);
  if (d.nw > d.ntau) return GW_ESHAPE;    // the frequency-domain intermediate lives in the first nw slices of the Wt buffer
  const size_t len = (size_t)d.nq * d.naux * d.naux;
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(s2::transform_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_t)) != cudaSuccess) return (int)e;
  if ((e = cudaFuncSetAttribute(s2::dyson_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_d)) != cudaSuccess) return (int)e;
  if (info) s2::set_info_kernel2<<<1, 1, 0, st>>>(info);
  s2::transform_kernel<<<pl.grid_t, s2::NTHR, pl.smem_t, st>>>(d.nw, d.ntau, (const c128 *)p->T_wt, P0t, Wt, len, pl.nblocks);
  s2::DysonParams D;
  D.n = d.naux; D.nb = pl.nb; D.batch = d.nw * d.nq; D.nq = d.nq; D.q0 = d.q0; D.ldpan = pl.ldpan; D.ldn = pl.ldn; D.prow = pl.prow;
  D.PW = Wt; D.slabs = (c128 *)((char *)p->work + 256); D.info = info; D.phi = phi;
  s2::dyson_kernel<<<pl.grid_d, s2::NTHR_D, pl.smem_d, st>>>(D);
  s2::transform_kernel<<<pl.grid_t, s2::NTHR, pl.smem_t, st>>>(d.ntau, d.nw, (const c128 *)p->T_tw, Wt, Wt, len, pl.nblocks);
  return (int)cudaGetLastError();
}

int gw_launch_transform(int n_out, int n_in, const c128 *T, const c128 *X, c128 *Y, size_t len, cudaStream_t st) {
  if (n_out <= 0 || n_in <= 0 || n_out > GW_MAX_NTAU || n_in > GW_MAX_NTAU) return GW_ESHAPE;
  const int nsm = gwp::gw_num_sms();
  const size_t nb = (len + s2::NC - 1) / s2::NC;
  if (nb == 0) return GW_OK;
  if (nb > 0x7fffffffu) return GW_ESHAPE;
  const int grid = nb < (size_t)nsm ? (int)nb : nsm;
  const size_t smem = (size_t)((n_in + 3) / 4 * 4) * (s2::NC + 2) * sizeof(c128);
  cudaError_t e = cudaFuncSetAttribute(s2::transform_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  s2::transform_kernel<<<grid, s2::NTHR, smem, st>>>(n_out, n_in, T, X, Y, len, (int)nb);
  return (int)cudaGetLastError();
}
