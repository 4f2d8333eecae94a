/*
 * gwref.c — CPU ORACLE for one scGW iteration's self-energy build (arXiv 2206.07660).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code with the
 * CUDA path (paper_2206_07660_b200/csrc) and neither imports the other.
 *
 * Plain, slow, obviously-correct loops in complex FP64 ("All our calculations are
 * performed in double precision"), in the order of the paper's
 * Algorithm 1:
 *
 *   for q { for k { read V(k,k+q); for tau: Eq. 28b }   -> gwref_p0t_slice
 *           Eq. 28a                                      -> gwref_transform
 *           for Omega_n: Eq. 29                          -> gwref_dyson
 *           Eq. 30                                       -> gwref_transform
 *           for k { read V(k,k-q); for tau: Eq. 31 } }   -> gwref_sigma_slice
 *   Eq. 22 (static exchange)                             -> gwref_exchange_slice
 *   Eq. 37 summand tr{ln[I - P0(iOmega)] + P0(iOmega)}   -> gwref_phi
 *   loop closure (Fig. 4): Eq. 20 -> gwref_hartree; Eq. 16 -> gwref_dyson_update; Eq. 15 -> gwref_electron_count;
 *   chemical potential -> gwref_find_mu
 *
 * No blocking, fusion or reordering beyond the temporaries A, B, X, Y named in
 * SURVEY.md §8(c); the linear solve is Gaussian elimination with partial pivoting
 * (assumes nothing about definiteness).  No symmetry of the inputs is used:
 * V[k+q][k] is read itself, never replaced by conj(V[k][k+q]).
 *
 * Readings of the paper where it is ambiguous:
 *   R1 sign of Eq. 28b: G(-tau_t) = -G(beta - tau_t) = -G[ntau-1-t]; the leading "-1/N_k" of
 *      Eq. 28b is that antiperiodicity sign, so P0t = -(s/N_k) sum_k tr[V G(tau) V' G(beta-tau)]
 *      (negative semidefinite, I - P0(iOmega) HPD as a Cholesky solver needs).
 *   R2 spin: closed shell, factor spin_deg = 2 on P0 only (sum over sigma,sigma' in Eq. 28b).
 *   R3 "I is a unitary matrix" = identity.
 *   R4 transforms Eq. 28a / Eq. 30 are applied as the given matrices T_wt / T_tw (inputs).
 *
 * Layouts (row-major, complex128):
 *   V block (k1,k2): [naux][nao][nao]  = V^{k1 k2}_{ij}(Q)   (Eq. 6-7); blocks are
 *                    handed over as a table of nk*nk pointers (NULL = not resident) so that the
 *                    big configs can be checked on sampled slices without 71 GB of host memory.
 *   G_t   : [nk][nao][nao]   one tau node;  P/W slabs: [nk][naux][naux];  Sigma_t: [nk][nao][nao].
 *
 * Parity pins: tests/test_oracle_pins.py (closed form P1, Lindhard P2, invariants P3-P5,
 * brute-force Matsubara sum P6, trace identity P7, solve residual P8, exchange limit P9,
 * literal 4-index evaluation P10, scalar form / series / eigenvalue route of the Eq. 37 summand P11, fermionic
 * transform of a single pole P12; loop closure: non-interacting closed form of Eq. 16 in the generalised eigenbasis P13,
 * Fermi-function electron count and root of the chemical-potential search P14, literal einsum of Eq. 20 P15,
 * back transform of a single pole P16, non-interacting limit of a whole iteration P17, weighted Matsubara sum of Eq. 37 P20).
 * Spin (oracle/__init__.py writes the sigma sums out over these single-block routines): identical channels = closed shell P18, Lindhard per
 * channel P19, two-component blocks under a global spin rotation P21.
 * Nothing here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex c128;

typedef struct {
  int32_t nk1, nk2, nk3;
  int32_t nao, naux, ntau, nw;
  int32_t spin_deg;
  double beta;
} gwref_dims;

/* ---- Gamma-centred mesh arithmetic: k = (i1*nk2 + i2)*nk3 + i3 ---- */
static int mesh_combine(const gwref_dims *d, int k, int q, int sign) {
  int n1 = d->nk1, n2 = d->nk2, n3 = d->nk3;
  int k1 = k / (n2 * n3), k2 = (k / n3) % n2, k3 = k % n3;
  int q1 = q / (n2 * n3), q2 = (q / n3) % n2, q3 = q % n3;
  int r1 = ((k1 + sign * q1) % n1 + n1) % n1;
  int r2 = ((k2 + sign * q2) % n2 + n2) % n2;
  int r3 = ((k3 + sign * q3) % n3 + n3) % n3;
  return (r1 * n2 + r2) * n3 + r3;
}
int gwref_kadd(const gwref_dims *d, int k, int q) { return mesh_combine(d, k, q, +1); }
int gwref_ksub(const gwref_dims *d, int k, int q) { return mesh_combine(d, k, q, -1); }

/* ---- Eq. 28b, one (q, tau_t):
 *   P0[Q][Q'] = -(s/N_k) sum_k sum_abcd V^{k,k+q}_{da}(Q) G^{k+q}_{ab}(tau_t) V^{k+q,k}_{bc}(Q') G^{k}_{cd}(beta - tau_t)
 * G_t = G[t], G_tbar = G[ntau-1-t] (reading R1).  Returns 1 if a needed V block is missing. */
int gwref_p0t_slice(const gwref_dims *d, const c128 *const *Vblk, const c128 *G_t, const c128 *G_tbar,
                    int q, c128 *out) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao, naux = d->naux;
  const size_t n2 = (size_t)nao * nao;
  c128 *A = (c128 *)malloc(sizeof(c128) * naux * n2);
  c128 *B = (c128 *)malloc(sizeof(c128) * naux * n2);
  c128 *acc = (c128 *)calloc((size_t)naux * naux, sizeof(c128));
  int missing = 0;
  for (int k = 0; k < nk; k++) {
    const int kq = gwref_kadd(d, k, q);
    const c128 *V1 = Vblk[(size_t)k * nk + kq];  /* V[k][k+q] */
    const c128 *V2 = Vblk[(size_t)kq * nk + k];  /* V[k+q][k] */
    if (!V1 || !V2) { missing = 1; break; }
    const c128 *Gkq = G_t + (size_t)kq * n2;
    const c128 *Gk = G_tbar + (size_t)k * n2;
    /* A[Q][d][b] = sum_a V[k][kq][Q][d][a] * G[t][kq][a][b] */
    for (int Q = 0; Q < naux; Q++)
      for (int dd = 0; dd < nao; dd++)
        for (int b = 0; b < nao; b++) {
          c128 s = 0;
          for (int a = 0; a < nao; a++) s += V1[Q * n2 + dd * nao + a] * Gkq[a * nao + b];
          A[Q * n2 + dd * nao + b] = s;
        }
    /* B[Q'][b][d] = sum_c V[kq][k][Q'][b][c] * G[tbar][k][c][d] */
    for (int Q = 0; Q < naux; Q++)
      for (int b = 0; b < nao; b++)
        for (int dd = 0; dd < nao; dd++) {
          c128 s = 0;
          for (int c = 0; c < nao; c++) s += V2[Q * n2 + b * nao + c] * Gk[c * nao + dd];
          B[Q * n2 + b * nao + dd] = s;
        }
    /* acc[Q][Q'] += sum_{d,b} A[Q][d][b] * B[Q'][b][d] */
    for (int Q = 0; Q < naux; Q++)
      for (int Qp = 0; Qp < naux; Qp++) {
        c128 s = 0;
        for (int dd = 0; dd < nao; dd++)
          for (int b = 0; b < nao; b++) s += A[Q * n2 + dd * nao + b] * B[Qp * n2 + b * nao + dd];
        acc[(size_t)Q * naux + Qp] += s;
      }
  }
  if (!missing) {
    const double pref = -(double)d->spin_deg / (double)nk;
    for (size_t i = 0; i < (size_t)naux * naux; i++) out[i] = pref * acc[i];
  }
  free(A); free(B); free(acc);
  return missing;
}

/* Full stage 1: P0t[t][q][Q][Q'] for all q, t.  G: [ntau][nk][nao][nao]. */
int gwref_polarization(const gwref_dims *d, const c128 *const *Vblk, const c128 *G, c128 *P0t) {
  const int nk = d->nk1 * d->nk2 * d->nk3, ntau = d->ntau;
  const size_t gs = (size_t)nk * d->nao * d->nao, ps = (size_t)d->naux * d->naux;
  int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic) reduction(| : bad)
  for (int q = 0; q < nk; q++)
    for (int t = 0; t < ntau; t++)
      bad |= gwref_p0t_slice(d, Vblk, G + (size_t)t * gs, G + (size_t)(ntau - 1 - t) * gs, q,
                             P0t + ((size_t)t * nk + q) * ps);
  return bad;
}

/* ---- Eq. 28a / Eq. 30 as given matrices:  Y[o][m] = sum_i T[o][i] * X[i][m]
 * X, Y are [n][...] with element strides xs / ys between consecutive i / o; m runs over len entries. */
void gwref_transform(int n_out, int n_in, const c128 *T, const c128 *X, size_t xs, c128 *Y, size_t ys, size_t len) {
  for (int o = 0; o < n_out; o++)
    for (size_t m = 0; m < len; m++) {
      c128 s = 0;
      for (int i = 0; i < n_in; i++) s += T[(size_t)o * n_in + i] * X[(size_t)i * xs + m];
      Y[(size_t)o * ys + m] = s;
    }
}

/* ---- Eq. 29: X = (I - P)^-1 P by Gaussian elimination with partial pivoting.
 * Returns 0, or 1 if a pivot is exactly zero. */
int gwref_dyson(int n, const c128 *P, c128 *X) {
  c128 *M = (c128 *)malloc(sizeof(c128) * n * n);
  for (int i = 0; i < n; i++)
    for (int j = 0; j < n; j++) {
      M[(size_t)i * n + j] = (i == j ? 1.0 : 0.0) - P[(size_t)i * n + j];
      X[(size_t)i * n + j] = P[(size_t)i * n + j];
    }
  int fail = 0;
  for (int c = 0; c < n && !fail; c++) {
    int p = c;
    double best = cabs(M[(size_t)c * n + c]);
    for (int r = c + 1; r < n; r++) {
      double v = cabs(M[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    if (best == 0.0) { fail = 1; break; }
    if (p != c)
      for (int j = 0; j < n; j++) {
        c128 tmp = M[(size_t)c * n + j]; M[(size_t)c * n + j] = M[(size_t)p * n + j]; M[(size_t)p * n + j] = tmp;
        tmp = X[(size_t)c * n + j]; X[(size_t)c * n + j] = X[(size_t)p * n + j]; X[(size_t)p * n + j] = tmp;
      }
    for (int r = c + 1; r < n; r++) {
      c128 f = M[(size_t)r * n + c] / M[(size_t)c * n + c];
      if (f == 0) continue;
      for (int j = c; j < n; j++) M[(size_t)r * n + j] -= f * M[(size_t)c * n + j];
      for (int j = 0; j < n; j++) X[(size_t)r * n + j] -= f * X[(size_t)c * n + j];
    }
  }
  if (!fail)
    for (int c = n - 1; c >= 0; c--) {
      for (int j = 0; j < n; j++) {
        c128 s = X[(size_t)c * n + j];
        for (int r = c + 1; r < n; r++) s -= M[(size_t)c * n + r] * X[(size_t)r * n + j];
        X[(size_t)c * n + j] = s / M[(size_t)c * n + c];
      }
    }
  free(M);
  return fail;
}

/* ---- Summand of Eq. 37: phi = tr{ ln[I - P] + P } for one matrix.
 * tr ln M = ln det M, and det M is the product of the pivots of Gaussian elimination with partial pivoting (times the
 * sign of the row permutation).  I - P0(iOmega) is Hermitian positive definite under reading R7, so det M > 0 and
 * ln det M = Σ_c ln|u_cc|; the imaginary part of tr P (zero for Hermitian P) is dropped.  Returns 1 on a zero pivot. */
int gwref_phi(int n, const c128 *P, double *phi) {
  c128 *M = (c128 *)malloc(sizeof(c128) * n * n);
  double tr = 0.0, lndet = 0.0;
  for (int i = 0; i < n; i++) {
    tr += creal(P[(size_t)i * n + i]);
    for (int j = 0; j < n; j++) M[(size_t)i * n + j] = (i == j ? 1.0 : 0.0) - P[(size_t)i * n + j];
  }
  int fail = 0;
  for (int c = 0; c < n; c++) {
    int p = c;
    double best = cabs(M[(size_t)c * n + c]);
    for (int r = c + 1; r < n; r++) {
      double v = cabs(M[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    if (best == 0.0) { fail = 1; break; }
    if (p != c)
      for (int j = 0; j < n; j++) { c128 tmp = M[(size_t)c * n + j]; M[(size_t)c * n + j] = M[(size_t)p * n + j]; M[(size_t)p * n + j] = tmp; }
    lndet += log(best);
    for (int r = c + 1; r < n; r++) {
      c128 f = M[(size_t)r * n + c] / M[(size_t)c * n + c];
      if (f == 0) continue;
      for (int j = c; j < n; j++) M[(size_t)r * n + j] -= f * M[(size_t)c * n + j];
    }
  }
  free(M);
  *phi = lndet + tr;
  return fail;
}

/* Stage 2 for ONE q (Algorithm 1 lines "Eq. 28a(q); for Omega_n: Eq. 29(q,Omega_n); Eq. 30(q)").
 * P0t_q / Wt_q: element stride tstride between consecutive tau nodes (nk*naux^2 inside the full arrays,
 * naux^2 for a packed per-q slab).  P0w_q / Ww_q: optional packed [nw][naux][naux] outputs (may be NULL). */
int gwref_screened_interaction_q(const gwref_dims *d, const c128 *T_wt, const c128 *T_tw, const c128 *P0t_q,
                                 size_t tstride_in, c128 *Wt_q, size_t tstride_out, c128 *P0w_q, c128 *Ww_q) {
  const int naux = d->naux, ntau = d->ntau, nw = d->nw;
  const size_t ps = (size_t)naux * naux;
  c128 *pw = P0w_q ? P0w_q : (c128 *)malloc(sizeof(c128) * nw * ps);
  c128 *ww = Ww_q ? Ww_q : (c128 *)malloc(sizeof(c128) * nw * ps);
  int fail = 0;
  gwref_transform(nw, ntau, T_wt, P0t_q, tstride_in, pw, ps, ps);          /* Eq. 28a */
  for (int n = 0; n < nw; n++) fail |= gwref_dyson(naux, pw + n * ps, ww + n * ps); /* Eq. 29 */
  gwref_transform(ntau, nw, T_tw, ww, ps, Wt_q, tstride_out, ps);          /* Eq. 30 */
  if (!P0w_q) free(pw);
  if (!Ww_q) free(ww);
  return fail;
}

/* Full stage 2.  P0t, Wt: [ntau][nk][naux][naux]; P0w, Ww: optional [nw][nk][naux][naux] (NULL to skip). */
int gwref_screened_interaction(const gwref_dims *d, const c128 *T_wt, const c128 *T_tw, const c128 *P0t, c128 *Wt,
                               c128 *P0w, c128 *Ww) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nw = d->nw;
  const size_t ps = (size_t)d->naux * d->naux;
  int fail = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : fail)
  for (int q = 0; q < nk; q++) {
    c128 *pw = (c128 *)malloc(sizeof(c128) * nw * ps), *ww = (c128 *)malloc(sizeof(c128) * nw * ps);
    fail |= gwref_screened_interaction_q(d, T_wt, T_tw, P0t + q * ps, (size_t)nk * ps, Wt + q * ps, (size_t)nk * ps, pw, ww);
    for (int n = 0; n < nw; n++) {
      if (P0w) memcpy(P0w + ((size_t)n * nk + q) * ps, pw + n * ps, sizeof(c128) * ps);
      if (Ww) memcpy(Ww + ((size_t)n * nk + q) * ps, ww + n * ps, sizeof(c128) * ps);
    }
    free(pw); free(ww);
  }
  return fail;
}

/* ---- Eq. 31, one (k, tau_t):
 *   Sigma[i][j] = -(1/N_k) sum_q sum_ab sum_QQ' G^{k-q}_{ab}(tau) V^{k,k-q}_{ia}(Q) P~^{q}_{QQ'}(tau) V^{k-q,k}_{bj}(Q')
 * G_t: [nk][nao][nao], Wt_t: [nk][naux][naux] at the same tau node. */
int gwref_sigma_slice_qrange(const gwref_dims *d, const c128 *const *Vblk, const c128 *G_t, const c128 *Wt_t, int k,
                             int q_begin, int q_end, c128 *out);
int gwref_sigma_slice(const gwref_dims *d, const c128 *const *Vblk, const c128 *G_t, const c128 *Wt_t, int k, c128 *out) {
  return gwref_sigma_slice_qrange(d, Vblk, G_t, Wt_t, k, 0, d->nk1 * d->nk2 * d->nk3, out);
}
/* same with the q sum restricted to q_begin <= q < q_end (one rank's partial sum) */
int gwref_sigma_slice_qrange(const gwref_dims *d, const c128 *const *Vblk, const c128 *G_t, const c128 *Wt_t, int k,
                             int q_begin, int q_end, c128 *out) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao, naux = d->naux;
  const size_t n2 = (size_t)nao * nao, ps = (size_t)naux * naux;
  c128 *X = (c128 *)malloc(sizeof(c128) * naux * n2);
  c128 *Y = (c128 *)malloc(sizeof(c128) * naux * n2);
  c128 *acc = (c128 *)calloc(n2, sizeof(c128));
  int missing = 0;
  for (int q = q_begin; q < q_end; q++) {
    const int kmq = gwref_ksub(d, k, q);
    const c128 *V1 = Vblk[(size_t)k * nk + kmq];  /* V[k][k-q] */
    const c128 *V2 = Vblk[(size_t)kmq * nk + k];  /* V[k-q][k] */
    if (!V1 || !V2) { missing = 1; break; }
    const c128 *Gp = G_t + (size_t)kmq * n2;
    const c128 *W = Wt_t + (size_t)q * ps;
    /* X[Q][i][b] = sum_a V[k][kmq][Q][i][a] * G[t][kmq][a][b] */
    for (int Q = 0; Q < naux; Q++)
      for (int i = 0; i < nao; i++)
        for (int b = 0; b < nao; b++) {
          c128 s = 0;
          for (int a = 0; a < nao; a++) s += V1[Q * n2 + i * nao + a] * Gp[a * nao + b];
          X[Q * n2 + i * nao + b] = s;
        }
    /* Y[Q'][i][b] = sum_Q X[Q][i][b] * Wt[t][q][Q][Q'] */
    for (int Qp = 0; Qp < naux; Qp++)
      for (size_t ib = 0; ib < n2; ib++) {
        c128 s = 0;
        for (int Q = 0; Q < naux; Q++) s += X[Q * n2 + ib] * W[(size_t)Q * naux + Qp];
        Y[Qp * n2 + ib] = s;
      }
    /* acc[i][j] += sum_{Q',b} Y[Q'][i][b] * V[kmq][k][Q'][b][j] */
    for (int i = 0; i < nao; i++)
      for (int j = 0; j < nao; j++) {
        c128 s = 0;
        for (int Qp = 0; Qp < naux; Qp++)
          for (int b = 0; b < nao; b++) s += Y[Qp * n2 + i * nao + b] * V2[Qp * n2 + b * nao + j];
        acc[i * nao + j] += s;
      }
  }
  if (!missing)
    for (size_t i = 0; i < n2; i++) out[i] = -acc[i] / (double)nk;
  free(X); free(Y); free(acc);
  return missing;
}

/* Full stage 3: Sigma[t][k][i][j]. */
int gwref_selfenergy(const gwref_dims *d, const c128 *const *Vblk, const c128 *G, const c128 *Wt, c128 *Sigma) {
  const int nk = d->nk1 * d->nk2 * d->nk3, ntau = d->ntau;
  const size_t gs = (size_t)nk * d->nao * d->nao, ws = (size_t)nk * d->naux * d->naux, n2 = (size_t)d->nao * d->nao;
  int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic) reduction(| : bad)
  for (int k = 0; k < nk; k++)
    for (int t = 0; t < ntau; t++)
      bad |= gwref_sigma_slice(d, Vblk, G + (size_t)t * gs, Wt + (size_t)t * ws, k, Sigma + (size_t)t * gs + (size_t)k * n2);
  return bad;
}

/* ---- Eq. 22, one k:
 *   K[i][j] = -(1/N_k) sum_k' sum_ab sum_Q V^{k k'}_{ia}(Q) gamma^{k'}_{ab} V^{k' k}_{bj}(Q) */
int gwref_exchange_slice_qrange(const gwref_dims *d, const c128 *const *Vblk, const c128 *gamma, int k, int q_begin, int q_end, c128 *out);
int gwref_exchange_slice(const gwref_dims *d, const c128 *const *Vblk, const c128 *gamma, int k, c128 *out) {
  return gwref_exchange_slice_qrange(d, Vblk, gamma, k, 0, d->nk1 * d->nk2 * d->nk3, out);
}
/* same with the k' sum restricted to k' = k - q, q_begin <= q < q_end */
int gwref_exchange_slice_qrange(const gwref_dims *d, const c128 *const *Vblk, const c128 *gamma, int k, int q_begin, int q_end, c128 *out) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao, naux = d->naux;
  const size_t n2 = (size_t)nao * nao;
  c128 *acc = (c128 *)calloc(n2, sizeof(c128));
  c128 *T = (c128 *)malloc(sizeof(c128) * n2);
  int missing = 0;
  for (int q = q_begin; q < q_end && !missing; q++) {
    const int kp = gwref_ksub(d, k, q);
    const c128 *V1 = Vblk[(size_t)k * nk + kp], *V2 = Vblk[(size_t)kp * nk + k];
    if (!V1 || !V2) { missing = 1; break; }
    const c128 *g = gamma + (size_t)kp * n2;
    for (int Q = 0; Q < naux; Q++) {
      /* T[i][b] = sum_a V[k][k'][Q][i][a] * gamma[k'][a][b] */
      for (int i = 0; i < nao; i++)
        for (int b = 0; b < nao; b++) {
          c128 s = 0;
          for (int a = 0; a < nao; a++) s += V1[Q * n2 + i * nao + a] * g[a * nao + b];
          T[i * nao + b] = s;
        }
      for (int i = 0; i < nao; i++)
        for (int j = 0; j < nao; j++) {
          c128 s = 0;
          for (int b = 0; b < nao; b++) s += T[i * nao + b] * V2[Q * n2 + b * nao + j];
          acc[i * nao + j] += s;
        }
    }
  }
  if (!missing)
    for (size_t i = 0; i < n2; i++) out[i] = -acc[i] / (double)nk;
  free(acc); free(T);
  return missing;
}

int gwref_exchange(const gwref_dims *d, const c128 *const *Vblk, const c128 *gamma, c128 *K) {
  const int nk = d->nk1 * d->nk2 * d->nk3;
  const size_t n2 = (size_t)d->nao * d->nao;
  int bad = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : bad)
  for (int k = 0; k < nk; k++) bad |= gwref_exchange_slice(d, Vblk, gamma, k, K + (size_t)k * n2);
  return bad;
}

/* =====================================================================================================================
 * Loop closure: the rest of one scGW iteration, Fig. 4 steps 1, 3, 4.
 * Same rules as above: plain loops, the paper's order, no symmetry used.
 * ===================================================================================================================== */

/* ---- Hartree term, Eq. 20 (the printed label "(19)" is lost in the text, the second line is Eq. 20):
 *   J[k][i][j] = (1/N_k) sum_k' sum_sigma1 sum_ab sum_Q V^{kk}_{ij}(Q) gamma^{k'}_{a sigma1, b sigma1} V^{k'k'}_{ba}(Q)
 * gamma: [nk][nao][nao] per spin channel; the sum over sigma1 of a closed shell is the factor spin_deg (reading R3).
 * Only the diagonal blocks V[k][k] are read.  Returns 1 if one of them is missing. */
int gwref_hartree(const gwref_dims *d, const c128 *const *Vblk, const c128 *gamma, c128 *J) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao, naux = d->naux;
  const size_t n2 = (size_t)nao * nao;
  for (int k = 0; k < nk; k++) if (!Vblk[(size_t)k * nk + k]) return 1;
  for (int k = 0; k < nk; k++)
    for (int i = 0; i < nao; i++)
      for (int j = 0; j < nao; j++) {
        c128 s = 0;
        for (int kp = 0; kp < nk; kp++) {
          const c128 *Vkk = Vblk[(size_t)k * nk + k], *Vpp = Vblk[(size_t)kp * nk + kp], *g = gamma + (size_t)kp * n2;
          for (int a = 0; a < nao; a++)
            for (int b = 0; b < nao; b++)
              for (int Q = 0; Q < naux; Q++) s += Vkk[Q * n2 + i * nao + j] * g[a * nao + b] * Vpp[Q * n2 + b * nao + a];
        }
        J[(size_t)k * n2 + i * nao + j] = (double)d->spin_deg / (double)nk * s;
      }
  return 0;
}

/* ---- Dyson equation, Eq. 16, one (k, i omega_n):
 *   G = [ (i omega_n + mu) S - F - Sigma_w ]^-1,   F = H0 + Sigma_inf (static part, Eq. 17-18), Sigma_w = Sigma~(i omega_n) or NULL
 * "The inverse is defined as a matrix inversion in spin-orbital space": Gaussian elimination with partial
 * pivoting on [A | I], then back substitution.  Returns 1 on a zero pivot. */
int gwref_dyson_update_one(int n, double omega, double mu, const c128 *S, const c128 *F, const c128 *Sigma_w, c128 *G) {
  c128 *A = (c128 *)malloc(sizeof(c128) * n * n);
  const c128 z = mu + I * omega;
  for (int i = 0; i < n; i++)
    for (int j = 0; j < n; j++) {
      A[(size_t)i * n + j] = z * S[(size_t)i * n + j] - F[(size_t)i * n + j] - (Sigma_w ? Sigma_w[(size_t)i * n + j] : 0);
      G[(size_t)i * n + j] = (i == j) ? 1.0 : 0.0;
    }
  int fail = 0;
  for (int c = 0; c < n && !fail; c++) {
    int p = c;
    double best = cabs(A[(size_t)c * n + c]);
    for (int r = c + 1; r < n; r++) { double v = cabs(A[(size_t)r * n + c]); if (v > best) { best = v; p = r; } }
    if (best == 0.0) { fail = 1; break; }
    if (p != c)
      for (int j = 0; j < n; j++) {
        c128 t = A[(size_t)c * n + j]; A[(size_t)c * n + j] = A[(size_t)p * n + j]; A[(size_t)p * n + j] = t;
        t = G[(size_t)c * n + j]; G[(size_t)c * n + j] = G[(size_t)p * n + j]; G[(size_t)p * n + j] = t;
      }
    for (int r = c + 1; r < n; r++) {
      const c128 f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      if (f == 0) continue;
      for (int j = c; j < n; j++) A[(size_t)r * n + j] -= f * A[(size_t)c * n + j];
      for (int j = 0; j < n; j++) G[(size_t)r * n + j] -= f * G[(size_t)c * n + j];
    }
  }
  if (!fail)
    for (int c = n - 1; c >= 0; c--)
      for (int j = 0; j < n; j++) {
        c128 s = G[(size_t)c * n + j];
        for (int r = c + 1; r < n; r++) s -= A[(size_t)c * n + r] * G[(size_t)r * n + j];
        G[(size_t)c * n + j] = s / A[(size_t)c * n + c];
      }
  free(A);
  return fail;
}

/* Eq. 16 for all (n, k).  S, F: [nk][nao][nao]; Sigma_w, G_w: [nwf][nk][nao][nao] (Sigma_w may be NULL); omega: [nwf]. */
int gwref_dyson_update(const gwref_dims *d, int nwf, const double *omega, double mu, const c128 *S, const c128 *F,
                       const c128 *Sigma_w, c128 *G_w) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao;
  const size_t n2 = (size_t)nao * nao;
  int fail = 0;
#pragma omp parallel for collapse(2) schedule(dynamic) reduction(| : fail)
  for (int n = 0; n < nwf; n++)
    for (int k = 0; k < nk; k++)
      fail |= gwref_dyson_update_one(nao, omega[n], mu, S + k * n2, F + k * n2,
                                     Sigma_w ? Sigma_w + ((size_t)n * nk + k) * n2 : NULL, G_w + ((size_t)n * nk + k) * n2);
  return fail;
}

/* ---- Electron count, Eq. 15:  N_e = (1/N_k) sum_k tr[gamma^k S^k] over spin orbitals, gamma^k = -G^k(tau = beta^-).
 * G(beta^-) is obtained from the sampled G(i omega_n) with the given evaluation vector: G(beta^-) = sum_n t_beta[n] G_w[n]
 * (reading R6: the grids and their maps are inputs).  The spin trace of a closed shell is the factor spin_deg. */
double gwref_electron_count(const gwref_dims *d, int nwf, const c128 *t_beta, const c128 *S, const c128 *G_w) {
  const int nk = d->nk1 * d->nk2 * d->nk3, nao = d->nao;
  const size_t n2 = (size_t)nao * nao;
  c128 tot = 0;
  for (int k = 0; k < nk; k++)
    for (int i = 0; i < nao; i++)
      for (int j = 0; j < nao; j++) {
        c128 gb = 0;                                              /* G^k_ij(beta^-) */
        for (int n = 0; n < nwf; n++) gb += t_beta[n] * G_w[((size_t)n * nk + k) * n2 + i * nao + j];
        tot += -gb * S[(size_t)k * n2 + j * nao + i];             /* tr[gamma S] = sum_ij gamma_ij S_ji */
      }
  return (double)d->spin_deg / (double)nk * creal(tot);
}

/* ---- Chemical potential (Fig. 4 step 3): adjust mu until N_e(mu) equals n_target ("threshold value of 1e-9").
 * Bisection on the monotone function N_e(mu) of Eq. 15-16 (reading R16):
 *   1. widen [lo, hi] by its own width (at most 60 times) until N_e(lo) <= n_target <= N_e(hi);
 *   2. halve it until hi - lo <= mu_tol (at most 200 times): mid goes to lo if N_e(mid) < n_target, else to hi;
 *   3. mu = (lo + hi)/2; *ne_out = N_e(mu).
 * Returns 0; 1 if a pivot vanished; 2 if no bracket was found.  Gw_scratch: [nwf][nk][nao][nao]. */
int gwref_find_mu(const gwref_dims *d, int nwf, const double *omega, const c128 *t_beta, const c128 *S, const c128 *F,
                  const c128 *Sigma_w, double n_target, double mu_lo, double mu_hi, double mu_tol, c128 *Gw_scratch,
                  double *mu_out, double *ne_out) {
  double lo = mu_lo, hi = mu_hi;
  int fail = 0;
#define NE(mu_) (fail |= gwref_dyson_update(d, nwf, omega, (mu_), S, F, Sigma_w, Gw_scratch), gwref_electron_count(d, nwf, t_beta, S, Gw_scratch))
  double nlo = NE(lo), nhi = NE(hi);
  int it = 0;
  while ((nlo > n_target || nhi < n_target) && it < 60) {
    const double w = hi - lo;
    if (nlo > n_target) { lo -= w; nlo = NE(lo); } else { hi += w; nhi = NE(hi); }
    it++;
  }
  if (nlo > n_target || nhi < n_target) return 2;
  for (it = 0; it < 200 && hi - lo > mu_tol; it++) {
    const double mid = 0.5 * (lo + hi);
    if (NE(mid) < n_target) lo = mid; else hi = mid;
  }
  *mu_out = 0.5 * (lo + hi);
  *ne_out = NE(*mu_out);
#undef NE
  return fail;
}

/* ---- Dynamical part of the GW Luttinger-Ward functional, Eq. 37:
 *   Phi~_GW = (1/(2 N_k)) sum_q (1/beta) sum_n tr{ ln[I - P0^q(i Omega_n)] + P0^q(i Omega_n) }
 * evaluated on the sampled frequencies with the caller's quadrature weights w[n] for the Matsubara sum (reading R18: the
 * paper prints none; for n >= 0 grids the weights carry the factor 2 of the n < 0 mirror images):
 *   Phi~_GW = (1/(2 N_k beta)) sum_q sum_n w[n] phi[n][q],   phi from gwref_phi.   phi: [nw][nq] (nq = nk for the full mesh). */
double gwref_phi_gw(int nk, int nq, int nw, double beta, const double *w, const double *phi) {
  double tot = 0.0;
  for (int q = 0; q < nq; q++)
    for (int n = 0; n < nw; n++) tot += w[n] * phi[(size_t)n * nq + q];
  return tot / (2.0 * (double)nk * beta);
}

/* Y = a X + b Y (simple mixing of two iterates, PAPER.md:326-330 mentions DIIS; plain damping is the baseline it improves on) */
void gwref_axpby(size_t n, c128 a, const c128 *X, c128 b, c128 *Y) {
  for (size_t i = 0; i < n; i++) Y[i] = a * X[i] + b * Y[i];
}

/* number of OpenMP threads the loops above will use (reported as cpu_baseline.cores) */
#ifdef _OPENMP
#include <omp.h>
int gwref_num_threads(void) { return omp_get_max_threads(); }
#else
int gwref_num_threads(void) { return 1; }
#endif
