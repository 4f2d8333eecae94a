/*
 * gw.h — C ABI of libgw_b200: one scGW iteration's self-energy build on one B200 (sm_100a).
 *
 * Method: "Fully self-consistent finite-temperature GW in Gaussian Bloch orbitals for solids",
 * arXiv 2206.07660.  The four calls follow Algorithm 1 and the static
 * exchange of Eq. 22; citations per function below.  All arithmetic is complex FP64.
 *
 * Conventions
 *   - gw_c128 is layout-compatible with C99 `double complex`, std::complex<double>, cuDoubleComplex,
 *     torch.complex128.  All arrays are dense, row-major, 16-byte aligned.
 *   - "device" pointers are CUDA global memory of the current device; the caller owns every buffer,
 *     the library allocates nothing on the four hot calls, keeps no state between calls (apart from the cached
 *     address of the driver's tensor-map encoder, a process-wide constant) and never
 *     frees caller memory.  Inputs are const and unmodified; outputs are fully overwritten.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  The calls only
 *     enqueue work; they never synchronise the host.
 *   - k-mesh: Γ-centred nk1 x nk2 x nk3, nk = nk1*nk2*nk3, k = (i1*nk2+i2)*nk3+i3,
 *     k±q and −k component-wise modulo (momentum conservation).
 *   - q sharding ("first layer of parallelization"): a call works on the q-points
 *     q_begin <= q < q_end only; nq = q_end - q_begin.  P0t / Wt hold nq q-points (index q - q_begin);
 *     Sigma / K then hold this shard's partial sums, to be summed over shards by the caller
 *     (one all-reduce).  q_begin = 0, q_end = nk is the single-GPU case.
 *   - Preconditions (documented, not "fixed" silently): the τ grid is mirror symmetric,
 *     τ[ntau-1-t] = β − τ[t], so that G(−τ_t) = −G(β−τ_t) = −G[ntau-1-t] (Eq. 28b);
 *     I − P̃0(q,iΩ) is Hermitian positive definite (true for time-reversal symmetric inputs; the paper
 *     solves Eq. 29 with a Cholesky solver).  A non-positive pivot is reported through
 *     `info`, never by abort.
 *   - Return value: 0 = GW_OK; negative = caller error (GW_E*); positive = cudaError_t of a failed
 *     launch.  No C++ exception crosses this boundary.
 */
#ifndef GW_B200_H
#define GW_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } gw_c128;

enum {
  GW_OK = 0,
  GW_EINVAL = -1,   /* null / misaligned pointer, non-positive size, bad q range */
  GW_ENOMEM = -2,   /* workspace too small */
  GW_EARCH = -3,    /* current device is not sm_100 */
  GW_ESHAPE = -4,   /* size outside what the kernels support; checked before anything is launched and before the workspace
                       check (gw_workspace_bytes returns 0 for such a problem):
                         nao > 64;  ntau > 200 or nw > 200 (the paper's range is N_tau = 10-200);
                         nw > ntau (stage 2 keeps the frequency-domain intermediate in the first nw slices of the Wt buffer);
                         naux > 896 (stage 1: panel columns = 2 CTAs x 2 column passes x 224; the paper's N_aux/N_orb = 3-10,
                         PAPER.md:96, gives naux <= 640 at nao = 64) */
  GW_ENOBRACKET = -6, /* gw_find_mu only: N_e(mu) did not bracket the target after 60 widenings of [mu_lo, mu_hi] */
  GW_ESTATIC = -7,  /* gw_hartree_static only: naux > GW_STATIC_MAX_NAUX, the problem does not fit the library's static scratch */
  GW_ENOTPD = -5    /* gw_sigma_iteration_host only: a Cholesky factorisation of I - P0(q, iOmega_n) met a non-positive pivot
                       (the device calls report that through `info` instead); Sigma / Wt are then not meaningful */
};

typedef struct {
  int32_t nk1, nk2, nk3;   /* k-mesh */
  int32_t nao;             /* N_orb */
  int32_t naux;            /* N_aux */
  int32_t ntau;            /* N_tau */
  int32_t nw;              /* N_omega: bosonic Matsubara sampling points */
  int32_t spin_deg;        /* s of the spin sum in Eq. 28b: 2 = closed shell, 1 = one spin channel */
  int32_t q_begin, q_end;  /* q shard [q_begin, q_end) */
  double beta;             /* inverse temperature (informational; the grids enter through T_wt/T_tw) */
  const gw_c128 *V;        /* device [nk][nk][naux][nao][nao]: V^{k1 k2}_{ij}(Q), Eq. 6-7; or a q-slab (v_layout) */
  const gw_c128 *T_wt;     /* device [nw][ntau]: bosonic τ→iΩ transform matrix, Eq. 28a */
  const gw_c128 *T_tw;     /* device [ntau][nw]: bosonic iΩ→τ transform matrix, Eq. 30 */
  void *work;              /* device scratch shared by the four calls (L2-resident intermediates, solver copies), */
  size_t work_bytes;       /*   at least gw_workspace_bytes(p) bytes, 256-byte aligned; contents are don't-care    */
  int32_t symmetry;        /* 0 = evaluate Algorithm 1 literally (default); GW_SYM_TR = the caller asserts time-reversal   */
                           /*   symmetric inputs (see GW_SYM_TR below)                                                     */
  int32_t ns;              /* spin blocks of G: 0 or 1 = one; 2 = two collinear channels (spin-polarised, e.g. */
                           /*   the paper's AFM MnO); 4 = two-component (all sigma sigma' blocks) — "Spin blocks" below  */
  int32_t v_layout;        /* GW_V_FULL (0) or GW_V_QSLAB: how p->V is laid out — see "V layouts" below                      */
  int32_t reserved;        /* must be 0                                                                                    */
} gw_problem;

/* Spin blocks.  The spin index is the LEADING index of G, Sigma ([ns][ntau][nk][nao][nao]) and gamma, K ([ns][nk][nao][nao]).
 *   ns = 2 : collinear channels G^{sigma sigma}, sigma = up, down (no spin-orbit coupling), in that order.
 *   ns = 4 : two-component, all blocks G^{sigma sigma'} in the order uu, ud, du, dd ("H0 exhibits a spin dependence with non-zero
 *            off-diagonal spin components ... spin-orbit coupling").
 *   gw_polarization : P0t = -(spin_deg/N_k) Σ_{sigma sigma'} Σ_k V G^{sigma sigma'}(k+q,tau) V G^{sigma' sigma}(k,-tau)   (Eq. 28b as printed; with
 *                     ns = 2 only sigma = sigma' is non-zero); the spin sum runs inside the stage-1 k loop.  Pass spin_deg = 1 with ns > 1; two
 *                     identical collinear channels with spin_deg = 1 equal one channel with spin_deg = 2.
 *   gw_selfenergy, gw_exchange : one Sigma^{sigma sigma'} / K^{sigma sigma'} per block from G^{sigma sigma'} / gamma^{sigma sigma'} and the common Wt
 *                     (Eq. 31, and Eq. 22 which prints the general K_{i sigma, j sigma'}).
 *   gw_hartree      : J (spin independent, [nk][nao][nao]) from the spin-diagonal blocks of gamma (Eq. 20's Σ_sigma1), times spin_deg.
 * P0t, Wt, V and the transforms carry no spin index. */

/* V layouts.
 *   GW_V_FULL  : p->V is the whole tensor [nk][nk][naux][nao][nao] (block (k1,k2) at index k1*nk + k2).
 *   GW_V_QSLAB : p->V holds only the blocks the q shard [q_begin, q_end) touches, [nq][nk][2][naux][nao][nao]:
 *                  slot (q - q_begin, k, 0) = V[k][k+q],   slot (q - q_begin, k, 1) = V[k+q][k].
 *                Stage 1 reads V[k][k+q] and V[k+q][k]; stages 3 and 4 read V[k][k-q] = slot (q, k-q, 1) and V[k-q][k] = slot (q, k-q, 0):
 *                the same 2 nk blocks per q serve every stage, which is what lets V be streamed through HBM one q-slab at a time
 *                (gw_sigma_iteration_stream; the paper reads V "a k-batch at a time").  gw_hartree needs the
 *                diagonal blocks V[k][k], i.e. a shard that contains q = 0 (else GW_EINVAL). */
enum { GW_V_FULL = 0, GW_V_QSLAB = 1 };

/* gw_problem.symmetry flag.  Time reversal: G[t][−k] = conj(G[t][k]) and V[−k1][−k2] = conj(V[k1][k2]) element-wise (the same
 * property that makes I − P̃0(iΩ) Hermitian for the Cholesky solve; the paper exploits k ↔ −k too), together with
 * V[k1][k2][Q][i][j] = conj(V[k2][k1][Q][j][i]) and Hermitian G[t][k] (true of the BASELINE.json inputs and of any physical G).  Then
 * P̃0^q(τ) is Hermitian,
 * P̃0^q(β−τ) = P̃0^q(τ) and Σ^{−k}(τ) = conj Σ^{k}(τ), and the library evaluates only the irreducible half and copies the rest:
 *   gw_polarization : tau nodes t <= ntau-1-t are computed, P0t[ntau-1-t] is a copy of P0t[t]; for the full q range and
 *                     nk <= 128 also only q <= −q, and P0t[t][−q] = transpose(P0t[t][q])  (216 -> 112 q points);
 *                     of each Q panel only the column tiles up to its diagonal block are computed, the rest is the conjugate mirror;
 *   gw_selfenergy   : k <= −k are computed, Sigma[t][−k] = conj(Sigma[t][k])  (only for the full q range and nk <= 128);
 * the other calls ignore the flag; with ns = 4 the flag is refused (GW_EINVAL: the relations above are those of a spin-diagonal G).
 * Computed elements are bit-identical to the literal evaluation.  If the inputs do not
 * have the symmetry the copied elements are wrong — nothing checks it. */
enum { GW_SYM_TR = 1 };

/* Stage 1 — Eq. 28b, Algorithm 1 first k loop:
 *   P0t[t][q-q_begin][Q][Q'] = -(s/N_k) Σ_k Σ_abcd V[k][k+q][Q][d][a] G[t][k+q][a][b] V[k+q][k][Q'][b][c] G[ntau-1-t][k][c][d]
 * (the printed "-1/N_k" is the antiperiodicity sign of G(−τ); reading R1).
 *   G   : device [ntau][nk][nao][nao]      in   ([ns][ntau][nk][nao][nao] with ns = 2, summed over the channel)
 *   P0t : device [ntau][nq][naux][naux]    out */
int gw_polarization(const gw_problem *p, const gw_c128 *G, gw_c128 *P0t, void *stream);

/* Stage 2 — Eq. 28a, 29, 30, Algorithm 1 middle part, for every q of the shard:
 *   P0w[n] = Σ_t T_wt[n][t] P0t[t];   Ww[n] = (I − P0w[n])^-1 P0w[n]  (Cholesky);   Wt[t] = Σ_n T_tw[t][n] Ww[n]
 *   P0t : device [ntau][nq][naux][naux]    in
 *   Wt  : device [ntau][nq][naux][naux]    out; may alias P0t (then P0t is overwritten)
 *   info: device int32[2], 8-byte aligned, or NULL.  Set to {-1,-1} on success, else {q, n} of ONE failing factorisation:
 *         the one with the smallest n, then the smallest q (a single 64-bit atomic minimum, so the pair is never mixed
 *         between two failing matrices and the report is deterministic). */
int gw_screened_interaction(const gw_problem *p, const gw_c128 *P0t, gw_c128 *Wt, int32_t *info, void *stream);

/* Stage 2 plus the integrand of the dynamical part of the GW Luttinger-Ward functional, Eq. 37:
 *   phi[n][q-q_begin] = tr{ ln[I − P0w[n][q]] + P0w[n][q] }      (real; ln det from the Cholesky diagonal of stage 2b)
 * so that  Φ̃_GW = (1/2N_k) Σ_q (1/β) Σ_n phi[n][q]; the Matsubara sum over the sparse grid needs the caller's
 * quadrature weights (the paper gives none), so the summand is returned, not the sum.
 *   phi : device double [nw][nq]   out (8-byte aligned, required).  Other arguments and errors as above;
 *   an entry whose factorisation failed (see info) is unspecified. */
int gw_screened_interaction_phi(const gw_problem *p, const gw_c128 *P0t, gw_c128 *Wt, int32_t *info, double *phi, void *stream);

/* Phi~_GW itself, Eq. 37, from the summand above and the caller's quadrature weights of the Matsubara sum
 * (the paper prints none for its sparse grid; reading R18; on an n >= 0 grid the weights carry the factor 2 of
 * the mirror images n < 0):
 *   *out = (1/(2 N_k beta)) Σ_q Σ_n w[n] phi[n][q]          (a q shard yields its partial sum: add the shards)
 *   nk = N_k of the whole mesh;  w : device double [nw];  phi : device double [nw][nq];  out : device double.  Fixed summation order. */
int gw_phi_gw(int32_t nk, int32_t nq, int32_t nw, double beta, const double *w, const double *phi, double *out, void *stream);

/* Generic imaginary-axis grid transform — the kernel of Eq. 28a / Eq. 30 exposed for the next workflow step, the fermionic
 * τ→iω_n transform of Σ̃ (Eq. 13; Fig. 4 step after the hot path):
 *   Y[o][m] = Σ_i T[o][i] X[i][m],   o < n_out, i < n_in, m < len      (complex T; n_out, n_in <= 200)
 *   T : device [n_out][n_in];  X : device [n_in][len];  Y : device [n_out][len], may alias X (each column block is read
 *   completely before it is written).  Returns GW_EINVAL / GW_ESHAPE / GW_EARCH or a launch error. */
int gw_transform(int32_t n_out, int32_t n_in, const gw_c128 *T, const gw_c128 *X, gw_c128 *Y, size_t len, void *stream);

/* Stage 3 — Eq. 31, Algorithm 1 second k loop:
 *   Sigma[t][k][i][j] = -(1/N_k) Σ_{q in shard} Σ_QQ' Σ_ab V[k][k-q][Q][i][a] G[t][k-q][a][b] Wt[t][q-q_begin][Q][Q'] V[k-q][k][Q'][b][j]
 *   G     : device [ntau][nk][nao][nao]    in
 *   Wt    : device [ntau][nq][naux][naux]  in
 *   Sigma : device [ntau][nk][nao][nao]    out */
int gw_selfenergy(const gw_problem *p, const gw_c128 *G, const gw_c128 *Wt, gw_c128 *Sigma, void *stream);

/* Stage 4 — static exchange, Eq. 22:
 *   K[k][i][j] = -(1/N_k) Σ_{q in shard, k'=k-q} Σ_Q Σ_ab V[k][k'][Q][i][a] gamma[k'][a][b] V[k'][k][Q][b][j]
 *   gamma : device [nk][nao][nao]  in (density matrix γ^k = −G^k(β⁻))
 *   K     : device [nk][nao][nao]  out */
int gw_exchange(const gw_problem *p, const gw_c128 *gamma, gw_c128 *K, void *stream);

/* Scratch (p->work) needed by the four calls for this problem: the maximum over the stages (bytes; host-side
 * arithmetic only, p->work / p->work_bytes are ignored). */
size_t gw_workspace_bytes(const gw_problem *p);

/* Whole iteration with HOST buffers (the end-to-end path timed as `e2e` by bench.py): uploads V, G, gamma,
 * T_wt, T_tw, runs the four stages above on `stream`, downloads Sigma and K, and synchronises the stream.
 * All pointers here (including p->V, p->T_wt, p->T_tw) are HOST memory (pinned memory makes the copies
 * asynchronous).  Device memory is allocated and freed inside the call.  Optional outputs may be NULL:
 *   P0t_out, Wt_out : host [ntau][nq][naux][naux];  stage_ms: host float[6] = H2D, stage 1..4, D2H times (ms).
 * Returns GW_ENOTPD if stage 2 reported a non-positive pivot (the outputs are still copied back), else as the device calls. */
int gw_sigma_iteration_host(const gw_problem *p, const gw_c128 *G, const gw_c128 *gamma, gw_c128 *Sigma, gw_c128 *K,
                            gw_c128 *P0t_out, gw_c128 *Wt_out, float *stage_ms, void *stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Loop closure: the remaining steps of one scGW iteration (Fig. 4).  The fermionic tau <-> i omega_n
 * transforms of Eq. 13 / 14 are gw_transform with the caller's fermionic matrices; G(tau = beta^-)
 * (gamma = -G(beta^-)) is gw_transform with a 1 x ntau evaluation vector.  Grids are inputs (reading R6).
 * ------------------------------------------------------------------------------------------------------------------ */

/* Hartree term, Eq. 20 (the label "(19)" is lost in the text):
 *   J[k][i][j] = (s/N_k) Σ_k' Σ_ab Σ_Q V[k][k][Q][i][j] gamma[k'][a][b] V[k'][k'][Q][b][a]        (s = spin_deg: the sum over sigma_1)
 *   gamma : device [nk][nao][nao] in;  J : device [nk][nao][nao] out.  Reads only the diagonal blocks V[k][k]; uses p->work
 *   (any q shard: J does not depend on q_begin / q_end). */
int gw_hartree(const gw_problem *p, const gw_c128 *gamma, gw_c128 *J, void *stream);

/* The same Hartree term for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): gw_hartree with its one intermediate, rho[Q] = Σ_k' Σ_ab gamma[k'][a][b] V[k'][k'][Q][b][a],
 * kept in a static device array inside the library instead of p->work.
 *   Arguments, layouts and result as gw_hartree (bit-identical: same sums, same order); p->work / p->work_bytes are ignored
 *   and may be NULL / 0.  The call allocates nothing (no cudaMalloc, cudaFree or allocating library routine); its only set-up
 *   is one symbol-address lookup per device, on the first call with that device current.
 *   Limit: naux <= GW_STATIC_MAX_NAUX (= gw_static_max_naux()); beyond it the call returns GW_ESTATIC and launches nothing.
 *   Cost: GW_STATIC_MAX_NAUX * 16 bytes = 8 KB of device memory on every GPU that loads the library, held until exit.
 *   Sharing: every call on a device uses the same array.  Nothing in it has to start at zero (each entry is written before it
 *   is read within a call), but calls that overlap on the GPU — different streams without an ordering between them, or two
 *   host threads on one device — race on it: order them (same stream, or an event). */
#define GW_STATIC_MAX_NAUX 512
int gw_hartree_static(const gw_problem *p, const gw_c128 *gamma, gw_c128 *J, void *stream);
int gw_static_max_naux(void);

/* Dyson equation, Eq. 16, for every (n, k):
 *   G_w[n][k] = [ (i omega[n] + mu) S[k] − F[k] − Sigma_w[n][k] ]^-1        ("matrix inversion in spin-orbital space")
 *   omega : device double [nwf] (fermionic Matsubara frequencies);  S, F : device [nk][nao][nao] (overlap; F = H0 + Sigma_inf,
 *   Eq. 17-18);  Sigma_w : device [nwf][nk][nao][nao] or NULL;  G_w : device [nwf][nk][nao][nao] out (must not alias Sigma_w's
 *   other matrices; the same matrix is read completely before it is written, so G_w == Sigma_w is allowed).
 *   In-kernel Gauss-Jordan elimination with partial pivoting, one CTA per matrix; nao <= 64 (GW_ESHAPE).
 *   info : device int32[2], 8-byte aligned, or NULL: {-1,-1}, else {n, k} of one singular matrix (smallest k, then n). */
int gw_dyson_update(int32_t nk, int32_t nao, int32_t nwf, const double *omega, double mu, const gw_c128 *S, const gw_c128 *F,
                    const gw_c128 *Sigma_w, gw_c128 *G_w, int32_t *info, void *stream);

/* Electron count, Eq. 15:  *ne = (s/N_k) Σ_k tr[gamma^k S^k],  gamma^k = −Σ_n t_beta[n] G_w[n][k]
 *   t_beta : device [nwf] (evaluation vector G(beta^-) = Σ_n t_beta[n] G(i omega_n));  partial : device scratch [nk];
 *   ne : device double out.  Fixed summation order (deterministic). */
int gw_electron_count(int32_t nk, int32_t nao, int32_t nwf, int32_t spin_deg, const gw_c128 *t_beta, const gw_c128 *S,
                      const gw_c128 *G_w, gw_c128 *partial, double *ne, void *stream);

/* Chemical potential (Fig. 4 step 3: mu is adjusted until N_e is right to 1e-9): bisection on N_e(mu) of
 * Eq. 15-16 (reading R16): widen [mu_lo, mu_hi] by its own width (<= 60 times) until it brackets n_target, halve it
 * until its width <= mu_tol (<= 200 times), return the midpoint and N_e there; G_w then holds G(i omega_n) at that mu.
 * Every N_e evaluation is one gw_dyson_update + gw_electron_count on `stream`; this call SYNCHRONISES the stream after each
 * (it reads N_e back), unlike the calls above.  mu_out, ne_out, n_eval (optional) are HOST pointers.
 * Returns GW_OK, GW_ENOTPD if a matrix was singular, GW_ENOBRACKET when no bracket was found. */
int gw_find_mu(int32_t nk, int32_t nao, int32_t nwf, int32_t spin_deg, const double *omega, const gw_c128 *t_beta, const gw_c128 *S,
               const gw_c128 *F, const gw_c128 *Sigma_w, double n_target, double mu_lo, double mu_hi, double mu_tol, gw_c128 *G_w,
               gw_c128 *partial, double *ne_dev, double *mu_out, double *ne_out, int32_t *n_eval, void *stream);

/* Y[i] = (a_re + i a_im) X[i] + (b_re + i b_im) Y[i], i < n (damping of two iterates, F = H0 + J + K, gamma = −G(beta^-)).
 * Y is not read when b == 0.  X, Y : device, may be equal. */
int gw_axpby(size_t n, double a_re, double a_im, const gw_c128 *X, double b_re, double b_im, gw_c128 *Y, void *stream);

/* Whole iteration with V OUT OF CORE (the paper keeps V on disk / in host memory and reads it a k-batch at a
 * time): as gw_sigma_iteration_host (all pointers HOST memory, p->V in the GW_V_FULL layout, pinned memory
 * recommended), but V never resides in HBM as a whole: the q shard is processed in slabs of nqs q-points; the 2 nk V blocks of each
 * q are gathered into one of TWO device slab buffers (GW_V_QSLAB layout, together at most v_budget_bytes) by cudaMemcpyAsync on an
 * internal copy stream while the previous slab computes; stages 1-4 run per slab and Sigma / K continue their q sums across slabs in
 * the same order as the resident evaluation (bit-identical results).
 *   stats : host float[4] or NULL = {total ms, GB copied host->device, number of slabs, q-points per slab}
 * Returns GW_ENOMEM if v_budget_bytes does not hold two slabs of one q-point, GW_ENOTPD / launch errors as the host call. */
int gw_sigma_iteration_stream(const gw_problem *p, const gw_c128 *G, const gw_c128 *gamma, gw_c128 *Sigma, gw_c128 *K,
                              size_t v_budget_bytes, float *stats, void *stream);

/* Executed FP64 flops of the last configuration of each stage kernel for `p` (what the kernels actually
 * issue, padding and recomputation included; 2 flops per real FMA).  out: host double[4] = stage 1..4. */
int gw_executed_flops(const gw_problem *p, double *out);

/* Number of kernels the four hot calls launch for `p` (host arithmetic; used for bench.py's gpu_launches). */
int gw_launch_count(const gw_problem *p);

/* Register-resident DMMA.8x8x4 loop on all SMs for about `ms` milliseconds; returns sustained FP64 TFLOP/s
 * in *tflops (the "measured FP64 peak" the roofline divides by; MEASURED_PEAKS.json has no FP64 entry). */
int gw_fp64_peak(double ms, double *tflops, void *stream);

/* The same measurement with a register-resident plain DFMA loop (no tensor-core instruction).  The roofline denominator of
 * bench.py is the larger of the two. */
int gw_fp64_peak_dfma(double ms, double *tflops, void *stream);

/* Inner loop of the main GEMMs alone (operands resident in shared memory, 8 warps per CTA, one CTA per SM) for about `ms` milliseconds, for
 * the three ways of forming a complex 8x8x4 tile product on DMMA.8x8x4 that profiles/r02_3m_vs_4m.md compares:
 *   mode 0: 4M (four real DMMAs);  mode 1: 3M Karatsuba with the operand sums formed by DADD in registers (what the kernels run);
 *   mode 2: 3M with the B operand's sums pre-formed in shared memory.
 * *tflops = ALGORITHMIC TFLOP/s, 8 flops per complex multiply-add. */
int gw_complex_mma_probe(int32_t mode, double ms, double *tflops, void *stream);

/* Diagnostic: which warps share an FP64 tensor pipe.  One CTA of 16 warps per SM; only the warps whose bit is set in warp_mask run a
 * register-resident DMMA.8x8x4 loop (12 independent accumulators), the others exit.  *tflops = executed TFLOP/s over the chip.
 * On B200 every SM sub-partition (warp id mod 4) has its own pipe: mask 0x000F (one warp on each) reaches the chip's peak, mask
 * 0x1111 (four warps on one sub-partition) a quarter of it (profiles/r02_fp64_subcores.md).  warp_mask != 0, bits 0..15. */
int gw_fp64_subcore_probe(uint32_t warp_mask, double *tflops, void *stream);

const char *gw_strerror(int code);
int gw_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GW_B200_H */
