// gw_static.cu — gw_hartree_static: the Hartree term (Eq. 20) for callers that cannot allocate device
// memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// gw_hartree (gw_loop.cu) keeps its one intermediate, rho[Q] = Σ_k' Σ_ab gamma[k'][a][b] V[k'][k'][Q][b][a], in the caller's
// workspace p->work.  This variant keeps it in a file-scope __device__ array of GW_STATIC_MAX_NAUX complex numbers (8 KB)
// that every GPU which loads the library holds until the process exits; p->work is not read.  The call allocates nothing:
// no cudaMalloc / cudaFree, no allocating library routine; set-up is one cudaGetSymbolAddress per device.
//
// The two kernels below are the kernels of gw_hartree with the same sums in the same order (the result is bit-identical).
// Sharing: every call on a device uses the same array.  Nothing in it has to start at zero (each rho[Q], Q < naux, is written
// by the first kernel before the second one reads it; entries beyond naux keep an earlier call's contents and are never
// read), but two calls that overlap on the GPU (different streams, no ordering between them) race on it.
#include <mutex>
#include "gw_common.cuh"

namespace gst {

constexpr int NT = 256;
constexpr int MAX_DEVICES = 64;

// The scratch.  In host code this name is a host-side stand-in, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress (rho_address below).
static __device__ __align__(256) c128 g_rho[GW_STATIC_MAX_NAUX];

// fixed-order tree reduction over the CTA (as lp::block_sum of gw_loop.cu); result valid in thread 0
__device__ __forceinline__ c128 block_sum(c128 v, c128 *red) {
  red[threadIdx.x] = v;
  __syncthreads();
  for (int s = NT / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) { red[threadIdx.x].x += red[threadIdx.x + s].x; red[threadIdx.x].y += red[threadIdx.x + s].y; }
    __syncthreads();
  }
  return red[0];
}

// rho[Q] = Σ_sigma Σ_k' Σ_ab gamma[sigma][k'][a][b] V[k'][k'][Q][b][a]      (one CTA per Q)
__global__ void __launch_bounds__(NT) hartree_rho_static_kernel(const GwDims d, int ql0, const c128 *__restrict__ V, const c128 *__restrict__ gamma,
                                                                c128 *__restrict__ rho) {
  __shared__ c128 red[NT];
  const int Q = blockIdx.x, nao = d.nao, n2 = nao * nao;
  c128 acc = make_double2(0.0, 0.0);
  for (int sg = 0; sg < d.ns; sg++) {                      // the spin-diagonal blocks
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

// J[k][i][j] = (s/N_k) Σ_Q V[k][k][Q][i][j] rho[Q]
__global__ void __launch_bounds__(NT) hartree_j_static_kernel(const GwDims d, int ql0, const c128 *__restrict__ V, const c128 *__restrict__ rho,
                                                              c128 *__restrict__ J) {
  const int k = blockIdx.y, n2 = d.nao * d.nao, e = blockIdx.x * NT + threadIdx.x;
  if (e >= n2) return;
  const c128 *Vk = V + gw_vfwd(d, ql0, k, k) * d.naux * n2 + e;
  c128 acc = make_double2(0.0, 0.0);
  for (int Q = 0; Q < d.naux; Q++) cfma(acc, Vk[(size_t)Q * n2], rho[Q]);
  const double pref = (double)d.s / (double)d.nk;
  J[(size_t)k * n2 + e] = make_double2(pref * acc.x, pref * acc.y);
}

// Device address of g_rho on the current device, looked up once per device (with that device current) and kept.
static int rho_address(c128 **out) {
  static std::mutex mu;
  static c128 *addr[MAX_DEVICES];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return (int)e; }
  if (dev < 0 || dev >= MAX_DEVICES) return GW_EINVAL;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void *ptr = 0;
    e = cudaGetSymbolAddress(&ptr, g_rho);
    if (e != cudaSuccess) { cudaGetLastError(); return (int)e; }
    if (!ptr || (((uintptr_t)ptr) & 255)) return GW_EINVAL;
    addr[dev] = (c128 *)ptr;
  }
  *out = addr[dev];
  return GW_OK;
}

}  // namespace gst

extern "C" int gw_static_max_naux(void) { return GW_STATIC_MAX_NAUX; }

extern "C" int gw_hartree_static(const gw_problem *p, const gw_c128 *gamma, gw_c128 *J, void *stream) {
  // the argument checks of gw_hartree (gw_api.cu: check_problem), without the workspace
  if (!p) return GW_EINVAL;
  if (p->nk1 <= 0 || p->nk2 <= 0 || p->nk3 <= 0 || p->nao <= 0 || p->naux <= 0 || p->ntau <= 0 || p->nw <= 0) return GW_EINVAL;
  if (p->spin_deg != 1 && p->spin_deg != 2) return GW_EINVAL;
  if ((p->symmetry & ~GW_SYM_TR) || p->reserved || (p->ns != 0 && p->ns != 1 && p->ns != 2 && p->ns != 4) ||
      (p->v_layout != GW_V_FULL && p->v_layout != GW_V_QSLAB)) return GW_EINVAL;
  if (p->ns == 4 && (p->symmetry & GW_SYM_TR)) return GW_EINVAL;
  const int64_t nk = (int64_t)p->nk1 * p->nk2 * p->nk3;
  if (nk > (1 << 20) || p->q_begin < 0 || p->q_end > nk || p->q_begin >= p->q_end) return GW_EINVAL;
  if (!p->V || (((uintptr_t)p->V) & 15) || !gamma || (((uintptr_t)gamma) & 15) || !J || (((uintptr_t)J) & 15)) return GW_EINVAL;
  if (p->nao > GW_MAX_NAO || p->ntau > GW_MAX_NTAU || p->nw > GW_MAX_NTAU || p->nw > p->ntau || p->naux > GW_MAX_NAUX) return GW_ESHAPE;
  if (p->naux > GW_STATIC_MAX_NAUX) return GW_ESTATIC;      // beyond the static scratch: use gw_hartree with a workspace
  const GwDims d = gw_dims(p);
  if (d.vq && !(d.q0 <= 0 && 0 < d.q0 + d.nq)) return GW_EINVAL;   // a q-slab without q = 0 holds no diagonal blocks
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
    cudaGetLastError();
    return GW_EARCH;
  }
  if (major != 10) return GW_EARCH;
  c128 *rho = 0;
  const int rc = gst::rho_address(&rho);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int ql0 = -d.q0, n2 = d.nao * d.nao;
  gst::hartree_rho_static_kernel<<<d.naux, gst::NT, 0, st>>>(d, ql0, (const c128 *)p->V, (const c128 *)gamma, rho);
  gst::hartree_j_static_kernel<<<dim3((n2 + gst::NT - 1) / gst::NT, d.nk), gst::NT, 0, st>>>(d, ql0, (const c128 *)p->V, rho, (c128 *)J);
  return (int)cudaGetLastError();
}
