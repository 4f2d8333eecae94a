"""ctypes marshalling for include/gw.h.  Same names as the C ABI."""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgw_b200.so")
_lib = None


class GWError(RuntimeError):
    pass


GW_SYM_TR = 1   # gw_problem.symmetry flag (include/gw.h)
GW_V_FULL, GW_V_QSLAB = 0, 1   # gw_problem.v_layout


class _CProblem(ctypes.Structure):
    _fields_ = [("nk1", ctypes.c_int32), ("nk2", ctypes.c_int32), ("nk3", ctypes.c_int32),
                ("nao", ctypes.c_int32), ("naux", ctypes.c_int32), ("ntau", ctypes.c_int32), ("nw", ctypes.c_int32),
                ("spin_deg", ctypes.c_int32), ("q_begin", ctypes.c_int32), ("q_end", ctypes.c_int32),
                ("beta", ctypes.c_double),
                ("V", ctypes.c_void_p), ("T_wt", ctypes.c_void_p), ("T_tw", ctypes.c_void_p),
                ("work", ctypes.c_void_p), ("work_bytes", ctypes.c_size_t),
                ("symmetry", ctypes.c_int32), ("ns", ctypes.c_int32), ("v_layout", ctypes.c_int32), ("reserved", ctypes.c_int32)]


def lib_path():
    return _SO


def lib():
    """Load libgw_b200.so; fails loudly if it has not been built (python -m paper_2206_07660_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise GWError(f"{_SO} is missing: build it with `python paper_2206_07660_b200/build.py` "
                          "(there is no CPU fallback)")
        L = ctypes.CDLL(_SO)
        P = ctypes.POINTER(_CProblem)
        vp, sz = ctypes.c_void_p, ctypes.c_size_t
        L.gw_polarization.argtypes = [P, vp, vp, vp]
        L.gw_screened_interaction.argtypes = [P, vp, vp, vp, vp]
        L.gw_screened_interaction_phi.argtypes = [P, vp, vp, vp, vp, vp]
        L.gw_selfenergy.argtypes = [P, vp, vp, vp, vp]
        L.gw_transform.argtypes = [ctypes.c_int32, ctypes.c_int32, vp, vp, vp, ctypes.c_size_t, vp]
        L.gw_exchange.argtypes = [P, vp, vp, vp]
        L.gw_workspace_bytes.argtypes = [P]
        L.gw_workspace_bytes.restype = sz
        L.gw_sigma_iteration_host.argtypes = [P, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gw_sigma_iteration_stream.argtypes = [P, vp, vp, vp, vp, sz, vp, vp]
        L.gw_executed_flops.argtypes = [P, ctypes.POINTER(ctypes.c_double)]
        L.gw_launch_count.argtypes = [P]
        L.gw_fp64_peak.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
        L.gw_fp64_peak_dfma.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
        i32, dbl = ctypes.c_int32, ctypes.c_double
        L.gw_hartree.argtypes = [P, vp, vp, vp]
        L.gw_dyson_update.argtypes = [i32, i32, i32, vp, dbl, vp, vp, vp, vp, vp, vp]
        L.gw_electron_count.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, vp]
        L.gw_find_mu.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, dbl, dbl, dbl, dbl, vp, vp, vp,
                                 ctypes.POINTER(dbl), ctypes.POINTER(dbl), ctypes.POINTER(i32), vp]
        L.gw_axpby.argtypes = [sz, dbl, dbl, vp, dbl, dbl, vp, vp]
        L.gw_phi_gw.argtypes = [i32, i32, i32, dbl, vp, vp, vp, vp]
        L.gw_complex_mma_probe.argtypes = [i32, dbl, ctypes.POINTER(dbl), vp]
        L.gw_strerror.argtypes = [ctypes.c_int]
        L.gw_strerror.restype = ctypes.c_char_p
        for n in ("gw_polarization", "gw_screened_interaction", "gw_screened_interaction_phi", "gw_transform", "gw_selfenergy", "gw_exchange",
                  "gw_sigma_iteration_host", "gw_executed_flops", "gw_launch_count", "gw_fp64_peak", "gw_fp64_peak_dfma", "gw_version",
                  "gw_hartree", "gw_hartree_static", "gw_static_max_naux", "gw_dyson_update", "gw_electron_count", "gw_find_mu", "gw_axpby", "gw_sigma_iteration_stream", "gw_phi_gw", "gw_complex_mma_probe", "gw_fp64_subcore_probe"):
            getattr(L, n).restype = ctypes.c_int
        _lib = L
    return _lib


def gw_strerror(code):
    return lib().gw_strerror(int(code)).decode()


def gw_version():
    return int(lib().gw_version())


def _check(rc, what):
    if rc != 0:
        raise GWError(f"{what} failed: {gw_strerror(rc)} (code {rc})")


def _dev(t, shape, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise GWError(f"{name}: need a contiguous CUDA complex128 tensor")
    if tuple(t.shape) != tuple(shape):
        raise GWError(f"{name}: shape {tuple(t.shape)} != expected {tuple(shape)}")
    return ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class GWProblem:
    """The POD problem descriptor of gw.h plus the tensors it points to (kept alive here).

    V, T_wt, T_tw: CUDA complex128 tensors for the device calls, or CPU tensors for gw_sigma_iteration_host."""

    def __init__(self, mesh, nao, naux, ntau, nw, beta, V, T_wt, T_tw, spin_deg=2, q_begin=0, q_end=None, symmetry=0, ns=1, v_layout=GW_V_FULL):
        self.symmetry = int(symmetry)      # 0 = literal Algorithm 1; GW_SYM_TR = time-reversal symmetric inputs (gw.h)
        self.ns = int(ns) if int(ns) in (2, 4) else 1   # spin blocks: G, Sigma [ns][ntau][nk][nao][nao], gamma, K [ns][nk][nao][nao] when ns > 1
        self.v_layout = int(v_layout)      # GW_V_FULL: V [nk][nk][naux][nao][nao]; GW_V_QSLAB: V [nq][nk][2][naux][nao][nao] (gw.h)
        self.mesh = tuple(int(m) for m in mesh)
        self.nk = self.mesh[0] * self.mesh[1] * self.mesh[2]
        self.nao, self.naux, self.ntau, self.nw = int(nao), int(naux), int(ntau), int(nw)
        self.beta, self.spin_deg = float(beta), int(spin_deg)
        self.q_begin = int(q_begin)
        self.q_end = self.nk if q_end is None else int(q_end)
        self.nq = self.q_end - self.q_begin
        self.V, self.T_wt, self.T_tw = V, T_wt, T_tw
        vshape = (self.nk, self.nk, naux, nao, nao) if self.v_layout == GW_V_FULL else (self.nq, self.nk, 2, naux, nao, nao)
        for name, t, shape in (("V", V, vshape), ("T_wt", T_wt, (nw, ntau)), ("T_tw", T_tw, (ntau, nw))):
            if t.dtype != torch.complex128 or not t.is_contiguous() or tuple(t.shape) != shape:
                raise GWError(f"{name}: need contiguous complex128 of shape {shape}, got {tuple(t.shape)} {t.dtype}")
        self.c = _CProblem(self.mesh[0], self.mesh[1], self.mesh[2], self.nao, self.naux, self.ntau, self.nw,
                           self.spin_deg, self.q_begin, self.q_end, self.beta,
                           V.data_ptr(), T_wt.data_ptr(), T_tw.data_ptr(), None, 0, self.symmetry, self.ns, self.v_layout, 0)
        self.work = None
        if V.is_cuda:
            self.set_work(torch.empty(int(lib().gw_workspace_bytes(ctypes.byref(self.c))), dtype=torch.uint8, device=V.device))

    def gshape(self):
        """shape of G and Sigma"""
        base = (self.ntau, self.nk, self.nao, self.nao)
        return (self.ns,) + base if self.ns > 1 else base

    def kshape(self):
        """shape of gamma and K"""
        base = (self.nk, self.nao, self.nao)
        return (self.ns,) + base if self.ns > 1 else base

    def set_work(self, work):
        """Attach the device workspace (uint8 CUDA tensor of at least gw_workspace_bytes bytes)."""
        self.work = work
        self.c.work = work.data_ptr()
        self.c.work_bytes = work.numel()

    @property
    def on_device(self):
        return self.V.is_cuda

    def shard(self, q_begin, q_end):
        if self.v_layout != GW_V_FULL:
            raise GWError("shard(): a q-slab problem is already a shard")
        return GWProblem(self.mesh, self.nao, self.naux, self.ntau, self.nw, self.beta, self.V, self.T_wt, self.T_tw,
                         self.spin_deg, q_begin, q_end, self.symmetry, self.ns)

    def ref(self):
        return ctypes.byref(self.c)


def gw_workspace_bytes(prob):
    return int(lib().gw_workspace_bytes(prob.ref()))


def gw_polarization(prob, G, P0t=None, stream=None):
    """Stage 1, Eq. 28b.  G [ntau][nk][nao][nao] -> P0t [ntau][nq][naux][naux]."""
    g = _dev(G, prob.gshape(), "G")
    if P0t is None:
        P0t = torch.empty((prob.ntau, prob.nq, prob.naux, prob.naux), dtype=torch.complex128, device=G.device)
    _check(lib().gw_polarization(prob.ref(), g, _dev(P0t, (prob.ntau, prob.nq, prob.naux, prob.naux), "P0t"),
                                 _stream(stream)), "gw_polarization")
    return P0t


def gw_screened_interaction(prob, P0t, Wt=None, info=None, stream=None):
    """Stage 2, Eq. 28a + 29 + 30.  Wt may alias P0t (pass Wt=P0t)."""
    shape = (prob.ntau, prob.nq, prob.naux, prob.naux)
    if Wt is None:
        Wt = torch.empty(shape, dtype=torch.complex128, device=P0t.device)
    if info is None:
        info = torch.empty(2, dtype=torch.int32, device=P0t.device)
    _check(lib().gw_screened_interaction(prob.ref(), _dev(P0t, shape, "P0t"), _dev(Wt, shape, "Wt"),
                                         ctypes.c_void_p(info.data_ptr()), _stream(stream)), "gw_screened_interaction")
    return Wt, info


def gw_screened_interaction_phi(prob, P0t, Wt=None, info=None, phi=None, stream=None):
    """Stage 2 plus phi[n][q] = tr{ln[I - P0w] + P0w}, the summand of Eq. 37."""
    shape = (prob.ntau, prob.nq, prob.naux, prob.naux)
    if Wt is None:
        Wt = torch.empty(shape, dtype=torch.complex128, device=P0t.device)
    if info is None:
        info = torch.empty(2, dtype=torch.int32, device=P0t.device)
    if phi is None:
        phi = torch.empty((prob.nw, prob.nq), dtype=torch.float64, device=P0t.device)
    if phi.dtype != torch.float64 or tuple(phi.shape) != (prob.nw, prob.nq) or not phi.is_contiguous():
        raise GWError("phi must be a contiguous float64 tensor of shape (nw, nq)")
    _check(lib().gw_screened_interaction_phi(prob.ref(), _dev(P0t, shape, "P0t"), _dev(Wt, shape, "Wt"),
                                             ctypes.c_void_p(info.data_ptr()), ctypes.c_void_p(phi.data_ptr()),
                                             _stream(stream)), "gw_screened_interaction_phi")
    return Wt, info, phi


def gw_phi_gw(prob, w, phi, stream=None):
    """Eq. 37: Phi~_GW = (1/(2 N_k beta)) sum_q sum_n w[n] phi[n][q] (1-element CUDA float64 tensor; a q shard gives its partial sum)."""
    out = torch.empty(1, dtype=torch.float64, device=phi.device)
    if tuple(phi.shape) != (prob.nw, prob.nq) or tuple(w.shape) != (prob.nw,):
        raise GWError("gw_phi_gw: need w [nw] and phi [nw][nq]")
    _check(lib().gw_phi_gw(prob.nk, prob.nq, prob.nw, prob.beta, _f64(w, "w"), _f64(phi, "phi"), _f64(out, "out"), _stream(stream)), "gw_phi_gw")
    return out


def gw_transform(T, X, Y=None, stream=None):
    """Y[o][...] = sum_i T[o][i] X[i][...] along the leading axis (Eq. 13 / 28a / 30); Y may be X when the shapes agree."""
    if T.dtype != torch.complex128 or X.dtype != torch.complex128 or not T.is_cuda or not X.is_cuda:
        raise GWError("gw_transform: need CUDA complex128 tensors")
    if not T.is_contiguous() or not X.is_contiguous() or T.dim() != 2 or X.shape[0] != T.shape[1]:
        raise GWError("gw_transform: need contiguous T [n_out][n_in] and X [n_in][...]")
    n_out, n_in = int(T.shape[0]), int(T.shape[1])
    if Y is None:
        Y = torch.empty((n_out,) + tuple(X.shape[1:]), dtype=torch.complex128, device=X.device)
    if tuple(Y.shape) != (n_out,) + tuple(X.shape[1:]) or not Y.is_contiguous() or Y.dtype != torch.complex128:
        raise GWError("gw_transform: Y must be contiguous complex128 of shape (n_out,) + X.shape[1:]")
    ln = X.numel() // n_in
    _check(lib().gw_transform(n_out, n_in, ctypes.c_void_p(T.data_ptr()), ctypes.c_void_p(X.data_ptr()),
                              ctypes.c_void_p(Y.data_ptr()), ctypes.c_size_t(ln), _stream(stream)), "gw_transform")
    return Y


def gw_selfenergy(prob, G, Wt, Sigma=None, stream=None):
    """Stage 3, Eq. 31."""
    gshape = prob.gshape()
    if Sigma is None:
        Sigma = torch.empty(gshape, dtype=torch.complex128, device=G.device)
    _check(lib().gw_selfenergy(prob.ref(), _dev(G, gshape, "G"),
                               _dev(Wt, (prob.ntau, prob.nq, prob.naux, prob.naux), "Wt"),
                               _dev(Sigma, gshape, "Sigma"), _stream(stream)), "gw_selfenergy")
    return Sigma


def gw_exchange(prob, gamma, K=None, stream=None):
    """Stage 4, Eq. 22."""
    shape = prob.kshape()
    if K is None:
        K = torch.empty(shape, dtype=torch.complex128, device=gamma.device)
    _check(lib().gw_exchange(prob.ref(), _dev(gamma, shape, "gamma"), _dev(K, shape, "K"), _stream(stream)), "gw_exchange")
    return K


def gw_sigma_iteration(prob, G, gamma, bufs=None, stream=None):
    """The whole hot path on device-resident inputs: four C-ABI calls on one stream.  Returns dict of outputs."""
    b = bufs if bufs is not None else {}
    P0t = gw_polarization(prob, G, b.get("P0t"), stream)
    Wt, info = gw_screened_interaction(prob, P0t, b.get("Wt", P0t) if bufs is not None else None, b.get("info"), stream)
    Sigma = gw_selfenergy(prob, G, Wt, b.get("Sigma"), stream)
    K = gw_exchange(prob, gamma, b.get("K"), stream)
    return {"P0t": P0t, "Wt": Wt, "Sigma": Sigma, "K": K, "info": info}


def gw_sigma_iteration_host(prob, G, gamma, Sigma=None, K=None, want_P0t=False, want_Wt=False, stream=None):
    """End-to-end call with HOST buffers (pinned recommended); copies are inside the call."""
    if prob.on_device:
        raise GWError("gw_sigma_iteration_host needs a GWProblem built from CPU tensors")
    for name, t in (("G", G), ("gamma", gamma)):
        if t.is_cuda or t.dtype != torch.complex128 or not t.is_contiguous():
            raise GWError(f"{name}: need a contiguous CPU complex128 tensor")
    pin = G.is_pinned()
    mk = lambda shape: torch.empty(shape, dtype=torch.complex128, pin_memory=pin)
    if Sigma is None:
        Sigma = mk(prob.gshape())
    if K is None:
        K = mk(prob.kshape())
    pshape = (prob.ntau, prob.nq, prob.naux, prob.naux)
    P0t = mk(pshape) if want_P0t else None
    Wt = mk(pshape) if want_Wt else None
    ms = (ctypes.c_float * 6)()
    vp = lambda t: ctypes.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().gw_sigma_iteration_host(prob.ref(), vp(G), vp(gamma), vp(Sigma), vp(K), vp(P0t), vp(Wt),
                                         ctypes.cast(ms, ctypes.c_void_p), _stream(stream)), "gw_sigma_iteration_host")
    return {"Sigma": Sigma, "K": K, "P0t": P0t, "Wt": Wt, "stage_ms": list(ms)}


def gw_sigma_iteration_stream(prob, G, gamma, v_budget_bytes, Sigma=None, K=None, stream=None):
    """Out-of-core V (gw.h): the whole iteration with V in HOST memory (GW_V_FULL layout, pinned recommended), streamed through two
    device q-slab buffers of at most v_budget_bytes together.  Returns dict(Sigma, K, stats)."""
    if prob.on_device or prob.v_layout != GW_V_FULL:
        raise GWError("gw_sigma_iteration_stream needs a GWProblem built from CPU tensors in the full V layout")
    for name, t, shape in (("G", G, prob.gshape()), ("gamma", gamma, prob.kshape())):
        if t.is_cuda or t.dtype != torch.complex128 or not t.is_contiguous() or tuple(t.shape) != shape:
            raise GWError(f"{name}: need a contiguous CPU complex128 tensor of shape {shape}")
    pin = G.is_pinned()
    mk = lambda shape: torch.empty(shape, dtype=torch.complex128, pin_memory=pin)
    if Sigma is None:
        Sigma = mk(prob.gshape())
    if K is None:
        K = mk(prob.kshape())
    st = (ctypes.c_float * 4)()
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    _check(lib().gw_sigma_iteration_stream(prob.ref(), vp(G), vp(gamma), vp(Sigma), vp(K), ctypes.c_size_t(int(v_budget_bytes)),
                                           ctypes.cast(st, ctypes.c_void_p), _stream(stream)), "gw_sigma_iteration_stream")
    return {"Sigma": Sigma, "K": K, "stats": {"ms": st[0], "h2d_gb": st[1], "slabs": int(st[2]), "q_per_slab": int(st[3])}}


def gw_executed_flops(prob):
    out = (ctypes.c_double * 4)()
    _check(lib().gw_executed_flops(prob.ref(), out), "gw_executed_flops")
    return list(out)


def gw_launch_count(prob):
    return int(lib().gw_launch_count(prob.ref()))


def gw_fp64_peak(ms=200.0, stream=None):
    out = ctypes.c_double(0.0)
    _check(lib().gw_fp64_peak(ctypes.c_double(ms), ctypes.byref(out), _stream(stream)), "gw_fp64_peak")
    return out.value


def gw_complex_mma_probe(mode, ms=100.0, stream=None):
    """Algorithmic TFLOP/s of the main-GEMM inner loop alone: mode 0 = 4M, 1 = 3M with sums in registers, 2 = 3M with pre-summed B."""
    out = ctypes.c_double(0.0)
    _check(lib().gw_complex_mma_probe(int(mode), ctypes.c_double(ms), ctypes.byref(out), _stream(stream)), "gw_complex_mma_probe")
    return out.value


def gw_fp64_subcore_probe(warp_mask, stream=None):
    """Executed TFLOP/s of a DMMA loop run by the warps of warp_mask only (one 16-warp CTA per SM): which warps share an FP64 pipe."""
    out = ctypes.c_double(0.0)
    _check(lib().gw_fp64_subcore_probe(ctypes.c_uint32(int(warp_mask)), ctypes.byref(out), _stream(stream)), "gw_fp64_subcore_probe")
    return out.value


def gw_fp64_peak_dfma(ms=200.0, stream=None):
    out = ctypes.c_double(0.0)
    _check(lib().gw_fp64_peak_dfma(ctypes.c_double(ms), ctypes.byref(out), _stream(stream)), "gw_fp64_peak_dfma")
    return out.value


# ---------------------------------------------------------------------------------------------------------------------
# loop closure (gw.h "Loop closure"; Fig. 4 of the paper)
# ---------------------------------------------------------------------------------------------------------------------
def _c128(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise GWError(f"{name}: need a contiguous CUDA complex128 tensor")
    return ctypes.c_void_p(t.data_ptr())


def _f64(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise GWError(f"{name}: need a contiguous CUDA float64 tensor")
    return ctypes.c_void_p(t.data_ptr())


def gw_hartree(prob, gamma, J=None, stream=None):
    """Eq. 20: J[k] (spin independent) from gamma[k'] (summed over the spin channels) and the diagonal blocks V[k][k]."""
    shape = (prob.nk, prob.nao, prob.nao)
    if J is None:
        J = torch.empty(shape, dtype=torch.complex128, device=gamma.device)
    _check(lib().gw_hartree(prob.ref(), _dev(gamma, prob.kshape(), "gamma"), _dev(J, shape, "J"), _stream(stream)), "gw_hartree")
    return J


def gw_static_max_naux():
    """Largest naux gw_hartree_static accepts (the size of the library's static device scratch, in complex numbers)."""
    return int(lib().gw_static_max_naux())


def gw_hartree_static(prob, gamma, J, stream=None):
    """gw_hartree without any device allocation: the intermediate rho[Q] lives in a static device array of the library
    (naux <= gw_static_max_naux(), else GWError / GW_ESTATIC); prob.work is not used.  J is the caller's output buffer.
    Calls that overlap on one GPU race on the shared array (include/gw.h)."""
    shape = (prob.nk, prob.nao, prob.nao)
    _check(lib().gw_hartree_static(prob.ref(), _dev(gamma, prob.kshape(), "gamma"), _dev(J, shape, "J"), _stream(stream)), "gw_hartree_static")
    return J


def gw_dyson_update(omega, mu, S, F, Sigma_w=None, G_w=None, info=None, stream=None):
    """Eq. 16 for all (n, k): G_w[n][k] = [(i omega_n + mu) S[k] - F[k] - Sigma_w[n][k]]^-1."""
    nk, nao = int(S.shape[0]), int(S.shape[1])
    nwf = int(omega.numel())
    shape = (nwf, nk, nao, nao)
    if G_w is None:
        G_w = torch.empty(shape, dtype=torch.complex128, device=S.device)
    if info is None:
        info = torch.empty(2, dtype=torch.int32, device=S.device)
    _check(lib().gw_dyson_update(nk, nao, nwf, _f64(omega, "omega"), float(mu), _dev(S, (nk, nao, nao), "S"), _dev(F, (nk, nao, nao), "F"),
                                 _dev(Sigma_w, shape, "Sigma_w") if Sigma_w is not None else None, _dev(G_w, shape, "G_w"),
                                 ctypes.c_void_p(info.data_ptr()), _stream(stream)), "gw_dyson_update")
    return G_w, info


def gw_electron_count(t_beta, S, G_w, spin_deg=2, stream=None):
    """Eq. 15: N_e from G(i omega_n) (returns a 1-element CUDA float64 tensor; no host sync)."""
    nwf, nk, nao = int(G_w.shape[0]), int(G_w.shape[1]), int(G_w.shape[2])
    partial = torch.empty(nk, dtype=torch.complex128, device=S.device)
    ne = torch.empty(1, dtype=torch.float64, device=S.device)
    _check(lib().gw_electron_count(nk, nao, nwf, int(spin_deg), _dev(t_beta, (nwf,), "t_beta"), _dev(S, (nk, nao, nao), "S"),
                                   _c128(G_w, "G_w"), _c128(partial, "partial"), _f64(ne, "ne"), _stream(stream)), "gw_electron_count")
    return ne


def gw_find_mu(omega, t_beta, S, F, Sigma_w, n_target, mu_lo, mu_hi, mu_tol=1e-12, spin_deg=2, G_w=None, stream=None):
    """Chemical-potential search of Fig. 4 step 3 (synchronises the stream).  Returns (mu, N_e(mu), G_w at mu, evaluations)."""
    nk, nao = int(S.shape[0]), int(S.shape[1])
    nwf = int(omega.numel())
    shape = (nwf, nk, nao, nao)
    if G_w is None:
        G_w = torch.empty(shape, dtype=torch.complex128, device=S.device)
    partial = torch.empty(nk, dtype=torch.complex128, device=S.device)
    ne = torch.empty(1, dtype=torch.float64, device=S.device)
    mu_o, ne_o, ev = ctypes.c_double(0.0), ctypes.c_double(0.0), ctypes.c_int32(0)
    _check(lib().gw_find_mu(nk, nao, nwf, int(spin_deg), _f64(omega, "omega"), _dev(t_beta, (nwf,), "t_beta"), _dev(S, (nk, nao, nao), "S"),
                            _dev(F, (nk, nao, nao), "F"), _dev(Sigma_w, shape, "Sigma_w") if Sigma_w is not None else None,
                            float(n_target), float(mu_lo), float(mu_hi), float(mu_tol), _dev(G_w, shape, "G_w"), _c128(partial, "partial"),
                            _f64(ne, "ne"), ctypes.byref(mu_o), ctypes.byref(ne_o), ctypes.byref(ev), _stream(stream)), "gw_find_mu")
    return mu_o.value, ne_o.value, G_w, ev.value


def gw_axpby(a, X, b, Y, stream=None):
    """Y <- a X + b Y (complex scalars a, b)."""
    if X.shape != Y.shape:
        raise GWError("gw_axpby: shapes differ")
    a, b = complex(a), complex(b)
    _check(lib().gw_axpby(X.numel(), a.real, a.imag, _c128(X, "X"), b.real, b.imag, _c128(Y, "Y"), _stream(stream)), "gw_axpby")
    return Y


def gw_scgw_iteration(prob, fg, H0, S, G, n_target, mu_lo, mu_hi, alpha=1.0, mu_tol=1e-12, stream=None):
    """One scGW iteration in the order of Fig. 4, every step a C-ABI call (this function only sequences them):
    G(tau) -> gamma = -G(beta^-) -> J (Eq. 20), K (Eq. 22), Sigma~(tau) (Algorithm 1) -> Sigma~(i omega_n) (Eq. 13) -> mu (Eq. 15) ->
    G(i omega_n) (Eq. 16) -> G(tau) (Eq. 14) -> damping.  fg: dict of CUDA tensors omega, T_wt_f, T_tw_f, t_beta, e_beta
    (gwgen.make_fermionic_grids).  Returns a dict of CUDA tensors and the scalars mu, ne."""
    Gb = gw_transform(fg["e_beta"].reshape(1, -1), G, stream=stream)[0].contiguous()
    gamma = gw_axpby(-1.0, Gb, 0.0, torch.empty_like(Gb), stream)
    J = gw_hartree(prob, gamma, stream=stream)
    K = gw_exchange(prob, gamma, stream=stream)
    P0t = gw_polarization(prob, G, stream=stream)
    Wt, info = gw_screened_interaction(prob, P0t, P0t, stream=stream)
    Sigma_t = gw_selfenergy(prob, G, Wt, stream=stream)
    Sigma_w = gw_transform(fg["T_wt_f"], Sigma_t, stream=stream)
    F = gw_axpby(1.0, J, 1.0, gw_axpby(1.0, K, 1.0, H0.clone(), stream), stream)
    mu, ne, G_w, n_eval = gw_find_mu(fg["omega"], fg["t_beta"], S, F, Sigma_w, n_target, mu_lo, mu_hi, mu_tol, prob.spin_deg, stream=stream)
    G_new = gw_transform(fg["T_tw_f"], G_w, stream=stream)
    G_mix = gw_axpby(alpha, G_new, 1.0 - alpha, G.clone(), stream)
    return dict(gamma=gamma, J=J, K=K, Wt=Wt, info=info, Sigma_t=Sigma_t, Sigma_w=Sigma_w, F=F, mu=mu, ne=ne, G_w=G_w, G_new=G_new,
                G=G_mix, n_eval=n_eval)
