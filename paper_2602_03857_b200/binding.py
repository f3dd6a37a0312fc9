"""Thin Python binding of include/grav.h (argument marshalling only -- every step of the path runs in the CUDA
kernels of libgrav.so).  PyTorch supplies device memory and streams.  No CPU fallback: load() raises if the
extension is missing, and every entry point raises GravError on a non-OK status.

Names mirror the C ABI: mesh_create -> GravContext, forward, adjoint, depth_weights, dataspace_cg, store_g,
forward_stored, adjoint_stored, gram_diag, direct_solve, *_host.
"""
import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgrav.so")

MATRIX_FREE, STORED_F64, STORED_F32 = 0, 1, 2
PREC_F64, PREC_F32 = 0, 1

EXPORTS = [
    "grav_mesh_create", "grav_mesh_destroy", "grav_sizes", "grav_workspace_bytes", "grav_set_workspace",
    "grav_forward", "grav_adjoint", "grav_depth_weights", "grav_dataspace_cg", "grav_store_g",
    "grav_forward_stored", "grav_adjoint_stored", "grav_stored_g", "grav_gram_diag", "grav_direct_solve",
    "grav_forward_host", "grav_adjoint_host", "grav_dataspace_cg_host", "grav_invert", "grav_launch_count",
    "grav_fp64_peak_probe", "grav_last_error", "grav_debug_set_psi_variant", "grav_debug_psi_eval_host",
    "grav_debug_k0", "grav_debug_log2d_binades", "grav_debug_log2d_default", "grav_debug_set_log2d", "grav_set_comm",
    "grav_set_precision", "grav_debug_psi_eval_device", "grav_noalloc_setup", "grav_gemvt_noalloc",
]

# include/grav.h: grav_comm
#   int allreduce_sum(double* buf_dev, long long count, void* stream, void* user)
#   int allgather(const double* send_dev, double* recv_dev, long long count, void* stream, void* user)
ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p)
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p)


class _Comm(C.Structure):
    _fields_ = [("world", C.c_int), ("rank", C.c_int), ("allreduce_sum", ALLREDUCE_FN), ("allgather", ALLGATHER_FN),
                ("user", C.c_void_p)]


class GravError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"grav status {status}: {msg}")
        self.status = status


class _CgState(C.Structure):
    _fields_ = [("x_dev", C.c_void_p), ("r_dev", C.c_void_p), ("p_dev", C.c_void_p), ("rho_dev", C.c_void_p),
                ("resume", C.c_int)]


_lib = None


def load():
    """dlopen libgrav.so (built in-tree by _build.build()).  Raises if it is not there: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built; run `python -c 'import __graft_entry__ as g; g.build()'`")
    L = C.CDLL(LIB_PATH)
    vp, dp, i, ll, d = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_longlong, C.c_double
    L.grav_mesh_create.restype = i
    L.grav_mesh_create.argtypes = [C.POINTER(vp), i, i, i, dp, dp, dp, ll, dp, dp, dp, d, i]
    L.grav_mesh_destroy.restype = None
    L.grav_mesh_destroy.argtypes = [vp]
    L.grav_sizes.restype = i
    L.grav_sizes.argtypes = [vp, C.POINTER(ll)]
    L.grav_workspace_bytes.restype = C.c_size_t
    L.grav_workspace_bytes.argtypes = [vp, i]
    L.grav_set_workspace.restype = i
    L.grav_set_workspace.argtypes = [vp, vp, C.c_size_t]
    for name in ("grav_forward", "grav_adjoint", "grav_forward_stored", "grav_adjoint_stored", "grav_gram_diag"):
        f = getattr(L, name)
        f.restype = i
        f.argtypes = [vp, vp, vp, vp]
    L.grav_depth_weights.restype = i
    L.grav_depth_weights.argtypes = [vp, d, d, vp, vp]
    L.grav_dataspace_cg.restype = i
    L.grav_dataspace_cg.argtypes = [vp, vp, vp, d, i, d, i, vp, C.POINTER(_CgState), vp, vp, vp, vp, vp]
    L.grav_store_g.restype = i
    L.grav_store_g.argtypes = [vp, i, vp]
    L.grav_stored_g.restype = i
    L.grav_stored_g.argtypes = [vp, C.POINTER(vp), C.POINTER(i)]
    L.grav_direct_solve.restype = i
    L.grav_direct_solve.argtypes = [vp, vp, vp, d, vp, vp, vp, vp]
    L.grav_forward_host.restype = i
    L.grav_forward_host.argtypes = [vp, vp, vp, vp]
    L.grav_adjoint_host.restype = i
    L.grav_adjoint_host.argtypes = [vp, vp, vp, vp]
    L.grav_dataspace_cg_host.restype = i
    L.grav_dataspace_cg_host.argtypes = [vp, vp, d, d, d, i, d, i, vp, vp, vp, vp]
    L.grav_launch_count.restype = ll
    L.grav_launch_count.argtypes = [vp]
    L.grav_fp64_peak_probe.restype = i
    L.grav_fp64_peak_probe.argtypes = [i, i, dp, dp]
    L.grav_invert.restype = i
    L.grav_invert.argtypes = [vp, vp, vp, d, vp, vp, i, i, d, d, i, vp, vp, vp, vp, C.POINTER(C.c_int),
                              C.POINTER(C.c_int), vp]
    L.grav_debug_set_psi_variant.restype = i
    L.grav_debug_set_psi_variant.argtypes = [vp, i]
    L.grav_debug_psi_eval_host.restype = d
    L.grav_debug_psi_eval_host.argtypes = [d, d, d, i, i]
    L.grav_debug_set_log2d.restype = i
    L.grav_debug_set_log2d.argtypes = [vp, i]
    L.grav_set_precision.restype = i
    L.grav_set_precision.argtypes = [vp, i]
    L.grav_debug_psi_eval_device.restype = i
    L.grav_debug_psi_eval_device.argtypes = [vp, i, ll, vp, vp, vp, vp, vp]
    L.grav_set_comm.restype = i
    L.grav_set_comm.argtypes = [vp, C.POINTER(_Comm)]
    L.grav_debug_k0.restype = i
    L.grav_debug_k0.argtypes = [vp]
    L.grav_debug_log2d_binades.restype = i
    L.grav_debug_log2d_binades.argtypes = [vp]
    L.grav_debug_log2d_default.restype = i
    L.grav_debug_log2d_default.argtypes = [vp]
    L.grav_noalloc_setup.restype = i
    L.grav_noalloc_setup.argtypes = [i]
    L.grav_gemvt_noalloc.restype = i
    L.grav_gemvt_noalloc.argtypes = [i, vp, i, ll, ll, vp, vp, vp, vp]
    L.grav_last_error.restype = C.c_char_p
    L.grav_last_error.argtypes = []
    _lib = L
    return L


def _check(st):
    if st != 0:
        raise GravError(st, load().grav_last_error().decode())


def _hp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, n, name):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and t.numel() == n):
        raise ValueError(f"{name}: need a contiguous CUDA float64 tensor of {n} elements")
    return C.c_void_p(t.data_ptr())


def _host(a, n, name):
    """numpy float64 array or pinned CPU torch tensor -> pointer (no copy)."""
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n:
            raise ValueError(f"{name}: need a contiguous CPU float64 tensor of {n} elements")
        return C.c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n):
        raise ValueError(f"{name}: need a contiguous float64 array of {n} elements")
    return C.c_void_p(a.ctypes.data)


NOALLOC_MAX_DOUBLES = 2 << 20        # include/grav.h GRAV_NOALLOC_MAX_DOUBLES


def noalloc_setup(device=0):
    """grav_noalloc_setup: look up the built-in scratch array's address on `device` (once; before a capture begins)."""
    _check(load().grav_noalloc_setup(int(device)))


def gemvt_noalloc(G, v, w=None, out=None):
    """grav_gemvt_noalloc: g = G^T v (w None) or W^-2 G^T v for a caller-held (N, M) float64 / float32 CUDA matrix, with
    the scratch in the library's built-in device array: no context, no workspace, no allocation inside the call (pass
    `out`; without it this wrapper allocates the result tensor itself).  Raises GravError beyond the array's limit."""
    if not (isinstance(G, torch.Tensor) and G.is_cuda and G.dim() == 2 and G.is_contiguous()
            and G.dtype in (torch.float64, torch.float32)):
        raise ValueError("G: need a contiguous 2-D CUDA tensor of float64 or float32")
    N, M = G.shape
    g = torch.empty(M, dtype=torch.float64, device=G.device) if out is None else out
    for t in (v, w, g):
        if t is not None and t.device != G.device:
            raise ValueError("all tensors must live on G's device")
    with torch.cuda.device(G.device):
        _check(load().grav_gemvt_noalloc(G.device.index, C.c_void_p(G.data_ptr()), G.element_size(), N, M,
                                         _dev(v, N, "v"), _dev(w, M, "w"), _dev(g, M, "g"), _stream()))
    return g


class CGState:
    """Device-resident CG state (x, r, p: N doubles; rho: 1 double)."""

    def __init__(self, N, device, x=None, r=None, p=None, rho=None):
        mk = lambda a: (torch.zeros(N, dtype=torch.float64, device=device) if a is None
                        else torch.as_tensor(np.asarray(a, dtype=np.float64)).to(device))
        self.x, self.r, self.p = mk(x), mk(r), mk(p)
        self.rho = torch.tensor([0.0 if rho is None else float(rho)], dtype=torch.float64, device=device)
        self.resume = x is not None


class GravContext:
    """grav_mesh_create + workspace.  Holds the workspace tensor so that it outlives every enqueued kernel."""

    def __init__(self, xn, yn, zn, xo, yo, zo, gamma, device=0, mode=MATRIX_FREE):
        L = load()
        self._lib = L
        xn, yn, zn, xo, yo, zo = [np.ascontiguousarray(a, dtype=np.float64) for a in (xn, yn, zn, xo, yo, zo)]
        if not (xo.size == yo.size == zo.size):
            raise ValueError("station arrays differ in length")
        self.device = torch.device("cuda", device)
        h = C.c_void_p()
        _check(L.grav_mesh_create(C.byref(h), xn.size - 1, yn.size - 1, zn.size - 1, _hp(xn), _hp(yn), _hp(zn),
                                  xo.size, _hp(xo), _hp(yo), _hp(zo), float(gamma), device))
        self._h = h
        sz = (C.c_longlong * 3)()
        _check(L.grav_sizes(h, sz))
        self.N, self.M, self.Nn = int(sz[0]), int(sz[1]), int(sz[2])
        self.mode = None
        self.ws = None
        self.set_mode(mode)

    def set_mode(self, mode):
        """(Re)allocate the workspace for `mode` (invalidates a stored G)."""
        nbytes = int(self._lib.grav_workspace_bytes(self._h, mode))
        if nbytes == 0:
            raise GravError(-1, "bad mode")
        if self.ws is None or self.ws.numel() < nbytes:
            self.ws = None
            self.ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        _check(self._lib.grav_set_workspace(self._h, C.c_void_p(self.ws.data_ptr()), self.ws.numel()))
        self.mode = mode

    def close(self):
        if getattr(self, "_h", None):
            torch.cuda.synchronize(self.device)
            self._lib.grav_mesh_destroy(self._h)
            self._h = None
            self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self, n):
        return torch.empty(n, dtype=torch.float64, device=self.device)

    # ---- device-pointer entry points -------------------------------------------------------------------
    def forward(self, u, out=None):
        d = self._new(self.N) if out is None else out
        _check(self._lib.grav_forward(self._h, _dev(u, self.M, "u"), _dev(d, self.N, "d"), _stream()))
        return d

    def adjoint(self, v, out=None):
        g = self._new(self.M) if out is None else out
        _check(self._lib.grav_adjoint(self._h, _dev(v, self.N, "v"), _dev(g, self.M, "g"), _stream()))
        return g

    def depth_weights(self, beta, z0, out=None):
        w = self._new(self.M) if out is None else out
        _check(self._lib.grav_depth_weights(self._h, float(beta), float(z0), _dev(w, self.M, "w"), _stream()))
        return w

    def dataspace_cg(self, dobs, w, lam, iters, rtol=0.0, mode=MATRIX_FREE, state=None, want_m=True, precond=None):
        """Returns dict(alpha, m, hist, ab) of device tensors.  precond: diag(G W^-2 G^T) from gram_diag() for Jacobi
        preconditioning (the library adds lambda), or None for plain CG."""
        alpha = self._new(self.N)
        m = self._new(self.M) if want_m else None
        hist = self._new(iters + 1)
        ab = self._new(max(2 * iters, 1))
        st = None
        if state is not None:
            st = _CgState(state.x.data_ptr(), state.r.data_ptr(), state.p.data_ptr(), state.rho.data_ptr(),
                          1 if state.resume else 0)
        _check(self._lib.grav_dataspace_cg(self._h, _dev(dobs, self.N, "dobs"), _dev(w, self.M, "w"), float(lam),
                                           int(iters), float(rtol), int(mode), _dev(precond, self.N, "precond"),
                                           C.byref(st) if st else None,
                                           _dev(alpha, self.N, "alpha"), _dev(m, self.M, "m"),
                                           C.c_void_p(hist.data_ptr()), C.c_void_p(ab.data_ptr()), _stream()))
        return dict(alpha=alpha, m=m, hist=hist, ab=ab[:2 * iters].view(-1, 2) if iters else ab[:0])

    def invert(self, dobs, w, lam, mref=None, max_outer=30, max_inner=20, tol_outer=1e-4, tol_inner=1e-4,
               mode=MATRIX_FREE, want_dpred=True, precond=None):
        """The paper's outer model-update loop (include/grav.h: grav_invert).  Returns dict(m, dpred, hist, steps,
        inner, n_outer, stop); hist / steps / inner (CG iterations per update) are numpy arrays."""
        m = self._new(self.M)
        dpred = self._new(self.N) if want_dpred else None
        hist = np.zeros(max_outer + 1)
        steps = np.zeros(max(max_outer, 1))
        n_outer = C.c_int(0)
        inner = (C.c_int * max(max_outer, 1))()
        _check(self._lib.grav_invert(self._h, _dev(dobs, self.N, "dobs"), _dev(w, self.M, "w"), float(lam),
                                     _dev(mref, self.M, "mref"), _dev(precond, self.N, "precond"), int(max_outer),
                                     int(max_inner), float(tol_outer), float(tol_inner), int(mode),
                                     _dev(m, self.M, "m"), _dev(dpred, self.N, "dpred"), C.c_void_p(hist.ctypes.data),
                                     C.c_void_p(steps.ctypes.data), inner, C.byref(n_outer), _stream()))
        k = n_outer.value
        stop = "tolerance" if hist[k] <= tol_outer else ("max_outer" if k == max_outer else "no_decrease")
        tried = min(k + (1 if stop == "no_decrease" else 0), max_outer)
        return dict(m=m, dpred=dpred, hist=hist[:k + 1], steps=steps[:k], inner=np.array(inner[:tried]), n_outer=k,
                    stop=stop)

    def store_g(self, fp32=False):
        want = STORED_F32 if fp32 else STORED_F64
        need = int(self._lib.grav_workspace_bytes(self._h, want))
        if self.ws.numel() < need:
            self.set_mode(want)
        _check(self._lib.grav_store_g(self._h, 1 if fp32 else 0, _stream()))

    def stored_g(self):
        """View of the stored G as an (N, M) tensor (float64 or float32) aliasing the workspace."""
        p, e = C.c_void_p(), C.c_int()
        _check(self._lib.grav_stored_g(self._h, C.byref(p), C.byref(e)))
        if not e.value:
            return None
        off = p.value - self.ws.data_ptr()
        dt = torch.float64 if e.value == 8 else torch.float32
        return self.ws[off:off + self.N * self.M * e.value].view(dt).view(self.N, self.M)

    def forward_stored(self, u, out=None):
        d = self._new(self.N) if out is None else out
        _check(self._lib.grav_forward_stored(self._h, _dev(u, self.M, "u"), _dev(d, self.N, "d"), _stream()))
        return d

    def adjoint_stored(self, v, out=None):
        g = self._new(self.M) if out is None else out
        _check(self._lib.grav_adjoint_stored(self._h, _dev(v, self.N, "v"), _dev(g, self.M, "g"), _stream()))
        return g

    def gram_diag(self, w):
        dg = self._new(self.N)
        _check(self._lib.grav_gram_diag(self._h, _dev(w, self.M, "w"), _dev(dg, self.N, "diag"), _stream()))
        return dg

    def direct_solve(self, dobs, w, lam, want_m=True):
        A = self._new(self.N * self.N)
        alpha = self._new(self.N)
        m = self._new(self.M) if want_m else None
        _check(self._lib.grav_direct_solve(self._h, _dev(dobs, self.N, "dobs"), _dev(w, self.M, "w"), float(lam),
                                           C.c_void_p(A.data_ptr()), _dev(alpha, self.N, "alpha"),
                                           _dev(m, self.M, "m"), _stream()))
        return alpha, m

    # ---- host-buffer (end-to-end) entry points ---------------------------------------------------------
    def forward_host(self, u_host, d_host):
        _check(self._lib.grav_forward_host(self._h, _host(u_host, self.M, "u"), _host(d_host, self.N, "d"), _stream()))
        return d_host

    def adjoint_host(self, v_host, g_host):
        _check(self._lib.grav_adjoint_host(self._h, _host(v_host, self.N, "v"), _host(g_host, self.M, "g"), _stream()))
        return g_host

    def dataspace_cg_host(self, dobs_host, beta, z0, lam, iters, alpha_host, m_host=None, hist_host=None, rtol=0.0,
                          mode=MATRIX_FREE):
        _check(self._lib.grav_dataspace_cg_host(self._h, _host(dobs_host, self.N, "dobs"), float(beta), float(z0),
                                                float(lam), int(iters), float(rtol), int(mode),
                                                _host(alpha_host, self.N, "alpha"), _host(m_host, self.M, "m"),
                                                _host(hist_host, iters + 1, "hist"), _stream()))
        return alpha_host

    def set_comm(self, comm):
        """Observation-sharded operation (include/grav.h: grav_set_comm).  `comm` has attributes world, rank and methods
        allreduce_sum(ptr, count, stream) / allgather(send_ptr, recv_ptr, count, stream) on raw device addresses, both
        ordered on the CUDA stream they are handed; None restores single-rank operation.  The workspace is re-allocated
        for the new layout (a stored G is lost)."""
        if comm is None or comm.world <= 1:
            self._comm = None
            _check(self._lib.grav_set_comm(self._h, None))
        else:
            def guard(fn):
                def tramp(*a):
                    try:
                        fn(*[int(v or 0) for v in a[:-1]])
                        return 0
                    except Exception:           # no exception may cross the C ABI
                        import traceback
                        traceback.print_exc()
                        return 1
                return tramp

            cs = _Comm(int(comm.world), int(comm.rank), ALLREDUCE_FN(guard(comm.allreduce_sum)),
                       ALLGATHER_FN(guard(comm.allgather)), None)
            self._comm = (comm, cs)               # keep the trampolines alive as long as the context uses them
            _check(self._lib.grav_set_comm(self._h, C.byref(cs)))
        mode, self.ws, self.mode = self.mode, None, None
        self.set_mode(mode)

    def set_precision(self, fp32):
        """Matrix-free evaluation in Float32 (True; the paper's precision, FP64 accumulation) or FP64 (False, default)."""
        _check(self._lib.grav_set_precision(self._h, PREC_F32 if fp32 else PREC_F64))

    def psi_eval_device(self, variant, X, Y, Z):
        """Psi (+ the k0 offset for variants 0, 2, 3) of the device evaluator `variant` at the argument triples given as
        CUDA float64 tensors (include/grav.h: grav_debug_psi_eval_device)."""
        n = X.numel()
        out = self._new(n)
        _check(self._lib.grav_debug_psi_eval_device(self._h, int(variant), n, _dev(X, n, "X"), _dev(Y, n, "Y"),
                                                    _dev(Z, n, "Z"), _dev(out, n, "out"), _stream()))
        return out

    def set_psi_variant(self, variant):
        """0: hand-built evaluator (default); 1: CUDA libm (cross-check)."""
        _check(self._lib.grav_debug_set_psi_variant(self._h, int(variant)))

    def set_log2d(self, mode):
        """-1: the context's default log table; 0: 256-entry table; 1: exponent-and-mantissa table (diagnostic)."""
        _check(self._lib.grav_debug_set_log2d(self._h, int(mode)))

    @property
    def k0(self):
        return int(self._lib.grav_debug_k0(self._h))

    @property
    def log2d_binades(self):
        return int(self._lib.grav_debug_log2d_binades(self._h))

    @property
    def log2d_default(self):
        return bool(self._lib.grav_debug_log2d_default(self._h))

    @property
    def launches(self):
        return int(self._lib.grav_launch_count(self._h))


def psi_eval_host(X, Y, Z, k0=0, log2d=False):
    """Host emulation of the device Psi evaluator of csrc/psi.cuh (diagnostic; needs no GPU); log2d selects the
    exponent-and-mantissa log table."""
    return float(load().grav_debug_psi_eval_host(float(X), float(Y), float(Z), int(k0), 1 if log2d else 0))


def fp64_peak_probe(device=0, iters=200000):
    """(FP64 thread-instructions per second, ms) of a DFMA-only kernel on the whole device."""
    n, ms = C.c_double(), C.c_double()
    _check(load().grav_fp64_peak_probe(device, iters, C.byref(n), C.byref(ms)))
    return n.value / (ms.value * 1e-3), ms.value
