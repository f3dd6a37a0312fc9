"""ctypes binding of the CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, `__graft_entry__.smoke()` and bench.py's cpu_baseline / `--impl reference` legs may import this
package.  It imports nothing from `paper_2602_03857_b200` and shares no code with the CUDA path.
Every function takes / returns numpy float64 arrays on the host.  Citations are to /root/reference/PAPER.md
lines (P:nn), see oracle.cpp for the per-function passages.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        llp = C.POINTER(C.c_longlong)
        mesh = [C.c_int, C.c_int, C.c_int, dp, dp, dp]
        obs = [C.c_longlong, dp, dp, dp]
        L.orc_psi.restype = C.c_double
        L.orc_psi.argtypes = [C.c_double] * 3 + [C.c_int]
        L.orc_prism_gz.restype = C.c_double
        L.orc_prism_gz.argtypes = [C.c_double] * 11 + [C.c_int]
        L.orc_forward.restype = None
        L.orc_forward.argtypes = mesh + obs + [C.c_double, dp, dp, C.c_int, C.c_int]
        L.orc_adjoint.restype = None
        L.orc_adjoint.argtypes = mesh + obs + [C.c_double, dp, C.c_longlong, llp, dp, C.c_int, C.c_int]
        L.orc_tabulate.restype = None
        L.orc_tabulate.argtypes = mesh + obs + [C.c_double, dp, C.c_int]
        L.orc_depth_weights.restype = None
        L.orc_depth_weights.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.c_double, C.c_double, dp]
        L.orc_dense_matvec.restype = None
        L.orc_dense_matvec.argtypes = [C.c_longlong, C.c_longlong, dp, dp, dp, C.c_int]
        L.orc_dense_rmatvec.restype = None
        L.orc_dense_rmatvec.argtypes = [C.c_longlong, C.c_longlong, dp, dp, dp, C.c_int]
        L.orc_gram_diag.restype = None
        L.orc_gram_diag.argtypes = [C.c_longlong, C.c_longlong, dp, dp, dp, C.c_int]
        L.orc_form_A.restype = None
        L.orc_form_A.argtypes = [C.c_longlong, C.c_longlong, dp, dp, C.c_double, dp, C.c_int]
        L.orc_cholesky_solve.restype = C.c_int
        L.orc_cholesky_solve.argtypes = [C.c_longlong, dp, dp, dp]
        L.orc_dataspace_direct.restype = C.c_int
        L.orc_dataspace_direct.argtypes = [C.c_longlong, C.c_longlong, dp, dp, C.c_double, dp, dp, dp, C.c_int]
        L.orc_modelspace_direct.restype = C.c_int
        L.orc_modelspace_direct.argtypes = [C.c_longlong, C.c_longlong, dp, dp, C.c_double, dp, dp, C.c_int]
        L.orc_cg.restype = None
        L.orc_cg.argtypes = ([C.c_longlong, C.c_longlong, dp] + mesh + [dp, dp, dp, C.c_double, dp, C.c_double, dp,
                             C.c_int, C.c_int, dp, dp, dp, dp, dp, dp, C.c_int, C.c_int])
        L.orc_pcg.restype = C.c_int
        L.orc_pcg.argtypes = [C.c_longlong, C.c_longlong, dp, dp, C.c_double, dp, dp, C.c_int, C.c_double, C.c_int,
                              dp, dp, dp, dp, dp, dp, C.c_int]
        L.orc_invert.restype = C.c_int
        L.orc_invert.argtypes = [C.c_longlong, C.c_longlong, dp, dp, C.c_double, dp, dp, dp, C.c_int, C.c_int,
                                 C.c_double, C.c_double, dp, dp, dp, dp, C.POINTER(C.c_int), dp, C.c_int]
        L.orc_hardware_threads.restype = C.c_int
        L.orc_hardware_threads.argtypes = []
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def hardware_threads() -> int:
    return int(lib().orc_hardware_threads())


def _nthreads(n):
    return hardware_threads() if n is None else int(n)


class Mesh:
    """Rectilinear prism mesh: node coordinates xn[nx+1], yn[ny+1], zn[nz+1] (z positive down)."""

    def __init__(self, xn, yn, zn):
        self.xn, self.yn, self.zn = _f64(xn), _f64(yn), _f64(zn)
        self.nx, self.ny, self.nz = len(self.xn) - 1, len(self.yn) - 1, len(self.zn) - 1
        self.M = self.nx * self.ny * self.nz

    def cargs(self):
        return [self.nx, self.ny, self.nz, _p(self.xn), _p(self.yn), _p(self.zn)]


def psi(X, Y, Z, prec=0) -> float:
    """Eq. 2-3."""
    return float(lib().orc_psi(float(X), float(Y), float(Z), int(prec)))


def prism_gz(station, box, rho, gamma, prec=0) -> float:
    """Eq. 1: gz of the prism box=(x1,x2,y1,y2,z1,z2) with density rho at station=(x,y,z)."""
    return float(lib().orc_prism_gz(*[float(s) for s in station], *[float(b) for b in box], float(rho),
                                    float(gamma), int(prec)))


def forward(mesh, xo, yo, zo, gamma, u, prec=0, nthreads=None):
    """d = G u, Eq. 5-6."""
    xo, yo, zo, u = _f64(xo), _f64(yo), _f64(zo), _f64(u)
    assert u.size == mesh.M
    d = np.empty(xo.size)
    lib().orc_forward(*mesh.cargs(), xo.size, _p(xo), _p(yo), _p(zo), float(gamma), _p(u), _p(d), int(prec),
                      _nthreads(nthreads))
    return d


def adjoint(mesh, xo, yo, zo, gamma, v, cells=None, prec=0, nthreads=None):
    """g = G^T v (transpose of Eq. 5), optionally only for the listed flat cell indices."""
    xo, yo, zo, v = _f64(xo), _f64(yo), _f64(zo), _f64(v)
    assert v.size == xo.size
    if cells is None:
        n, cp = mesh.M, None
    else:
        cells = np.ascontiguousarray(cells, dtype=np.int64)
        n, cp = cells.size, cells.ctypes.data_as(C.POINTER(C.c_longlong))
    g = np.empty(n)
    lib().orc_adjoint(*mesh.cargs(), xo.size, _p(xo), _p(yo), _p(zo), float(gamma), _p(v), n, cp, _p(g), int(prec),
                      _nthreads(nthreads))
    return g


def tabulate(mesh, xo, yo, zo, gamma, nthreads=None):
    """Dense G (N x M, row-major, prism index fastest), Eq. 6."""
    xo, yo, zo = _f64(xo), _f64(yo), _f64(zo)
    G = np.empty((xo.size, mesh.M))
    lib().orc_tabulate(*mesh.cargs(), xo.size, _p(xo), _p(yo), _p(zo), float(gamma), _p(G), _nthreads(nthreads))
    return G


def depth_weights(mesh, beta, z0):
    """w_k = (zc_k + z0)^(-beta/2)  (BASELINE.json north_star)."""
    w = np.empty(mesh.M)
    lib().orc_depth_weights(mesh.nx, mesh.ny, mesh.nz, _p(mesh.zn), float(beta), float(z0), _p(w))
    return w


def dense_matvec(G, u, nthreads=None):
    G, u = _f64(G), _f64(u)
    d = np.empty(G.shape[0])
    lib().orc_dense_matvec(G.shape[0], G.shape[1], _p(G), _p(u), _p(d), _nthreads(nthreads))
    return d


def dense_rmatvec(G, v, nthreads=None):
    G, v = _f64(G), _f64(v)
    g = np.empty(G.shape[1])
    lib().orc_dense_rmatvec(G.shape[0], G.shape[1], _p(G), _p(v), _p(g), _nthreads(nthreads))
    return g


def gram_diag(G, w, nthreads=None):
    """diag(G W^-2 G^T); its sum is the trace used for lambda (reading C7)."""
    G, w = _f64(G), _f64(w)
    dg = np.empty(G.shape[0])
    lib().orc_gram_diag(G.shape[0], G.shape[1], _p(G), _p(w), _p(dg), _nthreads(nthreads))
    return dg


def form_A(G, w, lam, nthreads=None):
    G, w = _f64(G), _f64(w)
    N = G.shape[0]
    A = np.empty((N, N))
    lib().orc_form_A(N, G.shape[1], _p(G), _p(w), float(lam), _p(A), _nthreads(nthreads))
    return A


def cholesky_solve(A, b):
    A = _f64(A).copy()
    b = _f64(b)
    x = np.empty_like(b)
    rc = lib().orc_cholesky_solve(A.shape[0], _p(A), _p(b), _p(x))
    if rc:
        raise np.linalg.LinAlgError(f"pivot {rc - 1} not positive")
    return x


def dataspace_direct(G, w, lam, dobs, nthreads=None):
    """Eq. 11 by Cholesky: returns (alpha, m)."""
    G, w, dobs = _f64(G), _f64(w), _f64(dobs)
    alpha, m = np.empty(G.shape[0]), np.empty(G.shape[1])
    rc = lib().orc_dataspace_direct(G.shape[0], G.shape[1], _p(G), _p(w), float(lam), _p(dobs), _p(alpha), _p(m),
                                    _nthreads(nthreads))
    if rc:
        raise np.linalg.LinAlgError(f"pivot {rc - 1} not positive")
    return alpha, m


def modelspace_direct(G, w, lam, dobs, nthreads=None):
    """Eq. 8 by Cholesky of the M x M normal equations (tiny inputs only)."""
    G, w, dobs = _f64(G), _f64(w), _f64(dobs)
    m = np.empty(G.shape[1])
    rc = lib().orc_modelspace_direct(G.shape[0], G.shape[1], _p(G), _p(w), float(lam), _p(dobs), _p(m),
                                     _nthreads(nthreads))
    if rc:
        raise np.linalg.LinAlgError(f"pivot {rc - 1} not positive")
    return m


class CGState:
    def __init__(self, x, r, p, rho):
        self.x, self.r, self.p, self.rho = x, r, p, float(rho)

    def copy(self):
        return CGState(self.x.copy(), self.r.copy(), self.p.copy(), self.rho)


def cg(w, lam, dobs, iters, G=None, mesh=None, obs=None, gamma=None, state=None, reverse=False, nthreads=None):
    """Textbook CG on (G W^-2 G^T + lam I) alpha = dobs (reading C8).

    G given: reuse the tabulated matrix; else matrix-free through the per-prism loops (needs mesh, obs, gamma).
    state=None: start from x=0, r=p=dobs.  Returns (CGState, hist[iters+1], ab[iters,2]).
    """
    w, dobs = _f64(w), _f64(dobs)
    N, M = dobs.size, w.size
    if state is None:
        st = CGState(np.zeros(N), np.zeros(N), np.zeros(N), 0.0)
        start = 1
    else:
        st = state.copy()
        start = 0
    hist = np.zeros(iters + 1)
    ab = np.zeros((max(iters, 1), 2))
    rho = C.c_double(st.rho)
    if G is not None:
        G = _f64(G)
        margs = [0, 0, 0, None, None, None, None, None, None, 0.0]
        gp = _p(G)
    else:
        xo, yo, zo = [_f64(a) for a in obs]
        margs = mesh.cargs() + [_p(xo), _p(yo), _p(zo), float(gamma)]
        gp = None
    lib().orc_cg(N, M, gp, *margs, _p(w), float(lam), _p(dobs), int(iters), start, _p(st.x), _p(st.r), _p(st.p),
                 C.byref(rho), _p(hist), _p(ab), int(bool(reverse)), _nthreads(nthreads))
    st.rho = rho.value
    return st, hist, ab[:iters]


def recover_model(G, w, alpha, nthreads=None):
    """m = W^-2 G^T alpha (Eq. 11)."""
    return dense_rmatvec(G, alpha, nthreads) / (_f64(w) ** 2)


def pcg(G, w, lam, dobs, iters, diag=None, rtol=0.0, state=None, nthreads=None):
    """Jacobi-preconditioned CG on (G W^-2 G^T + lam I) alpha = dobs with M = diag + lam (
    P:162), diag = gram_diag(G, w); diag=None is plain CG.  Stops after the iteration with ||r|| <= rtol ||dobs||.
    Returns (CGState with rho = r.z, hist[its+1] of ||r||_2, ab[its,2], its)."""
    G, w, dobs = _f64(G), _f64(w), _f64(dobs)
    N, M = G.shape
    if state is None:
        st, start = CGState(np.zeros(N), np.zeros(N), np.zeros(N), 0.0), 1
    else:
        st, start = state.copy(), 0
    hist = np.zeros(iters + 1)
    ab = np.zeros((max(iters, 1), 2))
    rho = C.c_double(st.rho)
    dg = None if diag is None else _f64(diag)
    its = lib().orc_pcg(N, M, _p(G), _p(w), float(lam), _p(dg), _p(dobs), int(iters), float(rtol), start, _p(st.x),
                        _p(st.r), _p(st.p), C.byref(rho), _p(hist), _p(ab), _nthreads(nthreads))
    st.rho = rho.value
    return st, hist[:its + 1], ab[:its], its


def invert(G, w, lam, dobs, mref=None, max_outer=30, max_inner=20, tol_outer=1e-4, tol_inner=1e-4, diag=None,
           nthreads=None, details=False):
    """The paper's outer model-update loop around the data-space update of Eq. 10-11,
    with a tabulated G (oracle.cpp orc_invert).  PARITY UNPINNED against the paper: it prints neither the residual
    norm nor the backtracking rule, so this follows readings R1-R4 of DESIGN.md 5.7 step by step.

    Returns (m, d_pred, hist, steps): hist[k] = ||r_k|| / ||d_obs||, steps[k] = accepted s of update k; with
    details=True also a dict(inner=CG iterations per update, trials=||r_k - 2^-h G dm||^2 per trial made,
    rejected=True when the loop ended on "no decrease")."""
    G, w, dobs = _f64(G), _f64(w), _f64(dobs)
    N, M = G.shape
    mr = None if mref is None else _f64(mref)
    dg = None if diag is None else _f64(diag)
    m, dpred = np.empty(M), np.empty(N)
    hist, steps = np.zeros(max_outer + 1), np.zeros(max(max_outer, 1))
    inner = (C.c_int * max(max_outer, 1))()
    trials = np.full((max(max_outer, 1), 11), np.nan)
    k = lib().orc_invert(N, M, _p(G), _p(w), float(lam), _p(dg), _p(dobs), _p(mr), int(max_outer), int(max_inner),
                         float(tol_outer), float(tol_inner), _p(m), _p(dpred), _p(hist), _p(steps), inner, _p(trials),
                         _nthreads(nthreads))
    out = (m, dpred, hist[:k + 1], steps[:k])
    if details:
        tried = k + (1 if k < max_outer and not np.isnan(trials[k, 0]) else 0) if max_outer else 0
        out += (dict(inner=np.array(inner[:tried]), trials=trials[:tried], rejected=tried > k),)
    return out
