"""The device Psi evaluators against the oracle's Psi (Eq. 2-3), argument by argument on the GPU
(grav_debug_psi_eval_device: MUFU seeds, shared-memory tables and all), and the Float32 matrix-free mode
(grav_set_precision; "using Float32 precision") against the FP64 oracle with the
error bound its arithmetic gives.

FP64 evaluators (hand-built with either log table, CUDA libm): error <= 1e-15 of the size of the three terms plus the
amplification of the rounding of R in R + Y that the plain formula has too (the scaling tests/test_fastmath_host.py
uses for the host emulation of the same source).  Float32: every term is rounded to 2^-24 relative, so
|err| <= C 2^-24 (|Z| pi/2 + |X ln| + |Y ln|) with a small C - and NO amplification term, because the evaluator forms
R + Y without the cancelling subtraction."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2602_03857_b200 import workloads

pytestmark = pytest.mark.gpu

LN2 = math.log(2.0)
EPS32 = 2.0 ** -24


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def host(t):
    return t.detach().cpu().numpy()


@pytest.fixture(scope="module")
def ctx():
    """A context whose geometry admits the 2-D log table with a wide range (stations 1 m above a 20 km mesh)."""
    from paper_2602_03857_b200 import binding
    xn = np.linspace(0.0, 20000.0, 5)
    zn = np.linspace(0.0, 8000.0, 5)
    xo = np.array([10.0, 19990.0, 10000.0])
    c = binding.GravContext(xn, xn, zn, xo, xo[::-1].copy(), np.full(3, -1.0), 6.674e-6, device=0)
    assert c.log2d_binades > 0
    yield c
    c.close()


def _args(rng, scale, n):
    X = rng.uniform(-scale, scale, n)
    Y = rng.uniform(-scale, scale, n)
    Z = rng.uniform(-1, 1, n) * scale * rng.choice([1, 0.01, 1e-3], n)
    return X, Y, Z


def _ref(X, Y, Z):
    return np.array([oracle.psi(x, y, z, 1) for x, y, z in zip(X, Y, Z)])       # long-double Psi


def _mag(X, Y, Z):
    R = np.sqrt(X * X + Y * Y + Z * Z)
    return np.abs(Z) * np.pi / 2 + np.abs(X * np.log(R + Y)) + np.abs(Y * np.log(R + X)), R


@pytest.mark.parametrize("variant", [0, 1, 3], ids=["table256", "libm", "log2d"])
def test_fp64_evaluators_on_device(ctx, variant):
    k0 = ctx.k0 if variant != 1 else 0
    rng = np.random.default_rng(40 + variant)
    worst = 0.0
    for scale in (30.0, 1e3, 1.5e4):          # 2 R stays inside the context's 2-D log table (Rmax = 29.4 km)
        X, Y, Z = _args(rng, scale, 3000)
        if variant == 3:      # arguments of the logarithms must lie inside the context's table: R + Y >= Zmin^2 / (2 Rmax)
            Z = np.where(np.abs(Z) < 1.0, np.copysign(1.0, Z) + Z, Z)
        got = host(ctx.psi_eval_device(variant, dev(X), dev(Y), dev(Z))) - (X + Y) * k0 * LN2
        mag, R = _mag(X, Y, Z)
        amp = np.abs(X) * R / (R + Y) + np.abs(Y) * R / (R + X)
        err = np.abs(got - _ref(X, Y, Z)) / (mag + amp + np.abs(X + Y) * abs(k0) * LN2)
        worst = max(worst, float(err.max()))
    print(f"variant {variant}: worst scaled error {worst:.2e}")
    assert worst <= (1e-15 if variant != 1 else 3e-15)


def test_fp64_guards_on_device(ctx):
    """Reading C6 on the device: Z = 0, X = 0, Y = 0, the station on a node, all finite and equal to the oracle's."""
    pts = np.array([(0, 0, 0), (0, -5, 0), (2, 3, 0), (0, 0, 5), (1, 1, 1), (3, -4, 0), (-3, 4, 1e-9), (0, 5, 2),
                    (5, 0, 2), (-5, 0, -2), (7, 7, 7), (7, -7, -7)], dtype=np.float64)
    X, Y, Z = (np.ascontiguousarray(pts[:, k]) for k in range(3))
    ref = _ref(X, Y, Z)
    for variant in (0, 1):
        k0 = ctx.k0 if variant == 0 else 0
        got = host(ctx.psi_eval_device(variant, dev(X), dev(Y), dev(Z))) - (X + Y) * k0 * LN2
        assert np.all(np.isfinite(got))
        assert (np.abs(got - ref) <= 1e-15 * np.maximum(1.0, np.abs(ref)) + 1e-14 * np.abs(X + Y) * abs(k0)).all()


def test_f32_evaluator_on_device(ctx):
    k0 = max(-100, min(100, ctx.k0))
    rng = np.random.default_rng(44)
    for scale in (30.0, 1e3, 2e4):
        X, Y, Z = _args(rng, scale, 3000)
        # the evaluator sees Float32 arguments: compare at exactly those
        X, Y, Z = (a.astype(np.float32).astype(np.float64) for a in (X, Y, Z))
        got = host(ctx.psi_eval_device(2, dev(X), dev(Y), dev(Z))) - (X + Y) * k0 * LN2
        R = np.sqrt(X * X + Y * Y + Z * Z)
        # term sizes with the logarithms as evaluated: ln((R + Y) / 2^k0)
        mag = np.abs(Z) * np.pi / 2 + np.abs(X) * (np.abs(np.log(R + Y) - k0 * LN2) + 1) + \
            np.abs(Y) * (np.abs(np.log(R + X) - k0 * LN2) + 1)
        err = np.abs(got - _ref(X, Y, Z)) / mag
        assert err.max() <= 8 * EPS32, err.max()
    # the cancelling corner Y -> -R: FP32 R + Y would be garbage; the evaluator's form is not
    X, Y, Z = np.full(64, 1.0), -np.logspace(1, 4.5, 64), np.full(64, 2.0)
    X, Y, Z = (a.astype(np.float32).astype(np.float64) for a in (X, Y, Z))
    got = host(ctx.psi_eval_device(2, dev(X), dev(Y), dev(Z))) - (X + Y) * k0 * LN2
    R = np.sqrt(X * X + Y * Y + Z * Z)
    mag = np.abs(Z) * np.pi / 2 + np.abs(X) * (np.abs(np.log(R + Y) - k0 * LN2) + 1) + \
        np.abs(Y) * (np.abs(np.log(R + X) - k0 * LN2) + 1)
    assert np.all(np.isfinite(got)) and (np.abs(got - _ref(X, Y, Z)) / mag).max() <= 8 * EPS32
    # guards (reading C6)
    pts = np.array([(0, 0, 0), (0, -5, 0), (2, 3, 0), (0, 0, 5), (3, -4, 0), (0, 5, 2), (5, 0, 2)], dtype=np.float64)
    X, Y, Z = (np.ascontiguousarray(pts[:, k]) for k in range(3))
    got = host(ctx.psi_eval_device(2, dev(X), dev(Y), dev(Z))) - (X + Y) * k0 * LN2
    assert np.all(np.isfinite(got)) and np.abs(got - _ref(X, Y, Z)).max() <= 1e-4


@pytest.mark.parametrize("shape", [(16, 16, 8, 50.0, 256, 0.0), (13, 9, 11, 30.0, 301, 40.0), (7, 20, 33, 25.0, 130, 10.0)])
def test_f32_matrix_free_mode(shape):
    """grav_set_precision(F32): forward / adjoint / CG with the Float32 evaluator against the FP64 oracle.  The gate is the
    bound the arithmetic gives - per node |err| <= C 2^-24 (|X| + |Y| + |Z|) (|ln| + 2), summed with the node weights -
    evaluated from the geometry, and the observed error is printed."""
    from paper_2602_03857_b200 import binding
    nx, ny, nz, h, nobs, topo = shape
    wl = workloads.make(1) if nobs == 256 else workloads.make_custom(nx, ny, nz, h, nobs, seed=2, topo_amp=topo)
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=0)
    rng = np.random.default_rng(5)
    u = wl.m_true
    v = rng.standard_normal(wl.N)
    d64 = host(ctx.forward(dev(u)))
    g64 = host(ctx.adjoint(dev(v)))
    ctx.set_precision(True)
    d32 = host(ctx.forward(dev(u)))
    g32 = host(ctx.adjoint(dev(v)))
    d_ref = oracle.forward(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, u)
    g_ref = oracle.adjoint(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, v)
    L = math.sqrt((wl.xn[-1] - wl.xn[0]) ** 2 + (wl.yn[-1] - wl.yn[0]) ** 2 + (wl.zn[-1] - wl.zn[0]) ** 2) * 1.3
    # node weights c = S^T u: at most 8 |u| per node; per-evaluation bound 8 eps (3 L)(|ln(L / 2^k0)| + 3)
    per_eval = 8 * EPS32 * 3 * L * (abs(math.log(L) - ctx.k0 * LN2) + 3)
    n_nodes = (wl.nx + 1) * (wl.ny + 1) * (wl.nz + 1)
    bound_d = wl.gamma * per_eval * 8 * np.abs(u).max() * n_nodes
    bound_g = wl.gamma * per_eval * 8 * np.abs(v).sum()
    err_d, err_g = np.abs(d32 - d_ref).max(), np.abs(g32 - g_ref).max()
    print(f"{wl.name}: FP32 matrix-free forward err {err_d / np.abs(d_ref).max():.2e} of max (bound "
          f"{bound_d / np.abs(d_ref).max():.1e}), adjoint {err_g / np.abs(g_ref).max():.2e} (bound "
          f"{bound_g / np.abs(g_ref).max():.1e})")
    assert err_d <= bound_d and err_g <= bound_g
    assert err_d <= 1e-3 * np.abs(d_ref).max() and err_g <= 1e-2 * np.abs(g_ref).max()     # and it is a usable operator
    assert err_d > 1e-10 * np.abs(d_ref).max()                # it IS the Float32 evaluator (the FP64 path is below this)
    # a few CG iterations run with the Float32 operator and stay close to the FP64 ones
    w = ctx.depth_weights(2.0, wl.z0)
    d = d_ref + 0.02 * np.abs(d_ref).max() * rng.standard_normal(wl.N)
    lam = 1e-2 * float(host(ctx.gram_diag(w)).mean())
    c32 = ctx.dataspace_cg(dev(d), w, lam, 4)
    ctx.set_precision(False)
    c64 = ctx.dataspace_cg(dev(d), w, lam, 4)
    assert np.array_equal(host(ctx.forward(dev(u))), d64) and np.array_equal(host(ctx.adjoint(dev(v))), g64)
    rel = np.abs(host(c32["hist"]) / host(c64["hist"]) - 1).max()
    print(f"{wl.name}: CG residual history FP32 vs FP64: {rel:.2e}")
    assert rel <= 5e-2
    ctx.close()
