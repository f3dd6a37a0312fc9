"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same seeded
inputs.  Tolerances (BASELINE.json north_star):
  forward / adjoint / stored entries : max |gpu - oracle| <= 1e-10 * max |oracle|   (reading C15: global max)
  CG                                  : protocol P1-P5 of SURVEY.md 8(c), 1e-8 relative where well-posed
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_03857_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_OP = 1e-10
TOL_CG = 1e-8


def relmax(a, b):
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(np.asarray(b)).max())


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def make_ctx(wl, mode=0):
    from paper_2602_03857_b200 import binding
    return binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=0, mode=mode)


@pytest.fixture(scope="module")
def c1(cfg1):
    ctx = make_ctx(cfg1["wl"], mode=1)
    yield ctx
    ctx.close()


# ---- operators, config 1 (full oracle) -----------------------------------------------------------------------
def test_forward_cfg1(cfg1, c1):
    wl, G = cfg1["wl"], cfg1["G"]
    u_w, _, _ = wl.test_vectors()
    for u in (np.ones(wl.M), wl.m_true, u_w):
        ref = oracle.dense_matvec(G, u)
        got = host(c1.forward(dev(u)))
        assert relmax(got, ref) <= TOL_OP


def test_adjoint_cfg1(cfg1, c1):
    wl, G = cfg1["wl"], cfg1["G"]
    _, v_w, v_s = wl.test_vectors()
    for v in (cfg1["d_obs"], v_s, v_w):
        ref = oracle.dense_rmatvec(G, v)
        got = host(c1.adjoint(dev(v)))
        assert relmax(got, ref) <= TOL_OP


def test_dot_product_test_gpu(cfg1, c1):
    wl = cfg1["wl"]
    u, v, _ = wl.test_vectors()
    d = host(c1.forward(dev(u)))
    g = host(c1.adjoint(dev(v)))
    a, b = float(d @ v), float(u @ g)
    assert abs(a - b) <= 1e-12 * np.linalg.norm(d) * np.linalg.norm(v)


def test_depth_weights_cfg1(cfg1, c1):
    wl = cfg1["wl"]
    for beta, z0 in ((2.0, 25.0), (3.0, 10.0), (0.0, 1.0)):
        ref = oracle.depth_weights(cfg1["mesh"], beta, z0)
        got = host(c1.depth_weights(beta, z0))
        assert np.abs(got / ref - 1).max() <= 4e-16


def test_gram_diag_cfg1(cfg1, c1):
    got = host(c1.gram_diag(dev(cfg1["w"])))
    assert np.abs(got / cfg1["diag"] - 1).max() <= 1e-11


def test_stored_g_cfg1(cfg1, c1):
    wl, G = cfg1["wl"], cfg1["G"]
    u, v, _ = wl.test_vectors()
    c1.store_g(fp32=False)
    Gd = host(c1.stored_g())
    assert relmax(Gd, G) <= TOL_OP
    assert relmax(host(c1.forward_stored(dev(u))), oracle.dense_matvec(G, u)) <= TOL_OP
    assert relmax(host(c1.adjoint_stored(dev(v))), oracle.dense_rmatvec(G, v)) <= TOL_OP
    c1.store_g(fp32=True)
    G32 = host(c1.stored_g())
    assert G32.dtype == np.float32
    assert np.array_equal(G32, Gd.astype(np.float32)) or relmax(G32, G) <= 1e-7
    # FP32 storage error is reported, not gated at 1e-10: bounded by float rounding of the entries
    assert relmax(host(c1.forward_stored(dev(u))), oracle.dense_matvec(G, u)) <= 2e-7
    assert relmax(host(c1.adjoint_stored(dev(v))), oracle.dense_rmatvec(G, v)) <= 2e-7
    c1.store_g(fp32=False)


# ---- ragged / irregular small workloads (several tiles, ragged tails, stretched mesh, topography) -------------
@pytest.mark.parametrize("shape", [(1, 1, 1, 1), (2, 3, 1, 5), (5, 7, 4, 23), (13, 9, 11, 301), (7, 20, 33, 130),
                                   (3, 3, 70, 257)])
def test_ragged_workloads(shape):
    nx, ny, nz, nobs = shape
    wl = workloads.make_custom(nx, ny, nz, 30.0, nobs, seed=11 + nx, topo_amp=40.0)
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    ctx = make_ctx(wl, mode=1)
    rng = np.random.default_rng(5)
    u, v = wl.m_true, rng.standard_normal(wl.N)
    d_ref = oracle.forward(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, u)
    g_ref = oracle.adjoint(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, v)
    assert relmax(host(ctx.forward(dev(u))), d_ref) <= TOL_OP
    assert relmax(host(ctx.adjoint(dev(v))), g_ref) <= TOL_OP
    ctx.store_g()
    assert relmax(host(ctx.stored_g()), oracle.tabulate(mesh, wl.xo, wl.yo, wl.zo, wl.gamma)) <= TOL_OP
    assert relmax(host(ctx.forward_stored(dev(u))), d_ref) <= TOL_OP
    assert relmax(host(ctx.adjoint_stored(dev(v))), g_ref) <= TOL_OP
    w = oracle.depth_weights(mesh, 2.0, wl.z0)
    G = oracle.tabulate(mesh, wl.xo, wl.yo, wl.zo, wl.gamma)
    assert np.abs(host(ctx.gram_diag(dev(w))) / oracle.gram_diag(G, w) - 1).max() <= 1e-10
    ctx.close()


def test_stations_inside_and_below_mesh():
    """Stations below the mesh top (Z < 0 for some nodes: borehole-like) and exactly on node planes / edges:
    principal-value atan (C3) and the guards of C6."""
    wl = workloads.make_custom(4, 4, 4, 10.0, 6, seed=2)
    wl.xo = np.array([5.0, 10.0, 20.0, 13.0, 0.0, -7.0])      # 10, 20, 0 are node x-planes
    wl.yo = np.array([4.0, 8.0, 3.0, 16.0, 0.0, 50.0])        # 8, 16, 0 are node y-planes
    wl.zo = np.array([15.0, 10.0, -2.0, 47.0, -1.0, 20.0])    # inside cells, on a node z-plane, below everything
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    ctx = make_ctx(wl)
    u = wl.m_true
    ref = oracle.forward(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, u)
    got = host(ctx.forward(dev(u)))
    assert np.all(np.isfinite(got))
    assert relmax(got, ref) <= TOL_OP
    v = np.array([1.0, -2.0, 0.5, 3.0, -1.0, 2.0])
    assert relmax(host(ctx.adjoint(dev(v))), oracle.adjoint(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, v)) <= TOL_OP
    ctx.close()


# ---- CG, config 1: protocol P1-P5 ------------------------------------------------------------------------------
def test_cg_cfg1_protocol(cfg1, c1):
    from paper_2602_03857_b200 import binding
    wl, G, w, lam, d = cfg1["wl"], cfg1["G"], cfg1["w"], cfg1["lam"], cfg1["d_obs"]
    wd, dd = dev(w), dev(d)
    # P2 prefix parity: first 5 iterates
    st5, hist5, ab5 = oracle.cg(w, lam, d, 5, G=G)
    r5 = c1.dataspace_cg(dd, wd, lam, 5)
    assert relmax(host(r5["alpha"]), st5.x) <= TOL_CG
    assert np.abs(host(r5["hist"]) / hist5 - 1).max() <= TOL_CG
    assert np.abs(host(r5["ab"]) / ab5 - 1).max() <= TOL_CG
    # P1 step parity: inject the oracle's state at j, run ONE GPU iteration
    for j in (0, 1, 10, 49):
        stj, _, _ = oracle.cg(w, lam, d, j, G=G)
        nxt, _, abn = oracle.cg(w, lam, d, 1, G=G, state=stj)
        gs = binding.CGState(wl.N, c1.device, x=stj.x, r=stj.r, p=stj.p, rho=stj.rho)
        out = c1.dataspace_cg(dd, wd, lam, 1, state=gs, want_m=False)
        assert np.abs(host(out["ab"])[0] / abn[0] - 1).max() <= 1e-9
        assert relmax(host(gs.x), nxt.x) <= 1e-9
        assert np.abs(host(gs.r) - nxt.r).max() <= 1e-9 * np.abs(d).max()
        assert np.abs(host(gs.p) - nxt.p).max() <= 1e-9 * np.abs(d).max()
        assert abs(float(gs.rho.item()) / nxt.rho - 1) <= 1e-8
    # P3 converged parity: k = 50 (config's count) and k = 100 vs oracle CG and oracle Cholesky
    alpha_dir, m_dir = oracle.dataspace_direct(G, w, lam, d)
    st50, hist50, _ = oracle.cg(w, lam, d, 50, G=G)
    r50 = c1.dataspace_cg(dd, wd, lam, 50)
    assert relmax(host(r50["alpha"]), st50.x) <= TOL_CG
    assert relmax(host(r50["alpha"]), alpha_dir) <= 5e-8      # CG truncation itself is 2.5e-9
    assert relmax(host(r50["m"]), oracle.recover_model(G, w, st50.x)) <= TOL_CG
    r100 = c1.dataspace_cg(dd, wd, lam, 100)
    assert relmax(host(r100["alpha"]), alpha_dir) <= TOL_CG
    assert relmax(host(r100["m"]), m_dir) <= TOL_CG
    # P4 fixed-k report against the oracle's own reorder sensitivity
    st50r, _, _ = oracle.cg(w, lam, d, 50, G=G, reverse=True)
    self_sens = relmax(st50r.x, st50.x)
    assert relmax(host(r50["alpha"]), st50.x) <= max(TOL_CG, 10 * self_sens)
    # P5 invariants: true residual vs recursive residual
    A = oracle.form_A(G, w, lam)
    true_res = np.linalg.norm(d - A @ host(r50["alpha"])) / np.linalg.norm(d)
    rec_res = host(r50["hist"])[-1] / np.linalg.norm(d)
    assert abs(true_res - rec_res) <= 1e-6 * max(true_res, 1e-9) + 1e-12
    # stored-G CG follows the same iterates
    c1.store_g()
    s50 = c1.dataspace_cg(dd, wd, lam, 50, mode=1)
    assert relmax(host(s50["alpha"]), st50.x) <= TOL_CG
    assert relmax(host(s50["m"]), oracle.recover_model(G, w, st50.x)) <= TOL_CG


def test_cg_rtol_freeze(cfg1, c1):
    w, lam, d = cfg1["w"], cfg1["lam"], cfg1["d_obs"]
    out = c1.dataspace_cg(dev(d), dev(w), lam, 60, rtol=1e-6)
    hist = host(out["hist"])
    k = int(np.argmax(hist <= 1e-6 * hist[0]))
    assert 0 < k < 60
    assert np.all(hist[k:] == hist[k])            # frozen after reaching the tolerance
    # the frozen result is exactly the k-iteration result of the same solver, and close to the oracle's k-th iterate
    fixed = c1.dataspace_cg(dev(d), dev(w), lam, k)
    assert np.array_equal(host(out["alpha"]), host(fixed["alpha"]))
    assert np.array_equal(host(out["m"]), host(fixed["m"]))
    ref, _, _ = oracle.cg(w, lam, d, k, G=cfg1["G"])
    assert relmax(host(out["alpha"]), ref.x) <= 1e-4


def test_direct_solve_cfg1(cfg1, c1):
    w, lam, d = cfg1["w"], cfg1["lam"], cfg1["d_obs"]
    c1.store_g()
    alpha, m = c1.direct_solve(dev(d), dev(w), lam)
    a_ref, m_ref = oracle.dataspace_direct(cfg1["G"], w, lam, d)
    assert relmax(host(alpha), a_ref) <= TOL_CG
    assert relmax(host(m), m_ref) <= TOL_CG


def test_host_entry_points(cfg1, c1):
    wl, w, lam, d = cfg1["wl"], cfg1["w"], cfg1["lam"], cfg1["d_obs"]
    u, v, _ = wl.test_vectors()
    up = torch.as_tensor(u).pin_memory()
    dh = torch.empty(wl.N, dtype=torch.float64).pin_memory()
    c1.forward_host(up, dh)
    assert np.array_equal(dh.numpy(), host(c1.forward(dev(u))))
    gh = np.empty(wl.M)
    c1.adjoint_host(np.ascontiguousarray(v), gh)
    assert np.array_equal(gh, host(c1.adjoint(dev(v))))
    ah, mh, hh = np.empty(wl.N), np.empty(wl.M), np.empty(11)
    c1.dataspace_cg_host(np.ascontiguousarray(d), wl.beta, wl.z0, lam, 10, ah, mh, hh)
    ref = c1.dataspace_cg(dev(d), c1.depth_weights(wl.beta, wl.z0), lam, 10)
    assert np.array_equal(ah, host(ref["alpha"])) and np.array_equal(mh, host(ref["m"]))
    assert np.array_equal(hh, host(ref["hist"]))


def test_determinism(cfg1, c1):
    wl = cfg1["wl"]
    u, v, _ = wl.test_vectors()
    a = host(c1.forward(dev(u)))
    b = host(c1.forward(dev(u)))
    assert np.array_equal(a, b)
    a = host(c1.adjoint(dev(v)))
    b = host(c1.adjoint(dev(v)))
    assert np.array_equal(a, b)


def test_error_paths(cfg1, c1):
    from paper_2602_03857_b200 import binding
    wl = cfg1["wl"]
    with pytest.raises(binding.GravError):
        binding.GravContext(wl.xn[::-1].copy(), wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma)   # decreasing nodes
    with pytest.raises(ValueError):
        c1.forward(torch.zeros(wl.M - 1, dtype=torch.float64, device="cuda"))
    with pytest.raises(binding.GravError):
        c1.dataspace_cg(dev(cfg1["d_obs"]), dev(cfg1["w"]), 1.0, 3, mode=7)
    fresh = make_ctx(wl)
    with pytest.raises(binding.GravError) as ei:
        fresh.forward_stored(dev(np.ones(wl.M)))
    assert ei.value.status == -4
    fresh.close()


def test_libm_variant_matches(cfg1):
    """The CUDA-libm evaluator (variant 1) and the hand-built one (variant 0, default) both match the oracle."""
    wl, G = cfg1["wl"], cfg1["G"]
    u, v, _ = wl.test_vectors()
    ctx = make_ctx(wl, mode=1)
    ctx.set_psi_variant(1)
    assert relmax(host(ctx.forward(dev(u))), oracle.dense_matvec(G, u)) <= TOL_OP
    assert relmax(host(ctx.adjoint(dev(v))), oracle.dense_rmatvec(G, v)) <= TOL_OP
    ctx.store_g()
    assert relmax(host(ctx.stored_g()), G) <= TOL_OP
    ctx.close()


@pytest.mark.parametrize("shape", [(9, 7, 12, 700), (3, 4, 70, 300), (2, 2, 1100, 40), (6, 5, 8, 333), (4, 6, 11, 90),
                                   (5, 3, 3, 64)])
def test_launch_variants_against_oracle(shape):
    """Both log tables (256-entry and exponent-and-mantissa), the CUDA-libm evaluator and every compiled KC of the
    adjoint kernel against the oracle, on ragged cases spanning several station tiles, several staged column tiles and
    a column deeper than the stage buffer (nz + 1 > 1024: unstaged fallback).  nz + 1 = 13, 71, 9, 12, 4 make the plan
    pick KC = 5, 8, 5, 6, 4 (csrc/grav_api.cu make_plan)."""
    nx, ny, nz, nobs = shape
    wl = workloads.make_custom(nx, ny, nz, 17.0, nobs, seed=5 + nz, topo_amp=25.0)
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    rng = np.random.default_rng(nz)
    u, v = rng.standard_normal(wl.M), rng.standard_normal(wl.N)
    d_ref = oracle.forward(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, u)
    g_ref = oracle.adjoint(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, v)
    G_ref = oracle.tabulate(mesh, wl.xo, wl.yo, wl.zo, wl.gamma) if wl.N * wl.M <= 4e6 else None
    ctx = make_ctx(wl, mode=1 if G_ref is not None else 0)
    # the 2-D log table exists for all but the 1100-layer mesh, which is 5e5 m deep under stations 1 m above it
    # (4 Rmax^2 / Zmin^2 > 2^40); it is the default only from 5e7 evaluations per product
    assert (ctx.log2d_binades > 0) == (nz < 1000) and not ctx.log2d_default
    for log2d in (0, 1):
        if log2d and ctx.log2d_binades == 0:
            with pytest.raises(Exception):
                ctx.set_log2d(1)
            continue
        ctx.set_log2d(log2d)
        assert relmax(host(ctx.forward(dev(u))), d_ref) <= TOL_OP, f"forward log2d={log2d}"
        assert relmax(host(ctx.adjoint(dev(v))), g_ref) <= TOL_OP, f"adjoint log2d={log2d}"
        if G_ref is not None:
            ctx.store_g()
            assert relmax(host(ctx.stored_g()), G_ref) <= TOL_OP, f"tabulate log2d={log2d}"
    ctx.close()


@pytest.mark.parametrize("shape", [(30, 34, 32, 1400), (26, 28, 50, 1500), (30, 26, 64, 1100), (10, 11, 150, 2800),
                                   (44, 50, 20, 1300)])
def test_default_paths_of_large_problems_on_midsize_shapes(shape):
    """Problems just above 5e7 evaluations per product take the code paths of the large configs by DEFAULT - the 2-D log
    table, the persistent launch, the (threads, KC) table of the adjoint: nz + 1 = 33, 51, 65, 151, 21 make make_plan
    pick KC = 11, 17, 13, 7 (column padded to 154) and 7 - yet stay small enough for oracle rows and columns: forward on
    sampled stations x all prisms, adjoint on sampled prisms (corners included) x all stations, Gram diagonal on sampled
    stations, and bit-identical repeats."""
    nx, ny, nz, nobs = shape
    wl = workloads.make_custom(nx, ny, nz, 35.0, nobs, seed=nz, topo_amp=50.0)
    assert wl.N * wl.n_nodes >= 5e7
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    rng = np.random.default_rng(nz)
    u, v = rng.standard_normal(wl.M), rng.standard_normal(wl.N)
    ctx = make_ctx(wl)
    assert ctx.log2d_default
    d, g = host(ctx.forward(dev(u))), host(ctx.adjoint(dev(v)))
    st = rng.choice(wl.N, size=40, replace=False)
    cells = np.unique(np.concatenate([rng.choice(wl.M, size=300, replace=False), [0, nz - 1, wl.M - nz, wl.M - 1]]))
    d_ref = oracle.forward(mesh, wl.xo[st], wl.yo[st], wl.zo[st], wl.gamma, u)
    g_ref = oracle.adjoint(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, v, cells=cells)
    assert np.abs(d[st] - d_ref).max() <= TOL_OP * np.abs(d).max()
    assert np.abs(g[cells] - g_ref).max() <= TOL_OP * np.abs(g).max()
    w = ctx.depth_weights(2.0, wl.z0)
    G6 = oracle.tabulate(mesh, wl.xo[st[:6]], wl.yo[st[:6]], wl.zo[st[:6]], wl.gamma)
    assert np.abs(host(ctx.gram_diag(w))[st[:6]] / oracle.gram_diag(G6, host(w)) - 1).max() <= 1e-10
    assert np.array_equal(host(ctx.forward(dev(u))), d) and np.array_equal(host(ctx.adjoint(dev(v))), g)
    ctx.close()


def test_survey_coordinates_with_large_offsets():
    """UTM-like coordinates (x ~ 5e5 m, y ~ 4e6 m, mesh top 1,250 m below datum): the kernels work on corner-minus-station
    differences, the exponent offset k0 and the log-table range come from distances, not from the absolute coordinates."""
    from paper_2602_03857_b200 import binding
    wl = workloads.make_custom(7, 6, 9, 40.0, 150, seed=21, topo_amp=60.0)
    xn, yn, zn = wl.xn + 512345.25, wl.yn + 4187654.5, wl.zn + 1250.0
    xo, yo, zo = wl.xo + 512345.25, wl.yo + 4187654.5, wl.zo + 1250.0
    mesh = oracle.Mesh(xn, yn, zn)
    rng = np.random.default_rng(8)
    u, v = rng.standard_normal(wl.M), rng.standard_normal(wl.N)
    ctx = binding.GravContext(xn, yn, zn, xo, yo, zo, wl.gamma, device=0)
    assert ctx.log2d_binades > 0
    for log2d in (0, 1):                                      # 256-entry table (small problem default) and 2-D table
        ctx.set_log2d(log2d)
        assert relmax(host(ctx.forward(dev(u))), oracle.forward(mesh, xo, yo, zo, wl.gamma, u)) <= TOL_OP
        assert relmax(host(ctx.adjoint(dev(v))), oracle.adjoint(mesh, xo, yo, zo, wl.gamma, v)) <= TOL_OP
    ctx.close()


def test_log2d_admissibility():
    """The exponent-and-mantissa log table is used only when the geometry bounds R+Y, R+X inside 40 binades: stations
    above the mesh enable it; stations level with a node layer (Z = 0 occurs) or 0.1 mm above the top (ratio 4 Rmax^2 /
    Zmin^2 > 2^40) disable it, and the results stay within tolerance either way (the guards of reading C6 live in the
    256-entry evaluator)."""
    from paper_2602_03857_b200 import binding
    base = workloads.make_custom(5, 4, 6, 10.0, 40, seed=3)
    mesh = oracle.Mesh(base.xn, base.yn, base.zn)
    u = np.random.default_rng(0).standard_normal(base.M)
    cases = ((base.zo, True), (np.full_like(base.zo, base.zn[2]), False), (np.full_like(base.zo, -1e-4), False))
    for zo, expect in cases:
        ctx = binding.GravContext(base.xn, base.yn, base.zn, base.xo, base.yo, zo, base.gamma, device=0)
        assert (ctx.log2d_binades > 0) == expect
        ref = oracle.forward(mesh, base.xo, base.yo, zo, base.gamma, u)
        assert relmax(host(ctx.forward(dev(u))), ref) <= TOL_OP
        g_ref = oracle.adjoint(mesh, base.xo, base.yo, zo, base.gamma, ref)
        assert relmax(host(ctx.adjoint(dev(ref))), g_ref) <= TOL_OP
        ctx.close()
    # stations INSIDE the mesh, between two node layers (3 m below layer 2): Z changes sign down a column but never
    # vanishes, so the table is admissible; force the 2-D variants and compare with the oracle (reading C3)
    zo = np.full_like(base.zo, base.zn[2] + 3.0)
    ctx = binding.GravContext(base.xn, base.yn, base.zn, base.xo, base.yo, zo, base.gamma, device=0)
    assert ctx.log2d_binades > 0
    ref = oracle.forward(mesh, base.xo, base.yo, zo, base.gamma, u)
    g_ref = oracle.adjoint(mesh, base.xo, base.yo, zo, base.gamma, ref)
    for log2d in (0, 1):
        ctx.set_log2d(log2d)
        assert relmax(host(ctx.forward(dev(u))), ref) <= TOL_OP
        assert relmax(host(ctx.adjoint(dev(ref))), g_ref) <= TOL_OP
    ctx.close()


class _TwinComm:
    """Stand-in for a 2-rank communicator whose other rank holds the SAME stations: an all-reduce doubles the buffer,
    an all-gather places two copies of the send buffer.  Runs on the stream it is handed."""

    def __init__(self, device):
        from paper_2602_03857_b200 import dist as gdist
        self._c = gdist.Comm(device)
        self.world, self.rank, self.calls = 2, 0, []

    def allreduce_sum(self, ptr, count, stream):
        with self._c._on(stream):
            self._c.view(ptr, count).mul_(2.0)
        self.calls.append(("allreduce", count))

    def allgather(self, send, recv, count, stream):
        with self._c._on(stream):
            r = self._c.view(recv, 2 * count)
            r[:count].copy_(self._c.view(send, count))
            r[count:].copy_(self._c.view(send, count))
        self.calls.append(("allgather", count))


def test_comm_exchange_placement(cfg1):
    """Observation sharding (include/grav.h: grav_set_comm).  Two IDENTICAL ranks, each holding the same stations S,
    form the global system [G_S; G_S].  By symmetry the sharded CG must then reproduce the single-rank CG of the problem
    with gamma*sqrt(2) (A = 2 G W^-2 G^T + lambda I): same alpha, residual history and model larger by sqrt(2).  Every
    exchange point has to be hooked for this to hold."""
    from paper_2602_03857_b200 import binding
    wl, w, lam, d = cfg1["wl"], cfg1["w"], cfg1["lam"], cfg1["d_obs"]
    its = 8
    for mode in (0, 1):
        sh = make_ctx(wl, mode=mode)
        comm = _TwinComm(sh.device)
        sh.set_comm(comm)
        ref = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma * np.sqrt(2.0), device=0,
                                  mode=mode)
        if mode == 1:
            sh.store_g()
            ref.store_g()
        comm.calls.clear()
        a = sh.dataspace_cg(dev(d), dev(w), lam, its, mode=mode)
        b = ref.dataspace_cg(dev(d), dev(w), lam, its, mode=mode)
        # the two runs differ by rounding only (gamma*sqrt(2) is rounded), amplified over 8 CG iterations
        # (~1e-9 at this depth); a missing or misplaced exchange changes the iterates at O(1)
        assert relmax(host(a["alpha"]), host(b["alpha"])) <= 1e-7
        assert np.abs(host(a["hist"]) / (np.sqrt(2.0) * host(b["hist"])) - 1).max() <= 1e-7
        assert relmax(host(a["m"]), np.sqrt(2.0) * host(b["m"])) <= 1e-7
        # node sums travel as gathered (hi, lo) planes, the stored-mode M-vector as an all-reduce
        big = ("allgather", 2 * wl.n_nodes) if mode == 0 else ("allreduce", wl.M)
        # [r.z | d.d | r.r], then per iteration: operator output, p.q, [r.z | r.r]; finally the model recovery
        assert comm.calls == [("allreduce", 768)] + [big, ("allreduce", 256), ("allreduce", 512)] * its + [big]
        # the adjoint is global (summed over the two ranks), the forward stays local
        v = cfg1["d_obs"]
        comm.calls.clear()
        g2 = host(sh.adjoint(dev(v)) if mode == 0 else sh.adjoint_stored(dev(v)))
        assert comm.calls == [big]
        sh.set_comm(None)
        if mode == 1:
            sh.store_g()
        g1 = host(sh.adjoint(dev(v)) if mode == 0 else sh.adjoint_stored(dev(v)))
        assert np.array_equal(g2, 2.0 * g1) and len(comm.calls) == 1
        with_hook_fwd = host(sh.forward(dev(wl.m_true)))
        assert relmax(with_hook_fwd, np.sqrt(0.5) * host(ref.forward(dev(wl.m_true)))) <= 1e-13
        sh.close()
        ref.close()
