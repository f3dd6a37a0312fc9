"""grav_gemvt_noalloc (include/grav.h): the stored-G adjoint product g = [W^-2] G^T v (Eq. 10-11: the
G^T of the data-space update and the model recovery) with its scratch in the library's built-in device array instead of a
caller workspace - for callers that cannot allocate.  Checked against the existing path (grav_adjoint_stored on a context
with a workspace; tests/test_gpu_parity.py holds that one to the oracle) on calls in a row that SHARE the array: different
shapes back to back, so that contents left by the previous call would show, and the same call repeated.

The file sorts last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the others:
the array's address is looked up lazily per device and nothing depends on what earlier calls left in it."""
import numpy as np
import pytest
import torch

from paper_2602_03857_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-12          # of max |g|: the two paths run the same kernels in the same order (bit-equal in practice)

# (nx, ny, nz, h, nobs): 4 row chunks with a ragged last one and even M; one chunk, odd M (the scalar-column branch)
SHAPES = [(24, 20, 12, 40.0, 777), (7, 9, 5, 25.0, 130)]


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def relmax(a, b):
    return float((a - b).abs().max() / b.abs().max())


def _case(shape, seed, fp32):
    """G tabulated by the library (kept as a caller-held copy), vectors, and the existing path's results."""
    from paper_2602_03857_b200 import binding
    nx, ny, nz, h, nobs = shape
    wl = workloads.make_custom(nx, ny, nz, h, nobs, seed=seed, topo_amp=20.0)
    ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=0,
                              mode=binding.STORED_F32 if fp32 else binding.STORED_F64)
    ctx.store_g(fp32=fp32)
    G = ctx.stored_g().clone()
    rng = np.random.default_rng(seed)
    v = dev(rng.standard_normal(wl.N))
    w = ctx.depth_weights(2.0, wl.z0).clone()
    ref = ctx.adjoint_stored(v).clone()                       # existing path: scratch in the context's workspace
    ref_w = ref / (w * w)
    ctx.close()
    return G, v, w, ref, ref_w


@pytest.mark.parametrize("fp32", [False, True], ids=["f64", "f32"])
def test_no_alloc_gemvt_matches_the_workspace_path_on_calls_in_a_row(fp32):
    from paper_2602_03857_b200 import binding
    binding.noalloc_setup(0)
    cases = [_case(s, 11 + k, fp32) for k, s in enumerate(SHAPES)]
    outs = [torch.empty(c[0].shape[1], dtype=torch.float64, device="cuda") for c in cases]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    # two calls in a row on the shared array, large shape then small and back: no allocation in between
    for k in (0, 1, 0, 1):
        G, v, w, ref, ref_w = cases[k]
        outs[k].fill_(float("nan"))
        got = binding.gemvt_noalloc(G, v, out=outs[k])
        assert got.data_ptr() == outs[k].data_ptr()
        assert relmax(got, ref) <= TOL, (k, relmax(got, ref))
        got = binding.gemvt_noalloc(G, v, w=w, out=outs[k])   # with the W^-2 scaling fused, straight after
        assert relmax(got, ref_w) <= TOL * 10                 # (ref_w is formed by torch: one more rounding)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    # the same call repeated gives the same bits (nothing stale is read)
    G, v, w, ref, _ = cases[0]
    a = binding.gemvt_noalloc(G, v).clone()
    binding.gemvt_noalloc(cases[1][0], cases[1][1])
    b = binding.gemvt_noalloc(G, v)
    assert torch.equal(a, b)
    assert torch.equal(a, ref)                                # same kernels, same chunking: bit-identical


def test_no_alloc_gemvt_rejects_sizes_beyond_the_array():
    import ctypes as C
    from paper_2602_03857_b200 import binding
    lib = binding.load()
    small = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = C.c_void_p(small.data_ptr())
    # sizes are checked before any pointer is used: 16 row chunks x M doubles just over the array
    N, M = 4097, binding.NOALLOC_MAX_DOUBLES // 16 + 2
    st = lib.grav_gemvt_noalloc(0, p, 8, N, M, p, None, p, None)
    msg = lib.grav_last_error().decode()
    assert st == -1 and "exceed" in msg and "16 MiB" in msg and str(16 * M) in msg
    assert lib.grav_gemvt_noalloc(0, p, 2, 1, 8, p, None, p, None) == -1          # bad element size
    assert lib.grav_gemvt_noalloc(0, p, 8, 0, 8, p, None, p, None) == -1          # empty
    # exactly at the limit (one row chunk, M = the whole array) it runs; one column more is refused
    M = binding.NOALLOC_MAX_DOUBLES
    G = torch.arange(M, dtype=torch.float64, device="cuda").reshape(1, M)
    v = torch.full((1,), 0.5, dtype=torch.float64, device="cuda")
    assert torch.equal(binding.gemvt_noalloc(G, v), 0.5 * G[0])
    G1 = torch.zeros((1, M + 1), dtype=torch.float64, device="cuda")
    with pytest.raises(binding.GravError):
        binding.gemvt_noalloc(G1, v)
    with pytest.raises(ValueError):
        binding.gemvt_noalloc(G.cpu(), v.cpu())
