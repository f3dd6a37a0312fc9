"""The observation-sharded product on TWO real GPUs ("observation domain partitioned across devices,
model-space variables replicated and synchronised"): two NCCL ranks, each with the station shard
of dist.ShardedContext and the exchange callbacks of dist.Comm, against the unsharded context on rank 0's device.

The NCCL test is skipped on a box with fewer than 2 GPUs (the development pool's boxes have one); there the second test
runs the same two ranks on ONE GPU with gloo collectives staged through host memory (dist.Comm.staged), which exercises
everything of the sharded product but NCCL itself.  (The CPU side of the plumbing is tests/test_dist_cpu.py, the
placement of the exchanges tests/test_gpu_parity.py::test_comm_exchange_placement.)
The workload is ragged and irregular (random stations over topography, the shape class of configs 4-5) and large
enough that the adjoint's (hi, lo) planes matter: the sharded adjoint must agree with the single-rank one to 1e-10 of
max (the operator tolerance), five CG iterates (prefix parity) and the recovered model to 1e-8."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

SHAPE = dict(nx=40, ny=36, nz=30, h=50.0, nobs=3001, seed=3, topo_amp=120.0)
CG_ITERS = 5


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _problem():
    from paper_2602_03857_b200 import workloads
    wl = workloads.make_custom(SHAPE["nx"], SHAPE["ny"], SHAPE["nz"], SHAPE["h"], SHAPE["nobs"], seed=SHAPE["seed"],
                               topo_amp=SHAPE["topo_amp"])
    rng = np.random.default_rng(77)
    return wl, rng.standard_normal(wl.N), rng.standard_normal(wl.M)


def _worker(rank, world, port, out, backend="nccl"):
    # backend "nccl": one device per rank.  "gloo": both ranks on cuda:0, the collectives staged through host memory by
    # dist.Comm - two REAL ranks of the product (distinct shards, rank order, gather layout) on a one-GPU box; the ranks'
    # kernels never wait on one another (the exchanges are host-driven, between launches).
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank if backend == "nccl" else 0))
    import torch.distributed as dist
    from paper_2602_03857_b200 import binding
    from paper_2602_03857_b200 import dist as gdist
    r, w, local = gdist.init_from_env(backend)
    try:
        torch.cuda.set_device(local)
        dev = torch.device("cuda", local)
        wl, v, u = _problem()
        to = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
        res = {}
        for mode in (binding.MATRIX_FREE, binding.STORED_F64):
            sh = gdist.ShardedContext(wl, rank, world, local, mode=mode)
            ctx = sh.ctx
            if mode == binding.STORED_F64:
                ctx.store_g()
            wgt = ctx.depth_weights(2.0, wl.z0)
            # lambda from the global trace: each rank's Gram diagonal covers its own stations
            tr = ctx.gram_diag(wgt).sum().reshape(1)
            tr = tr.cpu() if backend == "gloo" else tr              # the test's own collectives: host tensors under gloo
            dist.all_reduce(tr)
            lam = 1e-2 * float(tr.item()) / wl.N
            fwd = ctx.forward(to(u)) if mode == binding.MATRIX_FREE else ctx.forward_stored(to(u))
            adj = ctx.adjoint(sh.local(v)) if mode == binding.MATRIX_FREE else ctx.adjoint_stored(sh.local(v))
            cg = ctx.dataspace_cg(sh.local(v), wgt, lam, CG_ITERS, mode=mode)
            # a stream other than torch's current one: the callbacks must order the collectives on the stream they
            # are handed (dist.Comm._on), not on torch's current stream
            side = torch.cuda.Stream(device=dev)
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                adj_side = ctx.adjoint(sh.local(v)) if mode == binding.MATRIX_FREE else ctx.adjoint_stored(sh.local(v))
            side.synchronize()
            assert torch.equal(adj, adj_side)
            mine = adj.cpu() if backend == "gloo" else adj
            gather = [torch.empty_like(mine) for _ in range(world)]
            dist.all_gather(gather, mine)
            assert all(torch.equal(gather[0], g) for g in gather), "replicated model-space vector differs between ranks"
            res[mode] = dict(lo=sh.lo, hi=sh.hi, lam=lam, fwd=fwd.cpu().numpy(), adj=adj.cpu().numpy(),
                             alpha=cg["alpha"].cpu().numpy(), m=cg["m"].cpu().numpy(), hist=cg["hist"].cpu().numpy(),
                             calls=list(sh.comm.calls[-3:]))
            sh.close()
        out.put((rank, res))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs 2 GPUs (NCCL ranks on distinct devices)")
def test_two_nccl_ranks_match_the_unsharded_context():
    _run_two_ranks("nccl")


@pytest.mark.skipif(not torch.cuda.is_available(), reason="needs a GPU")
def test_two_ranks_on_one_gpu_match_the_unsharded_context():
    """The same comparison with both ranks on cuda:0 and gloo collectives staged through host memory: what a one-GPU box
    can verify of the sharded product - everything but NCCL itself."""
    _run_two_ranks("gloo")


def _run_two_ranks(backend):
    from paper_2602_03857_b200 import binding
    world = 2
    ctxmp = mp.get_context("spawn")
    out = ctxmp.Queue()
    port = _free_port()
    procs = [ctxmp.Process(target=_worker, args=(r, world, port, out, backend)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(out.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0

    wl, v, u = _problem()
    dev = torch.device("cuda", 0)
    to = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    rel = lambda a, b: float(np.abs(a - b).max() / np.abs(b).max())
    for mode in (binding.MATRIX_FREE, binding.STORED_F64):
        ref = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=0, mode=mode)
        if mode == binding.STORED_F64:
            ref.store_g()
        wgt = ref.depth_weights(2.0, wl.z0)
        lam = 1e-2 * float(ref.gram_diag(wgt).sum().item()) / wl.N
        fwd = (ref.forward(to(u)) if mode == binding.MATRIX_FREE else ref.forward_stored(to(u))).cpu().numpy()
        adj = (ref.adjoint(to(v)) if mode == binding.MATRIX_FREE else ref.adjoint_stored(to(v))).cpu().numpy()
        for rank in range(world):
            r = got[rank][mode]
            assert abs(r["lam"] / lam - 1) <= 1e-12
            assert rel(r["fwd"], fwd[r["lo"]:r["hi"]]) <= 1e-12          # same rows, same kernels: chunking order only
            assert rel(r["adj"], adj) <= 1e-10
        cg = ref.dataspace_cg(to(v), wgt, got[0][mode]["lam"], CG_ITERS, mode=mode)
        alpha, m, hist = (cg[k].cpu().numpy() for k in ("alpha", "m", "hist"))
        for rank in range(world):
            r = got[rank][mode]
            assert np.abs(r["alpha"] - alpha[r["lo"]:r["hi"]]).max() <= 1e-8 * np.abs(alpha).max()
            assert rel(r["m"], m) <= 1e-8
            assert np.abs(r["hist"] / hist - 1).max() <= 1e-8
        ref.close()
