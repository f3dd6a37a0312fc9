"""Multi-rank host logic on CPU (gloo, world_size 2): the station partition, the collectives of dist.Comm on raw
addresses, and the placement of the exchanges -- an observation-sharded CG that sums the adjoint
output and the dot-product partials over ranks reproduces the unsharded CG.  The local operators in that check are
the oracle's (tests may use it); the CUDA kernels cannot run here, their sharded use is covered on the GPU by
tests/test_gpu_parity.py::test_comm_exchange_placement and tests/test_gpu_multirank.py.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_03857_b200 import dist as gdist
from paper_2602_03857_b200 import workloads


def test_shard_range_partitions():
    for n in (1, 2, 7, 256, 178797):
        for world in (1, 2, 3, 8):
            edges = [gdist.shard_range(n, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        gdist.shard_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    r, w, _ = gdist.init_from_env("gloo")
    assert (r, w) == (rank, world)
    try:
        # ---- collectives on raw host addresses: in-place sum over ranks, gather in rank order
        comm = gdist.Comm("cpu")
        assert (comm.world, comm.rank) == (world, rank)
        buf = np.arange(10, dtype=np.float64) * (rank + 1)
        comm.allreduce_sum(buf.ctypes.data + 16, 5)         # elements 2..6 only
        exp = np.arange(10, dtype=np.float64) * (rank + 1)
        exp[2:7] = np.arange(2, 7) * sum(range(1, world + 1))
        assert np.array_equal(buf, exp)
        send = np.arange(4, dtype=np.float64) + 10 * rank
        recv = np.full(4 * world + 1, -1.0)
        comm.allgather(send.ctypes.data, recv.ctypes.data, 4)
        assert np.array_equal(recv[:-1], np.concatenate([np.arange(4.0) + 10 * r for r in range(world)])) and recv[-1] == -1
        assert comm.calls == [("allreduce", 5), ("allgather", 4)]
        assert gdist.max_over_ranks(float(rank + 1), "cpu") == float(world)

        # ---- exchange placement: sharded CG == unsharded CG (oracle operators, config 1)
        wl = workloads.make(1)
        mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
        lo, hi = gdist.shard_range(wl.N, world, rank)
        xo, yo, zo = wl.xo[lo:hi], wl.yo[lo:hi], wl.zo[lo:hi]
        wgt = oracle.depth_weights(mesh, wl.beta, wl.z0)
        G_full = oracle.tabulate(mesh, wl.xo, wl.yo, wl.zo, wl.gamma, nthreads=2)
        d_full = oracle.dense_matvec(G_full, wl.m_true) + 1e-3 * wl.noise()
        lam = 5e-5

        def allsum(a):
            t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1).copy())
            dist.all_reduce(t)
            return t.numpy().reshape(np.shape(a))

        d = d_full[lo:hi]
        x = np.zeros(hi - lo)
        res, p = d.copy(), d.copy()
        rho = float(allsum(np.array([res @ res]))[0])                     # exchange: partials of d.d
        for _ in range(5):                                   # prefix parity (P2): chaotic growth sets in by k ~ 8
            g = allsum(oracle.adjoint(mesh, xo, yo, zo, wl.gamma, p, nthreads=2))   # exchange: adjoint output
            q = oracle.forward(mesh, xo, yo, zo, wl.gamma, g / (wgt * wgt), nthreads=2) + lam * p
            delta = float(allsum(np.array([p @ q]))[0])                   # exchange: partials of p.q
            a = rho / delta
            x += a * p
            res -= a * q
            rho_new = float(allsum(np.array([res @ res]))[0])             # exchange: partials of r.r
            p = res + (rho_new / rho) * p
            rho = rho_new
        m = allsum(oracle.adjoint(mesh, xo, yo, zo, wl.gamma, x, nthreads=2)) / (wgt * wgt)
        ref, _, _ = oracle.cg(wgt, lam, d_full, 5, G=G_full, nthreads=2)
        m_ref = oracle.recover_model(G_full, wgt, ref.x, nthreads=2)
        err_a = np.abs(x - ref.x[lo:hi]).max() / np.abs(ref.x).max()
        err_m = np.abs(m - m_ref).max() / np.abs(m_ref).max()
        out.put((rank, float(err_a), float(err_m)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_hook_and_exchange_placement():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=300)
        assert p.exitcode == 0
    got = sorted(out.get(timeout=10) for _ in range(world))
    assert [g[0] for g in got] == [0, 1]
    for _, err_a, err_m in got:
        assert err_a <= 1e-8 and err_m <= 1e-8
