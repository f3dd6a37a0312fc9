"""Observation-sharded operation over several GPUs of one node (one process per GPU, torch.distributed / NCCL).

The path shards the way the paper shards it ("observation domain partitioned across devices,
model-space variables replicated and synchronised"): rank r owns a contiguous block of stations and the whole mesh.
  forward  d = G u      : rows of d are local -- no communication;
  adjoint  g = G^T v    : every rank forms the node sums T over ITS stations as compensated (hi, lo) pairs; one
                          all-gather of those planes (2 N_n doubles per rank, 54 MB at config 5) and an error-free
                          combination in rank order (csrc/adjoint.cu adjoint_reduce) make them global and bit-identical
                          on every rank -- the only data-path collective;
  CG                    : alpha, x, r, p, q are station vectors (local rows); each dot product all-reduces its 256
                          block partials, so every rank computes bit-identical scalars on the device.
The exchanges are issued by libgrav.so itself through the callbacks of include/grav.h (grav_set_comm); this module
only provides the callbacks (NCCL collectives on tensor views of the raw buffers) and the station partition.  Nothing
here computes any part of the method.
"""
import os

import numpy as np
import torch
import torch.distributed as dist


def shard_range(n: int, world: int, rank: int):
    """Contiguous, balanced partition of range(n): the first n % world ranks get one extra item."""
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("bad world / rank")
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


class _RawDeviceArray:
    """Zero-copy view of `count` doubles at a raw CUDA address (CUDA array interface, consumed by torch.as_tensor)."""

    def __init__(self, ptr, count):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": "<f8", "data": (int(ptr), False),
                                         "version": 2}


class Comm:
    """Collectives for GravContext.set_comm on raw addresses, over `group`.

    device = a CUDA device: buffers are viewed zero-copy as float64 tensors and the NCCL collective is issued under
    torch.cuda.stream(ExternalStream(stream)) - the stream libgrav.so hands over - so it is ordered with the library's
    kernels whatever torch's current stream is.
    device = "cpu": host addresses (gloo; used by the CPU tests of this plumbing)."""

    def __init__(self, device, group=None):
        self.device = torch.device(device)
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.calls = []           # ("allreduce" | "allgather", count) in call order
        # CUDA buffers over a CPU-only backend (gloo): stage through host memory.  The copies synchronise the stream the
        # library handed over, so the ordering with its kernels is kept; used to run two real ranks on ONE GPU in the
        # tests (NCCL needs a device per rank), never by bench.py.
        self.staged = (self.device.type == "cuda" and dist.is_initialized()
                       and "nccl" not in str(dist.get_backend(group)).lower())

    def view(self, ptr: int, count: int) -> torch.Tensor:
        if self.device.type == "cuda":
            return torch.as_tensor(_RawDeviceArray(ptr, count), device=self.device)
        import ctypes
        return torch.from_numpy(np.ctypeslib.as_array((ctypes.c_double * count).from_address(ptr)))

    def _on(self, stream: int):
        if self.device.type != "cuda":
            import contextlib
            return contextlib.nullcontext()
        if stream == 0:           # the legacy default stream cannot be wrapped; torch's default stream is that stream
            return torch.cuda.stream(torch.cuda.default_stream(self.device))
        return torch.cuda.stream(torch.cuda.ExternalStream(stream, device=self.device))

    def allreduce_sum(self, ptr: int, count: int, stream: int = 0):
        with self._on(stream):
            t = self.view(ptr, count)
            if self.staged:
                h = t.cpu()                                   # synchronises the stream
                dist.all_reduce(h, op=dist.ReduceOp.SUM, group=self.group)
                t.copy_(h)
            else:
                dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        self.calls.append(("allreduce", count))

    def allgather(self, send_ptr: int, recv_ptr: int, count: int, stream: int = 0):
        with self._on(stream):
            recv, send = self.view(recv_ptr, count * self.world), self.view(send_ptr, count)
            if self.staged:
                parts = [torch.empty(count, dtype=torch.float64) for _ in range(self.world)]
                dist.all_gather(parts, send.cpu(), group=self.group)
                recv.copy_(torch.cat(parts))
            else:
                dist.all_gather_into_tensor(recv, send, group=self.group)
        self.calls.append(("allgather", count))


def init_from_env(backend="nccl"):
    """torchrun environment -> (rank, world, local_rank); initialises the default process group once."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend == "nccl":
            torch.cuda.set_device(local)
            dist.init_process_group(backend, rank=rank, world_size=world, device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend, rank=rank, world_size=world)
    return rank, world, local


class ShardedContext:
    """GravContext on this rank's station shard with the exchange hook installed."""

    def __init__(self, wl, rank, world, local, mode=0):
        from . import binding
        self.rank, self.world = rank, world
        self.lo, self.hi = shard_range(wl.N, world, rank)
        sl = slice(self.lo, self.hi)
        self.ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo[sl], wl.yo[sl], wl.zo[sl], wl.gamma, device=local,
                                       mode=mode)
        self.comm = None
        if world > 1:
            self.comm = Comm(self.ctx.device)
            self.ctx.set_comm(self.comm)

    def local(self, a):
        """Rows of a station vector (numpy) owned by this rank, as a device tensor."""
        return torch.as_tensor(np.ascontiguousarray(a[self.lo:self.hi], dtype=np.float64)).to(self.ctx.device)

    def close(self):
        self.ctx.close()


def max_over_ranks(ms: float, device) -> float:
    """Device-timed milliseconds -> max over ranks (the contract's multi-GPU timing rule)."""
    if not dist.is_initialized():
        return ms
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
