"""q-sharded multi-GPU J/K build: one process per GPU, each rank holds
the columns B[:, q0:q1] of its own auxiliary-index range.  rho_q is local to its shard
(PAPER.md:45), J and K are sums over q, so the only exchange step is one
all-reduce(sum) of the contiguous [J; K] per build -- over NCCL/NVLink on GPUs, gloo in the CPU tests.

Shards are multiples of the 512-q block of the K path (R5), so the q-groups -- and
with them every INT8 digit -- are the same as in the single-GPU build.
"""
from __future__ import annotations

QBLOCK = 512


def shard_range(naux: int, rank: int, world: int, qblock: int = QBLOCK):
    """[q0, q1) of `rank`: 512-q blocks dealt out as evenly as possible, in order."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    nblk = (naux + qblock - 1) // qblock
    base, extra = divmod(nblk, world)
    b0 = rank * base + min(rank, extra)
    b1 = b0 + base + (1 if rank < extra else 0)
    return min(naux, b0 * qblock), min(naux, b1 * qblock)


def alloc_jk(nao: int, device=None):
    """(JK, J, K): one contiguous [2, nao, nao] FP64 buffer and its two halves, so that the exchange step
    is ONE all-reduce (46 MB at nao = 1200) instead of two."""
    import torch

    JK = torch.empty((2, nao, nao), dtype=torch.float64, device=device)
    return JK, JK[0], JK[1]


def _adjacent(J, K) -> bool:
    """K starts where J ends, in the same storage (the halves alloc_jk returns)."""
    return (J.is_contiguous() and K.is_contiguous() and J.dtype == K.dtype and J.device == K.device
            and J.untyped_storage().data_ptr() == K.untyped_storage().data_ptr()
            and K.storage_offset() == J.storage_offset() + J.numel())


def allreduce_jk(J, K, group=None):
    """The exchange step: J and K partial sums over this rank's q range -> full J, K (in place).  One
    all-reduce when J and K are adjacent halves of one buffer (alloc_jk), else one each."""
    import torch
    import torch.distributed as dist

    if dist.is_initialized() and dist.get_world_size(group) > 1:
        if _adjacent(J, K):
            flat = torch.as_strided(J, (J.numel() + K.numel(),), (1,))
            dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
        else:
            dist.all_reduce(J, op=dist.ReduceOp.SUM, group=group)
            dist.all_reduce(K, op=dist.ReduceOp.SUM, group=group)
    return J, K


def launcher_command(nproc: int, script: str, argv, port: int | None = None):
    """The command line that starts `script argv...` as `nproc` ranks on this node, one per GPU:
    torch.distributed.run with the rendezvous on 127.0.0.1 (the container hostname may not resolve),
    the same launch the driver uses for bench.py."""
    import socket
    import sys

    if port is None:
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(nproc)}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), script, *argv]


def df_jk_build_sharded(B_shard, nao, naux_shard, C_occ, nocc, D, tol, J, K, group=None, stream=None, plan=None):
    """This rank's df_jk_build over its shard of q (B_shard = B_packed[:, q0:q1], contiguous),
    then the all-reduce.  With an empty shard the rank contributes zeros.  plan: a binding.Plan of
    this rank's shard (B split once for the whole SCF), or None."""
    from . import binding

    if naux_shard > 0 and plan is not None:
        binding.df_jk_build_planned(plan, B_shard, nao, naux_shard, C_occ, nocc, D, tol, J, K, stream)
    elif naux_shard > 0:
        binding.df_jk_build(B_shard, nao, naux_shard, C_occ, nocc, D, tol, J, K, stream)
    else:
        J.zero_()
        K.zero_()
    return allreduce_jk(J, K, group)
