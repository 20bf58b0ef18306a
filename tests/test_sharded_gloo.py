"""world_size-2 gloo test of the multi-GPU host logic (paper_2601_08077_b200/sharded.py): the
q-shard partition and the one exchange step (all-reduce of J and K).  The per-shard partial
results come from the oracle here -- on GPUs they come from df_jk_build."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from df_inputs import generators as G
from oracle import df_oracle as O
from paper_2601_08077_b200 import sharded


def test_shard_range_covers_and_aligns():
    for naux in (1, 160, 512, 513, 1700, 4000, 6000):
        for world in (1, 2, 3, 4, 8):
            got = [sharded.shard_range(naux, r, world) for r in range(world)]
            assert got[0][0] == 0 and got[-1][1] == naux
            for (a0, a1), (b0, b1) in zip(got, got[1:]):
                assert a1 == b0 and a0 <= a1
            for q0, q1 in got:
                assert q0 % 512 == 0 or q0 == naux
            sizes = [(q1 - q0 + 511) // 512 for q0, q1 in got]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nao, naux, nocc, s = 24, 1300, 6, 3
    Bp = G.make_B_packed(nao, naux, seed=11)
    Cocc = G.make_C_occ(nao, nocc, seed=11)
    D = G.make_density(Cocc)
    q0, q1 = sharded.shard_range(naux, rank, world)
    Bs = np.ascontiguousarray(Bp[:, q0:q1])
    Jp, Kp = O.emul_df_jk(Bs, nao, Cocc, D, s)
    J, K = torch.from_numpy(Jp.copy()), torch.from_numpy(Kp.copy())
    sharded.allreduce_jk(J, K)
    if rank == 0:
        Jf, Kf = O.emul_df_jk(Bp, nao, Cocc, D, s)
        out.put((O.rel_frobenius(J.numpy(), Jf), O.rel_frobenius(K.numpy(), Kf)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_allreduce_equals_single_build():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    eJ, eK = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # same q-groups (shards are multiples of 512), only the FP64 summation order differs
    assert eJ <= 1e-14 and eK <= 1e-14
