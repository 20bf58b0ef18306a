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
    _JK, J, K = sharded.alloc_jk(nao)  # adjacent halves of one buffer: the exchange is ONE all-reduce
    J.copy_(torch.from_numpy(Jp))
    K.copy_(torch.from_numpy(Kp))
    calls = []
    real = dist.all_reduce
    dist.all_reduce = lambda t, *a, **kw: (calls.append(t.numel()), real(t, *a, **kw))[1]
    sharded.allreduce_jk(J, K)
    dist.all_reduce = real
    if rank == 0:
        Jf, Kf = O.emul_df_jk(Bp, nao, Cocc, D, s)
        out.put((O.rel_frobenius(J.numpy(), Jf), O.rel_frobenius(K.numpy(), Kf), calls))
    dist.barrier()
    dist.destroy_process_group()


def _oracle_build(calls, planned):
    """Stand-in for the binding's build call in the CPU test (no GPU here): the per-shard partial J, K
    come from the oracle, written into the caller's tensors exactly as df_jk_build does on a GPU."""
    def build(*args):
        if planned:
            _plan, Bs, nao, naux, Cocc, nocc, D, tol, J, K, _stream = args
        else:
            Bs, nao, naux, Cocc, nocc, D, tol, J, K, _stream = args
        calls.append(("planned" if planned else "plain", naux))
        Jp, Kp = O.emul_df_jk(Bs.numpy(), nao, Cocc.numpy(), D.numpy(), O.slices_for_tol(tol))
        J.copy_(torch.from_numpy(Jp))
        K.copy_(torch.from_numpy(Kp))
    return build


def _worker_sharded(rank, world, port, out, naux, use_plan):
    """df_jk_build_sharded itself on every rank: naux = 400 < 512 leaves rank 1 with an EMPTY shard
    (it must contribute zeros and still take part in the all-reduce); plan= takes the planned call."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2601_08077_b200 import binding
    calls = []
    binding.df_jk_build = _oracle_build(calls, False)
    binding.df_jk_build_planned = _oracle_build(calls, True)
    nao, nocc, tol = 20, 5, 1e-6
    Bp = G.make_B_packed(nao, naux, seed=12)
    Cocc = G.make_C_occ(nao, nocc, seed=12)
    D = G.make_density(Cocc)
    q0, q1 = sharded.shard_range(naux, rank, world)
    Bs = torch.from_numpy(np.ascontiguousarray(Bp[:, q0:q1]))
    J = torch.full((nao, nao), float("nan"), dtype=torch.float64)
    K = torch.full((nao, nao), float("nan"), dtype=torch.float64)
    sharded.df_jk_build_sharded(Bs, nao, q1 - q0, torch.from_numpy(Cocc), nocc, torch.from_numpy(D), tol, J, K,
                                plan=object() if use_plan else None)
    Jf, Kf = O.emul_df_jk(Bp, nao, Cocc, D, O.slices_for_tol(tol))
    out.put((rank, q1 - q0, calls, O.rel_frobenius(J.numpy(), Jf), O.rel_frobenius(K.numpy(), Kf)))
    dist.barrier()
    dist.destroy_process_group()


def _run_sharded(naux, use_plan):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_sharded, args=(r, 2, port, out, naux, use_plan)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=240) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return got


def test_sharded_build_empty_shard_contributes_zeros():
    (r0, n0, c0, eJ0, eK0), (r1, n1, c1, eJ1, eK1) = _run_sharded(400, False)
    assert (n0, n1) == (400, 0)  # one 512-q block: rank 1 owns nothing
    assert c0 == [("plain", 400)] and c1 == []  # no build call on the empty shard
    # every rank ends with the full J, K (rank 1 contributed zeros, not NaN or stale data)
    assert max(eJ0, eJ1) <= 1e-14 and max(eK0, eK1) <= 1e-14


def test_sharded_build_plan_branch():
    (r0, n0, c0, eJ0, eK0), (r1, n1, c1, eJ1, eK1) = _run_sharded(1300, True)
    assert (n0, n1) == (1024, 276)
    assert c0 == [("planned", 1024)] and c1 == [("planned", 276)]
    assert max(eJ0, eJ1) <= 1e-14 and max(eK0, eK1) <= 1e-14


def test_two_rank_allreduce_equals_single_build():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    eJ, eK, calls = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # same q-groups (shards are multiples of 512), only the FP64 summation order differs
    assert eJ <= 1e-14 and eK <= 1e-14
    assert calls == [2 * 24 * 24]  # one all-reduce over the contiguous [J; K]


def _bench(*argv):
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    return subprocess.run([sys.executable, os.path.join(root, "bench.py"), *argv], capture_output=True, text=True,
                          env=env, timeout=600)


def test_bench_gpus_2_starts_two_ranks_through_the_launcher():
    """`bench.py --gpus 2` started by hand (no WORLD_SIZE) re-executes itself under
    sharded.launcher_command -- torch.distributed.run, rendezvous on 127.0.0.1 -- as two ranks.  Driven
    here with the CPU arm (the oracle; no GPU needed): rank 0 prints the one JSON line, rank 1 exits 0."""
    import json

    r = _bench("--gpus", "2", "--impl", "reference", "--config", "tiny", "--steps", "1", "--warmup", "0", "--ref-q", "16")
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0


def test_bench_gpus_beyond_the_devices_fails_loudly():
    """The product arm never oversubscribes a GPU: more ranks than devices is an error, not n_gpus = 1."""
    import torch

    n = torch.cuda.device_count() + 1 if torch.cuda.is_available() else 2
    r = _bench("--gpus", str(max(2, n)), "--config", "tiny", "--steps", "1")
    assert r.returncode == 2
    assert "CUDA device" in r.stderr and not [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
