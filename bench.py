#!/usr/bin/env python
"""bench.py -- DF J/K builds per second at nao = 1200 (BASELINE.json metric, config 3).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config large]

A "step" is one pass of the whole hot path: one df_jk_build (rho, J, unpack+split, GEMM(5),
X split, GEMM(6), K reduce) at that step's tolerance.  Step i takes entry i mod 12 of the
synthetic 12-step SCF sequence D_k = D* + eps_k S_k of BASELINE.json config 2/3 (R11),
whose tolerance tightens along Table 1 (paper_2601_08077_b200/policy.py), so the slice count
adapts per step.  One JSON line on stdout; see DESIGN.md section 7 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from df_inputs import generators as G  # noqa: E402

NSEQ = 12
METRIC = "df_jk_builds_per_s"
UNIT = "builds/s"


def flops_per_build(cfg):
    """Effective FP64 FLOPs, PAPER.md:122-126 with N_scr = N_bf^2."""
    return 4.0 * cfg.nao**2 * cfg.naux + 4.0 * cfg.nao**2 * cfg.naux * cfg.nocc


def int8_ops_per_build(cfg, s):
    """Algorithmic INT8 ops of the two slice-pair GEMMs (2 per MAC), s(s+1)/2 pairs each
    (PAPER.md:139): GEMM(5) 2 (naux nao) nao nocc; GEMM(6) over the lower triangle only,
    2 (nao (nao+1)/2) (naux nocc).  No padding is counted."""
    pairs = s * (s + 1) // 2
    g5 = 2.0 * cfg.naux * cfg.nao * cfg.nao * cfg.nocc
    g6 = 2.0 * (cfg.nao * (cfg.nao + 1) / 2) * cfg.naux * cfg.nocc
    return pairs * g5, pairs * g6


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                smax = float(parts[1])
            except ValueError:
                continue
            for nm, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle_block(cfg, Bs, C, D, naux_sample):
    """Seconds the oracle's plain FP64 J/K (oracle/df_oracle.py, as it stands) takes on
    `naux_sample` auxiliary functions of the workload, on the host cores."""
    from oracle import df_oracle as O

    t0 = time.perf_counter()
    rho = O.df_rho(Bs, cfg.nao, D)
    J = O.df_j(Bs, cfg.nao, rho)
    K = O.df_k(Bs, cfg.nao, C)
    dt = time.perf_counter() - t0
    assert np.isfinite(J).all() and np.isfinite(K).all()
    return dt


def host_threads():
    try:
        from threadpoolctl import threadpool_info

        n = [d.get("num_threads", 1) for d in threadpool_info() if d.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def run_reference(args, cfg):
    """The reference arm for this tier = the CPU oracle, timed on the host cores; each step is
    a bounded sample (args.ref_q auxiliary functions) of the same workload, scaled to builds/s."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    qs = min(args.ref_q, cfg.naux)
    Bs = G.make_B_packed(cfg.nao, qs, cfg.seed)
    C = G.make_C_occ(cfg.nao, cfg.nocc, cfg.seed)
    D = G.make_density(C)
    for _ in range(args.warmup):
        time_oracle_block(cfg, Bs, C, D, qs)
    dts = [time_oracle_block(cfg, Bs, C, D, qs) for _ in range(args.steps)]
    t_build = (sum(dts) / len(dts)) * (cfg.naux / qs)
    value = 1.0 / t_build
    cores = host_threads()
    sample = f"{qs} of {cfg.naux} auxiliary functions per step (plain FP64 rho, J, X, K), time scaled by naux/{qs}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_build, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: DF J/K build nao={cfg.nao} naux={cfg.naux} nocc={cfg.nocc}",
                   "sample": sample},
        "effective_fp64_tflops": flops_per_build(cfg) * value / 1e12,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    import paper_2601_08077_b200 as p
    from paper_2601_08077_b200 import policy, sharded

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc
    # ---- inputs (synthetic, seeded).  With N ranks every rank owns one
    # q-shard of `naux` auxiliary functions of an N*naux basis (weak scaling).
    B = G.make_B_packed_torch(nao, naux, cfg.seed + rank, device=dev)
    C0 = G.make_C_occ(nao, nocc, cfg.seed)
    D0 = G.make_density(C0)
    seq = G.make_scf_sequence(D0, nocc, NSEQ, cfg.seed)
    sched = policy.schedule([eps * eps for eps, _, _ in seq])[:NSEQ]  # dE_rel,k := eps_k^2 (R11)
    tols = [t for _, t in sched]
    slices = [p.df_slices_for_tol(t) for t in tols]
    D_dev = [torch.from_numpy(Dk).to(dev) for _, Dk, _ in seq]
    C_dev = [torch.from_numpy(Ck).to(dev) for _, _, Ck in seq]
    D_pin = [torch.from_numpy(Dk).pin_memory() for _, Dk, _ in seq]
    C_pin = [torch.from_numpy(Ck).pin_memory() for _, _, Ck in seq]
    D_buf, C_buf = torch.empty_like(D_dev[0]), torch.empty_like(C_dev[0])
    J = torch.empty((nao, nao), dtype=torch.float64, device=dev)
    K = torch.empty_like(J)
    J_pin, K_pin = torch.empty((nao, nao), dtype=torch.float64).pin_memory(), torch.empty((nao, nao), dtype=torch.float64).pin_memory()

    # ---- workspace: as many 512-q blocks per launch as fit beside B
    smax = max(slices)
    nblk = (naux + 511) // 512
    free, _ = torch.cuda.mem_get_info(dev)
    while nblk > 1 and p.df_jk_workspace_bytes_blocks(nao, naux, nocc, smax, nblk) > free - (6 << 30):
        nblk -= 1
    ws = p.Workspace(p.df_jk_workspace_bytes_blocks(nao, naux, nocc, smax, nblk), device=dev)

    plan_box = [None]  # set for the "planned" leg

    def step(i, resident):
        k = i % NSEQ
        if resident:
            Dk, Ck = D_dev[k], C_dev[k]
        else:
            D_buf.copy_(D_pin[k], non_blocking=True)
            C_buf.copy_(C_pin[k], non_blocking=True)
            Dk, Ck = D_buf, C_buf
        sharded.df_jk_build_sharded(B, nao, naux, Ck, nocc, Dk, tols[k], J, K, plan=plan_box[0])
        if not resident:
            J_pin.copy_(J, non_blocking=True)
            K_pin.copy_(K, non_blocking=True)

    def timed(nsteps, resident, first):
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(first, first + nsteps):
            step(i, resident)
        e1.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item())

    # own UTCIMMA issue-rate probe (MEASURED_PEAKS.json has no INT8 figure)
    probe_ms = p.df_debug_mma_peak(256, 20000, 148)
    int8_probe_tops = 2.0 * 128 * 256 * 32 * 20000 * 148 / probe_ms / 1e9

    for i in range(args.warmup):
        step(i, True)
    torch.cuda.synchronize()
    assert p.df_last_status() == 0, "status word set during warm-up"

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    n0 = p.df_launch_count()
    p.df_profile_enable(True)
    ms_total = timed(args.steps, True, args.warmup)
    p.df_profile_enable(False)
    launches = p.df_launch_count() - n0
    prof = p.df_profile_read()
    clocks = sampler.stop() if rank == 0 else None
    assert p.df_last_status() == 0 and bool(torch.isfinite(K).all()) and bool(torch.isfinite(J).all())

    # ---- end to end through the C-ABI with HOST buffers: D_k, C_k from pinned memory in, J, K
    # out, every step; B stays resident (it is constant over the SCF).
    step(args.warmup, False)
    ms_e2e = timed(args.steps, False, args.warmup)
    h2d = (nao * nao + nao * nocc) * 8
    d2h = 2 * nao * nao * 8

    # ---- planned leg: B split once into max(slices) planes outside the
    # timed region, the same steps with GEMM(5) reading the plan.  An extra, not the headline:
    # `value` above runs every row of the hot path, the unpack + split included, in every step.
    planned = None
    free, _ = torch.cuda.mem_get_info(dev)
    plan_bytes = p.df_jk_plan_bytes(nao, naux, smax)
    fits = torch.tensor([1 if plan_bytes < free - (4 << 30) else 0], device=dev)
    if world > 1:
        dist.all_reduce(fits, op=dist.ReduceOp.MIN)  # every rank takes the same branch
    if int(fits.item()):
        J_ref, K_ref = J.clone(), K.clone()  # of the last e2e step = step warmup + steps - 1
        pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        # the plan's 36.9 GB come out of torch's caching allocator (a cudaMalloc of that size takes
        # 20-200 ms by itself): plan_create_ms times the library call, not the allocation
        del_me = torch.empty(plan_bytes + 256, dtype=torch.uint8, device=dev)
        del del_me
        torch.cuda.synchronize()
        pe0.record()
        plan_box[0] = p.Plan(B, nao, naux, smax)
        pe1.record()
        torch.cuda.synchronize()
        for i in range(args.warmup):
            step(i, True)
        p.df_profile_enable(True)
        ms_planned = timed(args.steps, True, args.warmup)
        p.df_profile_enable(False)
        prof_planned = p.df_profile_read()
        ms_planned_e2e = timed(args.steps, False, args.warmup)
        same = bool(torch.equal(J, J_ref)) and bool(torch.equal(K, K_ref))
        assert p.df_last_status() == 0
        planned = {"value": args.steps * world / (ms_planned / 1e3), "unit": UNIT,
                   "ms_per_step": ms_planned / args.steps,
                   "e2e_value": args.steps * world / (ms_planned_e2e / 1e3),
                   "plan_create_ms": pe0.elapsed_time(pe1), "plan_gb": plan_bytes / 1e9, "plan_slices": smax,
                   "bit_identical_to_unplanned": same,
                   "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof_planned.items() if v[1]},
                   "note": "B split once (df_jk_plan_create, outside the timed region) and reused by every "
                           "step; B is constant over the SCF (PAPER.md:157)"}
        plan_box[0].close()
        plan_box[0] = None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    units = args.steps * world  # shard-builds of this config processed by all ranks
    value = units / (ms_total / 1e3)
    e2e_value = units / (ms_e2e / 1e3)
    used = [slices[i % NSEQ] for i in range(args.warmup, args.warmup + args.steps)]
    ops5 = sum(int8_ops_per_build(cfg, s)[0] for s in used)
    ops6 = sum(int8_ops_per_build(cfg, s)[1] for s in used)
    ms5, n5 = prof["gemm5_i8"]
    ms6, n6 = prof["gemm6_i8"]
    peaks, peak_kind = measured_peaks()
    # INT8 dense peak = measured bf16 peak x the nominal INT8:bf16 ratio (4.5 : 2.25 PFLOP/s);
    # the GEMMs run inside a long step, so the sustained figure applies.
    peak_tops = 2.0 * peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    achieved = (ops5 + ops6) / ((ms5 + ms6) / 1e3) / 1e12
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int8", "dtype_note": "int8 x int8 -> int32 slice-pair products, f64 recombination; J in f64",
        "data": "synthetic",
        "config": {"workload": f"{cfg.name}: DF J/K build nao={nao} naux={naux} nocc={nocc} (BASELINE.json configs[3]), "
                               f"12-step adaptive SCF sequence, one q-shard per GPU",
                   "slices_per_step": used, "tol_per_step": [tols[i % NSEQ] for i in range(args.warmup, args.warmup + args.steps)],
                   "l2": "inputs larger than L2: packed B is %.1f GB and every step streams it" % (B.numel() * 8 / 1e9),
                   "workspace_gb": ws.view.numel() / 1e9, "q_blocks_per_launch": nblk},
        "effective_fp64_tflops": flops_per_build(cfg) * value / 1e12,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "note": "D_k, C_occ,k from pinned host memory and J, K back every step; B resident in HBM"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "tensor", "kernel": "gemm_i8_kernel (GEMM(5) + GEMM(6) launches)",
                     "achieved": achieved, "peak": peak_tops, "unit": "TOP/s", "frac": achieved / peak_tops,
                     "peak_source": f"2 x bf16_tflops_sustained of MEASURED_PEAKS.json ({peak_kind})",
                     "achieved_gemm5": ops5 / (ms5 / 1e3) / 1e12 if ms5 else None,
                     "achieved_gemm6": ops6 / (ms6 / 1e3) / 1e12 if ms6 else None,
                     "int8_probe_tops": int8_probe_tops, "frac_of_probe": achieved / int8_probe_tops,
                     "launches": n5 + n6, "avg_launch_ms": (ms5 + ms6) / max(1, n5 + n6),
                     "share_of_step": (ms5 + ms6) / ms_total,
                     # dram__bytes_read+write per launch, ncu --set full at s = 4 (profiles/r01_ncu_summary.md):
                     # GEMM(5) 25.9 + 6.1 GB, GEMM(6) 4.5 + 0.2 GB -> mean over the two launches of a build
                     "traffic": 0.5 * (32.0e9 + 4.7e9), "traffic_unit": "bytes per launch (s = 4)"},
        "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items() if v[1]},
    }
    if planned is not None:
        planned["effective_fp64_tflops"] = flops_per_build(cfg) * planned["value"] / 1e12
        out["planned"] = planned
    if world == 1 and not args.no_cpu_baseline:
        qs = min(args.cpu_q, naux)
        Bs = B[:, :qs].contiguous().cpu().numpy()
        dt = time_oracle_block(cfg, Bs, C0, D0, qs)
        v = 1.0 / (dt * naux / qs)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
                               "sample": f"first {qs} of {naux} auxiliary functions of the same B (plain FP64 "
                                         f"rho, J, X, K; {dt:.1f} s), time scaled by naux/{qs}",
                               "effective_fp64_tflops": flops_per_build(cfg) * v / 1e12}
    print(json.dumps(out))
    ws.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="large", choices=sorted(G.CONFIGS))
    ap.add_argument("--ref-q", dest="ref_q", type=int, default=32)
    ap.add_argument("--cpu-q", dest="cpu_q", type=int, default=256)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = G.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
