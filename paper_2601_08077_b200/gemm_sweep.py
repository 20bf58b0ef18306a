"""Config-1 sweep (BASELINE.json configs[1]): C = A.B emulated with s = 1..8 INT8 slices for square
M = N = K, timed with CUDA events; native FP64 `torch.matmul` time for context only (it is not on
the hot path).  Prints a markdown table.

    python -m paper_2601_08077_b200.gemm_sweep [--sizes 1024 2048 4096 8192 16384] [--slices 1 .. 8]
"""
from __future__ import annotations

import argparse
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def main():
    import torch

    import paper_2601_08077_b200 as p
    from df_inputs import generators as G

    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", type=int, nargs="+", default=[1024, 2048, 4096, 8192, 16384])
    ap.add_argument("--slices", type=int, nargs="+", default=list(range(1, 9)))
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    nmax = max(args.sizes)
    ws = p.Workspace(p.df_emul_gemm_workspace_bytes(nmax, nmax, nmax, max(args.slices)), device=dev)

    def timed(fn):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.reps

    print("| N | s | emulated GEMM ms (split + INT8 GEMM) | INT8 GEMM ms | INT8 TOP/s | effective FP64 TFLOP/s "
          "| rel. Frobenius error vs torch FP64 | native FP64 ms |")
    print("|---|---|---|---|---|---|---|---|")
    for n in args.sizes:
        if n <= 4096:
            A, B = (torch.from_numpy(x).to(dev) for x in G.make_gemm_inputs(n, n, n, seed=n))
        else:  # same distribution, generated on the device
            g = torch.Generator(device=dev)
            g.manual_seed(n)

            def one():
                e = torch.rand((n, n), generator=g, dtype=torch.float64, device=dev) * 30.0 - 30.0
                off = torch.randint(-10, 11, (n, 1), generator=g, device=dev).to(torch.float64)
                sgn = torch.where(torch.rand((n, n), generator=g, device=dev) < 0.5, -1.0, 1.0).to(torch.float64)
                return sgn * torch.exp2(e + off)

            A, B = one(), one()
        C = torch.empty((n, n), dtype=torch.float64, device=dev)
        ref = A @ B
        t_native = timed(lambda: torch.matmul(A, B, out=ref))
        ref_norm = float(torch.linalg.norm(ref))
        for s in args.slices:
            p.df_profile_read()
            p.df_profile_enable(True)
            t_all = timed(lambda: p.df_emul_gemm_slices(A, B, C, n, n, n, s))
            p.df_profile_enable(False)
            prof = p.df_profile_read()
            t_gemm = prof["emul_gemm_i8"][0] / max(1, prof["emul_gemm_i8"][1])
            err = float(torch.linalg.norm(C - ref)) / ref_norm
            ops = 2.0 * n**3 * s * (s + 1) / 2
            print(f"| {n} | {s} | {t_all:.3f} | {t_gemm:.3f} | {ops / t_gemm / 1e9:.0f} | "
                  f"{2.0 * n**3 / t_all / 1e9:.1f} | {err:.2e} | {t_native:.3f} |", flush=True)
        del A, B, C, ref
    ws.close()


if __name__ == "__main__":
    main()
