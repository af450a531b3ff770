"""BASELINE.json configs[4]: the dense-contraction / sparse-gather sweep.  Prints one line per
(envs, nodes, contact fraction): ms per step through the tensor-core contraction, the bf16 gather
form and the fp32 gather kernel, with the S1 / fused split of the dense path.  The command behind
the cfg-5 table of DESIGN.md §8.

    python -m paper_2604_20295_b200.examples.sweep_cfg5 [--envs 4096] [--nodes 256 1024 4096 8192] [--fp32]
"""
import argparse

import torch

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W


def time_path(wl, precision, path, iters):
    eng = T.Etac(wl, precision=precision)
    try:
        T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        stream = torch.cuda.current_stream().cuda_stream
        args = eng.args(wl.n_envs, dev)
        for _ in range(3):
            T.etac_step(eng.ctx, stream, args)
        torch.cuda.synchronize()
        ms, (s1, rest) = T.etac_time_steps(eng.ctx, stream, args, iters, per_kernel=True)
    finally:
        eng.close()
    return ms, s1, rest


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--envs", type=int, nargs="+", default=[4096])
    ap.add_argument("--nodes", type=int, nargs="+", default=[256, 1024, 4096, 8192])
    ap.add_argument("--fracs", type=float, nargs="+", default=[0.01, 0.05, 0.20])
    ap.add_argument("--fp32", action="store_true", help="also time the fp32 gather kernel (slow at large N)")
    ap.add_argument("--iters", type=int, default=10)
    a = ap.parse_args()
    print("envs nodes curved frac | dense ms (S1 + fused) | gather bf16 ms | gather fp32 ms")
    for E in a.envs:
        for N in a.nodes:
            curved = N >= 4096
            for f in a.fracs:
                wl = W.config5(E, N, curved, f, "bf16")
                d, s1, fu = time_path(wl, "bf16", T.ETAC_PATH_DENSE, a.iters)
                g, _, _ = time_path(wl, "bf16", T.ETAC_PATH_SPARSE, a.iters)
                g32 = time_path(wl, "fp32", T.ETAC_PATH_SPARSE, max(2, a.iters // 3))[0] if a.fp32 else float("nan")
                print(f"{E} {N} {int(curved)} {f:.2f} | {d:.3f} ({s1:.3f} + {fu:.3f}) | {g:.3f} | {g32:.3f}", flush=True)


if __name__ == "__main__":
    main()
