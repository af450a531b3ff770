"""Times one ETAC_RESID_POINTNET step on the cfg-3 hand workload (4096 envs): the command behind
profiles/r01c_pointnet_backward_launch_list.md.

    python -m paper_2604_20295_b200.examples.pointnet_step
"""
import dataclasses

import torch

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W


def main():
    wl = dataclasses.replace(W.config3(0, 4096), weights=W.make_pointnet_weights(3, 0, std=0.02))
    eng = T.Etac(wl)
    dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
    stream = torch.cuda.current_stream().cuda_stream
    args = eng.args(wl.n_envs, dev)
    for _ in range(3):
        T.etac_step(eng.ctx, stream, args)
    torch.cuda.synchronize()
    ms, (s1, rest) = T.etac_time_steps(eng.ctx, stream, args, 20, per_kernel=True)
    print(f"pointnet cfg3 4096 envs: {ms:.3f} ms/step (S1 {s1:.3f}, encode + global + decode {rest:.3f})")
    eng.close()


if __name__ == "__main__":
    main()
