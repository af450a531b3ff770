"""Times etac_backward (dL/dalpha, dL/dW, dL/ddelta from dL/dU) on the cfg-3 hand workload (4096 envs):
the command behind profiles/r01c_pointnet_backward_launch_list.md.

    python -m paper_2604_20295_b200.examples.backward_step
"""
import torch

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W


def main():
    wl = W.config3(0, 4096)
    eng = T.Etac(wl)
    dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
    stream = torch.cuda.current_stream().cuda_stream
    G = torch.randn((wl.n_envs, eng.N, 3), device=eng.device)
    g_alpha = torch.empty(1, device=eng.device)
    g_w = torch.empty(T.ETAC_GRAD_WEIGHTS_LEN, device=eng.device)
    g_pen = torch.empty((wl.n_envs, eng.N), device=eng.device)
    for with_pen in (False, True):
        kw = dict(dev, grad_penetration=g_pen) if with_pen else dev
        for _ in range(2):
            T.etac_backward(eng.ctx, stream, wl.n_envs, G, g_alpha, g_w, **kw)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            T.etac_backward(eng.ctx, stream, wl.n_envs, G, g_alpha, g_w, **kw)
        e1.record()
        torch.cuda.synchronize()
        print(f"etac_backward cfg3 4096 envs{' + dL/ddelta' if with_pen else ''}: {e0.elapsed_time(e1) / 5:.2f} ms per call")
    eng.close()


if __name__ == "__main__":
    main()
