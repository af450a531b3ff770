"""Calibration of alpha and Phi by gradient descent (Eq. 3) on synthetic data.

The paper fits alpha and the residual network to FEM displacements; no FEM data exists here, so the
targets are the displacements of a *teacher*: the same library with hidden parameters (alpha*, Phi*).
The student starts from a wrong alpha and perturbed weights; every iteration is one etac_step
(forward), one etac_backward (dL/dalpha, dL/dW from dL/dU = U - U*) and one etac_update_params.
torch.optim.Adam only holds the optimiser state.

    python -m paper_2604_20295_b200.examples.calibrate [--envs 256] [--iters 200]
"""
import argparse
import dataclasses

import numpy as np
import torch

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--envs", type=int, default=256)
    ap.add_argument("--iters", type=int, default=200)
    a = ap.parse_args()
    wl = dataclasses.replace(W.config3(0, a.envs), weights=W.make_weights(3, 0, std=0.1))
    dev_kw = dict(indenters=wl.indenters, patch_pose=wl.patch_pose)
    teacher = T.Etac(wl)
    target = teacher.step(wl.n_envs, teacher.upload(**dev_kw)).clone()
    teacher.close()

    rng = np.random.default_rng(1)
    alpha = torch.tensor(wl.alpha * 0.6, dtype=torch.float32, requires_grad=True)
    weights = {k: torch.tensor(v + rng.normal(0, 0.03, v.shape).astype(np.float32), requires_grad=True)
               for k, v in wl.weights.items()}
    opt = torch.optim.Adam([{"params": [alpha], "lr": 0.01}, {"params": list(weights.values()), "lr": 2e-3}])
    eng = T.Etac(dataclasses.replace(wl, alpha=alpha.detach().numpy(), weights={k: v.detach().numpy() for k, v in weights.items()}))
    dev = eng.upload(**dev_kw)
    stream = torch.cuda.current_stream().cuda_stream
    g_alpha = torch.empty(1, device=eng.device)
    g_w = torch.empty(T.ETAC_GRAD_WEIGHTS_LEN, device=eng.device)
    for it in range(a.iters):
        G = (eng.step(wl.n_envs, dev) - target).contiguous()
        loss = 0.5 * float((G * G).sum()) / wl.n_envs
        T.etac_backward(eng.ctx, stream, wl.n_envs, G, g_alpha, g_w, **dev)
        alpha.grad = g_alpha.cpu() / wl.n_envs
        for k, g in T.split_grad_weights(g_w.cpu()).items():
            weights[k].grad = g.clone() / wl.n_envs
        opt.step()
        with torch.no_grad():
            alpha.clamp_(min=1e-3)
        T.etac_update_params(eng.ctx, alpha=alpha.detach().numpy(), weights={k: v.detach().numpy() for k, v in weights.items()})
        if it % 20 == 0 or it == a.iters - 1:
            print(f"iter {it:4d}  loss/env {loss:10.4e}  alpha {float(alpha.detach()):.4f} (teacher {float(wl.alpha[0]):.4f})")
    eng.close()


if __name__ == "__main__":
    main()
