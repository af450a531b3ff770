"""Where is the object?  Pose estimation from a tactile field with the pose gradients of etac_backward.

ETac is differentiable (Table I): the penetration comes from the objects' SDFs, so
dL/dU chains through dL/ddelta to the poses of the indenters and of the patches.  Here the displacement field of a
sphere pressed into a fingertip cap at a hidden position is the observation; the estimate starts half a millimetre
off, and every iteration is one etac_step, one etac_backward (grad_indenter_pose: rows (dL/dt, dL/dtheta)) and an
Adam step on the translation.

The context runs in ETAC_ACTIVE_PROPAGATE mode: with the mask M_p of Eq. 2 (the default) the row of a node jumps
from its propagated value to u^ = -delta n when the node enters contact, the loss is then discontinuous in the pose
and a descent stalls at the jumps; without the mask the field is continuous in the penetration.

    python -m paper_2604_20295_b200.examples.pose_from_touch [--envs 64] [--iters 200]
"""
import argparse

import numpy as np
import torch

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--envs", type=int, default=64)
    ap.add_argument("--iters", type=int, default=200)
    a = ap.parse_args()
    wl = W.config2(0, a.envs)                                       # fingertip cap, 1024 nodes, fp32
    rng = np.random.default_rng(0)
    ind = wl.indenters.copy()
    ind["type"][:, 1:] = W.IND_NONE
    ind["type"][:, 0] = W.IND_SPHERE
    ind["param"][:, 0, 0] = 4.0
    cand = np.nonzero(wl.mesh.normal[:, 2] > 0.8)[0]
    c = rng.choice(cand, size=a.envs)
    t_star = (wl.mesh.pos[c] + wl.mesh.normal[c] * (4.0 - 0.9)).astype(np.float32)    # pressed 0.9 mm into node c
    ind["pose"][:, 0, 0:3] = t_star
    ind["pose"][:, 0, 3:7] = [0, 0, 0, 1]
    eng = T.Etac(wl, precision="fp32", active_mode=T.ETAC_ACTIVE_PROPAGATE)
    stream = torch.cuda.current_stream().cuda_stream
    target = eng.step(wl.n_envs, eng.upload(indenters=ind)).clone()
    off = rng.normal(size=(a.envs, 3))
    t = t_star.astype(np.float64) + 0.5 * off / np.linalg.norm(off, axis=1, keepdims=True)   # 0.5 mm off, any direction
    g_alpha = torch.empty(len(wl.alpha), device=eng.device)
    g_pen = torch.empty((wl.n_envs, eng.N), device=eng.device)
    g_ind = torch.empty((wl.n_envs, wl.max_indenters, 6), device=eng.device)
    m1, m2 = np.zeros_like(t), np.zeros_like(t)
    for it in range(1, a.iters + 1):
        ind["pose"][:, 0, 0:3] = t.astype(np.float32)
        dev = eng.upload(indenters=ind)
        G = eng.step(wl.n_envs, dev) - target
        T.etac_backward(eng.ctx, stream, wl.n_envs, G.contiguous(), g_alpha, None, grad_penetration=g_pen,
                        grad_indenter_pose=g_ind, **dev)
        g = g_ind[:, 0, 0:3].cpu().numpy().astype(np.float64)
        m1, m2 = 0.9 * m1 + 0.1 * g, 0.999 * m2 + 0.001 * g * g
        t = t - 0.02 * (m1 / (1 - 0.9 ** it)) / (np.sqrt(m2 / (1 - 0.999 ** it)) + 1e-12)
        if it % 25 == 0 or it == 1:
            err = np.linalg.norm(t - t_star, axis=1)
            print(f"iter {it:4d}  loss {0.5 * float((G * G).sum()):10.4g}  |t - t*| median {np.median(err):.4f} max {err.max():.4f} mm")
    eng.close()


if __name__ == "__main__":
    main()
