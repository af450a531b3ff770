#!/usr/bin/env python
"""bench.py -- ETac tactile hot path on B200: one JSON line (contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--envs E]

A "step" is one pass of the whole hot path (S1 SDF penetration -> S2 propagation -> S3 residual
MLP -> S4 combine) over one batch of 4,096 synthetic environments of the
dexterous-hand sensor set (BASELINE.json configs[2]; N = 5,696 nodes, 16 patches, bf16 tensor
path with fp32 accumulation).  metric = tactile env-steps/s (whole job), also node-updates/s.
Multi-GPU: environments are independent, every rank owns its own 4,096 envs,
no data-path collective -> "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2604_20295_b200 import workloads as W  # noqa: E402

METRIC = "tactile_env_steps_per_s"
UNIT = "env-steps/s"
N_INPUT_SETS = 4
MLP_FLOP_PER_NODE_ENV = 2 * (9 * 64 + 64 * 64 + 64 * 3)      # 9,728
# dram__bytes_read.sum + dram__bytes_write.sum of one dense_bf16_kernel launch, from the
# `ncu --set full` capture summarised in profiles/r01d_dense_ncu_full.md (79.2 MB read + 232.4 MB
# write; the kernel also zero-fills the rows of contact-free (env, patch) pairs); cfg 4: the counters
# in profiles/r01d_cfg4_item_order.md, first column (1.47 GB read + 0.41 GB write).
NCU_TRAFFIC_BYTES = 311.54e6
NCU_TRAFFIC_BYTES_CFG4 = 1877.3e6


WORKLOADS = {
    "cfg3": ("cfg3_dexterous_hand_5696 (BASELINE.json configs[2])", lambda seed, envs: W.config3(seed, envs)),
    # not the headline: the single dense K[8192 x 8192] case, same metric (python bench.py --workload cfg4)
    "cfg4": ("cfg4_curved_sheet_8192 (BASELINE.json configs[3])", lambda seed, envs: W.config4(seed, envs)),
}


def chosen_of(wl):
    """[E, P] contact pairs the generator placed (cfg 4: every env presses on its single patch)."""
    return wl.meta["chosen"] if "chosen" in wl.meta else np.ones((wl.n_envs, wl.mesh.n_patches), dtype=bool)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "src": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "src": "fallback"}


def work_model(wl, chosen):
    """Algorithmic work of one step from the realised contact pairs."""
    npat = np.diff(wl.mesh.patch_offset).astype(np.float64)
    pairs_per_patch = chosen.sum(0).astype(np.float64)
    w_nodeenv = float((pairs_per_patch * npat).sum())
    f_prop_dense = 6.0 * float((pairs_per_patch * npat * npat).sum())
    f_mlp = MLP_FLOP_PER_NODE_ENV * w_nodeenv
    E, N, P = wl.n_envs, wl.mesh.n_nodes, wl.mesh.n_patches
    b_out = 12.0 * E * N
    b_in = 48.0 * E * wl.max_indenters + 28.0 * E * P
    b_k = 2.0 * float((npat * npat).sum())
    return {"w_nodeenv": w_nodeenv, "f_prop_dense": f_prop_dense, "f_mlp": f_mlp,
            "b_hbm_min": b_out + b_in + b_k + 20e3, "pairs": float(pairs_per_patch.sum())}


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        time.sleep(0.15)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.f.name)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any("Active" == r[3 + k].strip() for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "power_w_max": max(float(r[2]) for r in rows),
                "samples": len(rows), "reasons": reasons}


def time_oracle(wl, n_sample, repeats=1):
    """The CPU oracle as it stands, on a strided sample of the workload's environments."""
    from oracle import etac_oracle as O
    from threadpoolctl import threadpool_info
    m = O.model_from_workload(wl)
    envs = list(range(0, wl.n_envs, max(1, wl.n_envs // n_sample)))[:n_sample]
    for p in range(m.n_patches):
        O.kernel_block(m, p)                       # K is create-time work on both sides
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose, envs=envs)
        best = min(best, time.perf_counter() - t0)
    threads = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    return len(envs) / best, len(envs), best, threads


def run_reference(a):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    label, make = WORKLOADS[a.workload]
    wl = make(0, a.envs)
    # each step = the oracle on a strided sample of the batch, sized from a probe so that the whole
    # --steps K --warmup W run stays within about two minutes
    probe_rate = time_oracle(wl, min(a.envs, 8))[0]
    n_sample = int(max(4, min(a.envs, 96, 120.0 * probe_rate / max(1, a.steps + a.warmup))))
    t_w = [time_oracle(wl, n_sample)[0] for _ in range(a.warmup)]
    t0 = time.perf_counter()
    envs_done = 0
    threads = 1
    for _ in range(a.steps):
        rate, n, _, threads = time_oracle(wl, n_sample)
        envs_done += n
    dt = time.perf_counter() - t0
    v = envs_done / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "node_updates_per_s": v * wl.mesh.n_nodes,
        "config": {"workload": label, "n_envs": a.envs,
                   "n_nodes": wl.mesh.n_nodes, "n_patches": wl.mesh.n_patches},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"each step = {n_sample} of {a.envs} envs (stride {max(1, a.envs // n_sample)})"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(a):
    import torch
    from paper_2604_20295_b200 import build as B
    from paper_2604_20295_b200 import etac as T
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the ETac hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.build()
    peaks = load_peaks()

    # weak scaling: every rank owns a batch of a.envs environments (its own seeds)
    label, make = WORKLOADS[a.workload]
    sets = [make(rank * N_INPUT_SETS + k, a.envs) for k in range(N_INPUT_SETS)]
    wl = sets[0]
    eng = T.Etac(wl, device=local)
    stream = torch.cuda.current_stream().cuda_stream
    if a.l2_group_mb:
        T.etac_set_option(eng.ctx, T.ETAC_OPT_L2_GROUP_BYTES, a.l2_group_mb << 20)
    devs = [eng.upload(indenters=s.indenters, patch_pose=s.patch_pose) for s in sets]
    argv = [eng.args(a.envs, d) for d in devs]

    def sync_all():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for i in range(a.warmup):
        T.etac_step(eng.ctx, stream, argv[i % N_INPUT_SETS])
    pairs = T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_CONTACT_PAIRS)
    last_set = sets[(a.warmup - 1) % N_INPUT_SETS]
    assert pairs == int(chosen_of(last_set).sum()), "realised contact pairs differ from the generator's placement"

    # ---- device-resident timing
    sync_all()
    clk = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(a.steps):
        T.etac_step(eng.ctx, stream, argv[i % N_INPUT_SETS])
    e1.record()
    sync_all()
    ms = e0.elapsed_time(e1)
    launches = a.steps * T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_LAUNCHES)
    # per-kernel split, live, same inputs (CUDA events on the launching stream inside the library)
    _, (ms_s1, ms_fused) = T.etac_time_steps(eng.ctx, stream, argv[0], max(5, min(a.steps, 20)), per_kernel=True)
    clocks = clk.stop() if clk else None
    # special-function pipe rate, measured live on this device (denominator of the "alu" roofline)
    sfu_ops_s, sfu_per_clk_sm = T.etac_measure_sfu_rate(stream) if rank == 0 else (0.0, 0.0)

    # ---- end to end: host buffers in, host buffer out, through the C-ABI call
    posed = sets[0].patch_pose is not None
    pin = [(torch.from_numpy(np.ascontiguousarray(s.indenters).view(np.uint8).reshape(-1)).pin_memory(),
            torch.from_numpy(np.ascontiguousarray(s.patch_pose)).pin_memory() if posed else None) for s in sets]
    d_ind = torch.empty_like(pin[0][0], device="cuda")
    d_pose = torch.empty_like(pin[0][1], device="cuda") if posed else None
    h_out = torch.empty((a.envs, eng.N, 3), dtype=torch.float32).pin_memory()
    e2e_args = T.make_step_args(a.envs, eng.out, indenters=d_ind, patch_pose=d_pose)
    n_e2e = max(3, min(a.steps, 10))

    # Two result buffers and a copy stream: the device->host read of step i runs while step i+1 is copied in
    # and computed (every step's copies are still inside the timed region; the loop ends with a full sync).
    d_outs = [eng.out, torch.empty_like(eng.out)]
    h_outs = [h_out, torch.empty((a.envs, eng.N, 3), dtype=torch.float32).pin_memory()]
    e2e_argv = [e2e_args, T.make_step_args(a.envs, d_outs[1], indenters=d_ind, patch_pose=d_pose)]
    s_main, s_copy = torch.cuda.current_stream(), torch.cuda.Stream()
    ev_done = [torch.cuda.Event(), torch.cuda.Event()]
    ev_free = [torch.cuda.Event(), torch.cuda.Event()]

    def e2e_step(i):
        k, b = i % N_INPUT_SETS, i % 2
        s_main.wait_event(ev_free[b])                      # the read of step i-2 has left this result buffer
        d_ind.copy_(pin[k][0], non_blocking=True)
        if posed:
            d_pose.copy_(pin[k][1], non_blocking=True)
        T.etac_step(eng.ctx, stream, e2e_argv[b])
        ev_done[b].record(s_main)
        s_copy.wait_event(ev_done[b])
        with torch.cuda.stream(s_copy):
            h_outs[b].copy_(d_outs[b][: a.envs], non_blocking=True)
            ev_free[b].record(s_copy)

    e2e_step(0), e2e_step(1)
    sync_all()
    t0 = time.perf_counter()
    for i in range(n_e2e):
        e2e_step(i)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0)
    h2d = pin[0][0].numel() + (pin[0][1].numel() * 4 if posed else 0)
    d2h = h_out.numel() * 4

    # the same loop with the result packed as bf16 by the kernel (etac_step_args.out_dtype): the PCIe
    # copy of the result dominates the end-to-end number, this halves it.  Extra information only:
    # "e2e" above is the fp32 result.
    d_out16 = torch.empty((a.envs, eng.N, 3), dtype=torch.bfloat16, device="cuda")
    h_out16 = torch.empty((a.envs, eng.N, 3), dtype=torch.bfloat16).pin_memory()
    e2e16_args = T.make_step_args(a.envs, d_out16, indenters=d_ind, patch_pose=d_pose, out_dtype=T.ETAC_OUT_BF16)

    def e2e16_step(k):
        d_ind.copy_(pin[k][0], non_blocking=True)
        if posed:
            d_pose.copy_(pin[k][1], non_blocking=True)
        T.etac_step(eng.ctx, stream, e2e16_args)
        h_out16.copy_(d_out16, non_blocking=True)

    e2e16_step(0)
    sync_all()
    t0 = time.perf_counter()
    for i in range(n_e2e):
        e2e16_step(i % N_INPUT_SETS)
    torch.cuda.synchronize()
    e2e16_ms = 1e3 * (time.perf_counter() - t0)

    t = torch.tensor([ms, e2e_ms, e2e16_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms, e2e16_ms = float(t[0]), float(t[1]), float(t[2])
    if rank != 0:
        eng.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    ms_step = ms / a.steps
    value = world * a.envs / (ms_step * 1e-3)
    wm = work_model(wl, np.mean([chosen_of(s) for s in sets], axis=0) * 1.0)
    flops = wm["f_prop_dense"] + wm["f_mlp"]
    peak = peaks["bf16_tflops_sustained"]
    achieved = flops / (ms_fused * 1e-3) / 1e12
    t_tensor = flops / (peak * 1e12)
    t_hbm = wm["b_hbm_min"] / (peaks["hbm_gbs"] * 1e9)
    t_roof = max(t_tensor, t_hbm)
    # Floors of the fused kernel on the three units it loads: tensor pipe, HBM, and the special-function pipe
    # (128 SiLUs = 128 MUFU.TANH per node-environment of a contacting pair).  "roofline" is the contract's
    # (tensor peak / HBM); the activation-pipe bound is reported beside it as "roofline_sfu"
    # against a rate measured live, and does not replace the contract fraction.
    acts = 128.0 * wm["w_nodeenv"]
    t_sfu = acts / sfu_ops_s
    t_hbm_fused = (wm["b_hbm_min"] + 4.0 * wm["w_nodeenv"]) / (peaks["hbm_gbs"] * 1e9)
    roof_tensor = {"bound": "tensor", "kernel": "dense_bf16_kernel", "achieved": achieved, "peak": peak,
                   "unit": "TFLOP/s", "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES if a.workload == "cfg3" else NCU_TRAFFIC_BYTES_CFG4,
                   "peak_src": f"MEASURED_PEAKS.json bf16_tflops_sustained ({peaks['src']})", "flops_per_launch": flops}
    roof_sfu = {"bound": "alu", "kernel": "dense_bf16_kernel", "achieved": acts / (ms_fused * 1e-3) / 1e12,
                "peak": sfu_ops_s / 1e12, "unit": "Tactivation/s", "frac": t_sfu / (ms_fused * 1e-3),
                "traffic": NCU_TRAFFIC_BYTES if a.workload == "cfg3" else NCU_TRAFFIC_BYTES_CFG4,
                "peak_src": f"etac_measure_sfu_rate, live on this device: {sfu_per_clk_sm:.2f} MUFU results per clock and SM",
                "activations_per_launch": acts, "pipe": "MUFU (special-function unit)"}
    cpu_rate, cpu_n, cpu_t, cpu_threads = time_oracle(wl, a.envs if a.workload == "cfg3" else 48)   # ~10 s of CPU work
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "node_updates_per_s": value * eng.N,
        "config": {"workload": label, "n_envs_per_gpu": a.envs,
                   "n_nodes": eng.N, "n_patches": eng.P, "precision": "bf16 operands, fp32 accumulate",
                   "contact_pairs_per_step": wm["pairs"], "node_envs_per_step": wm["w_nodeenv"],
                   "l2": f"{N_INPUT_SETS} rotating seeded input sets; {12 * a.envs * eng.N / 1e6:.0f} MB output + "
                         f"{10 * a.envs * eng.N / 1e6:.0f} MB workspace per step > 126 MB L2",
                   "algorithmic_bytes_fused": wm["b_hbm_min"] + 4.0 * wm["w_nodeenv"],
                   "parallelism": f"env-sharded x{world}, no collective"},
        "clocks": clocks,
        "e2e": {"value": world * a.envs * n_e2e / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": n_e2e,
                "note": "pinned host indenters+patch poses -> device, etac_step, full [E,N,3] fp32 result -> pinned host; the read of step i overlaps step i+1 (two result buffers, copy stream)"},
        "e2e_bf16_output": {"value": world * a.envs * n_e2e / (e2e16_ms * 1e-3), "unit": UNIT, "d2h_bytes_per_step": d2h // 2,
                            "note": "same loop, result written as bf16 by the kernel (out_dtype); not the headline"},
        "gpu_launches": launches,
        "kernels_ms": {"s1_sdf_kernel_incl_memsets": ms_s1, "dense_bf16_kernel": ms_fused},
        "roofline": roof_tensor, "roofline_sfu": roof_sfu,
        "roofline_floors_us": {"tensor": t_tensor * 1e6, "hbm": t_hbm_fused * 1e6, "sfu": t_sfu * 1e6},
        "roofline_step": {"t_roof_us": t_roof * 1e6, "t_tensor_us": t_tensor * 1e6, "t_hbm_us": t_hbm * 1e6,
                          "roof_dense_frac": t_roof / (ms_step * 1e-3),
                          "hbm_frac_of_measured": wm["b_hbm_min"] / (ms_step * 1e-3) / (peaks["hbm_gbs"] * 1e9),
                          "t_act_us_1mufu": t_sfu * 1e6},
        "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": cpu_threads, "kind": "oracle",
                         "sample": f"{cpu_n} of {a.envs} envs (strided), {cpu_t:.1f} s, numpy fp64"},
    }
    print(json.dumps(out))
    eng.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--envs", type=int, default=4096)
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--l2-group-mb", type=int, default=0,
                    help="experiments: ETAC_OPT_L2_GROUP_BYTES in MiB (0 = library default, 1024 = one group)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    (run_reference if args.impl == "reference" else run_ours)(args)
