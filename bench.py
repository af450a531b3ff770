#!/usr/bin/env python
"""bench.py -- ETac tactile hot path on B200: one JSON line (contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg1|cfg2|cfg3|cfg4|cfg5] [--envs E]

A "step" is one pass of the whole hot path (S1 SDF penetration -> S2 propagation -> S3 residual
MLP -> S4 combine) over one batch of synthetic environments.  The default
workload is BASELINE.json configs[2] (the configuration its `metric` is quoted on): 4,096 envs of the
dexterous-hand sensor set, N = 5,696 nodes, 16 patches, bf16 tensor path with fp32 accumulation.
metric = tactile env-steps/s (whole job), also node-updates/s.  The other configs of BASELINE.json are
selected with --workload (cfg1/cfg2: fp32 contexts; cfg4: one dense K[8192 x 8192]; cfg5: the dense /
sparse sweep, one line whose "sweep" key holds a row per (N, contact fraction, path)).
Multi-GPU: environments are independent, every rank owns its own batch,
no data-path collective -> "scaling": "weak"; `--gpus N` without a torchrun environment re-launches
itself under torch.distributed.run with N ranks.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
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
# --phi: the residual network of the timed context.  "pernode" = BASELINE.json's per-node MLP (the metric's config);
# "pointnet" = the paper's own form of Phi (widths = DESIGN.md R10).  Algorithmic flop and SiLU
# count per node-environment of a contacting pair: encoder 9->64->64, decoder 128->64->3 (the kernels run the
# encoder twice -- once for the max-pool, once in the decoder pass -- which these figures do not count), + the
# global MLP 64->64 once per pair.
PHI = {"pernode": {"flop_node": MLP_FLOP_PER_NODE_ENV, "act_node": 128.0, "flop_pair": 0.0, "act_pair": 0.0},
       "pointnet": {"flop_node": 2 * (9 * 64 + 64 * 64 + 128 * 64 + 64 * 3), "act_node": 192.0,
                    "flop_pair": 2 * 64 * 64, "act_pair": 64.0}}
PHI_SEL = "pernode"
FP32_FMA_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12              # 74.4: 148 SMs x 128 fp32 lanes x 2 flop at 1965 MHz

# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the `ncu --set full`
# capture named beside it; "src_sha" = sha1 (first 12 hex digits) of the kernel's source file at capture time.
# bench.py prints the figure only while the source still has that hash -- a changed kernel gives traffic: null.
NCU_TRAFFIC = {
    "cfg3": {"bytes": 312.55e6, "profile": "profiles/r02_fused_ncu_full.md", "src": "k_fused.cu",
             "src_sha": "bf720de59a78"},
    "cfg4": {"bytes": 1700.55e6, "profile": "profiles/r02_fused_ncu_full.md", "src": "k_fused.cu",
             "src_sha": "bf720de59a78"},
}

CFG5_NODES = (256, 1024, 4096, 8192)
CFG5_FRACS = (0.001, 0.003, 0.01, 0.05, 0.20)


def make_workload(name, seed, envs, **kw):
    wl = _make_workload(name, seed, envs, **kw)
    if PHI_SEL == "pointnet":      # same geometry and contact, the paper's form of Phi (N(0, 0.02) weights like the configs')
        import dataclasses
        wl = dataclasses.replace(wl, weights=W.make_pointnet_weights(int(name[3:]), 0, std=0.02))
    return wl


def _make_workload(name, seed, envs, **kw):
    if name == "cfg1":
        return W.config1(seed, envs)
    if name == "cfg2":
        return W.config2(seed, envs)
    if name == "cfg3":
        return W.config3(seed, envs)
    if name == "cfg4":
        return W.config4(seed, envs)
    if name == "cfg5":
        return W.config5(envs, kw.get("n_nodes", 4096), kw.get("curved", True), kw.get("frac", 0.05),
                         kw.get("precision", "bf16"), seed)
    raise ValueError(name)


LABELS = {
    "cfg1": ("cfg1_flat_pad_256 (BASELINE.json configs[0])", 1),
    "cfg2": ("cfg2_fingertip_cap_1024 (BASELINE.json configs[1])", 64),
    "cfg3": ("cfg3_dexterous_hand_5696 (BASELINE.json configs[2])", 4096),
    "cfg4": ("cfg4_curved_sheet_8192 (BASELINE.json configs[3])", 4096),
    "cfg5": ("cfg5_dense_sparse_sweep (BASELINE.json configs[4])", 4096),
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "src": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "src": "fallback"}


def src_sha(fname):
    p = os.path.join(ROOT, "paper_2604_20295_b200", "csrc", fname)
    return hashlib.sha1(open(p, "rb").read()).hexdigest()[:12] if os.path.exists(p) else None


def ncu_traffic(workload):
    t = NCU_TRAFFIC.get(workload)
    if not t or src_sha(t["src"]) != t["src_sha"]:
        return None, (f"no ncu capture of the current {t['src']}" if t else "no ncu capture for this workload")
    return t["bytes"], t["profile"]


def work_model(wl, m_ep):
    """Algorithmic work of one step from the REALISED contact.
    m_ep [E, P] = active nodes of patch p in env e (from the masks the GPU path produced)."""
    npat = np.diff(wl.mesh.patch_offset).astype(np.float64)
    m = m_ep.astype(np.float64)
    hit = m > 0
    w_nodeenv = float((hit * npat).sum())
    n_active = float(m.sum())
    E, N, P = m_ep.shape[0], wl.mesh.n_nodes, wl.mesh.n_patches
    return {
        "w_nodeenv": w_nodeenv, "n_active": n_active, "pairs": float(hit.sum()),
        "f_prop_dense": 6.0 * float((hit * npat * npat).sum()),          # what a dense K_p . U^ executes
        "f_prop_alg": 6.0 * float((m * (npat - m)).sum()),               # the method: Omega is (n - m) x m (L87)
        "f_prop_gather": 6.0 * float((m * npat).sum()),                  # gather over the active nodes, all rows
        "f_mlp": PHI[PHI_SEL]["flop_node"] * w_nodeenv + PHI[PHI_SEL]["flop_pair"] * float(hit.sum()),   # Phi on every row of a contacting pair
        "f_mlp_alg": PHI[PHI_SEL]["flop_node"] * (w_nodeenv - n_active) + PHI[PHI_SEL]["flop_pair"] * float(hit.sum()),  # passive rows only
        "acts": PHI[PHI_SEL]["act_node"] * w_nodeenv + PHI[PHI_SEL]["act_pair"] * float(hit.sum()),
        "b_hbm_min": 12.0 * E * N + 48.0 * E * wl.max_indenters + (28.0 * E * P if wl.patch_pose is not None else 0.0)
                     + 2.0 * float((npat * npat).sum()) + 20e3,
        "contact_frac": n_active / max(1.0, w_nodeenv),
    }


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


def time_oracle(wl, n_sample):
    """The CPU oracle as it stands (numpy float64; a Python loop over environments and patches, only the
    K[:, act] @ u^ products and the MLP matmuls run in the BLAS thread pool), on a strided sample of the
    workload's environments.  Returns env-steps/s, sample size, wall seconds and the AVERAGE number of host
    threads it kept busy (process CPU time / wall time)."""
    from oracle import etac_oracle as O
    from threadpoolctl import threadpool_info
    m = O.model_from_workload(wl, resid_arch="pointnet" if "E1" in wl.weights else "pernode")
    envs = list(range(0, wl.n_envs, max(1, wl.n_envs // n_sample)))[:n_sample]
    for p in range(m.n_patches):
        O.kernel_block(m, p)                       # K is create-time work on both sides
    c0, t0 = time.process_time(), time.perf_counter()
    O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose, envs=envs)
    wall, cpu = time.perf_counter() - t0, time.process_time() - c0
    pool = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    return {"rate": len(envs) / wall, "n": len(envs), "wall": wall, "threads_busy": round(cpu / wall, 2),
            "nproc": os.cpu_count(), "blas_pool": pool}


def cpu_baseline_dict(r, n_envs):
    return {"value": r["rate"], "unit": UNIT, "cores": r["threads_busy"], "kind": "oracle",
            "host_cores": r["nproc"], "blas_pool_threads": r["blas_pool"],
            "sample": f"{r['n']} of {n_envs} envs (strided), {r['wall']:.1f} s wall; oracle/etac_oracle.py: numpy float64, "
                      f"Python loop over envs and patches, BLAS threads only inside the matmuls "
                      f"(cores = process CPU time / wall time)"}


def run_reference(a):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    label, _ = LABELS[a.workload]
    wl = make_workload(a.workload, 0, a.envs)
    # each step = the oracle on a strided sample of the batch, sized from a probe so that the whole
    # --steps K --warmup W run stays within about two minutes
    probe = time_oracle(wl, min(a.envs, 8))
    n_sample = int(max(1, min(a.envs, 96, 120.0 * probe["rate"] / max(1, a.steps + a.warmup))))
    for _ in range(a.warmup):
        time_oracle(wl, n_sample)
    t0 = time.perf_counter()
    envs_done, last = 0, probe
    for _ in range(a.steps):
        last = time_oracle(wl, n_sample)
        envs_done += last["n"]
    dt = time.perf_counter() - t0
    v = envs_done / dt
    cb = cpu_baseline_dict(last, a.envs)
    cb["value"] = v
    cb["sample"] = f"each step = {n_sample} of {a.envs} envs (stride {max(1, a.envs // n_sample)}); " + cb["sample"]
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "node_updates_per_s": v * wl.mesh.n_nodes,
        "config": {"workload": label, "n_envs": a.envs, "phi": PHI_SEL,
                   "n_nodes": wl.mesh.n_nodes, "n_patches": wl.mesh.n_patches},
        "cpu_baseline": cb,
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def realised_contact(T, torch, eng, wl, dev):
    """[E, P] active-node counts of one input set, from the mask the GPU path writes (untimed extra step)."""
    E, N = wl.n_envs, eng.N
    mask = torch.zeros((E, (N + 31) // 32), dtype=torch.int32, device=eng.device)
    stream = torch.cuda.current_stream().cuda_stream
    T.etac_step(eng.ctx, stream, T.make_step_args(E, eng.out, mask_out=mask, **dev))
    torch.cuda.synchronize()
    w = mask.cpu().numpy().view(np.uint32)
    bits = ((w[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(E, -1)[:, :N]
    off = np.asarray(wl.mesh.patch_offset)
    return np.add.reduceat(bits.astype(np.int64), off[:-1], axis=1)


def time_point(T, torch, wl, precision, path, iters):
    """cfg-5 sweep point: ms per step (whole step, S1, fused) of one context on one path."""
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
        taken = T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_PATH)
        m_ep = realised_contact(T, torch, eng, wl, dev)
    finally:
        eng.close()
    return ms, s1, rest, taken, m_ep


def run_sweep(a, T, torch, peaks):
    """--workload cfg5: BASELINE.json configs[4], E = --envs, N x contact fraction x path."""
    rows = []
    names = {T.ETAC_PATH_DENSE: "dense", T.ETAC_PATH_SPARSE: "sparse", T.ETAC_PATH_AUTO: "auto"}
    iters = max(3, min(a.steps, 10))
    headline = None
    for n_nodes in (a.nodes or CFG5_NODES):
        curved = n_nodes >= 4096
        for frac in (a.fracs or CFG5_FRACS):
            wl = make_workload("cfg5", 0, a.envs, n_nodes=n_nodes, curved=curved, frac=frac)
            row = {"n_nodes": n_nodes, "curved": curved, "target_frac": frac}
            for path in (T.ETAC_PATH_DENSE, T.ETAC_PATH_SPARSE, T.ETAC_PATH_AUTO):
                ms, s1, fused, taken, m_ep = time_point(T, torch, wl, "bf16", path, iters)
                wm = work_model(wl, m_ep)
                t_dense = max((wm["f_prop_dense"] + wm["f_mlp"]) / (peaks["bf16_tflops_sustained"] * 1e12),
                              wm["b_hbm_min"] / (peaks["hbm_gbs"] * 1e9))
                t_alg = max((wm["f_prop_alg"] + wm["f_mlp_alg"]) / (peaks["bf16_tflops_sustained"] * 1e12),
                            wm["b_hbm_min"] / (peaks["hbm_gbs"] * 1e9))
                row["realised_frac"] = wm["contact_frac"]
                row[names[path]] = {"ms": ms, "s1_ms": s1, "fused_ms": fused, "path_taken": names[taken],
                                    "roof_dense": t_dense / (ms * 1e-3), "roof_alg": t_alg / (ms * 1e-3)}
            if a.fp32:
                ms, s1, fused, _, _ = time_point(T, torch, wl, "fp32", T.ETAC_PATH_SPARSE, max(2, iters // 3))
                row["fp32"] = {"ms": ms, "s1_ms": s1, "fused_ms": fused}
            rows.append(row)
            print(f"[cfg5] E={a.envs} N={n_nodes} target {frac:.3f} realised {row['realised_frac']:.4f}: "
                  + " ".join(f"{k} {row[k]['ms']:.3f} ms" for k in ("dense", "sparse", "auto", "fp32") if k in row),
                  file=sys.stderr, flush=True)
            if headline is None or (n_nodes == 4096 and abs(frac - 0.05) < 1e-9):
                headline = row
    ms = headline["auto"]["ms"]
    return rows, headline, ms


def run_ours(a):
    import torch
    from paper_2604_20295_b200 import build as B
    from paper_2604_20295_b200 import etac as T
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert world == a.gpus, f"--gpus {a.gpus} but WORLD_SIZE={world}"
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the ETac hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.build()
    peaks = load_peaks()
    label, _ = LABELS[a.workload]

    if a.workload == "cfg5":
        if rank != 0:
            return
        clk = ClockSampler(local)
        rows, head, ms_step = run_sweep(a, T, torch, peaks)
        clocks = clk.stop()
        value = a.envs / (ms_step * 1e-3)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic", "node_updates_per_s": value * head["n_nodes"],
            "config": {"workload": label, "n_envs_per_gpu": a.envs,
                       "headline_point": {k: head[k] for k in ("n_nodes", "curved", "target_frac", "realised_frac")},
                       "note": "value = the AUTO path at the headline point; every point is in 'sweep'"},
            "clocks": clocks, "sweep": rows}))
        return

    # weak scaling: every rank owns a batch of a.envs environments (its own seeds)
    sets = [make_workload(a.workload, rank * N_INPUT_SETS + k, a.envs) for k in range(N_INPUT_SETS)]
    wl = sets[0]
    bf16 = wl.precision == "bf16"
    eng = T.Etac(wl, device=local)
    stream = torch.cuda.current_stream().cuda_stream
    devs = [eng.upload(indenters=s.indenters, patch_pose=s.patch_pose) for s in sets]
    argv = [eng.args(a.envs, d) for d in devs]

    def sync_all():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for i in range(a.warmup):
        T.etac_step(eng.ctx, stream, argv[i % N_INPUT_SETS])
    torch.cuda.synchronize()

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
    path_taken = T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_PATH)
    # per-kernel split, live, same inputs (CUDA events on the launching stream inside the library)
    _, (ms_s1, ms_fused) = T.etac_time_steps(eng.ctx, stream, argv[0], max(5, min(a.steps, 20)), per_kernel=True)
    clocks = clk.stop() if clk else None
    # special-function pipe rate, measured live on this device (denominator of the "alu" roofline)
    sfu_ops_s, sfu_per_clk_sm = T.etac_measure_sfu_rate(stream) if rank == 0 else (0.0, 0.0)
    # realised contact of every input set (untimed): [E, P] active-node counts from the GPU masks
    m_eps = [realised_contact(T, torch, eng, s, d) for s, d in zip(sets, devs)]
    for s, m_ep in zip(sets, m_eps):
        if "chosen" in s.meta:
            assert np.array_equal(m_ep > 0, s.meta["chosen"]), "realised contact pairs differ from the generator's placement"

    # ---- end to end: host buffers in, host buffer out, through the C-ABI call
    posed = sets[0].patch_pose is not None
    pin = [(torch.from_numpy(np.ascontiguousarray(s.indenters).view(np.uint8).reshape(-1)).pin_memory(),
            torch.from_numpy(np.ascontiguousarray(s.patch_pose)).pin_memory() if posed else None) for s in sets]
    d_ind = torch.empty_like(pin[0][0], device="cuda")
    d_pose = torch.empty_like(pin[0][1], device="cuda") if posed else None
    n_e2e = max(3, min(a.steps, 10))
    # Two result buffers and a copy stream: the device->host read of step i runs while step i+1 is copied in
    # and computed (every step's copies are still inside the timed region; the loop ends with a full sync).
    d_outs = [eng.out, torch.empty_like(eng.out)]
    h_outs = [torch.empty((a.envs, eng.N, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    e2e_argv = [T.make_step_args(a.envs, d_outs[b], indenters=d_ind, patch_pose=d_pose) for b in range(2)]
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
    d2h = h_outs[0].numel() * 4

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
    wms = [work_model(s, m) for s, m in zip(sets, m_eps)]
    wm = {k: float(np.mean([w[k] for w in wms])) for k in wms[0]}      # the timed steps rotate over the sets
    hbm = peaks["hbm_gbs"] * 1e9
    t_hbm = wm["b_hbm_min"] / hbm
    power_capped = bool(clocks and "sw_power_cap" in clocks.get("reasons", []))
    traffic, traffic_src = ncu_traffic(a.workload) if PHI_SEL == "pernode" else (None, "no ncu capture for --phi pointnet")
    if bf16:
        # roofline.frac: the dominant kernel against the bf16 tensor peak -- the BURST figure when no sw_power_cap
        # sample was seen during the timed region (the kernel then runs at the clocks of a kernel timed alone), the
        # SUSTAINED figure otherwise (MEASURED_PEAKS.json; B200_PROFILING.md).
        peak = peaks["bf16_tflops_sustained"] if power_capped else peaks["bf16_tflops"]
        peak_name = "bf16_tflops_sustained (sw_power_cap seen)" if power_capped else "bf16_tflops (burst; no sw_power_cap sample)"
        kernel = "fused_mlp_kernel" if path_taken == T.ETAC_PATH_DENSE else "fused_mlp_kernel (gather form)"
        if PHI_SEL == "pointnet":
            kernel += " x 2 (PointNet: encoder + max-pool pass, pn_global_kernel, decoder pass; timed together)"
        flops = wm["f_prop_dense"] + wm["f_mlp"]
        flops_alg = wm["f_prop_alg"] + wm["f_mlp_alg"]
        achieved = flops / (ms_fused * 1e-3) / 1e12
        t_tensor, t_tensor_alg = flops / (peak * 1e12), flops_alg / (peak * 1e12)
        # Floors of the fused kernel on the three units it loads: tensor pipe, HBM, and the special-function pipe
        # (128 SiLUs per node-environment of a contacting pair).  "roofline" is the contract's (tensor
        # peak / HBM); the activation-pipe bound is reported beside it as "roofline_sfu" against a rate measured
        # live, and does not replace the contract fraction.
        acts = wm["acts"]
        t_sfu = acts / sfu_ops_s
        t_hbm_fused = (wm["b_hbm_min"] + 4.0 * wm["w_nodeenv"]) / hbm
        roofline = {"bound": "tensor", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                    "frac": achieved / peak, "traffic": traffic, "traffic_src": traffic_src,
                    "peak_src": f"MEASURED_PEAKS.json {peak_name} ({peaks['src']})", "flops_per_launch": flops,
                    "frac_vs_burst": achieved / peaks["bf16_tflops"], "frac_vs_sustained": achieved / peaks["bf16_tflops_sustained"],
                    "ceiling_frac_if_sfu_bound": t_tensor / t_sfu,
                    "note": "flops = F_prop,dense + F_mlp (SURVEY.md §8(d)); ceiling_frac_if_sfu_bound = tensor floor / MUFU floor "
                            "with one MUFU op per SiLU: the fraction this kernel would show if it ran AT its special-function floor"}
        extra = {
            "roofline_sfu": {"bound": "alu", "kernel": kernel, "achieved": acts / (ms_fused * 1e-3) / 1e12,
                             "peak": sfu_ops_s / 1e12, "unit": "Tactivation/s", "frac": t_sfu / (ms_fused * 1e-3),
                             "peak_src": f"etac_measure_sfu_rate, live on this device: {sfu_per_clk_sm:.2f} MUFU results per clock and SM",
                             "activations_per_launch": acts, "pipe": "MUFU (special-function unit), one op per SiLU"},
            "roofline_floors_us": {"tensor": t_tensor * 1e6, "hbm": t_hbm_fused * 1e6, "sfu_1_mufu_per_act": t_sfu * 1e6},
        }
        t_roof, t_roof_alg = max(t_tensor, t_hbm), max(t_tensor_alg, t_hbm)
        dtype = "bf16"
    else:
        # fp32 contexts (cfg 1, 2): plain FP32 FMA arithmetic; peak derived from the guide's unit counts and clock
        peak = FP32_FMA_TFLOPS
        flops = wm["f_prop_gather"] + wm["f_mlp"]
        flops_alg = wm["f_prop_alg"] + wm["f_mlp_alg"]
        achieved = flops / (ms_fused * 1e-3) / 1e12
        kernel32 = "gather_fp32_kernel" if PHI_SEL == "pernode" else "fp32 PointNet kernels (propagation + encode, global, decode; timed together)"
        roofline = {"bound": "alu", "kernel": kernel32, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                    "frac": achieved / peak, "traffic": traffic, "traffic_src": traffic_src,
                    "peak_src": "derived: 148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts)",
                    "flops_per_launch": flops}
        extra = {}
        t_roof, t_roof_alg = max(flops / (peak * 1e12), t_hbm), max(flops_alg / (peak * 1e12), t_hbm)
        dtype = "f32"
    n_cpu = a.envs if a.workload in ("cfg1", "cfg2", "cfg3") else min(a.envs, 64)      # ~10 s of CPU work
    if PHI_SEL != "pernode":                                                            # slower oracle branch: size the sample from a probe
        n_cpu = int(min(n_cpu, max(8, 10.0 * time_oracle(wl, min(a.envs, 8))["rate"])))
    cpu = time_oracle(wl, n_cpu)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": dtype, "data": "synthetic",
        "node_updates_per_s": value * eng.N,
        "config": {"workload": label, "n_envs_per_gpu": a.envs, "phi": PHI_SEL,
                   "n_nodes": eng.N, "n_patches": eng.P,
                   "precision": "bf16 operands, fp32 accumulate" if bf16 else "fp32",
                   "path": {T.ETAC_PATH_DENSE: "dense", T.ETAC_PATH_SPARSE: "sparse"}.get(path_taken, str(path_taken)),
                   "contact_pairs_per_step": wm["pairs"], "node_envs_per_step": wm["w_nodeenv"],
                   "active_nodes_per_step": wm["n_active"], "realised_contact_frac_of_contacting_patches": wm["contact_frac"],
                   "l2": f"{N_INPUT_SETS} rotating seeded input sets; {12 * a.envs * eng.N / 1e6:.0f} MB output + "
                         f"{10 * a.envs * eng.N / 1e6:.0f} MB workspace per step vs 126 MB L2",
                   "algorithmic_bytes_fused": wm["b_hbm_min"] + 4.0 * wm["w_nodeenv"],
                   "parallelism": f"env-sharded x{world}, no collective"},
        "clocks": clocks,
        "e2e": {"value": world * a.envs * n_e2e / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": n_e2e,
                "note": "pinned host indenters (+ patch poses) -> device, etac_step, full [E,N,3] fp32 result -> pinned host; the read of step i overlaps step i+1 (two result buffers, copy stream)"},
        "e2e_bf16_output": {"value": world * a.envs * n_e2e / (e2e16_ms * 1e-3), "unit": UNIT, "d2h_bytes_per_step": d2h // 2,
                            "note": "same loop, result written as bf16 by the kernel (out_dtype); not the headline"},
        "gpu_launches": launches,
        "kernels_ms": {"s1_sdf_kernel_incl_memsets": ms_s1, "fused_s2_s3_s4_kernel": ms_fused},
        "roofline": roofline,
        "roofline_step": {"roof_dense": t_roof / (ms_step * 1e-3), "roof_alg": t_roof_alg / (ms_step * 1e-3),
                          "t_roof_dense_us": t_roof * 1e6, "t_roof_alg_us": t_roof_alg * 1e6, "t_hbm_us": t_hbm * 1e6,
                          "f_prop_dense": wm["f_prop_dense"], "f_prop_alg": wm["f_prop_alg"], "f_mlp": wm["f_mlp"],
                          "hbm_frac_of_measured": wm["b_hbm_min"] / (ms_step * 1e-3) / hbm,
                          "note": "whole step vs max(F/P, B/BW), SURVEY.md §8(d): roof_dense with F_prop,dense = 6 sum N_p^2 over contacting "
                                  "pairs (the north_star's >= 0.60 target refers to it), roof_alg with F_prop,alg = 6 sum m (N_p - m) "
                                  "and the MLP on passive rows only (the method's own work, Omega is (n-m) x m)"},
        "cpu_baseline": cpu_baseline_dict(cpu, a.envs),
    }
    out.update(extra)
    print(json.dumps(out))
    eng.close()
    if dist is not None:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--envs", type=int, default=0, help="environments per GPU (default: the config's own batch)")
    ap.add_argument("--workload", default="cfg3", choices=sorted(LABELS))
    ap.add_argument("--phi", default="pernode", choices=sorted(PHI),
                    help="residual network: pernode = BASELINE.json's MLP (the metric's config), pointnet = the paper's form of Phi")
    ap.add_argument("--nodes", type=int, nargs="+", default=None, help="cfg5: mesh sizes (default 256 1024 4096 8192)")
    ap.add_argument("--fracs", type=float, nargs="+", default=None, help="cfg5: contact fractions (default 0.001 .. 0.20)")
    ap.add_argument("--fp32", action="store_true", help="cfg5: also time the fp32 context at every point")
    args = ap.parse_args()
    PHI_SEL = args.phi
    if args.phi != "pernode" and args.workload == "cfg5":
        raise SystemExit("--phi pointnet: cfg1 .. cfg4 only")
    args.envs = args.envs or LABELS[args.workload][1]
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # one process per GPU: re-launch under torchrun (the driver's own launch line does the same)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    (run_reference if args.impl == "reference" else run_ours)(args)
