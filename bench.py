#!/usr/bin/env python
"""bench.py -- the LEB hot path on BASELINE.json's headline workload (config 5: 168-state tanh MLP,
B=64 candidate trajectories x T=100 timesteps, forward + VJP), one process per GPU.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input (DESIGN.md
"Measurement"): leb_nn_fwd -> leb_zonotope_inflate -> leb_zonotope_inflate_vjp -> leb_vjp, the forward in
CERTIFIED mode (the library's default: every rounding error of the 3xTF32 path bounded and added outward).
Rank 0 prints ONE JSON line.  `value` = bounded (timestep x state-dim) entries per second over all
ranks with inputs resident in HBM; `e2e` = the same through the C ABI with host buffers
(LEB_FLAG_HOST_IO: H2D/D2H copies inside the timed region); `roofline` = the dominant kernel's
algorithmic flops / its CUDA-event time, measured during the timed steps; `value_mode` = the same step with the
plain (parity-tested) forward; `configs` = the other BASELINE.json configurations (1 GPU, few steps) with the
analytic kernels' ALU roofline; `cpu_baseline` = the oracle timed on this box's host cores on a bounded sample.

--gpus N without a torchrun environment starts N ranks itself (one process per GPU, NCCL for the barrier and the
max-over-ranks only: tiles are independent, there is no collective on the data path).

--impl reference times the oracle (oracle/nn_oracle.py, as it stands) instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bounded (timestep x state-dim) entries/sec incl. VJP"
UNIT = "entries/s"
CONFIG_ID = 5
WORKLOAD = ("config5: MLP 224->512x4->168 tanh residual, Xavier-normal weights, B=64 x T=100 tiles per GPU, "
            "radii U[0.005,0.03], forward + VJP")
KC_NAMES = {0: "chain_gemm_tc2_fwd_kernel (CROWN back-substitution step, CTA pairs)", 1: "chain_gemm_tc2_bwd_kernel (reverse-sweep step, CTA pairs)"}


def _clock_sampler(gpu_index: int):
    q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    try:
        return subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "200",
                                 "-i", str(gpu_index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
    except Exception:
        return None


def _clock_summary(proc):
    if proc is None:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
    proc.terminate()
    try:
        out, _ = proc.communicate(timeout=5)
    except Exception:
        proc.kill()
        out = ""
    sm, smax, reasons = [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for line in out.strip().splitlines():
        f = [x.strip() for x in line.split(",")]
        if len(f) < 7:
            continue
        try:
            sm.append(float(f[0])); smax.append(float(f[1]))
        except ValueError:
            continue
        for name, v in zip(names, f[3:7]):
            if v.lower().startswith("active"):
                reasons.add(name)
    sm.sort()
    return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
            "samples": len(sm), "reasons": sorted(reasons)}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0, "_source": "fallback"}


def _traffic(kernel_key: str):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = line.strip().split(",")
        if len(f) >= 2 and f[0] == kernel_key:
            try:
                return float(f[1])
            except ValueError:
                return None
    return None


def _cpu_oracle_sample(w, tiles: int):
    """Oracle forward + VJP on `tiles` seeded tiles of the workload; returns (entries/s, seconds, threads)."""
    import numpy as np
    from oracle import inflate_oracle, nn_oracle
    threads = 1
    try:
        from threadpoolctl import threadpool_info
        threads = max([int(i.get("num_threads", 1)) for i in threadpool_info()] + [1])
    except Exception:
        pass
    idx = np.linspace(0, w.B * w.T - 1, tiles).astype(int)
    nom, rad = w.nom.reshape(-1, w.N)[idx], w.rad.reshape(-1, w.N)[idx]
    gc, gR = w.g_lo.reshape(-1, w.n)[idx], w.g_hi.reshape(-1, w.n)[idx]
    t0 = time.perf_counter()
    r_lo, r_hi = nn_oracle.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom, rad)
    inflate_oracle.inflate(r_lo, r_hi, 1e-6)
    g_lo, g_hi = inflate_oracle.inflate_vjp(gc, gR)
    nn_oracle.leb_nn_vjp(w.mlp.W, w.mlp.b, w.mlp.act, nom, rad, g_lo, g_hi)
    dt = time.perf_counter() - t0
    return tiles * w.n / dt, dt, threads


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2607_01203_b200 import workloads as wl
    w = wl.make_config(CONFIG_ID)
    tiles_per_step = 3
    for _ in range(args.warmup):
        _cpu_oracle_sample(w, 1)
    t0 = time.perf_counter()
    threads = 1
    for _ in range(args.steps):
        _, _, threads = _cpu_oracle_sample(w, tiles_per_step)
    dt = time.perf_counter() - t0
    value = args.steps * tiles_per_step * w.n / dt
    sample = f"{tiles_per_step} seeded tiles of config 5 per step (forward + fold + VJP), numpy FP64"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_01203_b200 import leb, sharding, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the LEB library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    # weak scaling: every rank owns one full config-5 batch (B=64 x T=100); tiles are independent, so there
    # is no collective on the data path
    w = wl.make_config(CONFIG_ID)
    ctx = leb.context_for_workload(w, local)
    nom, rad = torch.from_numpy(w.nom).to(dev), torch.from_numpy(w.rad).to(dev)
    gc, gR = torch.from_numpy(w.g_lo).to(dev), torch.from_numpy(w.g_hi).to(dev)     # cotangents of (c_bar, R_diag)
    h_nom, h_rad = torch.from_numpy(w.nom).pin_memory(), torch.from_numpy(w.rad).pin_memory()
    h_gc, h_gR = torch.from_numpy(w.g_lo).pin_memory(), torch.from_numpy(w.g_hi).pin_memory()

    REUSE = leb.FLAG_REUSE_FWD      # the VJP starts from the coefficient blocks the step's forward left in HBM (108 GB resident)

    def step_device(fwd_flags=0):
        # fwd_flags = 0: certified forward (N6), the library's default and the mode north_star sanctions for tensor cores;
        # LEB_FLAG_NO_MARGIN: value mode, the mode the parity tests compare with the oracle at this size
        r_lo, r_hi = ctx.leb_nn_fwd(nom, rad, flags=fwd_flags)
        ctx.leb_zonotope_inflate(r_lo, r_hi, 1e-6)
        g_lo, g_hi = ctx.leb_zonotope_inflate_vjp(gc, gR)
        return ctx.leb_vjp(1, nom, rad, g_lo, g_hi, flags=fwd_flags | REUSE)

    HOST = leb.FLAG_HOST_IO
    e2e_bytes = {"h2d": 0, "d2h": 0}
    pin = lambda *shape: torch.empty(shape, dtype=torch.float32, pin_memory=True)
    hb = {k: pin(w.B, w.T, w.n) for k in ("r_lo", "r_hi", "c", "R", "g_lo", "g_hi")}
    hb.update({k: pin(w.B, w.T, w.N) for k in ("gn", "gr")})

    def step_host(count=False):
        r_lo, r_hi = ctx.leb_nn_fwd(h_nom, h_rad, r_lo=hb["r_lo"], r_hi=hb["r_hi"], flags=HOST)
        c, R = ctx.leb_zonotope_inflate(r_lo, r_hi, 1e-6, flags=HOST, c_bar=hb["c"], R_diag=hb["R"])
        g_lo, g_hi = ctx.leb_zonotope_inflate_vjp(h_gc, h_gR, flags=HOST, g_lo=hb["g_lo"], g_hi=hb["g_hi"])
        gn, gr = ctx.leb_vjp(1, h_nom, h_rad, g_lo, g_hi, grad_nom=hb["gn"], grad_rad=hb["gr"], flags=HOST | REUSE)
        if count:
            nb = lambda *ts: sum(t.numel() * t.element_size() for t in ts)
            e2e_bytes["h2d"] = nb(h_nom, h_rad) + nb(r_lo, r_hi) + nb(h_gc, h_gR) + nb(h_nom, h_rad, g_lo, g_hi)
            e2e_bytes["d2h"] = nb(r_lo, r_hi) + nb(c, R) + nb(g_lo, g_hi) + nb(gn, gr)
        return gn, gr

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for _ in range(args.warmup):
        step_device()
    barrier()
    sampler = _clock_sampler(local) if rank == 0 else None
    ctx.leb_profile_reset()
    ctx.leb_profile(True)
    launches0 = ctx.leb_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step_device()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.leb_launch_count() - launches0
    ctx.leb_profile(False)
    kstats = {kc: ctx.leb_profile_read(kc) for kc in (0, 1, 5)}
    clocks = _clock_summary(sampler) if rank == 0 else None
    ms_max = sharding.max_over_ranks(ms, dev)
    launches_total = int(sharding.sum_over_ranks(launches, dev))
    entries_per_rank = w.entries * args.steps
    value = world * entries_per_rank / (ms_max * 1e-3)

    # ---- end to end through the C ABI with host buffers
    for _ in range(max(1, min(args.warmup, 2))):
        step_host(count=True)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_host()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    dt_max = sharding.max_over_ranks(dt, dev)
    e2e_value = world * entries_per_rank / dt_max

    assert ctx.leb_nn_state()[1:] == (True, True), "the timed step did not reuse its certified forward state"
    value_mode = None
    if rank == 0:
        # outside the timed region: what the certified margin costs in tightness, against the value-mode (parity) result
        c_lo, c_hi = ctx.leb_nn_fwd(nom, rad, flags=0)
        v_lo, v_hi = ctx.leb_nn_fwd(nom, rad, flags=leb.FLAG_NO_MARGIN)
        width = (v_hi - v_lo).clamp_min(1e-12)
        ex = torch.maximum(c_hi - v_hi, v_lo - c_lo) / width
        # the same step with the forward in value mode (the mode the parity tests compare with the oracle)
        step_device(leb.FLAG_NO_MARGIN)
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(args.steps):
            step_device(leb.FLAG_NO_MARGIN)
        c1.record()
        torch.cuda.synchronize()
        vm_ms = c0.elapsed_time(c1) / max(args.steps, 1)
        value_mode = {"ms_per_step": vm_ms, "value": w.entries / (vm_ms * 1e-3),
                      "certified_excess_over_value_mode_median": float(ex.median()),
                      "certified_excess_over_value_mode_max": float(ex.max()),
                      "unit": "fraction of the enclosure width", "certified_contains_value_mode": bool((ex >= -1e-5).all())}
        # CROWN-IBP (LEB_FLAG_IBP_HIDDEN, value mode): the cheap, loose variant -- hidden bounds by interval propagation
        IBPF = leb.FLAG_NO_MARGIN | leb.FLAG_IBP_HIDDEN
        step_device(IBPF)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(args.steps):
            step_device(IBPF)
        c1.record()
        torch.cuda.synchronize()
        ib_ms = c0.elapsed_time(c1) / max(args.steps, 1)
        i_lo, i_hi = ctx.leb_nn_fwd(nom, rad, flags=IBPF)
        ic_lo, ic_hi = ctx.leb_nn_fwd(nom, rad, flags=leb.FLAG_IBP_HIDDEN)          # certified CROWN-IBP: tightness cost only
        value_mode["crown_ibp"] = {"ms_per_step": ib_ms, "value": w.entries / (ib_ms * 1e-3),
                                   "enclosure_width_over_full_crown": float((i_hi - i_lo).sum() / (v_hi - v_lo).sum()),
                                   "certified_excess_over_value_mode_max": float((torch.maximum(ic_hi - i_hi, i_lo - ic_lo)
                                                                                  / (i_hi - i_lo).amax(dim=2, keepdim=True)).max())}
    if rank == 0:
        peaks = _peaks()
        dom = max((0, 1), key=lambda kc: kstats[kc][0])
        k_ms, k_flops, k_n = kstats[dom]
        tot_ms = sum(kstats[kc][0] for kc in kstats)
        # 3xTF32 tcgen05 contraction: tensor-bound.  One FP32-equivalent product costs three TF32 MMAs, so the peak for
        # ALGORITHMIC flops is (TF32 dense peak) / 3; TF32 peak = measured bf16 peak x 0.5 (the guide's nominal ratio).
        # The kernel is timed inside a long step, so the sustained bf16 figure is the denominator.
        bf16_peak = float(peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops", 1400.0)))
        tf32_peak = 0.5 * bf16_peak
        peak = tf32_peak / 3.0
        achieved = (k_flops / 1e12) / (k_ms * 1e-3) if k_ms > 0 else 0.0
        other = 1 - dom
        roofline = {"bound": "tensor", "kernel": KC_NAMES[dom], "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                    "frac": achieved / peak, "traffic": _traffic("chain_fwd" if dom == 0 else "chain_bwd"),
                    "peak_source": f"{peaks['_source']} bf16 sustained {bf16_peak:.1f} TFLOP/s x 0.5 (TF32) / 3 (3xTF32 split)",
                    "executed_tf32_tflops": 3.0 * achieved, "tf32_peak": tf32_peak,
                    "launches": k_n, "avg_launch_ms": k_ms / max(k_n, 1),
                    "kernel_share_of_step": k_ms / ms if ms > 0 else None,
                    "all_chain_gemm_share_of_step": (kstats[0][0] + kstats[1][0]) / ms if ms > 0 else None,
                    "other_kernel": {"kernel": KC_NAMES[other], "achieved": (kstats[other][1] / 1e12) / max(kstats[other][0] * 1e-3, 1e-12),
                                     "frac": (kstats[other][1] / 1e12) / max(kstats[other][0] * 1e-3, 1e-12) / peak,
                                     "launches": kstats[other][2]},
                    "algorithmic_tflop_per_step": (kstats[0][1] + kstats[1][1]) / 1e12 / max(args.steps, 1)}
        cpu = None
        if world == 1:
            tiles = 12
            v, secs, threads = _cpu_oracle_sample(w, tiles)
            cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                   "sample": f"{tiles} seeded tiles of config 5 (forward + fold + VJP), {secs:.1f} s, numpy FP64"}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_max / max(args.steps, 1), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOAD, "global_batch": 64 * world, "horizon": 100, "tiles": w.B * w.T * world,
                           "parallelism": f"dp{world} (independent tiles, no collective)",
                           "l2": "working set (82 GB of coefficient blocks, streamed once per chain step) exceeds the 126 MB L2; no flush needed",
                           "mode": "certified forward (rounding errors of the 3xTF32 tcgen05 contractions bounded and added outward), VJP "
                                   "from the step's resident forward state (LEB_FLAG_REUSE_FWD); `value_mode` = the same step with the "
                                   "plain forward the parity tests compare with the oracle"},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e_bytes["h2d"], "d2h_bytes_per_step": e2e_bytes["d2h"],
                        "ms_per_step": 1e3 * dt_max / max(args.steps, 1)},
                "gpu_launches": launches_total, "roofline": roofline, "cpu_baseline": cpu, "value_mode": value_mode}
        ctx.close()
        ctx = None
        if world == 1 and not args.no_configs:
            line["configs"] = {f"config{c}": _config_record(c, 3, 2, peaks) for c in (1, 2, 3, 4)}
            line["configs"]["tube"] = _tube_record(peaks)
            line["configs"]["next_rows"] = _next_rows_record(max(args.steps, 3), 2)
        print(json.dumps(line))
    if ctx is not None:
        ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def _alu_peak(peaks):
    """FP32 ALU roofline of the analytic kernels: interval arithmetic is directed-rounding FADD / FMUL and FMNMX, one FP32
    operation per lane and instruction (no FMA contraction: every endpoint product is rounded on its own and goes through a
    min / max), so peak = 148 SMs x 128 FP32 lanes x sm_max clock."""
    return 148 * 128 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12


def _config_record(cfg, steps, warmup, peaks):
    """One of the other BASELINE.json configurations on cuda:0: the same step (forward -> fold -> fold VJP -> VJP),
    device-resident inputs, few steps.  Parity-test cases, not the bench line."""
    import torch
    from paper_2607_01203_b200 import leb, workloads as wl
    dev = torch.device("cuda", 0)
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w, 0)
    nom, rad = torch.from_numpy(w.nom).to(dev), torch.from_numpy(w.rad).to(dev)
    gc, gR = torch.from_numpy(w.g_lo).to(dev), torch.from_numpy(w.g_hi).to(dev)
    kind = 0 if w.kind == "analytic" else 1

    def fwd():
        return ctx.leb_analytic_fwd(nom, rad) if kind == 0 else ctx.leb_nn_fwd(nom, rad)

    def step():
        r_lo, r_hi = fwd()
        ctx.leb_zonotope_inflate(r_lo, r_hi, 1e-6)
        g_lo, g_hi = ctx.leb_zonotope_inflate_vjp(gc, gR)
        return ctx.leb_vjp(kind, nom, rad, g_lo, g_hi, flags=leb.FLAG_REUSE_FWD if kind else 0)

    def timed(f, n):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / max(n, 1)

    for _ in range(warmup):
        step()
    launches0 = ctx.leb_launch_count()
    ctx.leb_profile_reset()
    ctx.leb_profile(True)
    ms = timed(step, steps)
    ctx.leb_profile(False)
    launches = ctx.leb_launch_count() - launches0
    rec = {"workload": f"{w.name}: {w.kind}, B={w.B} x T={w.T} tiles, n={w.n}, N={w.N}", "ms_per_step": ms,
           "entries_per_s": w.entries / (ms * 1e-3), "gpu_launches_per_step": launches // max(steps, 1)}
    if kind == 0:
        peak = _alu_peak(peaks)
        st = ctx.leb_analytic_tape_stats()
        rec["tape"] = st
        for name, kc in (("fwd_kernel", 2), ("vjp_kernel", 3)):
            k_ms, k_flops, k_n = ctx.leb_profile_read(kc)
            ach = (k_flops / 1e12) / (k_ms * 1e-3) if k_ms > 0 else 0.0
            rec[name] = {"bound": "alu", "avg_launch_ms": k_ms / max(k_n, 1), "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                         "frac": ach / peak, "algorithmic_gflop_per_launch": k_flops / max(k_n, 1) / 1e9}
    rec["ms_forward_only"] = timed(fwd, steps)
    ctx.close()
    return rec


def _tube_record(peaks, B=16, T=100, n=168, m=56):
    """Tube propagation (27)-(28) and J_err (35) at config-5 shape: HBM-bound streams over the closed-loop responses
    (B = 16 trajectories: 12 GB of Phi, far beyond L2).  Synthetic responses drawn on the device, Phi^x_{j+1,j} = I."""
    import torch
    from paper_2607_01203_b200 import leb
    dev = torch.device("cuda", 0)
    g = torch.Generator(device=dev)
    g.manual_seed(20260706)
    nb = T * (T + 1) // 2
    Phi = torch.empty((B, nb, n + m, n), dtype=torch.float32, device=dev)
    for b in range(B):
        Phi[b].normal_(0.0, 1.0 / n ** 0.5, generator=g)
    for j in range(T):
        Phi[:, (j + 1) * j // 2 + j, :n] = torch.eye(n, device=dev)
    c = torch.randn((B, T, n), device=dev, generator=g) * 0.05
    R = torch.rand((B, T, n), device=dev, generator=g) * 0.1 + 1e-3
    E = torch.rand((n,), device=dev, generator=g) * 0.05
    ctx = leb.Context(0)
    rec = {"workload": f"tube propagation + J_err: B={B} x T={T}, n={n}, m={m}, Phi {Phi.numel() * 4 / 1e9:.1f} GB (synthetic)"}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    for name, f in (("tube_kernel", lambda: ctx.leb_tube_propagate(Phi, c, R, m, E)), ("jerr_kernel", lambda: ctx.leb_jerr(Phi, R, m, E))):
        for _ in range(2):
            f()
        ctx.leb_profile_reset()
        ctx.leb_profile(True)
        for _ in range(3):
            f()
        ctx.leb_profile(False)
        k_ms, k_bytes, k_n = ctx.leb_profile_read(6)
        ach = (k_bytes / 1e9) / (k_ms * 1e-3) if k_ms > 0 else 0.0
        rec[name] = {"bound": "hbm", "avg_launch_ms": k_ms / max(k_n, 1), "achieved": ach, "peak": hbm, "unit": "GB/s",
                     "frac": ach / hbm, "algorithmic_gb_per_launch": k_bytes / max(k_n, 1) / 1e9}
    ctx.close()
    return rec


def _next_rows_record(steps, warmup):
    """Timings of the SURVEY 8(f) variants (device-resident inputs, CUDA events): non-centred boxes on configs 4 and 5, input-
    domain partitioning with its VJP and PGD refinement on config 2, optimised slopes on config 3.  Parity-test cases, timing only."""
    import numpy as np
    import torch
    from paper_2607_01203_b200 import leb, workloads as wl
    dev = torch.device("cuda", 0)

    def timed(f, n):
        for _ in range(warmup):
            f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / max(n, 1)

    def dv(a):
        return torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    rec = {}
    # non-centred boxes, analytic (config 4) and NN (config 5, certified, 16 trajectories)
    for cfg, kw in ((4, {}), (5, {"B": 16})):
        w = wl.make_config(cfg, **kw)
        ctx = leb.context_for_workload(w, 0)
        nom, rad, mu = dv(w.nom), dv(w.rad), dv(wl.make_mu(w, 1.0))
        g_lo, g_hi = dv(w.g_lo), dv(w.g_hi)
        kind = 0 if w.kind == "analytic" else 1
        fwd = (lambda: ctx.leb_analytic_fwd(nom, rad, mu=mu)) if kind == 0 else (lambda: ctx.leb_nn_fwd(nom, rad, mu=mu))

        def step():
            fwd()
            ctx.leb_vjp_mu(kind, nom, rad, mu, g_lo, g_hi, flags=leb.FLAG_REUSE_FWD if kind else 0)
        ms_f, ms_s = timed(fwd, steps), timed(step, steps)
        rec[f"mu_config{cfg}"] = {"workload": f"{w.name}, B={w.B} x T={w.T} tiles, |mu| <= sigma", "ms_forward": ms_f, "ms_forward_plus_vjp": ms_s,
                                  "entries_per_s": w.entries / (ms_s * 1e-3)}
        ctx.close()
    # partitioning (12 sub-boxes per tile) with its VJP, and 8 PGD steps, config 2
    w = wl.make_config(2)
    ctx = leb.context_for_workload(w, 0)
    nom, rad, g_lo, g_hi = dv(w.nom), dv(w.rad), dv(w.g_lo), dv(w.g_hi)
    splits = np.ones(w.N, dtype=int)
    splits[[3, 4, 12]] = (2, 3, 2)
    rec["partition_config2"] = {"workload": f"{w.name}, {w.B * w.T} tiles x 12 sub-boxes",
                                "ms_forward": timed(lambda: ctx.leb_analytic_partition_fwd(nom, rad, splits), steps),
                                "ms_vjp": timed(lambda: ctx.leb_analytic_partition_vjp(nom, rad, splits, g_lo, g_hi), steps)}
    eps = 0.5 * rad
    rec["pgd_config2"] = {"workload": f"{w.name}, {w.B * w.T} tiles, 8 projected gradient steps on the nominal point",
                          "ms": timed(lambda: ctx.leb_analytic_pgd(nom, rad, eps, nom + 0.4 * rad, 8, 0.03), steps)}
    ctx.close()
    # optimised lower slopes, config 3 (certified result)
    w = wl.make_config(3)
    ctx = leb.context_for_workload(w, 0)
    nom, rad = dv(w.nom), dv(w.rad)
    ms = timed(lambda: ctx.leb_nn_alpha_fwd(nom, rad, 6, 10.0), steps)
    lo, hi, w0, wb = ctx.leb_nn_alpha_fwd(nom, rad, 6, 10.0, flags=leb.FLAG_NO_MARGIN)
    rec["alpha_config3"] = {"workload": f"{w.name}, {w.B * w.T} tiles, 6 slope steps + certified evaluation", "ms": ms,
                            "width_over_adaptive_slopes_median": float((wb / w0).median())}
    ctx.close()
    return rec


def _spawn_worker(local_rank, world, port, argv):
    os.environ.update({"RANK": str(local_rank), "LOCAL_RANK": str(local_rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.argv = argv
    sys.exit(main())


def run_other_config(args):
    """--config 1..4: the same step (forward -> fold -> fold VJP -> VJP) on one of the other BASELINE.json configurations,
    1 GPU, device-resident inputs.  These are parity-test cases, not the bench line (the contract's line is config 5);
    this mode exists so that the numbers quoted in DESIGN.md / profiles/ come from a committed command."""
    import torch
    from paper_2607_01203_b200 import leb, workloads as wl
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the LEB library has no CPU fallback")
    dev = torch.device("cuda", 0)
    w = wl.make_config(args.config)
    ctx = leb.context_for_workload(w, 0)
    nom, rad = torch.from_numpy(w.nom).to(dev), torch.from_numpy(w.rad).to(dev)
    gc, gR = torch.from_numpy(w.g_lo).to(dev), torch.from_numpy(w.g_hi).to(dev)
    kind = 0 if w.kind == "analytic" else 1

    def fwd():
        return ctx.leb_analytic_fwd(nom, rad) if kind == 0 else ctx.leb_nn_fwd(nom, rad)

    def step():
        r_lo, r_hi = fwd()
        ctx.leb_zonotope_inflate(r_lo, r_hi, 1e-6)
        g_lo, g_hi = ctx.leb_zonotope_inflate_vjp(gc, gR)
        return ctx.leb_vjp(kind, nom, rad, g_lo, g_hi, flags=leb.FLAG_REUSE_FWD if kind else 0)

    def timed(f, n):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / max(n, 1)

    for _ in range(args.warmup):
        step()
    launches0 = ctx.leb_launch_count()
    ms = timed(step, args.steps)
    launches = ctx.leb_launch_count() - launches0
    ms_fwd = timed(fwd, args.steps)
    line = {"metric": METRIC, "value": w.entries / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "ms_forward_only": ms_fwd, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config{args.config}: {w.kind}, B={w.B} x T={w.T} tiles, n={w.n}, N={w.N} (parity-test case, not the bench line)"},
            "gpu_launches": launches}
    print(json.dumps(line))
    ctx.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=CONFIG_ID, choices=[1, 2, 3, 4, 5],
                    help="5 (default) = the bench line; 1-4 = the other BASELINE.json configurations, timing only")
    ap.add_argument("--no-configs", action="store_true", help="skip the `configs` record (configs 1-4) of the bench line")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.config == CONFIG_ID:
        # launched without torchrun: start the N ranks here, one process per GPU
        import torch
        import torch.multiprocessing as mp
        if torch.cuda.device_count() < args.gpus:
            raise RuntimeError(f"--gpus {args.gpus} but only {torch.cuda.device_count()} CUDA devices are visible")
        import socket
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
        mp.spawn(_spawn_worker, args=(args.gpus, port, list(sys.argv)), nprocs=args.gpus, join=True)
        return 0
    if args.config != CONFIG_ID:
        return run_other_config(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
