#!/usr/bin/env python
"""bench.py — throughput of the vcs_step hot path on BASELINE.json's headline config.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload (N=1): BASELINE.json configs[3] — 65,536 envs over 256 seed-generated ROMs (128 x 4 KB, 128 x 8 KB F8),
uniform random actions, frameskip 4.  One "step" = one vcs_step(actions, 4) over the whole batch = one launch
of the persistent interpreter kernel.  `value` = env-steps/s with the action stream resident in HBM;
`e2e` = the same through the host-pointer C ABI (actions H2D, RAM + regs + screens D2H every step).
N>1 (torchrun): every rank runs its own 65,536-env shard, no collective on the data path (weak scaling).
`--impl reference` times the CPU oracle (oracle/) on host cores on a bounded sample of the same workload.
Prints ONE JSON line on rank 0."""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FRAMESKIP = 4
METRIC = "env-steps/s (frameskip 4) at batch 65536"
# SURVEY §8(d) lower-bound work model: thread-instructions per 6502 instruction / TIA segment / scanline
MODEL_PER_INSTR, MODEL_PER_SEGMENT, MODEL_PER_LINE = 40, 80, 40


def oracle_sample(w, n_envs: int, steps: int, threads: int):
    """Time the oracle, as it stands, on `n_envs` envs (spread over the ROMs) for `steps` env-steps."""
    from oracle.ovcs_py import OracleVCS
    idx = (np.arange(n_envs) * (w.batch // n_envs) + (np.arange(n_envs) * 37) % max(1, w.batch // n_envs)).astype(np.int64)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx], mappers=getattr(w, "mappers", None))
    acts = w.actions(0, steps + 1)
    o.step(acts[0][idx], FRAMESKIP, threads=threads)                    # untimed: first (short) frame, page-in
    c0 = o.regs()["cycles"].astype(np.int64).sum()
    d0 = [o.debug(e) for e in range(n_envs)]
    t0 = time.perf_counter()
    for t in range(1, steps + 1):
        o.step(acts[t][idx], FRAMESKIP, threads=threads)
    dt = time.perf_counter() - t0
    c1 = o.regs()["cycles"].astype(np.int64).sum()
    d1 = [o.debug(e) for e in range(n_envs)]
    per = n_envs * steps
    work = dict(instr=sum(b.n_instr - a.n_instr for a, b in zip(d0, d1)) / per,
                tia_writes=sum(b.n_tia_writes - a.n_tia_writes for a, b in zip(d0, d1)) / per,
                lines=(c1 - c0) / 76.0 / per, cycles=(c1 - c0) / per)
    return dict(value=per / dt, seconds=dt, cycles_per_s=(c1 - c0) / dt, work=work,
                sample=f"{n_envs} envs (one per {w.batch // n_envs} of {w.name}'s batch, spread over its ROMs) x {steps} env-steps of frameskip 4")


KERNEL_DRAM = os.path.join(ROOT, "profiles", "r02_kernel_dram.txt")


def csrc_hash() -> str:
    """sha256 over the kernel sources (what an ncu capture has to have been taken from to describe this build)"""
    import hashlib
    d = os.path.join(ROOT, "paper_2606_22447_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def kernel_dram_traffic(batch: int):
    """(bytes per launch | None, where it comes from): the committed ncu capture, if it matches batch and sources"""
    try:
        kv = dict(l.strip().split("=", 1) for l in open(KERNEL_DRAM) if "=" in l and not l.startswith("#"))
    except OSError:
        return None, "no capture committed"
    if int(kv.get("batch", -1)) != batch:
        return None, f"{os.path.relpath(KERNEL_DRAM, ROOT)} is for batch {kv.get('batch')}"
    if kv.get("csrc_sha256_16") != csrc_hash():
        return None, f"{os.path.relpath(KERNEL_DRAM, ROOT)} was captured from other kernel sources ({kv.get('csrc_sha256_16')} != {csrc_hash()}): stale"
    return float(kv["dram_bytes_read"]) + float(kv["dram_bytes_write"]), f"{os.path.relpath(KERNEL_DRAM, ROOT)} (ncu --set full, same kernel sources {kv['csrc_sha256_16']})"


class ClockSampler(threading.Thread):
    FIELDS = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index: int):
        super().__init__(daemon=True)
        self.gpu, self.rows, self.stop_flag, self.active = gpu_index, [], False, False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if self.active and out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "power_w_max": max(float(r[2]) for r in self.rows), "samples": len(self.rows)}


def run_paper_axis(args):
    """Instructions per second of 3,000-instruction rollouts over the batch size (the axis of PAPER.md Table 7)."""
    import torch
    import __graft_entry__ as g
    g.build()
    from paper_2606_22447_b200 import VCS
    from vcs_inputs import make_workload
    torch.cuda.set_device(0)
    rows = []
    mode = args.axis_mode                                  # hard | ste | full (the soft modes at the paper's corner alpha = 6, T = 0.14)
    for n in (1, 16, 64, 256, 1024, 4096, 16384, 65536):
        w = make_workload(2, batch=n)
        env = VCS(w.roms, w.seeds, w.env_rom)
        acts = torch.from_numpy(w.actions(0, 16)).cuda()
        if mode != "hard":
            so = torch.empty((n, 8), dtype=torch.float32, device="cuda")
            env.step_instructions = lambda a, k, _e=env, _so=so: _e.step_instructions_soft(a, k, 0.14, 6.0, mode == "full", out=_so)
        for t in range(3):
            env.step_instructions(acts[t], 3000)                   # warm-up rollouts
        torch.cuda.synchronize()
        reps = 10
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
        ev[0].record()
        for t in range(reps):
            env.step_instructions(acts[3 + t], 3000); ev[t + 1].record()
        torch.cuda.synchronize()
        ms = np.array([ev[i].elapsed_time(ev[i + 1]) for i in range(reps)])
        rows.append({"N": n, "ms_per_rollout_mean": float(ms.mean()), "ms_sd": float(ms.std()),
                     "instructions_per_s": n * 3000 / (float(ms.mean()) * 1e-3)})
        env.close()
    print(json.dumps({"metric": "emulated CPU instructions/s, 3,000-instruction rollouts (PAPER.md Table 7 axis)", "unit": "instructions/s",
                      "mode": {"hard": "hard (integer) mode, vcs_step_instructions", "ste": "SOFT-STE mode per instruction (alpha 6, T 0.14), vcs_step_instructions_soft",
                               "full": "FULL mode, the fully relaxed forward (alpha 6, T 0.14: its exact corner), vcs_step_instructions_soft"}[mode]
                              + "; the paper's rows are float32 soft mode on a GTX 1080 Ti with the Pong ROM",
                      "workload": "config 2: N envs sharing one seeded 4K ROM, per-env random actions", "rows": rows}), flush=True)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from vcs_inputs import make_workload
    import __graft_entry__ as g
    from oracle import ovcs_py
    ovcs_py.build()
    w = make_workload(4)
    cores = os.cpu_count() or 1
    n_envs = 32 * cores                                  # the same sample the cpu_baseline leg of the CUDA arm times
    from oracle.ovcs_py import OracleVCS
    idx = (np.arange(n_envs) * (w.batch // n_envs) + (np.arange(n_envs) * 37) % max(1, w.batch // n_envs)).astype(np.int64)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    W, K = max(args.warmup, 1), args.steps
    acts = w.actions(0, W + K)
    for t in range(W):                                   # untimed (the first one is the short frame after reset)
        o.step(acts[t][idx], FRAMESKIP, threads=cores)
    c0 = o.regs()["cycles"].astype(np.int64).sum()
    t0 = time.perf_counter()
    for t in range(W, W + K):
        o.step(acts[t][idx], FRAMESKIP, threads=cores)
    total = time.perf_counter() - t0
    c1 = o.regs()["cycles"].astype(np.int64).sum()
    value = n_envs * K / total
    sample = f"{n_envs} envs (one per {w.batch // n_envs} of config4's batch, spread over its ROMs) x 1 env-step of frameskip 4 per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "env-steps/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": "config4: 65536 envs/GPU, 256 seeded ROMs (half 4K, half 8K F8), uniform random actions, frameskip 4",
                       "batch_per_gpu": 65536, "frameskip": FRAMESKIP, "note": "each step is a bounded sample of the workload (see cpu_baseline.sample)"},
            "cpu_baseline": {"value": value, "unit": "env-steps/s", "cores": cores, "kind": "oracle", "sample": sample,
                             "emulated_cycles_per_s": float(c1 - c0) / total},
            "e2e": {"value": value, "unit": "env-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=120)      # ~1 s of timed steps: long enough for the clock sampler
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=65536, help="envs per GPU (default: BASELINE config 4)")
    ap.add_argument("--workload", type=int, default=4, choices=[2, 3, 4],
                    help="BASELINE config the envs run (default 4, the headline; 2/3 = one shared 4K ROM: the single-game "
                         "axis of the paper's Table 7, SURVEY §8(f) NEXT-2)")
    ap.add_argument("--cart", default=None, choices=["4K", "F8", "F6", "F4", "F8SC", "F6SC", "F4SC", "E0", "FE"],
                    help="with --workload 2: every env runs one seeded cartridge of this format instead of config 2's 4K ROM "
                         "(timing of the other bank-switching schemes, DESIGN.md section 10)")
    ap.add_argument("--soft-T", type=float, default=None,
                    help="run vcs_step_soft (SOFT-STE forward, BASELINE config 5: --workload 2 --batch 4096) at this temperature")
    ap.add_argument("--paper-axis", action="store_true",
                    help="the paper's own throughput axis (PAPER.md Table 7, L566-576; L582 one step = one CPU instruction): "
                         "3,000-instruction rollouts (vcs_step_instructions) of one shared 4K ROM at N in {1, 16, ..., 65536}; prints a table line")
    ap.add_argument("--axis-mode", default="hard", choices=["hard", "ste", "full"], help="with --paper-axis: which forward the rollouts run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.soft_T is not None:
        args.no_e2e = True
    if args.impl == "reference":
        return run_reference(args)
    if args.paper_axis:
        return run_paper_axis(args)

    import torch
    import torch.distributed as dist
    import __graft_entry__ as g
    g.build()
    from paper_2606_22447_b200 import VCS
    from vcs_inputs import make_workload

    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libvcsb200 has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K, W = args.steps, max(args.warmup, 3)
    B = args.batch
    n_roms = (256 if B % 16384 == 0 else 2 if B % 2 == 0 else 1) if args.workload == 4 else 1
    w = make_workload(args.workload, batch=B, n_roms=n_roms if args.workload == 4 else None)
    label = {4: f"config4: {B} envs/GPU, {n_roms} seeded ROMs (half 4K, half 8K F8), uniform random actions, frameskip 4",
             2: f"config2: {B} envs/GPU sharing one seeded 4K ROM, uniform random actions, frameskip 4",
             3: f"config3: {B} envs/GPU sharing one seeded 4K ROM (indexed/indirect, stack, BCD, timers), sticky actions, frameskip 4"}[args.workload]
    mappers = None
    if args.cart is not None:
        if args.workload != 2:
            raise SystemExit("--cart goes with --workload 2")
        from vcs_inputs import FEATURES, make_rom, superchip_rom, e0_rom, fe_rom
        gen = {"4K": lambda: make_rom(4242, FEATURES["4a"]), "F8": lambda: make_rom(4242, FEATURES["4b"]), "F6": lambda: make_rom(4242, FEATURES["f6"]),
               "F4": lambda: make_rom(4242, FEATURES["f4"]), "F8SC": lambda: superchip_rom("F8SC", 4242), "F6SC": lambda: superchip_rom("F6SC", 4242),
               "F4SC": lambda: superchip_rom("F4SC", 4242), "E0": lambda: e0_rom(4242), "FE": lambda: fe_rom(4242)}[args.cart]
        w.roms = [gen()]; mappers = [args.cart]; w.mappers = mappers
        label = f"{B} envs/GPU sharing one seeded {args.cart} cartridge ({len(w.roms[0])} bytes), uniform random actions, frameskip 4"
    if world > 1:                                   # every rank its own env seeds / action streams (same ROM set)
        from paper_2606_22447_b200.shard import rank_seeds
        w.seeds = rank_seeds(w.seeds, rank); w._act_seeds = rank_seeds(w._act_seeds, rank)
    env = VCS(w.roms, w.seeds, w.env_rom, mappers=mappers)
    acts_host = w.actions(0, W + K)
    acts = torch.from_numpy(acts_host).cuda()
    stream = torch.cuda.current_stream()
    if args.soft_T is not None:                     # SOFT-STE forward (alpha 4): same step, soft reads / branches on top
        label = f"config5 (soft mode, T={args.soft_T}, alpha=4) on " + label
        soft_out = torch.empty((B, 8), dtype=torch.float32, device="cuda")
        do_step = lambda a: env.step_soft(a, FRAMESKIP, args.soft_T, 4.0, out=soft_out)
    else:
        do_step = lambda a: env.step(a, FRAMESKIP)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local); sampler.start()
    for t in range(W):
        do_step(acts[t])
    barrier()
    cyc0 = env.regs_host()["cycles"].astype(np.int64).sum()
    l0 = env.launch_count()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    sampler.active = True
    barrier()
    evs[0].record(stream)
    for t in range(K):
        do_step(acts[W + t])
        evs[t + 1].record(stream)
    barrier()
    sampler.active = False
    launches = env.launch_count() - l0
    total_ms = evs[0].elapsed_time(evs[K])
    kern_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(K)]
    cyc1 = env.regs_host()["cycles"].astype(np.int64).sum()
    from paper_2606_22447_b200.shard import reduce_job
    total_ms, cycles = reduce_job(dist if world > 1 else None, total_ms, float(cyc1 - cyc0), device="cuda")
    value = world * B * K / (total_ms * 1e-3)

    # ---- e2e: host-pointer C ABI, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        Ke = max(2, min(K, 5))
        scr_host = torch.empty((B, 210, 160), dtype=torch.uint8).pin_memory().numpy()
        env.step_host(acts_host[0], FRAMESKIP); env.screen_host(out=scr_host)            # warm the staging buffers
        barrier()
        t0 = time.perf_counter()
        for t in range(Ke):
            env.step_host(acts_host[W + t], FRAMESKIP)
            env.ram_host(); env.regs_host(); env.screen_host(out=scr_host)
        barrier()
        dt = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        t0 = time.perf_counter()
        for t in range(Ke):
            env.step_host(acts_host[W + t], FRAMESKIP)
            env.ram_host(); env.regs_host()
        barrier()
        dt2 = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(dt2, op=dist.ReduceOp.MAX)
        e2e = {"value": world * B * Ke / float(dt.item()), "unit": "env-steps/s", "h2d_bytes_per_step": B,
               "d2h_bytes_per_step": B * (128 + 32 + 210 * 160), "steps": Ke,
               "what": "vcs_step_host + vcs_get_ram_host + vcs_get_regs_host + vcs_get_screen_host (pinned screen buffer)",
               "ram_regs_only": {"value": world * B * Ke / float(dt2.item()), "d2h_bytes_per_step": B * 160}}
    sampler.stop_flag = True
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    clocks = sampler.summary()
    cpu = None
    work = None
    if not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        wo = make_workload(args.workload)                # the config at its stated batch (a sample of it is timed)
        if args.cart is not None:
            wo.roms = w.roms; wo.mappers = mappers
        s = oracle_sample(wo, 32 * cores, 96, cores)     # ~10 s of wall clock on the box's 16 cores (~170 core-seconds)
        s1 = oracle_sample(wo, 64, 48, 1)                # the same oracle on ONE core (~9 s)
        work = s["work"]
        cpu = {"value": s["value"], "unit": "env-steps/s", "cores": cores, "kind": "oracle", "sample": s["sample"],
               "emulated_cycles_per_s": s["cycles_per_s"], "seconds": s["seconds"],
               "one_core": {"value": s1["value"], "unit": "env-steps/s", "cores": 1, "emulated_cycles_per_s": s1["cycles_per_s"],
                            "seconds": s1["seconds"], "sample": s1["sample"]}}
    # ---- roofline: integer-issue bound.  peak = 148 SM x 4 schedulers x 32 lanes x SM clock (1 warp-instruction
    # per scheduler per clock); achieved = SURVEY §8(d)'s lower-bound work model x envs / kernel time.
    sm_mhz = clocks.get("sm_mhz") or peaks.get("sm_max_mhz") or 1965.0
    nominal = 148 * 4 * 32 * sm_mhz * 1e6
    from paper_2606_22447_b200.binding import issue_peak
    peak_mixed, _ = issue_peak(1)                   # alu + fma pipes interleaved: the issue-slot ceiling, measured on this box
    peak_alu, _ = issue_peak(0)                     # alu pipe alone (16 lanes / scheduler / clk)
    peak = peak_mixed
    kms = float(np.mean(kern_ms))
    # DRAM bytes of one launch: from the committed `ncu --set full` capture (profiles/KERNEL_DRAM) — used only when that
    # capture was taken from the kernel sources this run was built from (hash of csrc/), else null
    traffic, traffic_note = kernel_dram_traffic(B)
    roof = {"bound": "alu", "unit": "thread-instr/s", "peak": peak,
            "peak_basis": "vcs_issue_peak(kind=1): LOP3+IMAD chains on all SMs, measured in this run",
            "peak_alu_pipe_only": peak_alu, "peak_nominal": nominal,
            "kernel": "vcs_step_kernel", "kernel_ms": kms, "traffic": traffic,
            "traffic_unit": "DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)", "traffic_source": traffic_note,
            "achieved_basis": "modelled: SURVEY 8(d) lower-bound work model (40 / 6502 instruction + 80 / TIA write + 40 / scanline) x counts "
                              "from the oracle's instrumentation in this run; the executed counters are in profiles/"}
    if work:
        ops = MODEL_PER_INSTR * work["instr"] + MODEL_PER_SEGMENT * work["tia_writes"] + MODEL_PER_LINE * work["lines"]
        roof.update(achieved=ops * B / (kms * 1e-3), algorithmic_thread_instr_per_env_step=ops, work_per_env_step=work)
        roof["frac"] = roof["achieved"] / peak
    hbm_bytes = B * (210 * 160 + 2 * (128 + 4 * 15 + 8) + 1)
    roof["hbm"] = {"algorithmic_bytes_per_launch": hbm_bytes, "achieved_gbs": hbm_bytes / (kms * 1e-3) / 1e9,
                   "peak_gbs": peaks.get("hbm_gbs"), "frac": (hbm_bytes / (kms * 1e-3) / 1e9) / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None}
    placement = None
    try:                                            # per-SM finishing times of the last step's blocks
        bt, perm = env.block_times()
        if len(perm) and (bt[:, 1] > bt[:, 0]).all():
            t0_ = bt[:, 0].min(); ends = {}
            for b in range(len(perm)):
                ends[int(bt[b, 2])] = max(ends.get(int(bt[b, 2]), 0.0), float(bt[b, 1] - t0_) * 1e-6)
            ev = np.array(list(ends.values()))
            placement = {"blocks": int(len(perm)), "sms_used": int(len(ev)), "sm_end_ms": {"min": float(ev.min()), "mean": float(ev.mean()), "max": float(ev.max())},
                         "identity": bool((perm == np.arange(len(perm))).all())}
    except Exception as ex:                         # diagnostics only
        placement = {"error": str(ex)}
    line = {"metric": METRIC if B == 65536 else METRIC.replace("65536", str(B)), "value": value, "unit": "env-steps/s", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8" if args.soft_T is None else "u8 + f32 soft reads", "data": "synthetic", "emulated_cycles_per_s": cycles / (total_ms * 1e-3), "frames_per_s": value * FRAMESKIP,
            "config": {"workload": label,
                       "batch_per_gpu": B, "frameskip": FRAMESKIP, "l2": "per-step working set 2.2 GB (screens) > 126 MB L2; no explicit flush",
                       "target_env_steps_per_s": 1e7},
            "clocks": clocks, "gpu_launches": int(launches), "placement": placement, "e2e": e2e, "roofline": roof, "cpu_baseline": cpu}
    if work:      # the paper's own unit (one step = one CPU instruction), from the oracle's instruction count per env-step
        line["emulated_instructions_per_s"] = value * work["instr"]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
