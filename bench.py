#!/usr/bin/env python
"""bench.py — env-steps/s of the batched differentiable rod step at BASELINE.json config 5 (4096 ropes x 128 verts).

BASELINE.json's metric is "fwd AND fwd+bwd env-steps/s": one run measures both and prints ONE JSON line.
  value / ms_per_step   one "step" = one pass of the whole hot path over one batch of synthetic input: a full forward
                        rollout (H frames of 5 substeps, checkpoints every `stride` frames) followed by the checkpointed
                        reverse pass.  value = B*H*n_gpus / time, CUDA events on the launching stream, inputs resident in HBM.
  forward               {value, ms_per_step, roofline}: the forward rollout alone (no checkpoints), timed the same way.
  e2e                   the fwd+bwd pass through the host-buffer C-ABI calls (host->device copies of x0, v0, actions and
                        device->host copies of x_T and the gradients inside the timed region).
  roofline              for the dominant kernel of the fwd+bwd pass (k_adjoint): algorithmic flops of its launches divided by
                        their durations, measured live with CUDA events on the launching stream (dlo_set_kernel_timing),
                        against the fp32 peak MEASURED in the same run by the library's FFMA-chain microbenchmark.
  cpu_baseline          the fp64 oracle, as it stands, on a bounded sample of the same workload (rank 0).
`--impl reference` times the oracle instead (the tier's reference arm).  `--mode fwd|fwdbwd` restricts a run to one mode.

Multi-GPU (torchrun): envs are independent, so ranks run disjoint shards of the batch with no collective on the data
path ("scaling": "weak"); every time is the max over ranks.
"""
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

from workloads.configs import make_problem, loss_and_seed, FULL_SIZES  # noqa: E402

METRIC = "env_steps_per_s"
UNIT = "env-steps/s"
# Algorithmic fp32 flops per env-step of config 5 (5 substeps, N=128, N_C=10, 4 primitives + 4 finger capsules), counted in
# DESIGN.md section 5 (FADD/FMUL = 1, FFMA = 2): forward kernel 0.5 Mflop, the same for the replay, adjoint kernel 0.85 Mflop.
# They are hand counts for config 5 only: no roofline is printed for another config.
ALG_FLOPS = {"k_forward": 0.5e6, "k_replay": 0.5e6, "k_adjoint": 0.85e6}
TAPE_ROWS_BASE = 22          # tape record rows besides the N_C multiplier rows (rod_warp.cuh: 14 state, dx 3, v1 3, S, mask)


class ClockSampler(threading.Thread):
    """samples nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def oracle_leg(problem, mode, budget_s, steps=1, warmup=0):
    """the fp64 oracle, as it stands, on a bounded sample of the same workload (rank 0, host cores).
    Returns (cpu_baseline dict, seconds per pass, passes actually timed)."""
    from oracle import dlo_oracle as orc
    cores = orc.num_threads()
    H_full, stride = problem["horizon"], problem["checkpoint_stride"]
    B = problem["config"]["batch"]

    def one(envs, H):
        sim = orc.OracleSim(problem, envs=envs)
        t0 = time.perf_counter()
        st = sim.rollout(H, max(1, min(stride, H)) if mode != "fwd" else 0)
        if mode != "fwd":
            sub = dict(problem, loss=dict(problem["loss"], target=problem["loss"]["target"][envs]))
            _, seed = loss_and_seed(sub, st["x"])
            sim.backward(seed)
        dt = time.perf_counter() - t0
        sim.close()
        return dt

    envs = np.arange(min(B, cores))
    probe_H = 4
    rate = len(envs) * probe_H / one(envs, probe_H)          # env-steps/s, rough
    # size one pass for ~budget_s / (passes + 1): grow the horizon first, then the number of envs
    units = max(rate * budget_s / (steps + warmup + 1), len(envs) * probe_H)
    H = int(min(H_full, max(probe_H, units // len(envs))))
    n_env = int(min(B, max(len(envs), (units // H) // cores * cores)))
    envs = np.arange(n_env)
    times = []
    for it in range(warmup + steps):
        dt = one(envs, H)
        if it >= warmup:
            times.append(dt)
    t = float(np.mean(times))
    return {"value": len(envs) * H / t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d envs x %d steps of config %d (%s, fp64%s), %.1f s per pass, %d passes timed" % (
                len(envs), H, problem.get("config_id", 5), mode, ", tape-AD reverse" if mode != "fwd" else "", t, len(times))}, t, len(times)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="both", choices=["both", "fwd", "fwdbwd"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--batch", type=int, default=None, help="per-GPU batch (default: the config's)")
    ap.add_argument("--horizon", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    full = FULL_SIZES[args.config]
    B = args.batch or full["batch"]
    H = args.horizon or full["horizon"]
    N = full["n_verts"]
    stride = full["stride"] if full["stride"] > 0 else H      # config 2 is forward-only in BASELINE.json: one segment if asked for a reverse pass
    stride = min(stride, H)
    main_mode = "fwd" if args.mode == "fwd" else "fwdbwd"
    workload = "config %d: %d ropes x %d verts per GPU, %d frames x 5 substeps, checkpoint stride %d" % (args.config, B, N, H, stride)
    base = {"metric": METRIC, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload, "mode": main_mode, "per_gpu_batch": B, "n_verts": N, "horizon": H,
                       "checkpoint_stride": stride if main_mode == "fwdbwd" else 0,
                       "cache": "inputs (actions %.0f MB) larger than L2" % (H * B * 2 * 6 * 4 / 1e6)}}

    if args.impl == "reference":
        if rank != 0:
            return
        problem = make_problem(args.config, batch=min(B, 256), horizon=H, stride=stride)
        cb, t, n_timed = oracle_leg(problem, main_mode, budget_s=60, steps=args.steps, warmup=min(args.warmup, 1))
        line = dict(base, impl="reference", value=cb["value"], ms_per_step=t * 1e3, dtype="f64", cpu_baseline=cb,
                    e2e={"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, gpu_launches=0)
        line["steps"] = n_timed
        line["warmup"] = min(args.warmup, 1)
        line["config"] = dict(line["config"], sample=cb["sample"])
        print(json.dumps(line))
        return

    import torch
    import torch.distributed as dist
    import paper_2606_04206_b200 as dlo
    from paper_2606_04206_b200.sharding import max_over_ranks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the DLO library has no CPU path")
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    # the denominator first, on an idle GPU: fp32 FFMA-chain microbenchmark of the library
    peak_tf, peak_ms, n_sm = dlo.dlo_measure_fp32_peak(torch.cuda.current_stream().cuda_stream)

    # each rank generates its own shard: same recipe, env ids offset by rank (weak scaling, no data-path collective)
    problem = make_problem(args.config, batch=B, horizon=H)
    if world > 1:
        rng = np.random.Generator(np.random.PCG64(977 + rank))
        problem["x0"] = problem["x0"] + rng.normal(0, 1e-5, problem["x0"].shape)
    sim = dlo.DloSim(problem, device=str(dev))
    G = sim.G
    target = torch.as_tensor(problem["loss"]["target"], dtype=torch.float32, device=dev)
    if target.dim() == 2:
        target = torch.zeros((B, 3, N), device=dev)
    seed_t, x_t = torch.zeros((B, 3, N), device=dev), torch.empty((B, 3, N), device=dev)
    grads = {"a": torch.zeros((H, B, max(G, 1), 6), device=dev), "x": torch.zeros((B, 3, N), device=dev),
             "v": torch.zeros((B, 3, N), device=dev), "m": torch.zeros((B, 5), device=dev)}

    def fwd_pass():
        dlo.dlo_rollout_forward(sim.h, H, 0)

    def fwdbwd_pass():
        dlo.dlo_rollout_forward(sim.h, H, stride)
        # loss head of the harness: mean squared distance to the target polyline -> dL/dx_T on the device
        dlo.dlo_get_state(sim.h, x_t)
        torch.sub(x_t, target, out=seed_t)
        seed_t.mul_(2.0 / N)
        dlo.dlo_backward(sim.h, seed_t, None, grads["a"] if G > 0 else None, grads["x"], grads["v"], grads["m"])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(one_pass):
        """W untimed + K timed passes, barrier + synchronize on both sides, CUDA events, max over ranks"""
        for _ in range(args.warmup):
            one_pass()
        barrier()
        dlo.dlo_set_kernel_timing(sim.h, True)
        l0 = dlo.dlo_launch_count(sim.h)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        ev[0].record()
        for k in range(args.steps):
            one_pass()
            ev[k + 1].record()
        barrier()
        launches = dlo.dlo_launch_count(sim.h) - l0
        kt = [dlo.dlo_get_kernel_timing(sim.h, c) for c in range(3)]
        dlo.dlo_set_kernel_timing(sim.h, False)
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
        ms = max_over_ranks(ev[0].elapsed_time(ev[-1]), dev) / args.steps
        return {"ms_per_step": ms, "value": B * H * world / (ms * 1e-3), "launches": int(launches), "ms_per_pass": per, "kernels": kt}

    def kernel_roofline(name, kt):
        """roofline object of one kernel class from its live event timing (config 5 only: the flop counts are config 5's)"""
        n, tot_ms, units = kt
        if args.config != 5 or n == 0:
            return None
        achieved = ALG_FLOPS[name] * units / (tot_ms * 1e-3) / 1e12
        r = {"bound": "alu", "kernel": name, "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf,
             "launches_timed": n, "ms_per_launch": tot_ms / n, "env_steps_per_launch": units // n,
             "algorithmic_flops_per_env_step": ALG_FLOPS[name],
             "peak_source": "measured: FFMA-chain microbenchmark of the library in this run (%d SMs, %.1f ms)" % (n_sm, peak_ms),
             "traffic": None}
        if name != "k_forward":
            # HBM bytes one launch has to move by construction: its tape records (written by the replay, read once by the adjoint)
            rec_bytes = (TAPE_ROWS_BASE + problem["config"]["n_proj_iters"]) * ((N + 3) // 4 * 4) * 4
            r["traffic"] = int(units // n * problem["config"]["n_substeps"] * rec_bytes)
            r["traffic_source"] = "tape layout: (22 + N_C) rows x NS x 4 B per env-substep x the env-substeps of one launch; ncu's dram bytes: profiles/"
            r["hbm_gbs"] = r["traffic"] / (tot_ms / n * 1e-3) / 1e9
            # replays of earlier segments run on a second stream under the adjoints of later ones: both kernels' event times span that overlap
            r["note"] = "launch durations include the time shared with the other stream's kernel (replay under adjoint); stand-alone durations: profiles/r02_ncu_summary.md"
        return r

    sampler = ClockSampler(local_rank)
    sampler.start()
    res_fb = timed(fwdbwd_pass) if args.mode in ("both", "fwdbwd") else None
    res_f = timed(fwd_pass) if args.mode in ("both", "fwd") else None
    clocks = sampler.stop()
    n_bad = sim.n_bad()

    # end to end through the host-buffer C-ABI calls (the fwd+bwd pass, or the forward pass in --mode fwd)
    e2e = None
    if not args.no_e2e:
        x0h = np.ascontiguousarray(problem["x0"], dtype=np.float32)
        v0h = np.ascontiguousarray(problem["v0"], dtype=np.float32)
        acth = np.ascontiguousarray(problem["actions"], dtype=np.float32)
        xTh = np.empty_like(x0h)
        tgt = np.ascontiguousarray(problem["loss"]["target"], dtype=np.float32)
        gah, gmh = np.empty_like(acth), np.empty((B, 5), dtype=np.float32)
        h2d = x0h.nbytes + v0h.nbytes + acth.nbytes
        d2h = xTh.nbytes
        if main_mode == "fwdbwd":
            h2d += x0h.nbytes
            d2h += gah.nbytes + gmh.nbytes

        def e2e_pass():
            dlo.dlo_rollout_forward_host(sim.h, x0h, v0h, None, acth, H, stride if main_mode == "fwdbwd" else 0, xTh, None)
            if main_mode == "fwdbwd":
                seed = ((xTh - tgt) * (2.0 / N)).astype(np.float32)
                dlo.dlo_backward_host(sim.h, seed, None, gah, None, None, gmh)
        e2e_pass()
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            e2e_pass()
        barrier()
        te = max_over_ranks((time.perf_counter() - t0) / n_e2e, dev)
        e2e = {"value": B * H * world / te, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "passes_timed": n_e2e}

    if rank != 0:
        return
    peaks, which = measured_peaks()
    main_res = res_fb if res_fb is not None else res_f
    line = dict(base, value=main_res["value"], ms_per_step=main_res["ms_per_step"], e2e=e2e, gpu_launches=main_res["launches"], clocks=clocks,
                envs_flagged=int(n_bad), ms_per_pass=main_res["ms_per_pass"],
                fp32_peak={"tflops": peak_tf, "source": "FFMA-chain microbenchmark (dlo_measure_fp32_peak), idle GPU, best of 3", "n_sm": n_sm,
                           "nominal_tflops": n_sm * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12, "hbm_gbs_" + which: peaks.get("hbm_gbs")})
    if res_fb is not None:
        line["roofline"] = kernel_roofline("k_adjoint", res_fb["kernels"][2])
        line["kernel_share"] = {name: {"launches": kt[0], "ms_per_step": kt[1] / args.steps}
                                for name, kt in zip(("k_forward", "k_replay", "k_adjoint"), res_fb["kernels"])}
        line["roofline_replay"] = kernel_roofline("k_replay", res_fb["kernels"][1])
    else:
        line["roofline"] = kernel_roofline("k_forward", res_f["kernels"][0])
    if res_f is not None and res_fb is not None:
        line["forward"] = {"value": res_f["value"], "unit": UNIT, "ms_per_step": res_f["ms_per_step"], "gpu_launches": res_f["launches"],
                           "ms_per_pass": res_f["ms_per_pass"], "roofline": kernel_roofline("k_forward", res_f["kernels"][0])}
    if not args.no_cpu_baseline:
        cb, _, _ = oracle_leg(make_problem(args.config, batch=256, horizon=H, stride=stride), main_mode, budget_s=40)   # one pass of ~10-20 s
        line["cpu_baseline"] = cb
    print(json.dumps(line))


if __name__ == "__main__":
    main()
