#!/usr/bin/env python
"""bench.py — env-steps/s of the batched differentiable rod step at BASELINE.json config 5 (4096 ropes x 128 verts).

One "step" of this benchmark = one pass of the whole hot path over one batch of synthetic input: a full
forward rollout (H frames of 5 substeps, checkpoints every `stride` frames) followed by the checkpointed reverse
pass (`--mode fwdbwd`, default) or the forward rollout alone (`--mode fwd`).  `value` = B*H*n_gpus / time,
timed with CUDA events on the launching stream, inputs resident in HBM.  `e2e` is the same metric through the
host-buffer C-ABI calls (host->device copies of x0, v0, actions and device->host copies of x_T and the
gradients inside the timed region).  `--impl reference` times the fp64 CPU oracle on a bounded sample instead.

Prints ONE JSON line.  Multi-GPU (torchrun): envs are independent, so ranks run disjoint shards of the batch
with no collective on the data path ("scaling": "weak"); the time is the max over ranks.
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
# Algorithmic fp32 flops per env-step of config 5 (5 substeps, N=128, N_C=10, 4 primitives + 4 finger capsules), counted
# in DESIGN.md section 7 (FADD/FMUL = 1, FFMA = 2): forward 0.10 Mflop per substep = 0.5 Mflop per env-step; the reverse of a
# substep 0.17 Mflop; forward+backward = forward + replay + reverse = 0.5 + 0.5 + 0.85 = 1.85 Mflop per env-step.
FLOPS_PER_ENV_STEP = {"fwd": 0.5e6, "fwdbwd": 1.85e6}
# DRAM bytes per env-substep of the dominant kernel (k_adjoint), from the `ncu --set full` capture summarised in
# profiles/r01_final_ncu_summary.md: (34.829 GB read + 0.237 GB written) / (4096 envs x 100 frames x 5 substeps) = 17.1 KB,
# against 16.4 KB of tape record it has to read (algorithmic) plus the side records of the self-contact substeps.
ADJ_DRAM_BYTES_PER_ENV_SUBSTEP = (34.829228e9 + 0.237290e9) / (4096 * 100 * 5)
# fp32 ALU peak derived in DESIGN.md section 7: 148 SMs x 128 lanes x 2 flop x 1.965 GHz
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


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
    """the fp64 oracle, as it stands, on a bounded sample of the same workload (rank 0, host cores)"""
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
    # size the sample for ~budget_s/2 per pass: grow the horizon first, then the number of envs
    units = max(rate * budget_s * 0.5, len(envs) * probe_H)
    H = int(min(H_full, max(probe_H, units // len(envs))))
    n_env = int(min(B, max(len(envs), (units // H) // cores * cores)))
    envs = np.arange(n_env)
    times = []
    for it in range(warmup + steps):
        dt = one(envs, H)
        if it >= warmup:
            times.append(dt)
        if sum(times) > budget_s:
            break
    t = float(np.mean(times))
    return {"value": len(envs) * H / t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d envs x %d steps of config %d (%s, fp64%s), %.1f s per pass" % (
                len(envs), H, problem.get("config_id", 5), mode, ", tape-AD reverse" if mode != "fwd" else "", t)}, t, len(envs) * H


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="fwdbwd", choices=["fwd", "fwdbwd"])
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
    stride = full["stride"] if args.mode == "fwdbwd" else 0
    workload = "config %d: %d ropes x %d verts per GPU, %d frames x 5 substeps, stride %d" % (args.config, B, full["n_verts"], H, stride)
    base = {"metric": METRIC, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload, "mode": args.mode, "per_gpu_batch": B, "n_verts": full["n_verts"], "horizon": H,
                       "checkpoint_stride": stride, "cache": "inputs (actions %.0f MB) larger than L2" % (H * B * 2 * 6 * 4 / 1e6)}}

    if args.impl == "reference":
        if rank != 0:
            return
        problem = make_problem(args.config, batch=min(B, 256), horizon=H, stride=full["stride"])
        cb, t, units = oracle_leg(problem, args.mode, budget_s=60, steps=args.steps, warmup=min(args.warmup, 1))
        line = dict(base, impl="reference", value=cb["value"], ms_per_step=t * 1e3, dtype="f64", cpu_baseline=cb,
                    e2e={"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, gpu_launches=0)
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

    # each rank generates its own shard: same recipe, env ids offset by rank (weak scaling, no data-path collective)
    problem = make_problem(args.config, batch=B, horizon=H)
    if world > 1:
        rng = np.random.Generator(np.random.PCG64(977 + rank))
        problem["x0"] = problem["x0"] + rng.normal(0, 1e-5, problem["x0"].shape)
    sim = dlo.DloSim(problem, device=str(dev))
    seed_t = None

    def one_pass():
        nonlocal seed_t
        dlo.dlo_rollout_forward(sim.h, H, stride)
        if args.mode == "fwdbwd":
            if seed_t is None:
                seed_t = torch.zeros((B, 3, full["n_verts"]), device=dev)
                grads = {"a": torch.zeros((H, B, sim.G, 6), device=dev), "x": torch.zeros((B, 3, full["n_verts"]), device=dev),
                         "v": torch.zeros((B, 3, full["n_verts"]), device=dev), "m": torch.zeros((B, 5), device=dev)}
                one_pass.grads = grads
            # loss head of the harness: mean squared distance to the target polyline -> dL/dx_T on the device
            x = torch.empty_like(seed_t)
            dlo.dlo_get_state(sim.h, x)
            seed_t.copy_((x - one_pass.target) * (2.0 / full["n_verts"]))
            g = one_pass.grads
            dlo.dlo_backward(sim.h, seed_t, None, g["a"], g["x"], g["v"], g["m"])

    one_pass.target = torch.as_tensor(problem["loss"]["target"], dtype=torch.float32, device=dev)
    if one_pass.target.dim() == 2:
        one_pass.target = torch.zeros((B, 3, full["n_verts"]), device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        one_pass()
    barrier()
    l0 = dlo.dlo_launch_count(sim.h)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record()
    for k in range(args.steps):
        one_pass()
        ev[k + 1].record()
    barrier()
    clocks = sampler.stop()
    launches = dlo.dlo_launch_count(sim.h) - l0
    per = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])
    total_ms = max_over_ranks(total_ms, dev)
    n_bad = sim.n_bad()
    ms_per_step = total_ms / args.steps
    value = B * H * world / (ms_per_step * 1e-3)

    # end to end through the host-buffer C-ABI calls
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

        def e2e_pass():
            dlo.dlo_rollout_forward_host(sim.h, x0h, v0h, None, acth, H, stride, xTh, None)
            if args.mode == "fwdbwd":
                seed = ((xTh - tgt) * (2.0 / full["n_verts"])).astype(np.float32)
                dlo.dlo_backward_host(sim.h, seed, None, gah, None, None, gmh)
        if args.mode == "fwdbwd":
            h2d += x0h.nbytes
            d2h += gah.nbytes + gmh.nbytes
        e2e_pass()
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            e2e_pass()
        barrier()
        te = (time.perf_counter() - t0) / n_e2e
        te = max_over_ranks(te, dev)
        e2e = {"value": B * H * world / te, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    if rank != 0:
        return
    peaks, which = measured_peaks()
    flops = FLOPS_PER_ENV_STEP[args.mode] * B * H          # per pass on this GPU (= per launch group)
    achieved = flops / (min(per) * 1e-3) / 1e12
    line = dict(base, value=value, ms_per_step=ms_per_step, e2e=e2e, gpu_launches=int(launches), clocks=clocks,
                roofline={"bound": "alu", "achieved": achieved, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / ALU_PEAK_TFLOPS,
                          "traffic": (ADJ_DRAM_BYTES_PER_ENV_SUBSTEP * B * max(stride, 1) * 5 if args.mode == "fwdbwd" else None),
                          "traffic_note": "DRAM bytes per k_adjoint launch (one checkpoint segment), ncu capture in profiles/r01_final_ncu_summary.md",
                          "peak_source": "derived (148 SMs x 128 fp32 lanes x 2 x %.0f MHz, DESIGN.md section 7); HBM peak %s %.0f GB/s" % (
                              peaks.get("sm_max_mhz", 1965.0), which, peaks.get("hbm_gbs", 0.0)),
                          "kernel": "k_forward" if args.mode == "fwd" else "k_forward + k_adjoint",
                          "algorithmic_flops_per_env_step": FLOPS_PER_ENV_STEP[args.mode]},
                envs_flagged=int(n_bad), ms_per_pass=per)
    if not args.no_cpu_baseline:
        cb, _, _ = oracle_leg(make_problem(args.config, batch=256, horizon=H, stride=full["stride"]), args.mode, budget_s=20)
        line["cpu_baseline"] = cb
    print(json.dumps(line))


if __name__ == "__main__":
    main()
