#!/usr/bin/env python
"""Benchmark of the batched EconoJax environment step (BASELINE.json metric: env agent-steps/s
at N=100 on one B200, and achieved HBM GB/s against peak).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (gather, craft, order placement, matching, expiry,
tax, rewards, observations, government statistics) over one batch of E economies.  The
workload is BASELINE.json's headline: configs[1]'s shape (N=100, R=2, 7 brackets, T=1000,
tax period 100) at north_star's E=4096, seeded synthetic uniform action streams
(DESIGN.md section 4).

  value      agent-steps/s of ej_rollout (persistent kernel), action streams resident in HBM,
             observations/rewards/done written to a ring deeper than L2.
  e2e        the same metric through ej_step_host: per step, actions H2D from pinned host
             memory and observations + rewards + done D2H, inside the timed region.
  roofline   algorithmic bytes (actions in + observations, rewards, done out) per launch of the
             step kernel / its CUDA-event duration, against MEASURED_PEAKS.json's HBM copy rate.
  cpu_baseline  the CPU oracle as it stands on the host cores, on a bounded sample of the workload.

With --impl reference the oracle itself is timed as the reference arm (rank 0 only).
"""
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2410_22165_b200 import inputs, sharding  # noqa: E402

METRIC = "agent_steps_per_sec"
UNIT = "agent-steps/s"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback


def workload_desc(name, cfg, E):
    p = cfg["params"]
    return "%s: E=%d N=%d R=%d prices=%d brackets=%d T=%d tax_period=%d actions=%s skills=%s" % (
        name, E, cfg["N"], cfg["R"], len(p["prices"]), len(p["thresholds"]) + 1, cfg["T"], p["tax_period"],
        cfg["action_mix"], ("uniform01", "pareto4_clip", "normal_clip+growth" if p["skill_growth_rate"] else "normal_clip")[p["skill_init"]])


def algorithmic_bytes_per_env_step(N, B, D_pop, D_gov):
    """Actions in + observations, rewards, done out: int32/fp32."""
    return 4 * N + 4 * B + 4 * N * D_pop + 4 * D_gov + 4 * (N + 1) + 4


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(cfg, n_envs_per_thread, steps, threads, seed):
    """The oracle as it stands: `threads` host threads, each stepping its own shard of envs
    (independent economies; ctypes releases the GIL).  Returns agent-steps/s."""
    import oracle

    N, R = cfg["N"], cfg["R"]
    envs, streams = [], []
    for k in range(threads):
        p = dict(cfg["params"], env_id_base=k * n_envs_per_thread)
        o = oracle.OracleEnv(n_envs_per_thread, N, R, p)
        o.reset(seed)
        envs.append(o)
        streams.append(inputs.action_stream(cfg, steps, seed=seed + k, E=n_envs_per_thread))

    def work(k):
        o, (acts, gov) = envs[k], streams[k]
        for t in range(steps):
            o.step(acts[t], gov[t])

    ths = [threading.Thread(target=work, args=(k,)) for k in range(threads)]
    t0 = time.perf_counter()
    for th in ths:
        th.start()
    for th in ths:
        th.join()
    dt = time.perf_counter() - t0
    return threads * n_envs_per_thread * N * steps / dt, dt


def run_reference(args, cfg, name):
    """Reference arm = the CPU oracle (this tier has no reference implementation to install)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = max(1, min(os.cpu_count() or 1, 32))
    per = 8  # envs per thread and step: a bounded sample of the E-env batch
    t_total = time.perf_counter()
    o_warm, _ = oracle_sample(cfg, per, max(args.warmup, 1), cores, cfg["seed"])
    value, dt = oracle_sample(cfg, per, args.steps, cores, cfg["seed"])
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_desc(name, cfg, cfg["E"]),
                   "note": "reference arm = CPU oracle; each step advances a bounded sample of %d of the %d envs" % (cores * per, cfg["E"])},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d envs x %d steps (%d threads x %d envs)" % (cores * per, args.steps, cores, per)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": time.perf_counter() - t_total,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=40)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="headline")
    ap.add_argument("--ring", type=int, default=16, help="output ring depth (16 x 51 MB > L2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    assert args.warmup >= 1 and args.steps >= 1

    name = args.workload
    cfg = inputs.configs()[name]
    if args.impl == "reference":
        run_reference(args, cfg, name)
        return

    import torch
    import torch.distributed as dist

    from paper_2410_22165_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    E, N, R, T = cfg["E"], cfg["N"], cfg["R"], cfg["T"]
    # envs are independent and keyed by global id: rank r owns global envs [r*E, (r+1)*E) (weak scaling)
    params = dict(cfg["params"], env_id_base=sharding.shard_env_base(rank, world, E))
    env = binding.Env(E, N, R, params, device=str(dev))
    env.set_action_cdf(inputs.action_cdf(cfg))
    use_policy = cfg["action_mix"] == "policy"
    if use_policy:  # configs[4]: actions come from the on-GPU policy MLPs (a12)
        env.set_policy(*inputs.policy_weights(cfg, seed=cfg["seed"]))
    B, K, W = env.B, args.steps, args.warmup
    depth = max(1, min(args.ring, K))
    chunk = min(K, 128)  # action streams are supplied per chunk of <= 128 steps (resident in HBM)
    acts_np, gov_np = inputs.action_stream(cfg, chunk, seed=cfg["seed"] + 1000 * rank)
    acts = torch.from_numpy(acts_np).to(dev)
    gov = torch.from_numpy(gov_np).to(dev)
    obs_ring, rew_ring, done_ring = env.new_obs(depth), env.new_rew(depth), env.new_done(depth)
    bytes_env_step = algorithmic_bytes_per_env_step(N, B, env.D_pop, env.D_gov)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def run_steps(n):
        """n batched steps through ej_rollout, in chunks that stay inside one episode."""
        done_steps = 0
        while done_steps < n:
            t_now = run_steps.t
            if t_now >= T:
                env.reset(cfg["seed"])
                run_steps.t = t_now = 0
            m = min(n - done_steps, chunk, T - t_now)
            env.rollout(m, ring_depth=depth, actions_in=None if use_policy else acts, gov_actions_in=None if use_policy else gov,
                        obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring)
            run_steps.t += m
            done_steps += m

    # Steady state by construction: orders live `order_expiry` steps (30), so the books are still filling
    # during the first steps of an episode.  Whatever --warmup says, every timed repetition starts at an episode
    # step >= 2 * order_expiry and (when K allows) ends inside the same episode.
    t_steady = min(2 * int(cfg["params"]["order_expiry"]), max(0, T - 1))

    def to_steady_state():
        """Every repetition times the SAME episode window [t_steady, t_steady + K): the cost of a step drifts over an
        episode (agents get richer, more bids are valid), so windows at different places are not comparable."""
        if run_steps.t != t_steady:
            if run_steps.t > t_steady:
                env.reset(cfg["seed"])
                run_steps.t = 0
            run_steps(t_steady - run_steps.t)

    env.reset(cfg["seed"])
    run_steps.t = 0
    run_steps(W)
    to_steady_state()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    REPS = 5
    rep_ms, rep_launches, windows = [], [], []
    for rep in range(REPS):
        to_steady_state()
        windows.append("%d..%d" % (run_steps.t, run_steps.t + K))
        l0 = env.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record()
        run_steps(K)
        ev1.record()
        barrier()
        rep_launches.append(env.launch_count() - l0)
        rep_ms.append(sharding.max_over_ranks(ev0.elapsed_time(ev1), dist, dev))
    clocks = sampler.stop()
    order = sorted(range(REPS), key=lambda i: rep_ms[i])
    mid = order[REPS // 2]
    ms, launches = rep_ms[mid], rep_launches[mid]      # the MEDIAN repetition is the reported one
    value = sharding.total_units(E * N * K, world) / (ms * 1e-3)

    # ---- per-launch ej_step path, device-resident inputs (reported beside the rollout) ----
    step_ms = None
    if True:
        obs1, rew1, done1 = env.new_obs(), env.new_rew(), env.new_done()
        ks = min(K, chunk, max(1, T - run_steps.t))
        for t in range(min(3, ks)):
            env.step(acts[t], gov[t], obs1, rew1, done1)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(ks):
            env.step(acts[t], gov[t], obs1, rew1, done1)
        e1.record()
        torch.cuda.synchronize()
        step_ms = e0.elapsed_time(e1) / ks
        run_steps.t += ks + min(3, ks)

    # ---- a12 alone (policy workloads): the tcgen05 policy kernel against the tensor roofline ----
    policy_kernel = None
    if use_policy:
        obs_p = env.observe()
        a_p = torch.zeros((E, N), dtype=torch.int32, device=dev)
        g_p = torch.zeros((E, B), dtype=torch.int32, device=dev)
        for _ in range(5):
            env.policy_act(obs_p, a_p, g_p)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps_p = 50
        e0.record()
        for _ in range(reps_p):
            env.policy_act(obs_p, a_p, g_p)
        e1.record()
        torch.cuda.synchronize()
        p_ms = e0.elapsed_time(e1) / reps_p
        L = len(cfg["params"]["rate_table"])
        flop = 2.0 * E * N * (env.D_pop * 128 + 128 * 128 + 128 * env.A) + 2.0 * E * (env.D_gov * 128 + 128 * 128 + 128 * B * L)
        try:
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                tpeak, tsrc = float(json.load(f)["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
        except Exception:
            tpeak, tsrc = 1590.0, "fallback (B200_PROFILING.md)"
        policy_kernel = {"kernel": "ej_policy_kernel (ej_policy_act, one launch, same obs every call: inputs L2-resident)", "bound": "tensor",
                         "us_per_launch": 1e3 * p_ms, "flop_per_launch": flop, "achieved": flop / (p_ms * 1e-3) / 1e12, "peak": tpeak,
                         "unit": "TFLOP/s", "frac": flop / (p_ms * 1e-3) / 1e12 / tpeak, "peak_source": tsrc}
        del obs_p, a_p, g_p

    # ---- f2: the same rollout with factored observations (private block + env-wide block), reported beside it ----
    fx = None
    if not use_policy and (N * (3 * R + 4)) % 4 == 0 and N * env.D_pop * 4 <= 64 * 1024:
        priv, shared, govr = env.new_factored_obs(depth)
        env.reset(cfg["seed"])
        kf = min(K, chunk)
        for _ in range(2):
            env.rollout(min(W, chunk), ring_depth=depth, actions_in=acts, gov_actions_in=gov, rew_ring=rew_ring, done_ring=done_ring,
                        obs_priv_ring=priv, obs_shared_ring=shared, obs_gov_ring=govr)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        env.rollout(kf, ring_depth=depth, actions_in=acts, gov_actions_in=gov, rew_ring=rew_ring, done_ring=done_ring,
                    obs_priv_ring=priv, obs_shared_ring=shared, obs_gov_ring=govr)
        e1.record()
        torch.cuda.synchronize()
        f_ms = e0.elapsed_time(e1) / kf
        fx_bytes = 4 * N + 4 * B + 4 * N * env.D_priv + 4 * env.D_shared + 4 * env.D_gov + 4 * (N + 1) + 4
        fx = {"api": "ej_rollout with obs_priv_ring / obs_shared_ring (SURVEY 8(f) f2)", "ms_per_step": f_ms,
              "value": E * N / (f_ms * 1e-3), "unit": UNIT, "bytes_per_env_step": fx_bytes, "steps": kf}
        del priv, shared, govr

    # ---- e2e: ej_step_host, pinned host buffers, H2D + D2H inside the timed region ----
    e2e = None
    if not args.no_e2e:
        Ke = min(K, chunk)
        h_acts = torch.from_numpy(acts_np[:Ke]).pin_memory()
        h_gov = torch.from_numpy(gov_np[:Ke]).pin_memory()
        h_obs = torch.zeros(env.obs_floats, dtype=torch.float32).pin_memory()
        h_rew = torch.zeros((E, N + 1), dtype=torch.float32).pin_memory()
        h_done = torch.zeros(E, dtype=torch.uint8).pin_memory()
        env.reset(cfg["seed"])
        lib = binding
        for t in range(3):
            lib.ej_step_host(env.h, h_acts[t].data_ptr(), h_gov[t].data_ptr(), h_obs.data_ptr(), h_rew.data_ptr(), h_done.data_ptr())
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(Ke):
            lib.ej_step_host(env.h, h_acts[t].data_ptr(), h_gov[t].data_ptr(), h_obs.data_ptr(), h_rew.data_ptr(), h_done.data_ptr())
        e1.record()
        barrier()
        e_ms = e0.elapsed_time(e1)
        e_ms = sharding.max_over_ranks(e_ms, dist, dev)
        e2e = {"value": world * E * N * Ke / (e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(4 * E * N + 4 * E * B),
               "d2h_bytes_per_step": int(4 * env.obs_floats + 4 * E * (N + 1) + E),
               "steps": Ke, "ms_per_step": e_ms / Ke, "api": "ej_step_host (pinned host buffers)"}

        # the same through ej_step_host_factored (f2): every observation value once, env-wide columns once per env
        if fx is not None:
            dpv, dsh = env.D_priv, env.D_shared_pad
            h_priv = torch.zeros((E, N, dpv), dtype=torch.float32).pin_memory()
            h_shared = torch.zeros((E, dsh), dtype=torch.float32).pin_memory()
            h_govr = torch.zeros((E, env.D_gov_pad), dtype=torch.float32).pin_memory()
            env.reset(cfg["seed"])
            step_fx = lambda t: lib.ej_step_host_factored(env.h, h_acts[t].data_ptr(), h_gov[t].data_ptr(), h_priv.data_ptr(),
                                                          h_shared.data_ptr(), h_govr.data_ptr(), h_rew.data_ptr(), h_done.data_ptr())
            for t in range(3):
                step_fx(t)
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for t in range(Ke):
                step_fx(t)
            e1.record()
            barrier()
            f_ms = sharding.max_over_ranks(e0.elapsed_time(e1), dist, dev)
            e2e["factored"] = {"value": world * E * N * Ke / (f_ms * 1e-3), "unit": UNIT, "ms_per_step": f_ms / Ke,
                               "h2d_bytes_per_step": int(4 * E * N + 4 * E * B),
                               "d2h_bytes_per_step": int(4 * E * (N * dpv + dsh + env.D_gov_pad) + 4 * E * (N + 1) + E),
                               "api": "ej_step_host_factored (pinned host buffers; same observation values, env-wide columns once per env)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    achieved = bytes_env_step * E * K / (ms * 1e-3) / 1e9  # GB/s per GPU (every rank runs the same work)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_desc(name, cfg, E), "E_per_gpu": E, "api": "ej_rollout (policy kernels + step kernel per step)" if use_policy else "ej_rollout (persistent kernel)",
                   "episode_steps": windows[mid],
                   "timing": "median of %d repetitions of K = %d steps, each bracketed by barrier + synchronize, every repetition over the same episode window starting at step %d (2 x order expiry: books in steady state)" % (REPS, K, t_steady),
                   "l2": "outputs go to a ring of %d steps x %.1f MB (> 126 MB L2); action streams %d steps x %.1f MB" % (
                       depth, bytes_env_step * E / 1e6, chunk, 4e-6 * E * (N + B))},
        "env_steps_per_sec": world * E * K / (ms * 1e-3),
        "repetitions": {"ms_per_step": [m / K for m in rep_ms], "episode_steps": windows, "best_ms_per_step": min(rep_ms) / K,
                        "median_ms_per_step": ms / K, "best_value": sharding.total_units(E * N * K, world) / (min(rep_ms) * 1e-3)},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "kernel": "ej_step_kernel", "peak_source": peak_src,
                     "bytes_per_env_step": bytes_env_step, "launches": launches,
                     "frac_of_nominal_8000": achieved / 8000.0},
        "e2e": e2e,
        "gpu_launches": int(launches),
        "per_launch_step": {"api": "ej_step (one launch per step, state in HBM between launches)",
                            "ms_per_step": step_ms, "value": E * N / (step_ms * 1e-3), "unit": UNIT},
        "clocks": clocks,
    }
    if fx:
        line["factored_obs"] = fx
    if policy_kernel:
        line["policy_kernel"] = policy_kernel
    traffic_path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_path):
        try:
            with open(traffic_path) as f:
                tr = json.load(f).get(name)
            if tr:  # ncu-measured DRAM bytes per env-step x env-steps per launch (per launch, like `achieved`)
                line["roofline"]["traffic"] = tr["bytes_per_env_step"] * E * K / max(1, launches)
                line["roofline"]["traffic_source"] = tr["source"]
        except Exception:
            pass
    if world == 1 and not args.no_cpu_baseline:
        cores = max(1, min(os.cpu_count() or 1, 32))
        per, osteps = 160, min(1000, T)
        # ~10-30 s of CPU work: (cores x 160 envs + 160 envs on one core) x 1000 steps, after a short warm-up
        oracle_sample(cfg, per, 5, cores, cfg["seed"])
        v, dt = oracle_sample(cfg, per, osteps, cores, cfg["seed"])
        v1, dt1 = oracle_sample(cfg, per, osteps, 1, cfg["seed"])
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "%d envs x %d steps of the same workload (%d threads x %d envs), %.1f s" % (
                                    cores * per, osteps, cores, per, dt),
                                "value_1core": v1}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
