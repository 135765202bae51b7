#!/usr/bin/env python
"""bench.py -- reaction firings/s of the random-time hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: one trajectory of
the workload's network run for its configured number of firings (cfg4: M=1e6, 1e4 firings) by ONE
launch of the persistent bundle kernel (a-0 init + every a-1..a-8 of every firing).  `value` is
timed with CUDA events on the launching stream through rt_run_dev (x0 resident in HBM); `e2e` is
the host-pointer rt_run (x0 H2D, x_out + result + trace D2H inside the timed region).
N > 1: the single large-M trajectory does not shard ("replicas only"), so every rank
runs an independent replica (trajectory id = rank), no collective on the data path.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import rt_workloads as W

METRIC = "reaction firings/sec on 1 B200 at M=10^6 (+ % of HBM roofline per firing)"
UNIT = "firings/s"
BYTES_PER_REACTION_FIRING = 32   # read T, P, a; write T
# Counters that a timed run cannot measure (DRAM bytes, shared-memory wavefronts, thread instructions)
# come from the committed ncu captures of THIS command line, one row per workload:
# profiles/r2_ncu_counters.csv (commands and commit in profiles/r2_ncu_counters.md).
NCU_COUNTERS_CSV = os.path.join(ROOT, "profiles", "r2_ncu_counters.csv")


def ncu_counters(workload):
    """Row of profiles/r2_ncu_counters.csv for `workload` (dict of str), or None."""
    import csv
    try:
        with open(NCU_COUNTERS_CSV, newline="") as f:
            for row in csv.DictReader(f):
                if row.get("workload") == workload:
                    return row
    except OSError:
        pass
    return None


# the other BASELINE.json configs, reported in the same JSON line under "secondary"
SECONDARY = ["cfg5a", "cfg5b", "cfg3", "cfg2"]
SECONDARY_STEPS = 2
# issue peak: 148 SMs x 4 schedulers x 32 lanes x 1.965 GHz (B200_PROFILING.md unit counts / clocks)
ALU_PEAK_GINSTR = 148 * 4 * 32 * 1.965


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5a", "cfg5b"])
    ap.add_argument("--firings", type=int, default=0, help="firings per step (0 = the config's)")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink N, M (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", dest="secondary", action="store_false",
                    help="skip the secondary workloads (cfg5a, cfg5b, cfg3, cfg2)")
    ap.add_argument("--option", action="append", default=[], help="name=value for rt_set_option")
    ap.add_argument("--breakpoints", type=int, default=0,
                    help="time-dependent rates (Eq.28): this many rate breakpoints spread over the step")
    return ap.parse_args()


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names)
                   if any(len(r) >= 6 and r[2 + i].lower() == "active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


def oracle_leg(net, x0, seed, traj, firings):
    """The oracle as it stands, single thread, timed on the host (wall clock around oracle_run,
    which includes its own init just as a GPU step includes a-0)."""
    import oracle
    t0 = time.perf_counter()
    o = oracle.run(net, x0, seed, traj, firings, math.inf, 0, want_state=False)
    dt = time.perf_counter() - t0
    return o["firings"] / dt, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    net, x0, par = W.make_config(args.workload, scale=args.scale)
    M = int(net["n_reactions"])
    # bounded sample: about 2e8 reaction-steps (~2-4 s) per step
    sample = max(20, min(par["max_firings"], int(2e8 // M)))
    for _ in range(min(args.warmup, 1)):
        oracle_leg(net, x0, par["seed"], 0, sample)
    times, fired = [], 0
    for _ in range(args.steps):
        v, dt = oracle_leg(net, x0, par["seed"], 0, sample)
        times.append(dt)
        fired += sample
    value = fired / sum(times)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": args.workload, "n_species": int(net["n_species"]),
                   "n_reactions": M, "firings_per_step": sample,
                   "note": "CPU oracle (oracle/rt_oracle.cpp, 1 thread); each step is a bounded "
                           f"sample: the first {sample} firings of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"first {sample} firings of {args.workload} x {args.steps} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def smem_roofline(M, kernel_s_per_firing, sm_mhz, num_sms, bytes_per_reaction):
    """The binding on-chip resource when (T, P, a) live in shared memory: aggregate shared-memory
    bandwidth = SMs x 128 B/clk x SM clock (B200_PROFILING.md unit counts)."""
    peak = num_sms * 128.0 * sm_mhz * 1e6 / 1e9                    # GB/s
    ach = bytes_per_reaction * M / kernel_s_per_firing / 1e9
    return {"smem_achieved": ach, "smem_peak": peak, "smem_frac": ach / peak,
            "smem_peak_source": f"{num_sms} SMs x 128 B/clk x {sm_mhz:.0f} MHz"}


def measure(rt, torch, dist, args, workload, steps, warmup, rank, world, local, headline):
    """K device-timed steps of one workload (CUDA events on the launching stream, L2 flushed
    between steps, clocks sampled during the timed region).  Returns the fields of a bench line."""
    dev = torch.device("cuda", local)
    scale = args.scale
    net, x0, par = W.make_config(workload, scale=scale)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    firings = (args.firings if headline else 0) or par["max_firings"]
    n_all = par["n_traj"]
    t_end = float(par.get("t_end", math.inf)) if workload in ("cfg1", "cfg2") else math.inf
    seed = par["seed"]
    if n_all > 1 and world > 1:
        # ensembles shard by trajectory id with no data-path collective: strong scaling
        first, n_traj = rt.shard_range(n_all, rank, world)
        traj0, scaling = first, "strong"
    else:
        n_traj, traj0, scaling = n_all, rank * n_all, "weak"      # replicas: own trajectory ids
    model = rt.Model(net, local)
    formulation = 0
    if headline:
        for kv in args.option:
            k, v = kv.split("=")
            model.set_option(k, int(v))
            if k == "formulation":
                formulation = int(v)

    x0_dev = torch.from_numpy(x0).to(dev)
    x_out_dev = torch.empty(max(n_traj, 1) * N, dtype=torch.int64, device=dev)
    res_dev = torch.zeros(max(n_traj, 1) * 3, dtype=torch.int64, device=dev)   # rt_result[n_traj]
    trace_cap = min(firings, par.get("trace", 0)) if n_all == 1 else 0
    tmu_dev = torch.empty(max(trace_cap, 1), dtype=torch.int32, device=dev)
    tt_dev = torch.empty(max(trace_cap, 1), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)              # > 126 MB L2

    def step_dev():
        if n_traj == 0:
            return
        if n_all == 1:
            rc = rt.rt_run_dev(model.handle, x0_dev, seed, traj0, firings, t_end, x_out_dev,
                               res_dev, tmu_dev, tt_dev, trace_cap)
        else:
            rc = rt.rt_ensemble_dev(model.handle, x0_dev, seed, traj0, n_traj, firings, t_end,
                                    x_out_dev, res_dev)
        if rc != rt.RT_OK:
            raise rt.RtError(rc, "rt_run_dev")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    breakpoints = args.breakpoints if headline else 0
    if breakpoints > 0:
        # learn how long (in simulated time) a step is, then spread the breakpoints over it:
        # factors alternate 1.5 / 0.5 on the even-numbered reactions
        step_dev()
        torch.cuda.synchronize()
        t_final = float(res_dev.cpu().numpy().view(rt.RESULT_DTYPE)["t"].max())
        tb = [t_final * (i + 1) / (breakpoints + 2) for i in range(breakpoints)]
        fa = [1.5 if i % 2 == 0 else 0.5 for i in range(breakpoints)]
        model.set_rate_schedule(tb, fa, (np.arange(M) % 2 == 0).astype(np.uint8))
    for _ in range(max(warmup, 3)):
        flush.fill_(1)
        step_dev()
    torch.cuda.synchronize()
    if rt.rt_sync(model.handle) != rt.RT_OK:
        raise SystemExit("bench.py: device reported an error during warm-up")
    done = res_dev.cpu().numpy().view(rt.RESULT_DTYPE)[:n_traj]
    assert (done["status"] == 0).all(), done
    if math.isinf(t_end):
        assert (done["firings"] == firings).all(), done
    elif n_traj:
        # (a Lotka-Volterra trajectory may also die out -> absorbed, or explode -> max_firings)
        assert (done["stop"] >= rt.RT_STOP_T_END).all() and (done["stop"] == rt.RT_STOP_T_END).mean() > 0.9, done
    fired_local = int(done["firings"].sum())         # trajectory-steps of one step on this rank
    fired_t = torch.tensor([fired_local], dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(fired_t)
    fired_per_step = int(fired_t.item())             # ... on all ranks

    # ---- timed region: K steps, device-timed; per-step events bracket the kernel launch only
    # (L2 flush sits between steps, outside the per-step events but inside the barrier bracket).
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(steps)]
    launches0 = model.info("kernel_launches")
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    for a, b in ev:
        flush.fill_(1)
        a.record()
        step_dev()
        b.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = model.info("kernel_launches") - launches0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_s = float(total_ms.item()) * 1e-3
    value = fired_per_step * steps / total_s

    out = {"workload": workload, "value": value, "ms_per_step": 1e3 * total_s / steps,
           "scaling": scaling, "gpu_launches": int(launches), "clocks": clocks}
    if headline:
        # ---- e2e: the host-pointer C-ABI call a user makes; copies inside the timed region
        x0_pin = torch.from_numpy(x0.copy()).pin_memory().numpy()

        def step_host():
            if n_traj == 0:
                return 0
            if n_all == 1:
                return model.run(x0_pin, seed, traj0, firings, t_end, trace_cap=trace_cap)["firings"]
            return int(model.ensemble(x0_pin, seed, traj0, n_traj, firings, t_end)["firings"].sum())

        step_host()
        barrier()
        t0 = time.perf_counter()
        got = 0
        for _ in range(steps):
            got += step_host()
        torch.cuda.synchronize()
        e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        got_t = torch.tensor([got], dtype=torch.int64, device=dev)
        if world > 1:
            dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
            dist.all_reduce(got_t)
        out["e2e"] = {"value": int(got_t.item()) / float(e2e_s.item()), "unit": UNIT,
                      "h2d_bytes_per_step": N * 8,
                      "d2h_bytes_per_step": n_traj * N * 8 + n_traj * 24 + trace_cap * 12}

    if rank == 0:
        peak, peak_src = peaks()
        kernel_s = (sum(step_ms) / len(step_ms)) * 1e-3          # one kernel launch per step (this rank)
        smem = bool(model.info("state_in_smem"))
        bundles = max(1, model.info("bundles"))
        us_per_firing = 1e6 * kernel_s / max(fired_local, 1) * max(n_traj, 1)
        out["config"] = {
            "workload": workload, "n_species": N, "n_reactions": M,
            "trajectories_per_step": n_all, "firings_per_step": fired_per_step,
            "parallelism": ("replicas only (one trajectory per GPU)" if n_all == 1 else
                            "independent trajectories" + (", sharded by trajectory id" if world > 1 else "")),
            "l2": "flushed between steps (256 MB fill)",
            "bundle_ctas": model.info("bundle_ctas"), "bundles": model.info("bundles"),
            "block_threads": model.info("block_threads"), "state_in_shared_memory": smem,
            "exchange": ("thread-block cluster (DSMEM)" if model.info("cluster_exchange") else
                         "L2 slots" if model.info("bundle_ctas") > 1 else "none"),
            "us_per_firing": us_per_firing, "ensemble_path": model.info("ensemble_path"),
            "formulation": "residual (Table 3)" if formulation else "(T, P) internal time",
            "rate_breakpoints": breakpoints}
        ctr = ncu_counters(workload)
        src = ("profiles/r2_ncu_counters.csv (ncu --set full, one launch of this command at commit "
               + ctr["commit"] + ")") if ctr else None
        if model.info("ensemble_path") == 1:
            # one thread per trajectory, state in shared memory: plain ALU issue is the bound
            ips = float(ctr["thread_inst_executed"]) / float(ctr["steps_per_launch"]) if ctr else None
            ginstr = ips * fired_local / kernel_s / 1e9 if ips else None
            out["roofline"] = {"bound": "alu", "achieved": ginstr, "peak": ALU_PEAK_GINSTR,
                               "unit": "Ginstr/s", "frac": ginstr / ALU_PEAK_GINSTR if ginstr else None,
                               "traffic": None, "kernel": "rt_tiny_kernel" if model.info("tiny_kernel") else "rt_thread_kernel",
                               "peak_source": "148 SMs x 4 schedulers x 32 lanes x 1.965 GHz (DESIGN.md 7)",
                               "thread_instructions_per_step": ips, "thread_instructions_source": src}
        else:
            # residual (Table 3) form: T and a read, T written -- no P: 24 bytes per reaction
            bpr = 24 if formulation else BYTES_PER_REACTION_FIRING
            alg_bytes = bpr * M * fired_local
            achieved = alg_bytes / kernel_s / 1e9
            traffic = None
            if ctr and int(ctr["steps_per_launch"]) > 0 and not (not smem and model.info("l2_persist")):
                # (with the persisting-L2 window no capture exists: under ncu's replay the window has no
                #  effect -- profiles/r2_bundle_kernel_cfg5a.md -- so `traffic` stays null there)
                # DRAM bytes of the captured launch, scaled if this run fires a different number
                traffic = (float(ctr["dram_bytes_read"]) + float(ctr["dram_bytes_write"])) * \
                          fired_local / float(ctr["steps_per_launch"])
            kernel = "rt_fast_kernel" if model.info("pipeline") else "rt_bundle_kernel"
            roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": traffic, "traffic_source": src,
                    "kernel": kernel, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg_bytes,
                    "frac_of_8TBs_nominal": achieved / 8000.0}
            if smem:
                sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
                # all bundles stream side by side: per-firing time of the chip = kernel_s / firings of
                # one bundle's queue; aggregate bytes per second is what the shared memories deliver
                roof.update(smem_roofline(M, kernel_s / max(fired_local, 1), sm_mhz,
                                          model.info("num_sms"), bpr))
                if ctr and ctr.get("smem_wavefronts"):
                    # measured shared-memory traffic: wavefronts x 128 B of the captured launch
                    smem_bytes = float(ctr["smem_wavefronts"]) * 128.0 / float(ctr["steps_per_launch"])
                    roof["smem_bytes_per_firing_measured"] = smem_bytes
                    roof["smem_bytes_per_firing_algorithmic"] = bpr * M
                roof["bound_actual"] = "latency (per-firing dependency chain) + shared-memory bandwidth"
                roof["note"] = ("state (T,P,a) resident in shared memory: `achieved` is ALGORITHMIC bytes per "
                                "second (north_star's definition), not DRAM throughput (see `traffic`); a "
                                "fraction above 1 only says the state never leaves the chip.  What binds is "
                                "the per-firing latency chain (exchange + refresh) and shared-memory "
                                "bandwidth: `smem_frac` (DESIGN.md 7)")
            else:
                persist = model.info("l2_persist")
                roof["note"] = ("state streamed from global memory; T (read and written every firing, half of "
                                "the algorithmic bytes) is kept as persisting lines in the 126 MB L2, so DRAM "
                                "traffic is BELOW the algorithmic bytes (`traffic`) and `frac` can exceed 1; "
                                "`hbm_streaming_only` is the same kernel with plain streaming"
                                if persist else
                                "state streamed from global memory: DRAM traffic = algorithmic bytes")
                if persist and not headline and world == 1:
                    # the plain-streaming figure (every byte from HBM every firing): the honest HBM roofline
                    model.set_option("l2_persist", 0)
                    flush.fill_(1); step_dev(); torch.cuda.synchronize()
                    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                           for _ in range(steps)]
                    for a, b in ev2:
                        flush.fill_(1)
                        a.record()
                        step_dev()
                        b.record()
                    torch.cuda.synchronize()
                    model.set_option("l2_persist", 1)
                    k2 = sum(a.elapsed_time(b) for a, b in ev2) / len(ev2) * 1e-3
                    ctr2 = ncu_counters(workload + "_stream")
                    roof["hbm_streaming_only"] = {
                        "value": fired_local / k2, "us_per_firing": 1e6 * k2 / max(fired_local, 1),
                        "achieved": alg_bytes / k2 / 1e9, "frac": alg_bytes / k2 / 1e9 / peak,
                        "traffic": ((float(ctr2["dram_bytes_read"]) + float(ctr2["dram_bytes_write"])) *
                                    fired_local / float(ctr2["steps_per_launch"])) if ctr2 else None}
            out["roofline"] = roof
        out["_cpu"] = (net, x0, seed, traj0, firings, t_end, n_traj, fired_local, M)
    model.close()
    del flush, x0_dev, x_out_dev, res_dev
    torch.cuda.empty_cache()
    return out


def cpu_baseline(workload, net, x0, seed, traj0, firings, t_end, n_traj, fired_local, M):
    """The oracle as it stands on the box's host cores, on a bounded sample (~1e9 reaction-steps)."""
    if n_traj == 1:
        sample = max(20, min(firings, int(1e9 // M)))    # ~1e9 reaction-steps: 10-30 s
        v, dt = oracle_leg(net, x0, seed, traj0, sample)
        return {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": f"first {sample} firings of {workload} (M={M}), {dt:.1f} s, single thread"}
    # ensembles: one independent oracle instance per host core on a subset of the trajectories,
    # sized for ~1e9 reaction-steps in total
    import oracle
    cores = os.cpu_count() or 1
    per_traj = max(1, fired_local // n_traj) * M
    sub = int(max(cores, min(n_traj, 1e9 // per_traj)))
    t0 = time.perf_counter()
    o = oracle.ensemble(net, x0, seed, traj0, sub, firings, t_end, n_threads=cores)
    dt = time.perf_counter() - t0
    return {"value": float(o["firings"].sum()) / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"trajectories {traj0}..{traj0 + sub - 1} of {workload} in full, {dt:.1f} s, "
                      "one oracle instance per core"}


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2103_00405_b200 as rt

    rt.lib()                                   # no extension -> ImportError; there is no fallback
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    head = measure(rt, torch, dist, args, args.workload, args.steps, args.warmup, rank, world, local, True)
    secondary = {}
    if args.secondary and world == 1 and args.scale == 1.0:
        # the other configs of BASELINE.json, each timed exactly like the headline (fewer steps)
        for wl in SECONDARY:
            if wl == args.workload:
                continue
            s = measure(rt, torch, dist, args, wl, SECONDARY_STEPS, 3, rank, world, local, False)
            s.pop("_cpu", None)
            s["unit"] = UNIT if s["config"]["trajectories_per_step"] == 1 else "trajectory-steps/s"
            s["steps"] = SECONDARY_STEPS
            secondary[wl] = s

    if rank == 0:
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": head["ms_per_step"],
            "higher_is_better": True, "scaling": head["scaling"], "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": head["config"], "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "clocks": head["clocks"], "roofline": head["roofline"],
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(args.workload, *head["_cpu"])
        if secondary:
            line["secondary"] = secondary
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_cuda(a)
