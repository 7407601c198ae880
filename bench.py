#!/usr/bin/env python
"""bench.py -- neutrons traced per second on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (RNG -> source -> slits -> sample -> Q -> I(Q) with the
quadrature loops -> detector histogram) over one batch of n_neutrons synthetic neutrons of the
headline workload, BASELINE.json configs[1] (polydisperse sphere + Percus-Yevick S(q), fp32 model,
1e8 neutrons, 256x256 detector).  `value` is timed with the descriptors and tables resident on the
device; `e2e` goes through the C ABI with host buffers every step (sas_set_model: H2D of parameters
and tables; sas_read_detector: D2H of the three histograms).  The other four configs are timed with
a short loop and reported under "configs".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 is launched by torch.distributed.run, one rank per GPU; rank r traces the id range
[r n, (r+1) n) (weak scaling) and the detectors are merged onto rank 0 by one reduction per step.
--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import sas_workloads as W  # noqa: E402

METRIC = "neutrons traced/sec on 1 B200 (SANS + SAS sample)"
UNIT = "neutrons/s"
HEADLINE = 1                      # BASELINE.json configs[1]


# ------------------------------------------------------------------ reference arm: the CPU oracle
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle as O
    c = W.config(HEADLINE)
    ins, mod = O.make_instrument(c["instrument"]), O.make_model(c["model"])
    sample = 1_000_000            # ids per step: a bounded prefix-like sample of the 1e8-neutron workload
    for w in range(args.warmup):
        O.trace_range(ins, mod, c["seed"], w * sample, sample, dump=False)
    t0 = time.perf_counter()
    for s in range(args.steps):
        O.trace_range(ins, mod, c["seed"], (args.warmup + s) * sample, sample, dump=False)
    dt = time.perf_counter() - t0
    value = sample * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": c["name"], "n_neutrons_per_step": sample,
                   "note": "CPU oracle, single thread, ids [0, steps*1e6) of the 1e8-neutron workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps} x {sample} neutron ids of {c['name']}"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------ clock sampling (NVML)
class ClockSampler(threading.Thread):
    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                break
            time.sleep(0.002)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------ helpers
def model_key_and_nodes(model):
    from paper_2501_06054_b200 import roofline as R  # noqa: F401
    m, prec = model["model"], model["precision"]
    pd = [n if k == "schulz" else 1 for k, n in zip(model["pd_kind"], model["pd_nodes"])]
    if is_event_model(model) and m == "cylinder":
        return "cylinder_event_fp64", 1
    if is_event_model(model) and m == "barbell":
        return "barbell_event_fp64", 64
    if m == "sphere":
        nodes = pd[0]
        eff = prec if nodes > 1 else "fp64"
        key = ("sphere_py_" if model["sq_kind"] != "none" else "sphere_") + eff
        return key, nodes
    if m == "cylinder" and model["orient_kind"] == "gauss_quad":
        return "cylinder_quad_fp32", model["n_theta"] * model["n_phi"] * (pd[0] + pd[1]) // 2
    if m == "core_shell_triaxial":
        return "cs_triaxial_iso_fp32", pd[0] * pd[1]
    if m == "cylinder":
        return "cylinder_iso_fp64", 1
    raise KeyError(m)


def is_event_model(model):
    return "gauss_mc" in model["pd_kind"]


def time_steps(torch, tracer, do_step, steps, warmup, flush):
    """Device time of `steps` steps: one CUDA-event pair per step on the tracer's stream, L2 flushed
    between steps outside the pairs; barrier + synchronize on both sides."""
    import torch.distributed as dist
    for i in range(warmup):
        do_step(i)
    torch.cuda.synchronize()
    if dist.is_initialized():
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    tracer.kernel_time_ms(reset=True)
    l0 = tracer.launch_info()["n_launches"]
    for i in range(steps):
        flush()
        ev[i][0].record()
        do_step(warmup + i)
        ev[i][1].record()
    torch.cuda.synchronize()
    if dist.is_initialized():
        dist.barrier()
    torch.cuda.synchronize()
    per_step = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(per_step)
    time_steps.last_per_step = per_step
    if dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    return total_ms, tracer.launch_info()["n_launches"] - l0


def bench_config(torch, S, cfg_index, steps, warmup, rank, world, flush, with_e2e):
    from paper_2501_06054_b200 import roofline as R
    from paper_2501_06054_b200.sharding import weak_shard, merge_detectors
    c = W.config(cfg_index)
    batch = "models" in c
    if batch:
        tr = S.BatchTracer(c["instruments"], c["models"])
        n_step = c["n_neutrons_each"] * len(c["models"])
        n_arg = c["n_neutrons_each"]
    else:
        tr = S.Tracer(c["instrument"], c["model"])
        n_step = n_arg = c["n_neutrons"]
    seed = c["seed"]
    first, _ = weak_shard(n_arg, rank)

    def do_step(i):
        tr.reset()
        if batch:
            tr.trace(n_arg, seed + rank)           # ranks use distinct streams of the same experiments
        else:
            tr.trace_range(first, n_arg, seed)
        if world > 1:
            merge_detectors([tr.sum_p, tr.sum_p2, tr.counts], dst=0)

    total_ms, launches = time_steps(torch, tr, do_step, steps, warmup, flush)
    kernel_ms, n_timed = tr.kernel_time_ms(reset=True)   # average per launch; a step may take several
    launches_per_step = max(1, int(n_timed) // steps)    # launches (one per kernel variant in a batch)
    kernel_ms *= launches_per_step                        # trace-kernel time per step
    info = tr.launch_info()
    cnt = tr.counters().astype(np.float64)
    ms_per_step = total_ms / steps
    value = n_step * world / (ms_per_step * 1e-3)
    per = sorted(getattr(time_steps, "last_per_step", [ms_per_step]))
    out = {"workload": c["name"], "n_neutrons_per_step": n_step, "ms_per_step": ms_per_step, "value": value,
           "ms_per_step_median": per[len(per) // 2], "ms_per_step_best": per[0],
           "kernel_ms": kernel_ms, "grid": info["grid"], "block": info["block"], "smem_bytes": info["smem_bytes"],
           "gpu_launches": int(launches), "detected_frac": cnt[6] / cnt[0], "survive_frac": 1.0 - cnt[1] / cnt[0],
           # survivors whose fp64 geometry ran (the others were certain detector misses, counters[7])
           "geometry_frac": 1.0 - cnt[1] / cnt[0] - cnt[7] / cnt[0]}
    # roofline of the (only) kernel of the step, from its own average launch duration
    if batch:
        ks = {}
        for m in c["models"]:
            k, n = model_key_and_nodes(m)
            ks[k] = n
        # mixed batch: weigh the per-detected cost of the two model families equally (half each)
        rl = None
        for k, n in ks.items():
            r = R.roofline(n_step / (kernel_ms * 1e-3), out["survive_frac"], out["detected_frac"], k, n,
                           workload=c["name"], frac_geometry=out["geometry_frac"])
            rl = r if rl is None else {**rl, "achieved": 0.5 * (rl["achieved"] + r["achieved"]),
                                       "frac": 0.5 * (rl["frac"] + r["frac"])}
        out["roofline"] = rl
    else:
        k, n = model_key_and_nodes(c["model"])
        out["roofline"] = R.roofline(n_step / (kernel_ms * 1e-3), out["survive_frac"], out["detected_frac"], k, n,
                                     workload=c["name"], frac_geometry=out["geometry_frac"])
    e2e = None
    if with_e2e and not batch:
        # the call a user makes, host buffers in and out, every step
        def e2e_step(i):
            tr.set_model(c["model"])                # H2D: parameters + quadrature tables
            tr.reset()
            tr.trace_range(first, n_arg, seed)
            return tr.read_detector()               # D2H: three histograms into host arrays

        for i in range(2):
            e2e_step(i)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(steps):
            sp, sp2, cn = e2e_step(i)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            import torch.distributed as dist
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        npix = sp.size
        e2e = {"value": n_step * world * steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(tr.upload_bytes()), "d2h_bytes_per_step": int(3 * 8 * npix)}
    tr.close()
    return out, e2e


def cpu_baseline(cfg_index, budget_s=12.0):
    from oracle import oracle as O
    c = W.config(cfg_index)
    ins, mod = O.make_instrument(c["instrument"]), O.make_model(c["model"])
    O.trace_range(ins, mod, c["seed"], 0, 100000, dump=False)
    t0 = time.perf_counter()
    O.trace_range(ins, mod, c["seed"], 0, 1_000_000, dump=False)
    rate = 1e6 / (time.perf_counter() - t0)
    n = int(min(max(rate * budget_s, 1e6), 1e8))
    t0 = time.perf_counter()
    O.trace_range(ins, mod, c["seed"], 0, n, dump=False)
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"ids [0, {n}) of {c['name']} ({dt:.1f} s, single thread)"}


def _oracle_worker(job):
    cfg_index, first, n = job
    from oracle import oracle as O
    c = W.config(cfg_index)
    O.trace_range(c["instrument"], c["model"], c["seed"], first, n, dump=False)
    return n


def cpu_baseline_all_cores(cfg_index, rate_1core, seconds=3.0):
    """The same oracle as K independent id-range processes (the paper's MPI scheme):
    K = the cores this process may run on."""
    import multiprocessing as mp
    k = len(os.sched_getaffinity(0))
    n = int(max(rate_1core * seconds, 2e5))
    with mp.get_context("spawn").Pool(k) as pool:
        pool.map(_oracle_worker, [(cfg_index, 0, 1000)] * k)          # start the workers, load the library
        t0 = time.perf_counter()
        pool.map(_oracle_worker, [(cfg_index, r * n, n) for r in range(k)])
        dt = time.perf_counter() - t0
    return {"value": k * n / dt, "cores": k, "sample": f"{k} processes x {n} ids ({dt:.1f} s)"}


def oracle_rate(cfg_index, n=300_000):
    """Oracle neutrons/s on one host core over ids [0, n) of a secondary config (c4: its first two experiments)."""
    from oracle import oracle as O
    c = W.config(cfg_index)
    if "models" in c:
        pairs = [(c["instruments"][e], c["models"][e], e) for e in (0, 1)]
    else:
        pairs = [(c["instrument"], c["model"], 0)]
    t0 = time.perf_counter()
    for ins, mod, e in pairs:
        O.trace_range(ins, mod, c["seed"], 0, n // len(pairs), exp_index=e, dump=False)
    return n / (time.perf_counter() - t0)


def run_sweep(torch, S):
    """Run time against the number of neutrons, the paper's own experiment (N from 1e5 to
    1e11): c0 (monodisperse sphere) and the paper's per-event scheme on its rod (n1), one launch sequence per N,
    CUDA events around it, after one warm-up at the same N."""
    out = {}
    for idx in (0, 5):
        c = W.config(idx)
        tr = S.Tracer(c["instrument"], c["model"])
        rows = []
        for n in (10**5, 10**6, 10**7, 10**8, 10**9, 10**10, 10**11):
            reps = 1 if n >= 10**10 else 2
            for r in range(reps):
                tr.reset()
                tr.kernel_time_ms(reset=True)
                t0 = time.perf_counter()
                tr.trace(n, c["seed"])
                cnt = tr.counters()                      # synchronises
                wall = time.perf_counter() - t0
                ms, nl = tr.kernel_time_ms(reset=True)
            rows.append({"n": n, "kernel_s": ms * nl * 1e-3, "wall_s": wall, "launches": int(nl),
                         "neutrons_per_s": n / (ms * nl * 1e-3), "detected": int(cnt[6])})
        tr.close()
        out[c["name"]] = rows
    print(json.dumps({"sweep": out}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--headline-only", action="store_true", help="skip the four secondary configs")
    ap.add_argument("--config", type=int, default=HEADLINE, help="workload timed as the main line (profiling)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="run time against N (1e5..1e11) for c0 and n1, then exit")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    import paper_2501_06054_b200 as S
    S.load_library()              # raises if libsas_b200.so is missing: no fallback

    if args.sweep:
        return run_sweep(torch, S)

    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def flush():
        flush_buf.fill_(1)

    sampler = ClockSampler(local)
    sampler.start()
    head, e2e = bench_config(torch, S, args.config, args.steps, max(args.warmup, 3) if args.warmup else 0,
                             rank, world, flush, True)
    sampler.stop_flag = True
    sampler.join()
    clocks = sampler.result()

    others = {}
    if not args.headline_only:
        for i in [j for j in range(7) if j != args.config]:
            o, _ = bench_config(torch, S, i, 3, 3, rank, world, flush, False)
            others[o["workload"]] = {k: o[k] for k in ("value", "ms_per_step", "kernel_ms", "n_neutrons_per_step",
                                                       "detected_frac", "grid", "smem_bytes")}
            others[o["workload"]]["roofline_frac"] = o["roofline"]["frac"]
            others[o["workload"]]["roofline_pipe"] = o["roofline"]["pipe"]
        # config 0 at 1e6 neutrons is launch-latency bound; the same experiment at 1e9 shows the path
        c0 = W.config(0)
        tr = S.Tracer(c0["instrument"], c0["model"])
        first = rank * 10**9
        tr.trace_range(first, 10**9, c0["seed"])
        torch.cuda.synchronize()
        tr.reset()
        tr.kernel_time_ms(reset=True)
        tr.trace_range(first, 10**9, c0["seed"])
        ms, nt = tr.kernel_time_ms(reset=True)
        ms *= nt
        from paper_2501_06054_b200 import roofline as R
        cnt = tr.counters().astype(np.float64)
        rl = R.roofline(1e9 / (ms * 1e-3), 1 - cnt[1] / cnt[0], cnt[6] / cnt[0], "sphere_fp64", 1,
                        frac_geometry=1 - cnt[1] / cnt[0] - cnt[7] / cnt[0])
        others["c0_sphere_fp64_1e9"] = {"value": 1e9 * world / (ms * 1e-3), "kernel_ms": ms,
                                        "roofline_frac": rl["frac"], "roofline_pipe": rl["pipe"]}
        tr.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args.config if args.config < 4 else HEADLINE)
        try:
            cpu["all_cores"] = cpu_baseline_all_cores(args.config if args.config < 4 else HEADLINE, cpu["value"])
        except Exception as exc:                          # a reported extra, never fatal
            cpu["all_cores"] = {"error": str(exc)}
        if not args.headline_only:
            names = {W.config(i)["name"]: i for i in range(7)}
            for k, v in others.items():
                if k in names:
                    v["oracle_1core"] = oracle_rate(names[k])

    if rank == 0:
        c = W.config(args.config)
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 model / f64 geometry+accumulation",
            "data": "synthetic",
            "config": {"workload": c["name"], "n_neutrons_per_step": head["n_neutrons_per_step"], "seed": c["seed"], "parallelism": f"ids sharded over {world} GPU(s)",
                       "l2": "flushed between timed steps (256 MiB write, outside the event pairs)",
                       "grid": head["grid"], "block": head["block"], "smem_bytes": head["smem_bytes"]},
            "clocks": clocks, "e2e": e2e, "gpu_launches": head["gpu_launches"],
            "ms_per_step_median": head["ms_per_step_median"], "ms_per_step_best": head["ms_per_step_best"],
            "kernel_ms": head["kernel_ms"], "roofline": head["roofline"], "cpu_baseline": cpu,
            "configs": others,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
