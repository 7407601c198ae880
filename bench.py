#!/usr/bin/env python
"""bench.py -- neutrons traced per second on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (RNG -> source -> slits -> sample -> Q -> I(Q) with the quadrature
loops -> detector histogram) over one batch of synthetic neutrons.  The headline workload is the largest
single-GPU one of BASELINE.json that the target names, configs[2]: oriented cylinders, fp32 model, 24 x 24
orientation nodes per detected neutron, 1e9 neutrons per step, 256 x 256 detector.  `value` is timed with the
descriptors and tables resident on the device; `e2e` goes through the C ABI with host buffers every step
(sas_set_model: H2D of parameters and tables; sas_read_detector: D2H of the three histograms).  Every other
workload -- c0 (1e6 as specified, and 1e9), c1 in fp32 AND fp64, c3, c4 (batch of 1024), n1, n2 -- is timed the
same way (>= 10 steps, its own clock record, roofline and e2e) and reported under "configs".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 is launched by torch.distributed.run, one rank per GPU (`python bench.py --gpus N` without a launcher
re-executes itself under it); rank r traces the id range [r n, (r+1) n) of every experiment (weak scaling) and
the detectors are merged onto rank 0 by one reduction per step.  --impl reference times the CPU oracle
(oracle/) on bounded 1e5-id steps of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import sas_workloads as W  # noqa: E402

METRIC = "neutrons traced/sec on 1 B200 (SANS + SAS sample)"
UNIT = "neutrons/s"
HEADLINE = 2                      # BASELINE.json configs[2]
# (name in "configs", workload index, precision override, neutrons per step override)
SECONDARY = [("c0_sphere_fp64", 0, None, None), ("c0_sphere_fp64_1e9", 0, None, 10**9),
             ("c1_polysphere_py_fp32", 1, "fp32", None), ("c1_polysphere_py_fp64", 1, "fp64", None),
             ("c3_coreshell_triaxial", 3, None, None), ("c4_batch", 4, None, None),
             ("n1_paper_cylinder", 5, None, None), ("n2_paper_barbell", 6, None, None),
             ("n3_paper_micelle", 7, None, None), ("n4_paper_hayter_msa", 8, None, None),
             ("n5_paper_hollow_prism", 9, None, None)]


# ------------------------------------------------------------------ reference arm: the CPU oracle
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle as O
    c = W.config(HEADLINE)
    ins, mod = O.make_instrument(c["instrument"]), O.make_model(c["model"])
    sample = 100_000              # ids per step: a bounded sample of the 1e9-neutron workload (~0.5 s each)
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
                   "note": "CPU oracle, single thread, ids [0, (warmup+steps)*1e5) of the 1e9-neutron workload"},
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
            time.sleep(0.001)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------ helpers
def is_event_model(model):
    return "gauss_mc" in model["pd_kind"]


def model_key_and_nodes(model):
    """Row of roofline.MODEL_COST that prices this model, and its node evaluations per detected neutron."""
    m, prec = model["model"], model["precision"]
    pd = [n if k == "schulz" else 1 for k, n in zip(model["pd_kind"], model["pd_nodes"])]
    if is_event_model(model) and m == "cylinder":
        return "cylinder_event_fp64", 0
    if is_event_model(model) and m == "barbell":
        return "barbell_event_fp64", 64
    if m == "polymer_micelle":
        return "micelle_event_fp64", 0
    if is_event_model(model) and m == "hollow_prism_thin":
        return "hollow_prism_event_fp64", 0
    if is_event_model(model) and m == "sphere" and model["sq_kind"] == "hayter_msa":
        return "sphere_msa_event_fp64", 32   # node pairs of the folded 64-node rule (models.cuh: msa_sq)
    if m == "sphere":
        nodes = pd[0]
        if nodes == 1:
            return "sphere_fp64", 0              # one evaluation, served in fp64
        return ("sphere_py_" if model["sq_kind"] != "none" else "sphere_") + prec, nodes
    if m == "cylinder" and model["orient_kind"] == "gauss_quad":
        return "cylinder_quad_fp32", model["n_theta"] * model["n_phi"] * pd[0] * pd[1]
    if m == "core_shell_triaxial":
        return "cs_triaxial_iso_fp32", pd[0] * pd[1]
    if m == "cylinder":
        return "cylinder_iso_fp64", 0
    raise KeyError(m)


def geometry_class(ins):
    return "fast" if ins["sample_shape"] == "box" and ins["mu_abs_2200"] == 0 and ins["mu_inc"] == 0 else "general"


VARIANT_OF = {"sphere": 0, "core_shell_sphere": 1, "cylinder": 2, "triaxial": 3, "core_shell_triaxial": 4}


def run_microbench(local):
    """Pipe rates of this GPU from csrc/microbench.cu (built by __graft_entry__.build / build.py --microbench)."""
    from paper_2501_06054_b200 import build as libbuild
    exe = os.path.join(ROOT, "paper_2501_06054_b200", "microbench")
    try:
        if not os.path.exists(exe):
            libbuild.build_microbench()
        env = dict(os.environ, CUDA_VISIBLE_DEVICES=os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")[local]
                   if os.environ.get("CUDA_VISIBLE_DEVICES") else str(local))
        out = subprocess.run([exe], capture_output=True, text=True, timeout=120, env=env).stdout
        return json.loads([ln for ln in out.splitlines() if ln.startswith("{")][-1])
    except Exception as exc:                              # the roofline then says it used the recorded rates
        return {"error": str(exc)}


def time_steps(torch, tracer, do_step, steps, warmup, flush):
    """Device time of `steps` steps: one CUDA-event pair per step on the tracer's stream, L2 flushed between
    steps outside the pairs; barrier + synchronize on both sides; MAX over ranks."""
    import torch.distributed as dist
    for i in range(warmup):
        do_step(i)
    torch.cuda.synchronize()
    if dist.is_initialized():
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    tracer.kernel_time_ms(reset=True)
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
    if dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    return total_ms, per_step


def bench_config(torch, S, cfg_index, precision, n_override, steps, warmup, rank, world, local, flush, rates, traffic):
    from paper_2501_06054_b200 import roofline as R
    from paper_2501_06054_b200.sharding import weak_shard, merge_detectors
    c = W.config(cfg_index, precision) if precision else W.config(cfg_index)
    batch = "models" in c
    dev = torch.device("cuda", local)
    if batch:
        tr = S.BatchTracer(c["instruments"], c["models"], device=dev)
        n_arg = n_override or c["n_neutrons_each"]
        n_step = n_arg * len(c["models"])
    else:
        tr = S.Tracer(c["instrument"], c["model"], device=dev)
        n_step = n_arg = n_override or c["n_neutrons"]
    seed = c["seed"]
    first, _ = weak_shard(n_arg, rank)                    # rank r owns ids [r n, (r+1) n) of every experiment

    def do_step(i):
        tr.reset()
        tr.trace_range(first, n_arg, seed)
        if world > 1:
            merge_detectors([tr.sum_p, tr.sum_p2, tr.counts], dst=0)

    sampler = ClockSampler(local)
    sampler.start()
    # the timed steps run as a user's production loop does, without the library's per-launch event pairs
    # (sas_set_launch_timing: ~6 us of stream operations per launch); the same steps are then repeated with them
    # on, for the per-launch kernel times the roofline is computed from
    tr.set_launch_timing(False)
    total_ms, per_step = time_steps(torch, tr, do_step, steps, warmup, flush)
    tr.set_launch_timing(True)
    tr.kernel_time_ms(reset=True)
    for i in range(steps):
        flush()
        do_step(warmup + i)
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    clocks = sampler.result()
    recs = tr.launch_records()                            # every trace-kernel launch of the repeated steps
    tr.kernel_time_ms(reset=True)
    tr.set_launch_timing(False)                           # end to end below: the production setting again
    info = tr.launch_info()
    cnt = tr.counters().astype(np.float64)
    ms_per_step = total_ms / steps
    per = sorted(per_step)
    kernel_ms = sum(r["ms"] for r in recs) / steps
    out = {"workload": c["name"], "precision_requested": (c["models"][0] if batch else c["model"])["precision"],
           "n_neutrons_per_step": n_step, "steps": steps, "ms_per_step": ms_per_step,
           "value": n_step * world / (ms_per_step * 1e-3),
           "ms_per_step_median": per[len(per) // 2], "ms_per_step_best": per[0], "kernel_ms": kernel_ms,
           "grid": info["grid"], "block": info["block"], "smem_bytes": info["smem_bytes"],
           "gpu_launches": len(recs) // steps + 1, "clocks": clocks,   # trace kernels + zero_detector_kernel
           "detected_frac": cnt[6] / cnt[0], "survive_frac": 1.0 - cnt[1] / cnt[0],
           # survivors whose fp64 geometry ran (the others were certain detector misses, counters[7])
           "geometry_frac": 1.0 - cnt[1] / cnt[0] - cnt[7] / cnt[0]}
    # roofline: one record per launch group (a batch launches one kernel per model form), each from its own
    # event time; the step's fraction is the sum of the groups' algorithmic lane-clocks over peak x kernel time
    models = c["models"] if batch else [c["model"]]
    inss = c["instruments"] if batch else [c["instrument"]]
    groups = {}
    for ins, m in zip(inss, models):
        key, nodes = model_key_and_nodes(m)
        g = groups.setdefault((VARIANT_OF.get(m["model"], -1), is_event_model(m)), dict(key=key, nodes=nodes, geo=geometry_class(ins), n_exp=0))
        g["n_exp"] += 1
    ms_of = {}
    for r in recs:
        k = (r["variant"] if r["variant"] != 6 else 2, bool(r["per_event"]))
        ms_of[k] = ms_of.get(k, 0.0) + r["ms"] / steps
    peak = R.N_SM * R.SMSP_PER_SM * 32 * R.SM_MAX_MHZ * 1e6
    lane_clocks, parts = 0.0, []
    for k, g in groups.items():
        ms = ms_of.get(k, kernel_ms if len(groups) == 1 else 0.0)
        n_g = n_arg * g["n_exp"]
        rl = R.roofline(n_g / (ms * 1e-3) if ms > 0 else 0.0, out["survive_frac"], out["detected_frac"], g["key"], g["nodes"],
                        frac_geometry=out["geometry_frac"], geometry=g["geo"], rates=rates,
                        sm_mhz_sampled=clocks.get("sm_mhz"), traffic=traffic.get(c["name"]))
        rl["model_cost_row"], rl["kernel_ms"], rl["n_exp"] = g["key"], ms, g["n_exp"]
        lane_clocks += rl["achieved"] * 1e9 * ms * 1e-3
        parts.append(rl)
    if len(parts) == 1:
        out["roofline"] = parts[0]
    else:
        top = max(parts, key=lambda p: p["kernel_ms"])
        out["roofline"] = dict(top, frac=lane_clocks / (peak * kernel_ms * 1e-3), achieved=lane_clocks / (kernel_ms * 1e-3) / 1e9,
                               note="per-launch records under 'launches'; frac = sum of their algorithmic lane-clocks / (peak x kernel time)",
                               launches=parts)
        out["roofline"].pop("frac_at_sampled_clock", None)

    # ---- end to end: the call a user makes, host buffers in and out, every step
    import paper_2501_06054_b200.binding as B
    if batch:
        host = [torch.empty((len(models),) + tuple(tr.shape[1:]), dtype=dt, pin_memory=True)
                for dt in (torch.float64, torch.float64, torch.int64)]
        tr.close()

        def e2e_step(i):
            bt = S.BatchTracer(c["instruments"], c["models"], device=dev)   # host descriptors -> tables -> H2D
            bt._host = host                                                    # caller-owned page-locked output
            bt.trace_range(first, n_arg, seed)
            res = bt.read_detector()                                           # D2H of every histogram
            up = bt.upload_bytes()
            bt.close()
            return res, up
    else:
        def e2e_step(i):
            tr.set_model(c["model"])                # H2D: parameters + quadrature tables
            tr.reset()
            tr.trace_range(first, n_arg, seed)
            return tr.read_detector(), tr.upload_bytes()   # D2H: three histograms into host arrays

    n_e2e = steps if not batch else max(3, steps // 3)
    for i in range(2):
        e2e_step(i)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(n_e2e):
        (sp, sp2, cn), up = e2e_step(i)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    if world > 1:
        import torch.distributed as dist
        t = torch.tensor([dt], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dt = float(t.item())
    out["e2e"] = {"value": n_step * world * n_e2e / dt, "unit": UNIT, "steps": n_e2e, "ms_per_step": 1e3 * dt / n_e2e,
                  "h2d_bytes_per_step": int(up), "d2h_bytes_per_step": int(3 * 8 * sp.size),
                  "includes": ("sas_create_batch + sas_trace_batch_range + sas_read_detector + sas_destroy" if batch else
                               "sas_set_model + sas_reset_detector + sas_trace_range + sas_read_detector")}
    if not batch:
        tr.close()
    return out


def bench_reduce(torch, S, local, hbm_gbs):
    """The ring average (sas_reduce_radial): one kernel reading sum_p and sum_p2 of a 512 x 512 detector (16 B per
    pixel), HBM-bound; its own roofline against the measured copy bandwidth."""
    c = W.config(3)
    tr = S.Tracer(c["instrument"], c["model"], device=torch.device("cuda", local))
    tr.trace(10**7, c["seed"])
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=tr.device)
    best = []
    for i in range(12):
        flush_buf.fill_(i)
        tr.reduce_radial(6.0, 0.001, 0.05, 200)
        best.append(tr.reduce_time_ms())
    tr.close()
    ms = float(np.median(best[2:]))
    npix = c["instrument"]["det_nx"] * c["instrument"]["det_ny"]
    gbs = 16.0 * npix / (ms * 1e-3) / 1e9
    return {"workload": "ring average of the 512 x 512 detector of c3 into 200 rings (L2 flushed before each call)",
            "kernel_ms_median": ms, "algorithmic_bytes": 16 * npix,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs if hbm_gbs else None,
                         "note": "4 MB read once: the kernel is launch-latency sized (a few microseconds), far from bandwidth-bound"}}


def _oracle_worker(job):
    cfg_index, precision, first, n, exps = job
    from oracle import oracle as O
    c = W.config(cfg_index, precision) if precision else W.config(cfg_index)
    if "models" in c:
        for e in exps:
            O.trace_range(c["instruments"][e], c["models"][e], c["seed"], first, n // len(exps), exp_index=e, dump=False)
    else:
        O.trace_range(c["instrument"], c["model"], c["seed"], first, n, dump=False)
    return n


def oracle_rates(cfg_index, precision, seconds=2.0):
    """The oracle as it stands on the host cores: one core, then K independent id-range processes (the paper's
    MPI scheme), K = the cores this process may run on."""
    import multiprocessing as mp
    exps = (0, 1)                                         # c4: its first sphere and its first cylinder
    t0 = time.perf_counter()
    _oracle_worker((cfg_index, precision, 0, 20000, exps))
    rate = 20000 / (time.perf_counter() - t0)
    n = int(min(max(rate * seconds, 2e4), 5e7))
    t0 = time.perf_counter()
    _oracle_worker((cfg_index, precision, 0, n, exps))
    dt1 = time.perf_counter() - t0
    k = len(os.sched_getaffinity(0))
    out = {"oracle_1core": n / dt1, "oracle_1core_sample": f"ids [0, {n}) ({dt1:.1f} s)"}
    try:
        with mp.get_context("spawn").Pool(k) as pool:
            pool.map(_oracle_worker, [(cfg_index, precision, 0, 1000, exps)] * k)   # start the workers, load the library
            t0 = time.perf_counter()
            pool.map(_oracle_worker, [(cfg_index, precision, r * n, n, exps) for r in range(k)])
            dtk = time.perf_counter() - t0
        out.update(oracle_kcores=k * n / dtk, cores=k, oracle_kcores_sample=f"{k} processes x {n} ids ({dtk:.1f} s)")
    except Exception as exc:                              # a reported extra, never fatal
        out["oracle_kcores_error"] = str(exc)
    return out


def cpu_model_name():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_sweep(torch, S):
    """Run time against the number of neutrons, the paper's own experiment (N from 1e5 to
    1e11): c0 (monodisperse sphere) and the paper's per-event scheme on its rod (n1) and on three of the models it
    found expensive (barbell n2, polymer micelle n3, Hayter MSA n4, thin-walled hollow prism n5), one launch sequence per N, CUDA
    events around it, after one warm-up at the same N."""
    out = {}
    for idx in (0, 5, 6, 7, 8, 9):
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
    ap.add_argument("--headline-only", action="store_true", help="skip the secondary workloads")
    ap.add_argument("--config", type=int, default=HEADLINE, help="workload timed as the main line (profiling)")
    ap.add_argument("--precision", default=None, help="precision override of --config (profiling)")
    ap.add_argument("--neutrons", type=int, default=None, help="neutrons per step override of --config (profiling)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="run time against N (1e5..1e11) for c0 and n1..n5, then exit")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: one rank per GPU under torch.distributed.run
        port = 29500 + os.getpid() % 2000
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                   "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])

    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE is {world}: launch one rank per GPU")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    import paper_2501_06054_b200 as S
    from paper_2501_06054_b200 import roofline as R
    from paper_2501_06054_b200 import build as libbuild
    if rank == 0:
        libbuild.build()          # no-op when the in-tree library is up to date; nvcc otherwise
    if world > 1:
        dist.barrier()
    S.load_library()              # raises if libsas_b200.so is missing: no fallback

    if args.sweep:
        return run_sweep(torch, S)

    mb = run_microbench(local)
    rates = R.rates_from_microbench(mb) if "error" not in mb else None
    traffic = R.read_traffic(os.path.join(ROOT, "profiles", "r2_dram_traffic.md"))
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def flush():
        flush_buf.fill_(1)

    warm = max(args.warmup, 3) if args.warmup else 0
    head = bench_config(torch, S, args.config, args.precision, args.neutrons, args.steps, warm, rank, world, local, flush, rates, traffic)

    others = {}
    if not args.headline_only:
        for name, idx, prec, n_over in SECONDARY:
            if idx == args.config and n_over is None and prec == args.precision:
                continue
            k = max(10, min(args.steps, 20)) if idx != 4 else 10
            o = bench_config(torch, S, idx, prec, n_over, k, 3, rank, world, local, flush, rates, traffic)
            others[name] = o
        if rank == 0:
            peaks = {}
            try:
                peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            except Exception:
                pass
            others["reduce_radial"] = bench_reduce(torch, S, local, peaks.get("hbm_gbs"))

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        c = W.config(args.config, args.precision) if args.precision else W.config(args.config)
        r = oracle_rates(args.config, args.precision, seconds=12.0)
        cpu = {"value": r["oracle_1core"], "unit": UNIT, "cores": 1, "kind": "oracle", "cpu": cpu_model_name(),
               "sample": f"{r['oracle_1core_sample']} of {c['name']}, single thread",
               "all_cores": {k: r.get(k) for k in ("oracle_kcores", "cores", "oracle_kcores_sample", "oracle_kcores_error") if k in r}}
        for name, idx, prec, n_over in SECONDARY:
            if name in others and n_over is None:
                others[name].update(oracle_rates(idx, prec, seconds=1.5))

    if rank == 0:
        c = W.config(args.config, args.precision) if args.precision else W.config(args.config)
        m0 = c["models"][0] if "models" in c else c["model"]
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": ("f32" if m0["precision"] == "fp32" else "f64") + " model / f64 RNG-to-uniform, geometry and accumulation",
            "data": "synthetic",
            "config": {"workload": c["name"], "n_neutrons_per_step": head["n_neutrons_per_step"], "seed": c["seed"],
                       "parallelism": f"neutron ids sharded over {world} GPU(s), one detector reduction per step",
                       "l2": "flushed between timed steps (256 MiB write, outside the event pairs)",
                       "grid": head["grid"], "block": head["block"], "smem_bytes": head["smem_bytes"]},
            "clocks": head["clocks"], "e2e": head["e2e"], "gpu_launches": head["gpu_launches"] * args.steps,
            "ms_per_step_median": head["ms_per_step_median"], "ms_per_step_best": head["ms_per_step_best"],
            "kernel_ms": head["kernel_ms"], "roofline": head["roofline"], "cpu_baseline": cpu,
            "microbench": mb, "configs": others,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
