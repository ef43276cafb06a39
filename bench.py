"""bench.py — samples/s of the whole hot path (Philox -> Hepp-sector sample + pdf -> all forest terms ->
conditioning check / double-double re-evaluation -> compensated sums) on BASELINE.json config 5:
seeded random 5-loop electron-vertex graphs without lepton loops, 14 variables after the merge of PAPER.md:222.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--graphs G] [--samples S] [--impl reference]

A "step" integrates --samples samples (per GPU) of each of the first --graphs graphs of the config-5 batch, by default all
32 (they come from the seeded generator in paper_1909_08015_b200/inputs.py; planning them takes a few minutes of host
time before the timed region).  Per step every graph gets a fresh range of sample ids, so no step repeats work.
value = whole-job samples/s per graph (all samples of all graphs / device time; graphs run one after another).  With
N > 1 every graph's range is split over the ranks by paper_1909_08015_b200.dist (no data-path collective; one all_gather
of the table of results per step, exact merge); value is the whole-job aggregate.  --impl reference times the CPU oracle
on the host cores instead.
"""
import argparse
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "integrand samples/sec per graph at 5 loops"
UNIT = "samples/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--graphs", type=int, default=32, help="how many graphs of the 32-graph config-5 batch to time")
    ap.add_argument("--graph-list", default="", help="comma-separated indices into the 32-graph batch (overrides --graphs), e.g. 0,17 for a profiler capture")
    ap.add_argument("--samples", type=int, default=1 << 22, help="samples per graph per step and per GPU")
    ap.add_argument("--pilot-samples", type=int, default=1 << 16, help="samples of the pilot stage that sets the acceptance tolerance")
    ap.add_argument("--impl", default="fg", choices=["fg", "reference"])
    ap.add_argument("--rel-tol", type=float, default=0.0)
    ap.add_argument("--target-samples", type=float, default=1e10, help="run length the acceptance tolerance is set for")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows = []; self.stop = False; self.index = index; self.t = None

    def start(self):
        def run():
            while not self.stop:
                try:
                    out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, timeout=5).stdout.strip()
                    if out:
                        self.rows.append([c.strip() for c in out.split(",")])
                except Exception:
                    pass
                time.sleep(0.2)
        self.t = threading.Thread(target=run, daemon=True); self.t.start()

    def finish(self):
        self.stop = True
        if self.t:
            self.t.join(3)
        sm = sorted(int(float(r[0])) for r in self.rows if r and r[0].replace(".", "").isdigit())
        mx = [int(float(r[1])) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


def cfg5_graphs(n_graphs, graph_list=""):
    from paper_1909_08015_b200 import inputs
    cfg = inputs.config(5)
    if graph_list:
        return [cfg["graphs"][int(i)] for i in graph_list.split(",")], cfg
    return cfg["graphs"][:n_graphs], cfg


def oracle_leg(args, graphs, steps, warmup, seconds):
    """The CPU oracle as it stands on the host cores: samples/s on a bounded sample of graph 0 (table build excluded,
    reported as build_s).  Precision policy as on the GPU's first rung: every sample in double precision (the oracle's
    higher-precision evaluations serve the parity tests; its __float128 rate is quoted in `sample` as context)."""
    from oracle import oracle as O
    x, ph = graphs[0]
    t0 = time.time(); orc = O.Oracle(x, ph, merge=True, printed=False); build_s = time.time() - t0
    t0 = time.time(); orc.integrate(1, 0, 256, quad=False); probe = (time.time() - t0) / 256
    t0 = time.time(); orc.integrate(1, 0, 32, quad=True); quad_rate = 32 / (time.time() - t0)
    per_step = max(256, int(seconds / max(steps, 1) / max(probe, 1e-9)))
    for w in range(warmup):
        orc.integrate(1, 10 ** 9 + w * 256, 256, quad=False)
    t0 = time.time(); done = 0
    for k in range(steps):
        orc.integrate(1, k * per_step, per_step, quad=False); done += per_step
    dt = time.time() - t0
    return dict(value=done / dt, unit=UNIT, cores=O.threads(), kind="oracle",
                sample="config-5 graph 0, %d samples x %d steps, every sample in double precision (spanning-tree sums, pattern loops); with the __float128 evaluation of every sample on top: %.0f samples/s; table build %.0f s not timed" % (per_step, steps, quad_rate, build_s),
                ms_per_step=1e3 * dt / steps, per_step=per_step, build_s=build_s)


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    graphs, _ = cfg5_graphs(1)
    r = oracle_leg(args, graphs, max(1, args.steps), args.warmup, seconds=min(120.0, 12.0 * max(1, args.steps)))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config5: seeded random 5-loop vertex graphs, M=14; CPU oracle on graph 0, %d samples/step" % r["per_step"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# DRAM traffic of the dominant kernel from the ncu capture of build cbfb73c (written up in profiles/r02_stream_kernel_ncu.md;
# a constant here: bench.py reads nothing under profiles/): dram__bytes_read.sum + dram__bytes_write.sum of one launch of
# fg_stream_kernel divided by the 606208 samples of that launch, config-5 graph 0 (graph 17: 54.1 KB per sample).
STREAM_KERNEL_DRAM_BYTES_PER_SAMPLE = 3754.0


def main_fg(args):
    import torch
    from paper_1909_08015_b200 import build, dist as fgdist, fg, sched
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local = int(os.environ.get("LOCAL_RANK", "0"))
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the library has no CPU path); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    graphs, cfg = cfg5_graphs(args.graphs, args.graph_list)
    S = args.samples                 # samples per graph per step PER GPU (weak scaling): a step integrates world * S per graph
    stream = torch.cuda.current_stream()
    # plans; acceptance tolerance (18) for the run length the config names: abs_tol = sigma_down(target)/4 from a pilot stage
    batch = sched.Batch([fg.plan_for(x, ph, merge_ext_lines=True, rel_tol=1e-6, abs_tol=0.0, device=local) for x, ph in graphs])
    plans = batch.plans
    batch.pilot(args.pilot_samples, cfg["seed"], first_sample=10 ** 12, target_samples=args.target_samples, rel_tol=args.rel_tol, stream=stream)
    info = [dict(graph=gi, x=x, photons=ph, abs_tol=batch.abs_tol[gi], **{k: plans[gi].stats[k] for k in ("n_terms", "n_records", "n_coefs", "flops_per_sample", "exec_flops_per_sample", "plan_seconds")})
            for gi, (x, ph) in enumerate(graphs)]
    peak_tf, _ = fg.dfma_peak(local, 200000, stream)
    peak_tf = max(peak_tf, fg.dfma_peak(local, 200000, stream)[0])
    dmma_tf = fg.dmma_peak(local, 20000, stream)[0]       # FP64 tensor path (shares the FP64 units with DFMA): context
    table = torch.zeros((len(plans), fgdist.RESULT_DOUBLES), dtype=torch.float64, device=dev)
    gathered = [None]

    def step_async(k):
        # product path of the multi-GPU case: every graph's sample range of this step is split over the ranks
        # (dist.shard_range), shard results stay on the device, one all_gather of the result table per step
        for gi, p in enumerate(plans):
            fgdist.integrate_sharded_async(p, world * S, cfg["seed"], rank, world, table[gi].data_ptr(), stream=stream, first_sample=k * world * S)
        gathered[0] = fgdist.gather_device(table, world)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for w in range(args.warmup):
        step_async(10 ** 6 + w)
    barrier()
    for p in plans:
        p.profile(True)              # four CUDA events per slab on the launching stream, resolved after the timed region
    clocks = ClockSampler(local) if rank == 0 else None
    if clocks:
        clocks.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(args.steps):
        step_async(k)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clk = clocks.finish() if clocks else None
    tim = [p.timing() for p in plans]
    for p in plans:
        p.profile(False)
    merged = fgdist.merge_gathered(gathered[0])          # last step, all ranks merged (exact double-double merge)
    # end to end through the blocking C call with host result buffers (d2h of the 88-byte result every call)
    flagged = flagged2 = rejected = 0
    barrier()
    e2e_steps = min(args.steps, 3)
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        for gi, p in enumerate(plans):
            r = fgdist.integrate_sharded(p, world * S, cfg["seed"], rank, world, device=dev, stream=stream, first_sample=(args.steps + k) * world * S)
            flagged += int(r.n_flagged); flagged2 += int(r.n_flagged2); rejected += int(r.n_rejected)
    torch.cuda.synchronize()
    ms_e2e = 1e3 * (time.perf_counter() - t0)
    t = torch.tensor([ms, ms_e2e], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, ms_e2e = float(t[0]), float(t[1])
    if rank != 0:
        if world > 1:
            dist.barrier(); dist.destroy_process_group()
        return
    total = float(world) * len(plans) * S * args.steps
    value = total / (ms * 1e-3)
    ms_d = sum(x["ms_double"] for x in tim); ms_q = sum(x["ms_dd"] for x in tim); launches = sum(x["launches"] for x in tim)
    algo = sum(p.stats["flops_per_sample"] for p in plans) * S * args.steps
    execf = sum(p.stats["exec_flops_per_sample"] for p in plans) * S * args.steps
    ach = algo / (ms_d * 1e-3) / 1e12
    for gi, x in enumerate(tim):       # per-graph throughput of the double-precision pass and its algorithmic FP64 rate
        info[gi]["samples_per_s"] = S * args.steps / (x["ms_double"] * 1e-3)
        info[gi]["algo_tflops"] = info[gi]["flops_per_sample"] * info[gi]["samples_per_s"] / 1e12
        info[gi]["frac"] = info[gi]["algo_tflops"] / peak_tf
        info[gi]["ext_ms_per_step"] = x["ms_dd"] / args.steps
        info[gi]["mean_last_step"] = merged[gi].mean; info[gi]["sigma_last_step"] = max(merged[gi].variance, 0.0) ** 0.5
    fr = sorted(g["frac"] for g in info)
    traffic = None if STREAM_KERNEL_DRAM_BYTES_PER_SAMPLE is None else STREAM_KERNEL_DRAM_BYTES_PER_SAMPLE * min(S, plans[0].wave_samples())
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "config5: %s of the 32 seeded random 5-loop vertex graphs (14 lines, M=14 after merge), %d samples per graph per step per GPU, graphs one after another, fresh Philox sample ids every step; value = whole-job samples/s per graph (all graphs' samples / device time)" % ("all 32" if len(plans) == 32 else ("graphs %s" % args.graph_list if args.graph_list else "the first %d" % len(plans)), S),
                       "l2": "inputs are generated on chip; the 2-9 MB coefficient stream per graph is L2-resident by design (re-read by every block), no flush applies",
                       "tolerance": "rel_tol %.1e, abs_tol = sigma_down(%.0e samples)/4 from a %d-sample pilot stage per graph (PAPER.md:286, (18))" % (args.rel_tol, args.target_samples, args.pilot_samples),
                       "graphs": info, "flagged_fraction": flagged / max(1.0, float(world) * len(plans) * S * e2e_steps), "flagged2": flagged2, "rejected": rejected,
                       "frac_per_graph": {"min": fr[0], "median": fr[len(fr) // 2], "max": fr[-1]},
                       "kernel_ms": {"double_pass": ms_d, "extended_passes": ms_q, "share_double": ms_d / max(ms_d + ms_q, 1e-9)},
                       "exec_tflops_double_pass": execf / (ms_d * 1e-3) / 1e12},
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf, "traffic": traffic,
                         "traffic_unit": "DRAM bytes per launch of fg_stream_kernel over one wave of graph 0 (ncu capture, profiles/r02_stream_kernel_ncu.md; algorithmic bytes: 0)",
                         "kernel": "fg_stream_kernel (with its fg_geom_kernel: the time is that of the double-precision pass, CUDA events around every slab in the timed region)",
                         "peak_source": "fg_dfma_peak measured in this run (MEASURED_PEAKS.json has no FP64 entry)", "dmma_peak": dmma_tf,
                         "frac_executed": execf / (ms_d * 1e-3) / 1e12 / peak_tf},
            "e2e": {"value": float(world) * len(plans) * S * e2e_steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 88 * len(plans),
                    "steps": e2e_steps, "note": "blocking fg_integrate_range per graph (host result struct, 88 bytes device to host per call); inputs are a seed and a sample range, nothing goes host to device"},
            "gpu_launches": launches, "clocks": clk}
    if not args.no_cpu_baseline and world == 1:
        r = oracle_leg(args, graphs, 3, 1, args.cpu_seconds)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.barrier(); dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        main_reference(a)
    else:
        main_fg(a)
