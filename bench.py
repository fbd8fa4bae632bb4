"""bench.py -- throughput of the hot path on BASELINE.json's config 3 (1e8 fp64 events, Ipatia+exp).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--events N]

A step is one pass of the whole hot path over the resident event array: parameter upload, prologue
(per-set constants, normalisation), streaming NLL kernel with its deterministic reduction, for ONE
parameter set (K = 1); the K = 9 gradient batch, the general shape P2 and the fit loop of config 2 are
timed beside it and reported in the same JSON line.  Inputs are generated on the device by the
method's own seeded toy generator (synthetic, the paper's workload: PAPER.md:343-351).  The array
(800 MB) is larger than L2 (126 MB), so every step streams from HBM.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import ipa_inputs as inp  # noqa: E402

LO, HI = inp.LO, inp.HI
METRIC = "unbinned fp64 NLL events/s (Ipatia+exp)"
UNIT = "events/s"
# Algorithmic FP64 work per event and parameter set: flops, FMA = 2.
FLOPS_PER_EVENT_SET = {"P1_geometric": None}  # filled from DESIGN.md numbers below
SM_COUNT, FP64_LANES, SM_MAX_HZ = 148, 64, 1.965e9
FP64_PEAK_NOMINAL = SM_COUNT * FP64_LANES * 2 * SM_MAX_HZ  # 37.2 TFLOP/s


def algorithmic_flops(degree):
    """FP64 flops one event x set needs in this method (table 'work per event'):
    core path 2*(degree) Horner + fixed part; the fixed part is counted from the SASS of the kernel
    (sqrt, region select, tail log, exp, log1p, accumulate)."""
    return 2.0 * degree + FIXED_FLOPS


FIXED_FLOPS = 260.0  # see DESIGN.md: SASS count of the non-polynomial FP64 work per event (v1 kernel)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [s.strip() for s in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def cpu_baseline(x_host, params, cores, budget_events):
    import oracle
    n = int(min(x_host.size, budget_events))
    t0 = time.perf_counter()
    v = oracle.nll(x_host[:n], params, LO, HI, nthreads=cores)
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} events of the workload, K=1, {cores} threads each on a contiguous chunk, {dt:.2f} s",
            "nll": float(v[0])}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cores = os.cpu_count() or 1
    n = int(min(args.events, 250_000 * cores))
    x = inp.standin_masses(3, n)
    P = inp.GEN
    for _ in range(args.warmup):
        oracle.nll(x[: n // 4], P, LO, HI, nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.nll(x, P, LO, HI, nthreads=cores)
    dt = time.perf_counter() - t0
    val = n * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (x87 long double inside)", "data": "synthetic",
            "config": {"workload": f"config 3 model (Ipatia+exp, lambda=zeta=1), bounded sample of {n} events per step",
                       "events_per_step": n, "K": 1},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{n} stand-in events per step, {cores} threads"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def timed(torch, fn, steps, stream):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=100_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import paper_1706_01420_b200 as ipa

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    stream = torch.cuda.current_stream()
    n = args.events
    P1 = inp.GEN
    batch9, h = inp.fd_batch(P1)

    # workload: config 3, generated on the device by the method's generator (seed 3 + rank)
    x, _, _ = ipa.ipa_toy_generate([3 + rank], P1, -1.0, -1.0, LO, HI, n)
    ws = ipa.workspace(n, 32)
    out1 = torch.empty(1, dtype=torch.float64, device="cuda")
    out9 = torch.empty(9, dtype=torch.float64, device="cuda")
    st1 = torch.empty(1, dtype=torch.int32, device="cuda")
    st9 = torch.empty(9, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()

    ipa.ipa_set_degree_policy(1)  # general-order path: no half-integer shortcut in the headline (reading D2)

    def step_k1():
        ipa.ipa_nll_eval(x, P1, LO, HI, ws=ws, stream=stream, out=out1, status=st1)

    def step_k9():
        ipa.ipa_nll_eval(x, batch9, LO, HI, ws=ws, stream=stream, out=out9, status=st9)

    for _ in range(args.warmup):
        step_k1()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    if dist:
        dist.barrier()
    dt = timed(torch, step_k1, args.steps, stream)
    if dist:
        t = torch.tensor([dt], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.barrier()
        dt = t.item()
    clocks = sampler.stop() if rank == 0 else None
    value = world * n * args.steps / dt
    nll1 = out1.item()

    extras = {}
    if not args.no_extras:
        for _ in range(2):
            step_k9()
        dt9 = timed(torch, step_k9, max(3, args.steps // 4), stream) / max(3, args.steps // 4)
        extras["k9_gradient_batch"] = {"ms_per_call": dt9 * 1e3, "event_sets_per_s": 9 * n / dt9,
                                       "events_per_s": n / dt9}
        ipa.ipa_set_degree_policy(0)
        for _ in range(2):
            step_k1()
        dta = timed(torch, step_k1, args.steps, stream) / args.steps
        extras["k1_adaptive_degree_half_integer_shortcut"] = {"ms_per_call": dta * 1e3, "events_per_s": n / dta}

        def step_p2():
            ipa.ipa_nll_eval(x, inp.P2, LO, HI, ws=ws, stream=stream, out=out1, status=st1)
        for _ in range(2):
            step_p2()
        dtp = timed(torch, step_p2, args.steps, stream) / args.steps
        extras["k1_general_shape_P2"] = {"ms_per_call": dtp * 1e3, "events_per_s": n / dtp}
        ipa.ipa_set_degree_policy(1)
        # FP64 peak probe (DFMA chains), for the roofline denominator
        iters = 200000
        ipa.ipa_fp64_peak_probe(1000)
        tp = timed(torch, lambda: ipa.ipa_fp64_peak_probe(iters), 1, stream)
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        extras["fp64_dfma_probe_tflops"] = sms * 8 * 256 * 8 * 2.0 * iters / tp / 1e12

    # end to end through the public API with HOST buffers: H2D of the events + D2H of the result inside
    e2e = None
    if rank == 0 or dist:
        xh = torch.empty(n, dtype=torch.float64, pin_memory=True)
        xh.copy_(x)
        torch.cuda.synchronize()
        ipa.nll_host(xh, P1, LO, HI, x_dev=x, ws=ws)
        e2e_steps = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            r = ipa.nll_host(xh, P1, LO, HI, x_dev=x, ws=ws)
        torch.cuda.synchronize()
        de = time.perf_counter() - t0
        if dist:
            t = torch.tensor([de], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            de = t.item()
        e2e = {"value": world * n * e2e_steps / de, "unit": UNIT, "h2d_bytes_per_step": 8 * n + 88,
               "d2h_bytes_per_step": 8, "steps": e2e_steps, "nll": float(r[0])}

    if rank != 0:
        return
    degree = 31  # geometric policy on the config-1 z-interval (prologue output)
    flops = algorithmic_flops(degree)
    achieved = flops * n * args.steps / dt / 1e12 / world * world  # per GPU == aggregate / world
    peak = FP64_PEAK_NOMINAL / 1e12
    roofline = {"bound": "alu", "achieved": flops * n / (dt / args.steps) / 1e12, "peak": peak, "unit": "TFLOP/s",
                "frac": flops * n / (dt / args.steps) / 1e12 / peak, "traffic": None,
                "peak_source": "nominal 148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (no FP64 entry in MEASURED_PEAKS.json); "
                               "measured DFMA probe in extras",
                "flops_per_event_set": flops,
                "hbm": {"achieved_gbs": 8.0 * n / (dt / args.steps) / 1e9, "algorithmic_bytes_per_event": 8}}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        roofline["hbm"]["peak_gbs"] = peaks.get("hbm_gbs")
        roofline["hbm"]["frac"] = roofline["hbm"]["achieved_gbs"] / peaks["hbm_gbs"]
    except Exception:
        roofline["hbm"]["peak_gbs"] = 6650.0
        roofline["hbm"]["frac"] = roofline["hbm"]["achieved_gbs"] / 6650.0
        roofline["hbm"]["peak_note"] = "of fallback"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config 3: 1e8 fp64 events on [5000,5600] from the Ipatia+exp model (device generator, "
                                   "seed 3), one NLL evaluation per step, K=1, general-order degree policy",
                       "events": n, "K": 1, "l2": "input (8 B x events) larger than L2, no flush needed",
                       "multi_gpu": "independent event shards per rank, no data-path collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": 2 * args.steps, "roofline": roofline, "nll": nll1}
    line.update(extras)
    if not args.no_cpu_baseline and world == 1:
        cores = os.cpu_count() or 1
        xs = x[: min(n, 1_000_000 * cores)].cpu().numpy()
        line["cpu_baseline"] = cpu_baseline(xs, P1, cores, 1_000_000 * cores)
    print(json.dumps(line))


if __name__ == "__main__":
    main()
