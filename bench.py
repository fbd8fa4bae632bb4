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
SM_COUNT, FP64_LANES, SM_MAX_HZ = 148, 64, 1.965e9
# B200 has 64 FP64 FMA lanes per SM (the DFMA-chain probe in extras measures 95 % of this)
FP64_PEAK_NOMINAL = SM_COUNT * FP64_LANES * 2 * SM_MAX_HZ  # 37.2 TFLOP/s


def algorithmic_flops(degree, p_core):
    """FP64 flops one event x set needs in this method (table 'work per event'),
    FMA = 2, add / mul / compare = 1; an event pays the core OR the tail arithmetic, never both:
      common  d (1), 2 compares (2), E_B (1 FMA), exp = 5 FMA + 1 add + 1 mul (12), 1+w (1), log on [1,2] = 6 FMA (12),
              2 adds                                                                          : 12 FMA + 8 other = 32
      core    q, sqrt (3 FMA + 2 mul), t, Horner (degree FMA), (beta-k) d                     : (6 + degree) FMA + 2 mul
      tail    u (1 FMA), log = 7 FMA + 1 add, -n log u + c (1 FMA), -k d (1 FMA)              : 10 FMA + 1 add = 21
    (table-driven exp / log of round 2: csrc/ipa_fastmath.cuh; the degree-11 / degree-8 polynomials of round 1 made
    this 55 / 27).  p_core = fraction of the events inside [mu - a sigma, mu + a2 sigma] (0.344 for the config model)."""
    core = 2.0 * (6 + degree) + 2.0
    return 32.0 + p_core * core + (1.0 - p_core) * 21.0


def core_cells(torch, ipa, x, P, policy):
    """Cells of the core of set P (ipa_core_cells) and the share of the core events of x in each: on a prepared (or
    sorted) array a warp lies in one cell and runs that cell's polynomial, so the Horner work of a core event is the
    degree of its cell; `degree_eff` is the mean over the core events.  An as-generated array runs the full polynomial."""
    info = ipa.ipa_core_cells(P, LO, HI, policy=policy)
    full = int(ipa.ipa_core_degree(P, LO, HI, policy=policy))
    if int(info[0]) == 0:
        return {"ncell": 0, "degree_full": full, "degree_eff": float(full)}
    core = x[(x >= P["mu"] - P["a"] * P["sigma"]) & (x <= P["mu"] + P["a2"] * P["sigma"])]
    hi = (core.view(torch.int64) >> 32).to(torch.int32)
    cnt = torch.zeros_like(hi)
    for b in info[5:11]:
        cnt += (hi >= int(b)).to(torch.int32)
    cell = (cnt - 3).abs()
    share = [float((cell == c).double().mean().item()) for c in range(4)]
    deg = [int(d) for d in info[1:5]]
    return {"ncell": 4, "degree_full": full, "cell_degrees": deg, "cell_share_of_core_events": share,
            "degree_eff": sum(a * b for a, b in zip(share, deg))}


def shape_stage_flops(degree, p_core):
    """Shape stage of a group of sets sharing (mu, sigma, lambda, zeta, beta, a, n, a2, n2) -- DESIGN.md section 5:
    d (1), 2 region compares (2), core: q, sqrt, t, Horner = (5 + degree) FMA + 2 mul; tail: u (1 FMA) + log
    (7 FMA + 1 add) + the product with -n (1 mul)."""
    return 3.0 + p_core * (2.0 * (5 + degree) + 2.0) + (1.0 - p_core) * (2.0 * 8 + 2.0)


MEMBER_STAGE_FLOPS = 32.0
"""Member stage per set: Delta = s d + (V + c): 1 add + 1 FMA (3); E_B (1 FMA: 2); exp (12); 1 + w (1);
log on [1,2] (12); 2 adds (2)."""


def gradient_flops(degree, p_core):
    """Analytic-gradient pass per event x set (ipa_eval_grad, five derivatives): common = d, 2 compares (3), exp (16),
    1+w (1), 1/(1+w) (4 FMA: 8), w/(1+w) (1), E_B (2), log (12), 2 adds, the five derivative terms (2 + 2 + 3 + 3 + 2) and
    6 accumulations = 63; core = q (2), sqrt (8), 1/r (8), t (2), value and derivative Horner 2 FMA per coefficient of the
    4 ceil((D+1)/4) slots, L - beta (3), Delta (2), dd (1), ds (3); tail = u (2), 1/u (8), log (15), Delta (4), dd (1),
    ds (5), db (2) = 37."""
    slots = 4 * (degree // 4) + 4
    core = 2.0 + 8 + 8 + 2 + 4.0 * slots + 3 + 2 + 1 + 3
    return 63.0 + p_core * core + (1.0 - p_core) * 37.0


def alu_roofline(flops_per_event, events, seconds, extra=None):
    """'alu' roofline entry: achieved = declared algorithmic FP64 flops / measured time, against the FP64 FMA peak."""
    ach = flops_per_event * events / seconds / 1e12
    d = {"bound": "alu", "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12, "unit": "TFLOP/s",
         "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "flops_per_event": flops_per_event, "ms": seconds * 1e3}
    if extra:
        d.update(extra)
    return d


def build_hash():
    """sha256 over the CUDA sources and the header the library was built from (profiles/*.md record the hash of the
    build an ncu capture was taken on; a capture of another build is not quoted)."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1706_01420_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh", ".inc")):
            h.update(open(os.path.join(csrc, name), "rb").read())
    h.update(open(os.path.join(ROOT, "include", "ipanll.h"), "rb").read())
    return h.hexdigest()[:16]


def measured_traffic(n):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the streaming kernel from the committed ncu raw
    page profiles/r02_nll_kernel_raw.csv (command in the .md beside it), quoted only if that capture was taken on
    THIS build (hash line in the .md) and scaled by the event count.  -> (bytes or None, note)."""
    import csv
    md, raw = os.path.join(ROOT, "profiles", "r02_nll_kernel_raw.md"), os.path.join(ROOT, "profiles", "r02_nll_kernel_raw.csv")
    if not (os.path.exists(md) and os.path.exists(raw)):
        return None, "no ncu --set full capture committed for this build"
    txt = open(md).read()
    h = build_hash()
    if ("build_hash: " + h) not in txt:
        return None, "profiles/r02_nll_kernel_raw.csv was captured on another build (this build: %s)" % h
    rows = list(csv.reader(open(raw)))
    hdr = next(r for r in rows if "Kernel Name" in r)
    ik, ir, iw = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    units = rows[rows.index(hdr) + 1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    vals = [float(r[ir].replace(",", "")) * scale[units[ir]] + float(r[iw].replace(",", "")) * scale[units[iw]]
            for r in rows[rows.index(hdr) + 2:] if len(r) > iw and "ipa_nll_kernel" in r[ik]]
    if not vals:
        return None, "no ipa_nll_kernel row in profiles/r02_nll_kernel_raw.csv"
    ev = 1e8
    for line in txt.splitlines():
        if line.startswith("events: "):
            ev = float(line.split()[1])
    return float(np.mean(vals)) * n / ev, ("ncu --set full, mean of %d launches of ipa_nll_kernel at %g events, "
                                           "profiles/r02_nll_kernel_raw.csv (same build %s), scaled by events" % (len(vals), ev, h))


class ClockSampler:
    """SM clock / throttle reasons during the timed region (B200_PROFILING.md recipe), sampled through
    NVML every 5 ms; falls back to nvidia-smi -lms when pynvml is not importable."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4))

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.thread, self.h = index, [], False, None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.nv = pynvml
        except Exception:
            self.h = None
            return
        self.thread = threading.Thread(target=self._loop, daemon=True)
        self.thread.start()

    def _loop(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                mx = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.rows.append((sm, mx, pw, rs))
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self):
        if self.h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["NVML unavailable"], "samples": 0}
        self.stop_flag = True
        self.thread.join(timeout=2)
        sm = [r[0] for r in self.rows]
        reasons = sorted({nm for r in self.rows for nm, bit in self.REASONS if r[3] & bit})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(r[1] for r in self.rows) if sm else None,
                "power_w_max": max(r[2] for r in self.rows) if sm else None, "samples": len(sm), "reasons": reasons}


def cpu_baseline(x_host, params, cores):
    """The oracle as it stands on the host cores: all-cores figure on the WHOLE workload (its NLL is the parity number of
    the line) and the single-thread figure on the first 1e6 events (SURVEY.md 8(d) 'Timing the oracle beside it')."""
    import oracle
    n = int(x_host.size)
    t0 = time.perf_counter()
    v = oracle.nll(x_host, params, LO, HI, nthreads=cores)
    dt = time.perf_counter() - t0
    n1 = min(n, 1_000_000)
    t0 = time.perf_counter()
    v1 = oracle.nll(x_host[:n1], params, LO, HI, nthreads=1)
    dt1 = time.perf_counter() - t0
    return ({"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
             "sample": f"all {n} events of the workload, K=1, {cores} threads each on a contiguous chunk, {dt:.2f} s",
             "nll": float(v[0])},
            {"value": n1 / dt1, "unit": UNIT, "cores": 1, "kind": "oracle",
             "sample": f"first {n1} events of the workload, K=1, single thread (the oracle proper), {dt1:.2f} s",
             "nll": float(v1[0])})


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


def other_rows(torch, ipa, x, ws, stream, n, p_core):
    """The other rows of SURVEY.md 8(a), timed at BASELINE.json's sizes in the same run (device time, CUDA events):
    config 2 (fit loop on 1e6 events), config 4 (toys), config 5 (binned path).  Reported beside the headline;
    parity of each is in tests/ (-m gpu)."""
    from paper_1706_01420_b200 import minimiser
    out = {}
    peaks_hbm = 6650.0
    try:
        peaks_hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass

    def t(fn, steps, warm=2):
        for _ in range(warm):
            fn()
        return timed(torch, fn, steps, stream) / steps

    # config 2: host minimiser loop, 1e6 events (seed 2), floating (mu, sigma, f, k)
    n2 = min(1_000_000, n)
    x2, _, _ = ipa.ipa_toy_generate([2], inp.GEN, -1.0, -1.0, LO, HI, n2)
    x2 = ipa.ipa_events_prepare(x2, LO, HI)
    ws2 = ipa.workspace(n2, 32)
    th0 = inp.as_array(inp.GEN)
    for name, d in inp.FIT_START_SHIFT.items():
        th0[inp.IDX[name]] += d

    def nll_batch_plain(th):                                    # the general-purpose wrapper: tensors allocated per call
        return ipa.ipa_nll_eval(x2, th, LO, HI, ws=ws2, stream=stream)[0].cpu().numpy()
    minimiser.minimise(nll_batch_plain, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    minimiser.minimise(nll_batch_plain, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE)
    wall_plain = time.perf_counter() - t0
    ev = ipa.NllEvaluator(x2, LO, HI, stream=stream)            # the fit loop's evaluator: buffers allocated once

    def nll_batch(th):
        return ev(th)
    minimiser.minimise(nll_batch, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = minimiser.minimise(nll_batch, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE)
    wall = time.perf_counter() - t0

    def grad_batch(th):
        nll, g = ev.gradient(th)
        return nll, g[:, :4]
    minimiser.minimise(nll_batch, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE, grad_batch=grad_batch)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res_a = minimiser.minimise(nll_batch, th0, inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE, grad_batch=grad_batch)
    wall_a = time.perf_counter() - t0
    b9, _ = inp.fd_batch(inp.GEN)
    o9 = torch.empty(9, dtype=torch.float64, device="cuda")
    d9 = t(lambda: ipa.ipa_nll_eval(x2, b9, LO, HI, ws=ws2, stream=stream, out=o9), 200, 10)
    out["config2_fit_1e6_events"] = {
        "wall_s": wall, "wall_s_general_wrapper": wall_plain, "nll_evaluations": res.n_evals, "batched_calls": res.n_calls, "edm": res.edm,
        "nll_evaluations_per_s_wall": res.n_evals / wall, "k9_call_ms_device": d9 * 1e3,
        "nll_evaluations_per_s_device_k9": 9 / d9,
        "fitted": {k: res.par[k] for k in inp.FLOATED}, "errors": {k: res.errors[k] for k in inp.FLOATED},
        "with_analytic_gradient": {"wall_s": wall_a, "evaluations": res_a.n_evals, "calls": res_a.n_calls, "edm": res_a.edm,
                                   "fitted": {k: res_a.par[k] for k in inp.FLOATED}}}

    # config 4: 1000 toys x ~1e5 events generated on the device, one segmented launch
    T = 1000
    seeds = inp.toy_seeds(T)
    cap = 101_000_000
    if n >= 100_000_000:
        xt = torch.empty(cap, dtype=torch.float64, device="cuda")
        wst = ipa.workspace(cap, T)
        holder = {}

        def gen():
            holder["off"] = ipa.ipa_toy_generate(seeds, inp.GEN, 30000.0, 70000.0, LO, HI, cap, ws=wst, x=xt, stream=stream,
                                                 policy=1)[1]
        dg = t(gen, 3, 1)
        off = holder["off"]
        ntot = int(off[-1].item())
        sets = inp.toy_param_sets(T)
        xs = torch.empty(ntot, dtype=torch.float64, device="cuda")
        dprep = t(lambda: ipa.ipa_events_prepare(xt[:ntot], LO, HI, off, out=xs, stream=stream), 5)
        seg = {}
        for pol, tag in ((1, "general_order"), (0, "adaptive_degree")):
            ds = t(lambda: ipa.ipa_nll_eval_segmented(xt, off, sets, LO, HI, ws=wst, stream=stream, policy=pol), 10)
            dss = t(lambda: ipa.ipa_nll_eval_segmented(xs, off, sets, LO, HI, ws=wst, stream=stream, policy=pol), 10)
            cl = core_cells(torch, ipa, xt[:ntot], inp.GEN, pol)      # (the toys' own sets differ from GEN by a fit error)
            deg = cl["degree_full"]
            seg[tag] = {"core_degree": deg, "core_cells": cl, "as_generated_ms": ds * 1e3, "prepared_per_toy_ms": dss * 1e3,
                        "toys_per_s": T / dss, "events_per_s": ntot / dss,
                        "roofline_prepared": alu_roofline(algorithmic_flops(cl["degree_eff"], p_core), ntot, dss,
                                                          {"note": "whole call: 1000-set prologue + segmented kernel + finalize"}),
                        "roofline_as_generated": alu_roofline(algorithmic_flops(deg, p_core), ntot, ds)}
        # generator: issue-slot model: a sub-partition issues one warp instruction per cycle and an
        # FP64 instruction holds the port for two.  Declared per event: signal fraction 0.3 x (bookkeeping Philox 100 +
        # attempts x (Philox 100 + core log G 8 int + (7 + D) FP64 + acceptance exp 15 FP64 + 12 int)) + background 0.7 x
        # (2 Philox 200 + inverse CDF log1p/expm1 ~ 60 FP64 + 20 int); list / refill bookkeeping 10 int.
        deg1 = int(ipa.ipa_core_degree(inp.GEN, LO, HI, policy=1))
        att = 1.11
        cyc = 0.3 * (100 + att * (100 + 8 + 12 + 2 * (7 + deg1 + 15))) + 0.7 * (2 * 100 + 20 + 2 * 60) + 10
        peak_issue = SM_COUNT * 4 * 32 * SM_MAX_HZ
        out["config4_toys"] = {"toys": T, "events": ntot, "generate_ms": dg * 1e3, "generate_events_per_s": ntot / dg,
                               "roofline_toygen": {"bound": "alu", "unit": "thread-issue-cycles/s", "achieved": cyc * ntot / dg,
                                                   "peak": peak_issue, "frac": cyc * ntot / dg / peak_issue,
                                                   "issue_cycles_per_event_declared": cyc, "attempts_per_signal_event": att,
                                                   "note": "peak = 148 SM x 4 schedulers x 32 lanes x 1.965 GHz; FP64 counted twice"},
                               "prepare_per_toy_ms": dprep * 1e3, "segmented_nll": seg}
        del xt, xs
    # config 5: histogram (HBM-bound), 100 x 100 scan, 10 000 Poisson toy histograms
    nbins = 1000
    dh = t(lambda: ipa.ipa_hist_fill(x, LO, HI, nbins, stream=stream), 20)
    counts = ipa.ipa_hist_fill(x, LO, HI, nbins, stream=stream)
    ns, nb, kk = inp.scan_grid(100, 100, n_obs=float(n))
    ws5 = ipa.workspace(0, 10000, nbins)
    dsc = t(lambda: ipa.ipa_binned_nll_scan(counts, LO, HI, inp.GEN, ns, nb, kk, ws=ws5, stream=stream), 20)
    nu = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 2500.0, n - 2500.0, -0.002)
    sd = np.arange(1, 10001, dtype=np.uint64)
    dp = t(lambda: ipa.ipa_poisson_hist_toys(nu, sd, ws=ws5, stream=stream), 20)
    # row f2: CLs for one signal hypothesis on the toy histograms above (statistic of 10 000 x 1000 counts is one
    # HBM pass over 40 MB)
    nu_b0 = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 0.0, float(n), -0.002)
    toys = ipa.ipa_poisson_hist_toys(nu, sd, ws=ws5, stream=stream)
    qobs = ipa.ipa_cls_teststat(counts, nu, nu_b0, ws=ws5, stream=stream)
    dq = t(lambda: ipa.ipa_cls_teststat(toys, nu, nu_b0, ws=ws5, stream=stream), 20)
    qt = ipa.ipa_cls_teststat(toys, nu, nu_b0, ws=ws5, stream=stream)
    dc = t(lambda: ipa.ipa_cls_count_ge(qt, qobs, stream=stream), 20)
    out["cls_f2"] = {"toy_histograms": int(sd.size), "bins": nbins, "teststat_ms": dq * 1e3, "count_ms": dc * 1e3,
                     "teststat_roofline": {"bound": "hbm", "achieved": 4.0 * sd.size * nbins / dq / 1e9, "peak": peaks_hbm,
                                           "unit": "GB/s", "frac": 4.0 * sd.size * nbins / dq / 1e9 / peaks_hbm}}
    # row f3: Gaussian-smeared signal shape on the bin grid feeding the same binned scan
    sig = ipa.ipa_signal_shape(nbins, LO, HI, inp.GEN, ws=ws5, stream=stream)
    dsm = t(lambda: ipa.ipa_gauss_smear(sig, LO, HI, 10.0, stream=stream), 20)
    sm = ipa.ipa_gauss_smear(sig, LO, HI, 10.0, stream=stream)
    dss = t(lambda: ipa.ipa_binned_nll_scan_shape(counts, LO, HI, sm, ns, nb, kk, ws=ws5, stream=stream), 20)
    out["smear_f3"] = {"bins": nbins, "sigma0": 10.0, "smear_ms": dsm * 1e3, "scan_with_smeared_shape_ms": dss * 1e3,
                       "scan_points_per_s": ns.size / dss}
    out["config5_binned"] = {
        "hist_fill_ms": dh * 1e3, "hist_events_per_s": n / dh,
        "hist_roofline": {"bound": "hbm", "achieved": 8.0 * n / dh / 1e9, "peak": peaks_hbm, "unit": "GB/s",
                          "frac": 8.0 * n / dh / 1e9 / peaks_hbm},
        "scan_points": int(ns.size), "scan_ms": dsc * 1e3, "scan_points_per_s": ns.size / dsc,
        # per (point, bin) term: table-driven exp (16) and log (15) of csrc/ipa_fastmath.cuh, nu (2 FMA: 4), n log nu and the
        # two sums (5) -> 40 flops; the call is four launches and three small uploads around a ~60 us kernel: latency-bound
        "roofline_scan": alu_roofline(40.0, ns.size * nbins, dsc, {"unit_of_work": "(scan point, bin) term",
                                                                   "note": "whole call: shape prologue + shape kernel + 3 small H2D copies + scan kernel"}),
        "poisson_toy_histograms": int(sd.size), "poisson_toys_ms": dp * 1e3, "poisson_draws_per_s": sd.size * nbins / dp}
    return out


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
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=100_000_000, help="events per GPU")
    ap.add_argument("--layout", default="prepared", choices=["prepared", "asis"],
                    help="headline event layout: prepared once by ipa_events_prepare (outside the timed region; its cost "
                         "and the break-even number of calls are in the line) or as generated")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import paper_1706_01420_b200 as ipa
    from paper_1706_01420_b200 import sharding

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
    batch9, _ = inp.fd_batch(P1)

    # workload: config 3 -- ONE seeded dataset of world x n events (seed 3) generated on the device by the method's
    # generator; rank r owns the contiguous shard of slots [r n, (r+1) n) (ipa_options.first_slot): weak scaling,
    # no data-path collective on the events, the K partial sums are combined in rank order inside the step
    x_asis, _, _ = ipa.ipa_toy_generate([3], P1, -1.0, -1.0, LO, HI, n, first_slot=rank * n)
    x_prep = torch.empty_like(x_asis)
    wsp = torch.empty(ipa.ipa_prepare_workspace_bytes(n, 0), dtype=torch.uint8, device="cuda")

    def step_prep():
        ipa.ipa_events_prepare(x_asis, LO, HI, out=x_prep, ws=wsp, stream=stream)
    step_prep()                                                 # one-off preparation, outside the headline's timed region
    x = x_prep if args.layout == "prepared" else x_asis
    p_core = float(((x_asis >= P1["mu"] - P1["a"] * P1["sigma"]) & (x_asis <= P1["mu"] + P1["a2"] * P1["sigma"]))
                   .double().mean().item())
    ws = ipa.workspace(n, 32)
    out1 = torch.empty(1, dtype=torch.float64, device="cuda")
    out9 = torch.empty(9, dtype=torch.float64, device="cuda")
    st1 = torch.empty(1, dtype=torch.int32, device="cuda")
    st9 = torch.empty(9, dtype=torch.int32, device="cuda")
    total = {}
    torch.cuda.synchronize()

    POL = 1  # general-order path: no half-integer shortcut in the headline (reading D2)

    def step_k1(arr=None):
        ipa.ipa_nll_eval(x if arr is None else arr, P1, LO, HI, ws=ws, stream=stream, out=out1, status=st1, policy=POL)
        if dist:
            total["nll"] = sharding.combine_nll(out1)           # 8 K bytes all-gathered over NCCL, added in rank order

    def step_k9(arr=None):
        ipa.ipa_nll_eval(x if arr is None else arr, batch9, LO, HI, ws=ws, stream=stream, out=out9, status=st9, policy=POL)

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
    nll_total = float(total["nll"].item()) if dist else float(out1.item())

    # prologue alone (same kernel, same arguments, through ipa_norm): the streaming kernel's average launch
    # duration is the step minus this, launch gaps included on the kernel's side
    norm_out = (torch.empty(1, dtype=torch.float64, device="cuda"), torch.empty(1, dtype=torch.float64, device="cuda"),
                torch.empty(1, dtype=torch.int32, device="cuda"))

    def prologue_gpu_time(params, out, reps=20, replays=10):
        """Device time of the prologue alone: `reps` launches captured in a CUDA graph and replayed, so that the Python /
        ctypes cost of a launch (~20 us, as long as the kernel itself) does not leave the GPU idle between them."""
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            ipa.ipa_norm(params, LO, HI, ws=ws, stream=side, out=out, policy=POL)
            side.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                for _ in range(reps):
                    ipa.ipa_norm(params, LO, HI, ws=ws, stream=torch.cuda.current_stream(), out=out, policy=POL)
            g.replay()
            side.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(side)
            for _ in range(replays):
                g.replay()
            e1.record(side)
            side.synchronize()
        stream.wait_stream(side)
        return e0.elapsed_time(e1) * 1e-3 / (reps * replays)
    dt_pro = prologue_gpu_time(P1, norm_out)
    t_step = dt / args.steps
    cells = core_cells(torch, ipa, x_asis, P1, POL)
    degree = cells["degree_full"]
    # Horner work per core event: the cell polynomials on the prepared layout, the full polynomial as generated
    deg_prep, deg_asis = cells["degree_eff"], float(degree)
    deg_x = deg_prep if args.layout == "prepared" else deg_asis
    deg_other = deg_asis if args.layout == "prepared" else deg_prep
    flops = algorithmic_flops(deg_x, p_core)

    def local_step_time(fn, steps, warm=2):
        for _ in range(warm):
            fn()
        return timed(torch, fn, steps, stream) / steps

    def k1_local(arr):
        ipa.ipa_nll_eval(arr, P1, LO, HI, ws=ws, stream=stream, out=out1, status=st1, policy=POL)
    # kernel time from a loop without the collective (identical to the step at N = 1)
    t_local = t_step if not dist else local_step_time(lambda: k1_local(x), args.steps)
    t_kernel = max(t_local - dt_pro, 1e-9)

    extras = {"p_core": p_core, "core_degree": degree, "core_cells": cells, "prologue_ms": dt_pro * 1e3, "nll_kernel_ms": t_kernel * 1e3,
              "build_hash": build_hash()}
    if not args.no_extras and rank == 0:
        k9steps = max(5, args.steps // 8)
        # one-off preparation (stable counting sort on a coarse bin index) and what it buys
        d_prep = local_step_time(step_prep, 10)
        other = x_asis if args.layout == "prepared" else x_prep
        oname = "asis" if args.layout == "prepared" else "prepared"
        d_other = local_step_time(lambda: k1_local(other), args.steps)
        t_asis, t_prepared = (d_other, t_local) if args.layout == "prepared" else (t_local, d_other)
        extras["prepare"] = {"ms": d_prep * 1e3, "events_per_s": n / d_prep,
                             "hbm_gbs": 24.0 * n / d_prep / 1e9,
                             "algorithmic_bytes_per_event": 24, "note": "two reads (count, scatter) + one write of 8 B",
                             "break_even_calls_k1": d_prep / max(t_asis - t_prepared, 1e-12),
                             "single_call_with_prepare_ms": (d_prep + t_prepared) * 1e3}
        extras[f"roofline_{oname}"] = alu_roofline(algorithmic_flops(deg_other, p_core), n, max(d_other - dt_pro, 1e-9),
                                                   {"layout": oname, "call_ms": d_other * 1e3})
        extras["roofline_asis_plus_prepare_single_call"] = alu_roofline(flops, n, d_prep + t_prepared,
                                                                        {"note": "new data every call: prepare + one NLL"})
        dt9 = local_step_time(step_k9, k9steps)
        # (the four displaced shapes of the batch have cells of their own; their degrees equal the base set's here)
        W9 = 5 * shape_stage_flops(deg_x, p_core) + 9 * MEMBER_STAGE_FLOPS
        W9o = 5 * shape_stage_flops(deg_other, p_core) + 9 * MEMBER_STAGE_FLOPS
        extras["k9_gradient_batch"] = {"ms_per_call": dt9 * 1e3, "event_sets_per_s": 9 * n / dt9, "events_per_s": n / dt9,
                                       "nll_calls_per_s": 9 / dt9}
        extras["roofline_k9"] = alu_roofline(W9, n, max(dt9 - dt_pro, 1e-9),
                                             {"note": "central-difference batch over (mu, sigma, f, k): 5 shape stages + 9 member "
                                                      "stages per event", "flops_per_event_set": W9 / 9})
        dto9 = local_step_time(lambda: step_k9(other), k9steps)
        extras[f"roofline_k9_{oname}"] = alu_roofline(W9o, n, max(dto9 - dt_pro, 1e-9), {"layout": oname, "call_ms": dto9 * 1e3})

        def step_adaptive():
            ipa.ipa_nll_eval(x, P1, LO, HI, ws=ws, stream=stream, out=out1, status=st1, policy=0)
        dta = local_step_time(step_adaptive, args.steps)
        extras["k1_adaptive_degree_half_integer_shortcut"] = {"ms_per_call": dta * 1e3, "events_per_s": n / dta}

        def step_p2():
            ipa.ipa_nll_eval(x, inp.P2, LO, HI, ws=ws, stream=stream, out=out1, status=st1, policy=0)
        dtp = local_step_time(step_p2, args.steps)
        extras["k1_general_shape_P2"] = {"ms_per_call": dtp * 1e3, "events_per_s": n / dtp}

        def step_t1():
            ipa.ipa_nll_eval(x, inp.T1, LO, HI, ws=ws, stream=stream, out=out1, status=st1, policy=POL)
        dtt = local_step_time(step_t1, args.steps)
        extras["k1_student_t_core_f4"] = {"ms_per_call": dtt * 1e3, "events_per_s": n / dtt}
        k1_local(x)
        # row f1: analytic gradient in one pass, beside the K = 9 finite-difference batch it replaces
        dtg = local_step_time(lambda: ipa.ipa_nll_grad_eval(x, P1, LO, HI, ws=ws, stream=stream, policy=POL), k9steps)
        extras["f1_analytic_gradient"] = {"ms_per_call": dtg * 1e3, "events_per_s": n / dtg,
                                          "speedup_vs_k9_finite_differences": dt9 / dtg}
        extras["roofline_grad"] = alu_roofline(gradient_flops(int(deg_x), p_core), n, dtg, {"note": "whole call (prologue with "
                                               "normalisation derivatives + gradient kernel)"})
        if world == 1:
            extras.update(other_rows(torch, ipa, x_asis, ws, stream, n, p_core))
        # FP64 peak probe (DFMA chains), for the roofline denominator
        iters = 200000
        ipa.ipa_fp64_peak_probe(1000)
        tp = timed(torch, lambda: ipa.ipa_fp64_peak_probe(iters), 1, stream)
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        extras["fp64_dfma_probe_tflops"] = sms * 8 * 256 * 8 * 2.0 * iters / tp / 1e12
    if dist:
        dist.barrier()
    k1_local(x)
    torch.cuda.synchronize()

    # end to end through the public API with HOST buffers: H2D of the events + D2H of the result inside the
    # timed region, events in the order the host holds them (as generated; no device-side preparation)
    e2e = None
    if rank == 0 or dist:
        xh = torch.empty(n, dtype=torch.float64, pin_memory=True)
        xh.copy_(x_asis)
        xd = torch.empty(n, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        ipa.nll_host(xh, P1, LO, HI, x_dev=xd, ws=ws, policy=POL)
        e2e_steps = max(2, min(args.steps, 5))
        if dist:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            r = ipa.nll_host(xh, P1, LO, HI, x_dev=xd, ws=ws, policy=POL)
        torch.cuda.synchronize()
        de = time.perf_counter() - t0
        if dist:
            t = torch.tensor([de], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            de = t.item()
        e2e = {"value": world * n * e2e_steps / de, "unit": UNIT, "h2d_bytes_per_step": 8 * n + 88,
               "d2h_bytes_per_step": 8, "steps": e2e_steps, "nll": float(r[0]), "layout": "as generated",
               "timer": "host wall clock around copy + call + result read"}
        del xd

    if rank != 0:
        return
    achieved = flops * n / t_kernel / 1e12
    peak = FP64_PEAK_NOMINAL / 1e12
    traffic, traffic_note = measured_traffic(n)
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_note,
                "kernel": "ipa_nll_kernel<false,false,true>", "kernel_ms": t_kernel * 1e3,
                "kernel_time_source": "CUDA events: step time minus the prologue's device time (20 prologue launches captured "
                                      "in a CUDA graph and replayed: no host gaps)",
                "frac_whole_step": flops * n / t_local / 1e12 / peak,
                "peak_source": "DESIGN.md section 6: 148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no "
                               "FP64 entry); measured DFMA-chain probe in fp64_dfma_probe_tflops",
                "flops_per_event_set": flops, "p_core": p_core, "core_degree": degree,
                "work_history": {
                    "note": "the declared work is what THIS build executes per event (ncu: FP64 instructions x 2 within 10 %); "
                            "every round-2 cut of it (table-driven exp / log, a-priori degree 27, cell polynomials of degree "
                            "13-14, one-step reduction, 1024-entry exp table) lowered W and the time, the time by less: the "
                            "integer half of the instruction stream did not shrink with it",
                    "r01_flops_per_event_set": 98.87, "r01_kernel_ms": 0.4045,
                    "frac_if_measured_against_r01_flops": 98.87 * n / t_kernel / 1e12 / peak},
                "hbm": {"achieved_gbs": 8.0 * n / t_kernel / 1e9, "algorithmic_bytes_per_event": 8}}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        roofline["hbm"]["peak_gbs"] = peaks["hbm_gbs"]
        roofline["hbm"]["frac"] = roofline["hbm"]["achieved_gbs"] / peaks["hbm_gbs"]
        roofline["hbm"]["peak_note"] = "of measured"
    except Exception:
        roofline["hbm"]["peak_gbs"] = 6650.0
        roofline["hbm"]["frac"] = roofline["hbm"]["achieved_gbs"] / 6650.0
        roofline["hbm"]["peak_note"] = "of fallback"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config 3: 1e8 fp64 events per GPU on [5000,5600] from the Ipatia+exp model (device generator, "
                                   "seed 3, one dataset of n_gpus x 1e8 events sharded contiguously), one NLL evaluation per "
                                   "step (prologue + streaming kernel" + (" + all-gather of the partial sums" if dist else "") +
                                   "), K=1, general-order degree policy",
                       "events": n * world, "events_per_gpu": n, "K": 1,
                       "layout": args.layout + (" (stable counting sort on a coarse bin index by ipa_events_prepare, once, before "
                                                "the timed region: cost and break-even in 'prepare'; as-generated order in "
                                                "roofline_asis)" if args.layout == "prepared" else ""),
                       "l2": "input (8 B x events) larger than L2, no flush needed",
                       "multi_gpu": "contiguous event shards of one dataset, K partial sums all-gathered and added in rank order"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": 2 * args.steps, "roofline": roofline, "nll": nll_total}
    line.update(extras)
    if not args.no_cpu_baseline and world == 1:
        cores = os.cpu_count() or 1
        allc, one = cpu_baseline(xh.numpy(), P1, cores)
        line["cpu_baseline"] = allc
        line["cpu_baseline_1core"] = one
        line["parity"] = {"gpu_nll": nll_total, "oracle_nll": allc["nll"],
                          "rel_diff": abs(nll_total - allc["nll"]) / abs(allc["nll"]), "tolerance": 1e-10,
                          "note": "same 1e8 seed-3 events: device sum over the prepared layout against the oracle's threaded "
                                  "pairwise sums over the as-generated order (single-thread oracle on the same events: "
                                  "tests/test_gpu_parity.py::test_full_size_sampled)"}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
