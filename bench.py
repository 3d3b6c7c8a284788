#!/usr/bin/env python3
"""bench.py - log-likelihoods/s of the batched LISA MBHB likelihood hot path on B200 (fp64).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0|1|2] [--impl ours|reference]

A step = one pass of the whole hot path (per-walker constants, PhenomHM + response on the sparse grid,
spline solve, fused dense interpolation + inner products, final reduction) over one batch of walkers.
Default workload: BASELINE.json configs[2] (B = 1024 walkers, 6 modes, S = 1024, N = 4 197 160 bins), the
configuration the north_star's roofline target is quoted on.  N > 1: one process per GPU (torchrun), data
replicated, walkers sharded - every rank runs its own batch of B walkers, no data-path collective
("scaling": "weak"); the only communication is the max over ranks of the timings.
--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload (rank 0 only).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "log-likelihoods/sec"
FLOP_PER_PAIR = 113.0     # per (walker, bin, active mode)
FLOP_PER_BIN = 40.0       # per (walker, active bin) epilogue
# the roofline numerator is the LESSER of the table count and what the kernel EXECUTES.  The executed
# count is taken per run from the tallies k_dense keeps (mbhl_last_dense_work: evaluator calls, each 4 bins x 32 lanes,
# in band or not) times the FP64 operations of one evaluation as written in csrc/mbhl_dense.cuh:
#   one mode at one bin: 45 DFMA + 4 DADD + 4 DMUL = 98 FLOPs (+1 DMUL when the amplitude is gated); a single-bin evaluation of
#   the global per-bin path (mode_contrib, the longer sincos polynomials): 48 DFMA + 4 DADD + 5 DMUL = 105 FLOPs,
#   epilogue per (walker, bin): 12 DFMA + 3 DMUL + 2.75 DADD (per-lane sums and the shuffle tree, per bin) = 29.75 FLOPs.
# profiles/r02_dense_flop_check.md compares this count with ncu's sm__sass_thread_inst_executed_op_d*_pred_on.
F_EVAL, F_EVAL_GATED, F_LANE, F_EPI = 98.0, 99.0, 105.0, 29.75
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 lanes x 2 x max SM clock
# dram__bytes_read.sum + dram__bytes_write.sum of ONE k_dense launch from the committed `ncu --set full` captures, by config
DENSE_TRAFFIC = {2: (2.0385e9, "profiles/r02_dense_c2_ncu.txt (dram__bytes_read.sum 2.0289 GB + dram__bytes_write.sum 9.6 MB)")}


def _stage_dict(stage):
    """Per-stage milliseconds by name.  Slot 2 of mbhl_stage_times (the former stand-alone spline kernel) is a zero-length
    interval between two back-to-back event records since the spline solve was fused into the sparse kernel: not reported."""
    return {k: float(stage[i]) for i, k in ((0, "consts"), (1, "sparse_spline_fused"), (3, "dense"), (4, "reduce"))}


def executed_flops(counts):
    """FP64 FLOPs k_dense executed, from its own tallies (uniform, gated, per-bin-record calls; lane evaluations; epilogues)."""
    n_uni, n_gat, n_rec, n_lane, n_epi = counts
    return 128.0 * (F_EVAL * n_uni + F_EVAL_GATED * (n_gat + n_rec) + F_EPI * n_epi) + F_LANE * n_lane


def dense_numerator(pairs, bins, counts):
    """(FLOPs for the roofline numerator, table FLOPs, executed FLOPs): the lesser of the two."""
    table = FLOP_PER_PAIR * pairs + FLOP_PER_BIN * bins
    execd = executed_flops(counts)
    return min(table, execd), table, execd


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def workload_name(cfg, B, N, S):
    return f"BASELINE.json configs[{cfg}]: B={B} walkers x 6 PhenomHM modes, S={S} sparse knots/mode, N={N} dense bins, A/E/T"


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


_ORACLE = {}


def _oracle_one(b):
    from oracle import likelihood as L
    wl = _ORACLE["wl"]
    return L.loglike_parts(_ORACLE["table"], wl["params"][b], wl["freqs"], wl["data"], wl["psd"], wl["S"], wl["t0"])[2]


def _oracle_template(args):
    from oracle import likelihood as L
    p, f, S = args
    return L.template(_ORACLE["table"], p, f, S)


class OraclePool:
    """The oracle, as it stands, over all host cores: one walker per worker process (fork; must be created before this
    process touches CUDA).  The workload is built once with the oracle's own injections and inherited by the workers."""

    def __init__(self, cfg):
        import multiprocessing as mp
        from oracle.constants import load_model_table
        from paper_2005_01827_b200 import workloads as W
        self.cores = host_cores()
        _ORACLE["table"] = load_model_table()
        ctx = mp.get_context("fork")
        with ctx.Pool(min(self.cores, 3)) as pool0:     # the injections (up to three templates) in parallel too
            cache = {}

            def tf(p, f, S):
                return cache[tuple(p)]
            # W.build asks for the injection templates one by one: precompute them in parallel from a dry run
            dry = []
            W.build(cfg, lambda p, f, S: (dry.append((p.copy(), f, S)), np.zeros((3, f.size), dtype=np.complex128))[1], with_noise=False)
            for (p, f, S), h in zip(dry, pool0.map(_oracle_template, dry)):
                cache[tuple(p)] = h
            _ORACLE["wl"] = W.build(cfg, tf)
        self.wl = _ORACLE["wl"]
        self.pool = ctx.Pool(self.cores)

    def sample(self, n):
        B = self.wl["params"].shape[0]
        return sorted(set(int(round(v)) for v in np.linspace(0, B - 1, min(n, B))))

    def time(self, idx):
        t0 = time.perf_counter()
        out = self.pool.map(_oracle_one, idx, chunksize=1)
        return time.perf_counter() - t0, out

    def close(self):
        self.pool.terminate()
        self.pool.join()


def run_reference(args):
    """--impl reference: the oracle, as it stands, on this box's host cores (one walker per process, numpy)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pool = OraclePool(args.config)
    wl = pool.wl
    B, N, S = wl["params"].shape[0], wl["freqs"].size, wl["S"]
    idx = pool.sample(min(16, max(3, pool.cores)))
    for _ in range(args.warmup):                # W untimed passes over the same sample, as the contract asks
        pool.time(idx)
    t = sum(pool.time(idx)[0] for _ in range(args.steps))
    pool.close()
    value = len(idx) * args.steps / t
    sample = f"{len(idx)} walkers {idx} of the batch per step (spread over the injection groups), full grid, one walker per process on {pool.cores} cores"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "logL/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, B, N, S), "sample": sample},
        "cpu_baseline": {"value": value, "unit": "logL/s", "cores": pool.cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "logL/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def _device_setup():
    import torch
    from paper_2005_01827_b200 import binding as M
    from paper_2005_01827_b200 import build as mbuild
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    mbuild.build()
    M.lib()
    return torch, M, torch.device("cuda", local), local


def _fp64_probe(torch, M, dev):
    sink = torch.zeros(8, dtype=torch.float64, device=dev)
    blocks, threads, iters = 148 * 8, 256, 20000
    M.mbhl_dfma_probe(blocks, threads, 200, sink)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    M.mbhl_dfma_probe(blocks, threads, iters, sink)
    p1.record()
    torch.cuda.synchronize()
    return 2.0 * blocks * threads * iters * 8 / (p0.elapsed_time(p1) * 1e-3) / 1e12


def _hbm_peak():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback of /opt/skills/guides/B200_PROFILING.md"


def run_sparse_isolation(args, collect=None):
    """BASELINE.json configs[3]: B = 16384 parameter sets, steps a1-a5 only (mbhl_sparse), no dense stage.
    collect: a list that receives the result line instead of stdout (the default run's `also` entry)."""
    torch, M, dev, local = _device_setup()
    from paper_2005_01827_b200 import workloads as W
    S, B = 1024, args.batch or 16384
    freqs = W.grid(1.33, int(0.1 * 1.33 * W.YEAR_JULIAN_S), 0.0)
    N = freqs.size
    ctx = M.mbhl_init(torch.as_tensor(freqs, device=dev), torch.zeros((3, N, 2), dtype=torch.float64, device=dev),
                      torch.ones((3, N), dtype=torch.float64, device=dev), sparse_points=S, max_batch=B, device=local)
    params = torch.as_tensor(W.sparse_batch(B), device=dev)
    M.mbhl_enable_stage_timing(ctx, True)
    for _ in range(max(args.warmup, 3)):
        M.mbhl_sparse(ctx, params, outputs=False)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    M.mbhl_stage_times(ctx)
    launches0 = M.mbhl_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        M.mbhl_sparse(ctx, params, outputs=False)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    stage = M.mbhl_stage_times(ctx)
    launches = M.mbhl_launch_count(ctx) - launches0
    clocks = sampler.stop()
    # algorithmic HBM bytes per parameter set: knots written once, coefficient records written once
    # (the knot values y stay in shared memory)
    bytes_set = 6 * S * 8 + 6 * (S - 1) * 256
    hbm, hbm_src = _hbm_peak()
    k_bytes = B * bytes_set
    achieved = k_bytes / (stage[1] * 1e-3) / 1e9
    fp64_peak = _fp64_probe(torch, M, dev)
    flops_set = 1730.0 * 6 * S                                       # ~1600 + 130 FLOPs per knot
    hbm_ms, fp64_ms = B * bytes_set / (hbm * 1e9) * 1e3, B * flops_set / (fp64_peak * 1e12) * 1e3
    line = ({
        "metric": "parameter sets/sec (sparse stage only)", "value": B / (ms * 1e-3), "unit": "sets/s", "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[3]: B={B} parameter sets (config-0 priors, M_T log-uniform 1e5-1e8), 6 modes x S={S} knots; "
                               "per-walker constants + PhenomHM + response + spline coefficients, no dense stage",
                   "l2": "outputs larger than L2 (coefficient records %.1f GB per step)" % (B * 6 * (S - 1) * 256 / 1e9),
                   "stage_ms": {"consts": float(stage[0]), "sparse_spline_fused": float(stage[1])}},
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "alu" if fp64_ms >= hbm_ms else "hbm", "kernel": "k_sparse_spline",
                     "frac": max(fp64_ms, hbm_ms) / stage[1], "frac_of_step": max(fp64_ms, hbm_ms) / ms,
                     "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac_hbm": achieved / hbm,
                     "traffic": None, "peak_source": hbm_src, "algorithmic_bytes_per_launch": k_bytes,
                     "whole_stage": {"hbm_bound_ms": hbm_ms, "fp64_bound_ms": fp64_ms, "measured_ms": ms, "fp64_peak_tflops": fp64_peak}}})
    M.mbhl_free(ctx)
    if collect is not None:
        collect.append(line)
    else:
        print(json.dumps(line))


def run_dense_sweep(args, collect=None):
    """BASELINE.json configs[4]: dense grid N x batch B sweep, random priors with M_T log-uniform [1e5, 1e8]; one line per point.
    collect: a list that receives the result lines instead of stdout (the default run's `also` entry)."""
    torch, M, dev, local = _device_setup()
    from paper_2005_01827_b200 import workloads as W
    S = 1024
    fp64_peak = _fp64_probe(torch, M, dev)
    hbm, _ = _hbm_peak()
    all_params = W.sparse_batch(4096, seed_offset=4)
    rng = np.random.default_rng(W.SEED0 + 4)
    for logn in ((args.logn,) if args.logn else (16, 18, 20, 22, 23)):
        N = 1 << logn
        df = 0.1 / N
        freqs = (1.0 + np.arange(N, dtype=np.float64)) * df           # N bins ending at 0.1 Hz
        psd = W.scird_psd_aet(freqs)
        f_d, psd_d = torch.as_tensor(freqs, device=dev), torch.as_tensor(psd, device=dev)
        ctx0 = M.mbhl_init(f_d, torch.zeros((3, N, 2), dtype=torch.float64, device=dev), torch.ones((3, N), dtype=torch.float64, device=dev),
                           sparse_points=S, device=local)
        scale_t = (1.0 / df) / (1.33 * W.YEAR_JULIAN_S)             # t_ref was drawn as a fraction of 1.33 yr: same fraction of T_obs = 1/df
        inj = all_params[:1].copy()
        inj[0, 10] *= scale_t
        data = M.mbhl_template(ctx0, torch.as_tensor(inj, device=dev))[0].cpu().numpy() + W.noise(rng, psd, df)
        M.mbhl_free(ctx0)
        ctx = M.mbhl_init(f_d, torch.as_tensor(data, device=dev), psd_d, sparse_points=S, max_batch=4096, device=local)
        M.mbhl_enable_stage_timing(ctx, True)
        for B in ((args.batch,) if args.batch else (1, 16, 256, 1024, 4096)):
            p = all_params[:B].copy()
            p[:, 10] *= scale_t
            params = torch.as_tensor(p, device=dev)
            logL = torch.empty(B, dtype=torch.float64, device=dev)
            for _ in range(3):
                M.mbhl_loglike(ctx, params, logL)
            torch.cuda.synchronize()
            M.mbhl_stage_times(ctx)
            steps = args.steps
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                M.mbhl_loglike(ctx, params, logL)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            stage = M.mbhl_stage_times(ctx)
            pairs, bins = M.mbhl_last_work(ctx)
            counts = M.mbhl_last_dense_work(ctx)
            flops, flops_table, flops_exec = dense_numerator(pairs, bins, counts)
            fp64_ms = flops / (fp64_peak * 1e12) * 1e3
            # HBM lower bound: every walker tile (<= 8 walkers) streams at least its largest walker's bins once (80 B per bin),
            # and every record of an in-band interval is read once
            hbm_ms = (80.0 * bins / min(B, 8) + B * 6 * (S - 1) * 256) / (hbm * 1e9) * 1e3
            line = ({"metric": METRIC, "value": B / (ms * 1e-3), "unit": "logL/s", "n_gpus": 1, "steps": steps, "ms_per_step": ms,
                              "dtype": "f64", "data": "synthetic",
                              "config": {"workload": f"BASELINE.json configs[4] point: N=2^{logn} bins ending at 0.1 Hz, B={B}, S={S}",
                                         "active_pairs_per_step": pairs, "active_bins_per_step": bins,
                                         "stage_ms": _stage_dict(stage)},
                              "roofline": {"bound": "alu" if fp64_ms >= hbm_ms else "hbm", "dense_fp64_bound_ms": fp64_ms, "dense_hbm_bound_ms": hbm_ms,
                                           "frac": max(fp64_ms, hbm_ms) / stage[3], "frac_of_step": max(fp64_ms, hbm_ms) / ms,
                                           "flops_table": flops_table, "flops_executed": flops_exec, "fp64_peak_tflops": fp64_peak,
                                           "dense_work_counts": dict(zip(("uniform_calls", "gated_calls", "perbin_record_calls", "lane_evals", "epilogues"), counts))},
                              "finite": bool(torch.isfinite(logL).all().item())})
            if collect is not None:
                collect.append(line)
            else:
                print(json.dumps(line), flush=True)
        M.mbhl_free(ctx)


def run_sampler(args):
    """the parallel-tempered stretch-move ensemble of PAPER.md:193-222 driving the likelihood on
    the device.  10 rungs (geometric ladder of base 2.04807, last rung at infinite temperature, :220-222) x 32 walkers
    (4 walkers for each of the 8 sky modes per temperature, :222) around the 1e6 Msun injection of the config-2 data."""
    torch, M, dev, local = _device_setup()
    from paper_2005_01827_b200 import workloads as W
    state = {}

    def gpu_template(p, f, S):
        if "ctx0" not in state:
            n = f.size
            state["ctx0"] = M.mbhl_init(torch.as_tensor(f, device=dev), torch.zeros((3, n, 2), dtype=torch.float64, device=dev),
                                        torch.ones((3, n), dtype=torch.float64, device=dev), sparse_points=S, device=local)
        h = M.mbhl_template(state["ctx0"], torch.as_tensor(p[None, :].copy(), device=dev))
        torch.cuda.synchronize()
        return h[0].cpu().numpy()

    wl = W.build(2, gpu_template)
    M.mbhl_free(state.pop("ctx0"))
    t = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=dev)
    T, K = 10, 32
    ctx = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=wl["S"], t0=wl["t0"], max_batch=T * K, device=local)
    betas = 2.04807 ** -np.arange(T, dtype=np.float64)
    betas[-1] = 0.0
    inj = wl["injections"][1]
    th0 = inj.copy()
    th0[0], th0[4], th0[10] = np.log(inj[0]), np.log(inj[4]), np.log(inj[10])
    th0[1] = 1.0 / inj[1] if inj[1] > 1.0 else inj[1]
    th0[6], th0[8] = np.cos(inj[6]), np.sin(inj[8])
    rng = np.random.default_rng(W.SEED0 + 5)
    theta = th0 + np.array([1e-5, 1e-4, 1e-4, 1e-4, 1e-3, 1e-3, 1e-3, 1e-3, 1e-3, 1e-3, 1e-7]) * rng.standard_normal((T, K, 11))
    pt = M.mbhl_pt_init(ctx, t(theta), betas, seed=W.SEED0, stretch_a=1.15)
    M.mbhl_pt_step(pt, max(args.warmup, 3))
    torch.cuda.synchronize()
    launches0 = M.mbhl_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    M.mbhl_pt_step(pt, args.steps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    launches = M.mbhl_launch_count(ctx) - launches0
    th, ll, acc, swp = M.mbhl_pt_state(pt, T, K, dev)
    steps_done = max(args.warmup, 3) + args.steps
    print(json.dumps({
        "metric": "log-likelihoods/sec through the parallel-tempered ensemble", "value": T * K / (ms * 1e-3), "unit": "logL/s", "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"PT ensemble {T} rungs x {K} walkers (two half-ensemble stretch moves of {T * K // 2} proposals + one swap sweep per step) "
                               f"on the BASELINE.json configs[2] data (N={wl['freqs'].size}, S={wl['S']}), walkers around the 1e6 Msun injection"},
        "gpu_launches": int(launches), "finite": bool(torch.isfinite(ll).all().item()),
        "acceptance_per_rung": [float(a) / (steps_done * K) for a in acc],
        "swap_fraction_per_pair": [float(x) / (steps_done * K) for x in swp]}))
    M.mbhl_pt_free(pt)
    M.mbhl_free(ctx)


def run_het(args):
    """the heterodyned likelihood variant against the brute-force path on the BASELINE.json configs[2] data.
    The batch keeps config 2's shape (1024 walkers in three groups around the three injections) but the walkers are drawn at
    posterior-like distances from their injection (relative width w; config 2's own 1e-3 is far outside what a heterodyne
    around ONE reference covers): each group is evaluated against its own reference = its injection.  One JSON line per
    (width, number of coarse bins): error against the brute-force logL of the same walkers, and throughput."""
    torch, M, dev, local = _device_setup()
    from paper_2005_01827_b200 import workloads as W
    state = {}

    def gpu_template(p, f, S):
        if "ctx0" not in state:
            n = f.size
            state["ctx0"] = M.mbhl_init(torch.as_tensor(f, device=dev), torch.zeros((3, n, 2), dtype=torch.float64, device=dev),
                                        torch.ones((3, n), dtype=torch.float64, device=dev), sparse_points=S, device=local)
        h = M.mbhl_template(state["ctx0"], torch.as_tensor(p[None, :].copy(), device=dev))
        torch.cuda.synchronize()
        return h[0].cpu().numpy()

    wl = W.build(2, gpu_template)
    M.mbhl_free(state.pop("ctx0"))
    t = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=dev)
    B, N, S = wl["params"].shape[0], wl["freqs"].size, wl["S"]
    ctx = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=S, t0=wl["t0"], max_batch=B, device=local)
    inj = wl["injections"]
    counts = [B - 2 * (B // 3), B // 3, B // 3]
    kn = M.mbhl_sparse(ctx, t(inj), want_coef=False)[0].cpu().numpy()                # knots of every reference's modes
    band = [(kn[i][kn[i][:, 0] > 0, 0].min(), kn[i][:, -1].max()) for i in range(3)]    # lowest f_lo, highest f_hi over the modes
    ev = lambda: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    for width in (1e-7, 1e-6, 1e-5):
        rng = np.random.default_rng(W.SEED0 + 40)
        groups = [t(W.perturb(rng, inj[i], counts[i], width)) for i in range(3)]
        walkers = torch.cat(groups)
        brute = M.mbhl_loglike_parts(ctx, walkers)
        e0, e1 = ev()
        e0.record()
        for _ in range(args.steps):
            M.mbhl_loglike_parts(ctx, walkers)
        e1.record()
        torch.cuda.synchronize()
        brute_ms = e0.elapsed_time(e1) / args.steps
        b_dh, b_hh, b_ll = [x.cpu().numpy() for x in brute]
        for nb in (512, 2048, 8192):
            i0, i1 = ev()
            i0.record()
            hets = [M.mbhl_het_init(ctx, t(inj[i]), W.het_edges(wl["freqs"], nb, band[i][0], band[i][1])) for i in range(3)]
            i1.record()
            torch.cuda.synchronize()
            outs = [M.mbhl_het_loglike(hets[i], groups[i]) for i in range(3)]
            for _ in range(3):
                for i in range(3):
                    M.mbhl_het_loglike(hets[i], groups[i])
            launches0 = M.mbhl_launch_count(ctx)
            e0, e1 = ev()
            e0.record()
            for _ in range(args.steps):
                for i in range(3):
                    M.mbhl_het_loglike(hets[i], groups[i])
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.steps
            launches = M.mbhl_launch_count(ctx) - launches0
            h_dh, h_hh, h_ll = [np.concatenate([o[j].cpu().numpy() for o in outs]) for j in range(3)]
            print(json.dumps({
                "metric": METRIC + " (heterodyned variant)", "value": B / (ms * 1e-3), "unit": "logL/s", "n_gpus": 1, "steps": args.steps,
                "warmup": 3, "ms_per_step": ms, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"BASELINE.json configs[2] data (N={N}, S={S}); B={B} walkers in three groups at relative width {width:g} around "
                                       f"their injection, one reference per group, {nb} coarse bins requested",
                           "walker_width": width, "coarse_bins": nb},
                "gpu_launches": int(launches),
                "brute_force": {"ms_per_step": brute_ms, "value": B / (brute_ms * 1e-3)},
                "speedup_over_brute_force": brute_ms / ms, "summary_ms_per_reference": i0.elapsed_time(i1) / 3.0,
                "error_vs_brute_force": {"max_abs_dlogL": float(np.max(np.abs(h_ll - b_ll))), "median_abs_dlogL": float(np.median(np.abs(h_ll - b_ll))),
                                         "max_rel_hh": float(np.max(np.abs(h_hh - b_hh) / b_hh)),
                                         "max_dh_over_hh": float(np.max(np.abs(h_dh - b_dh) / b_hh))}}), flush=True)
            for h in hets:
                M.mbhl_het_free(h)
    M.mbhl_free(ctx)


def _also_points(args, torch, M, dev, local, fp64_peak):
    """The short BASELINE configs, measured after the headline's timed region and outside it, so that the one JSON line of
    the default run carries them: config 3 (sparse-stage isolation, 5 steps), config 0 (B = 4, N = 2^16, 200 steps) and one
    config-4 point (N = 2^16, B = 1024).  Each entry: ms_per_step, the roofline fraction of its dominant kernel, the bound."""
    from types import SimpleNamespace
    from paper_2005_01827_b200 import workloads as W
    out = {}
    got = []
    run_sparse_isolation(SimpleNamespace(steps=5, warmup=3, batch=0), collect=got)
    r = got[-1]
    out["config3_sparse_isolation"] = {"ms_per_step": r["ms_per_step"], "frac": r["roofline"]["frac"], "bound": r["roofline"]["bound"],
                                       "kernel": "k_sparse_spline", "unit_per_step": "16384 parameter sets"}
    got = []
    run_dense_sweep(SimpleNamespace(steps=20, warmup=3, batch=1024, logn=16), collect=got)
    r = got[-1]
    out["config4_N2^16_B1024"] = {"ms_per_step": r["ms_per_step"], "frac": r["roofline"]["frac"], "bound": r["roofline"]["bound"],
                                  "kernel": "k_dense", "dense_ms": r["config"]["stage_ms"]["dense"]}
    # config 0: latency-bound (four kernels of a few microseconds each); frac is that of k_dense like the headline's
    state = {}

    def gpu_template(p, f, S):
        if "ctx0" not in state:
            n = f.size
            state["ctx0"] = M.mbhl_init(torch.as_tensor(f, device=dev), torch.zeros((3, n, 2), dtype=torch.float64, device=dev),
                                        torch.ones((3, n), dtype=torch.float64, device=dev), sparse_points=S, device=local)
        h = M.mbhl_template(state["ctx0"], torch.as_tensor(p[None, :].copy(), device=dev))
        torch.cuda.synchronize()
        return h[0].cpu().numpy()

    wl = W.build(0, gpu_template)
    M.mbhl_free(state.pop("ctx0"))
    t = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=dev)
    B = wl["params"].shape[0]
    ctx = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=wl["S"], t0=wl["t0"], max_batch=B, device=local)
    params, logL = t(wl["params"]), torch.empty(B, dtype=torch.float64, device=dev)
    M.mbhl_enable_stage_timing(ctx, True)
    for _ in range(10):
        M.mbhl_loglike(ctx, params, logL)
    torch.cuda.synchronize()
    steps, ms, dense = 200, 0.0, 0.0
    M.mbhl_stage_times(ctx)                          # forget the warm-up calls
    for _ in range(steps // 50):                     # the stage-event ring holds 64 calls: read (and reset) it every 50
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(50):
            M.mbhl_loglike(ctx, params, logL)
        e1.record()
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1) / steps
        dense += M.mbhl_stage_times(ctx)[3] * 50 / steps
    pairs, bins = M.mbhl_last_work(ctx)
    flops, _, _ = dense_numerator(pairs, bins, M.mbhl_last_dense_work(ctx))
    out["config0"] = {"ms_per_step": ms, "frac": flops / (dense * 1e-3) / 1e12 / fp64_peak, "bound": "latency (alu roofline of k_dense shown)",
                      "kernel": "k_dense", "dense_ms": dense, "walkers": B, "bins": int(wl["freqs"].size)}
    M.mbhl_free(ctx)
    return out


def run_ours(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cpu = None
    if args.cpu_baseline and rank == 0 and world == 1:
        # the oracle over all host cores on a bounded sample, BEFORE this process touches CUDA (the workers are forked)
        pool = OraclePool(args.config)
        idx = pool.sample(16 if args.config == 2 else 8)
        tcpu, _ = pool.time(idx)
        pool.close()
        cpu = {"value": len(idx) / tcpu, "unit": "logL/s", "cores": pool.cores, "kind": "oracle",
               "sample": f"{len(idx)} walkers {idx} of the batch (spread over the injection groups), full grid, one walker per process, {tcpu:.1f} s"}

    import torch
    import torch.distributed as dist

    from paper_2005_01827_b200 import binding as M
    from paper_2005_01827_b200 import build as mbuild
    from paper_2005_01827_b200 import shard
    from paper_2005_01827_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        mbuild.build()
    if world > 1:
        dist.barrier()
    M.lib()
    strong = args.scaling == "strong" and world > 1

    # ---- workload: grid, PSD, parameters from the seeded generators; injections from the library's own template ----
    state = {}

    def gpu_template(p, f, S):
        if "ctx0" not in state:     # a context on a zero data stream, used only to synthesise the injections
            n = f.size
            state["ctx0"] = M.mbhl_init(torch.as_tensor(f, device=dev), torch.zeros((3, n, 2), dtype=torch.float64, device=dev),
                                        torch.ones((3, n), dtype=torch.float64, device=dev), sparse_points=S, device=local)
        h = M.mbhl_template(state["ctx0"], torch.as_tensor(p[None, :].copy(), device=dev))
        torch.cuda.synchronize()
        return h[0].cpu().numpy()

    wl = W.build(args.config, gpu_template)
    M.mbhl_free(state.pop("ctx0"))
    B, N, S = wl["params"].shape[0], wl["freqs"].size, wl["S"]
    params_np = wl["params"]
    if rank > 0 and not strong:   # weak scaling: each rank gets its own walkers around the same injections
        rng = np.random.default_rng(W.SEED0 + 1000 + rank)
        params_np = params_np * (1.0 + 1e-4 * rng.standard_normal(params_np.shape) * (np.arange(11) == 0))
    t = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=dev)
    ctx = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=S, t0=wl["t0"], max_batch=B, device=local)
    params = t(params_np)
    logL = torch.empty(B, dtype=torch.float64, device=dev)
    params_pin = torch.from_numpy(params_np.copy()).pin_memory()
    logL_pin = torch.empty(B, dtype=torch.float64).pin_memory()
    if strong:
        # strong scaling: ONE batch of B walkers, rows sharded across the ranks by the product's own sharding
        # (paper_2005_01827_b200/shard.py: contiguous row ranges, all_gather of the logL slices over NCCL)
        lo, hi = shard.shard_rows(B, world, rank)

        def step():
            out = shard.sharded_loglike(lambda rows: M.mbhl_loglike(ctx, rows), params)
            logL.copy_(out)

        def step_host():
            M.mbhl_loglike_host(ctx, params_pin[lo:hi], logL_pin[lo:hi])
    else:
        def step():
            M.mbhl_loglike(ctx, params, logL)

        def step_host():
            M.mbhl_loglike_host(ctx, params_pin, logL_pin)     # synchronous: returns after the D2H copy landed

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        v = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(v, op=dist.ReduceOp.MAX)
        return float(v.item())

    # ---- device-resident timing ----
    M.mbhl_enable_stage_timing(ctx, True)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = M.mbhl_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    M.mbhl_stage_times(ctx)                 # resets the per-call event ring: the mean below covers the timed steps only
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    launches = M.mbhl_launch_count(ctx) - launches0
    stage = np.array(M.mbhl_stage_times(ctx)) * args.steps       # mean over the timed steps (CUDA events on the launch stream)
    pairs, bins = M.mbhl_last_work(ctx)
    counts = M.mbhl_last_dense_work(ctx)
    # ---- end to end: host buffers, H2D + D2H inside the timed region ----
    step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_host()
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    clocks = sampler.stop()
    if strong:
        assert np.array_equal(logL_pin.numpy()[lo:hi], logL.cpu().numpy()[lo:hi])
    else:
        assert np.array_equal(logL_pin.numpy(), logL.cpu().numpy())

    # ---- the same step replayed from a CUDA graph (one launch per step instead of four kernels and a memset) ----
    graph_ms = None
    if world == 1:
        gs = torch.cuda.Stream()
        with torch.cuda.stream(gs):
            ctx_g = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=S, t0=wl["t0"], max_batch=B, device=local, stream=gs)
            out_g = torch.empty(B, dtype=torch.float64, device=dev)
            for _ in range(3):
                M.mbhl_loglike(ctx_g, params, out_g)
            gs.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=gs):
                M.mbhl_loglike(ctx_g, params, out_g)
            for _ in range(3):
                graph.replay()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            for _ in range(args.steps):
                graph.replay()
            g1.record(gs)
            gs.synchronize()
            graph_ms = g0.elapsed_time(g1) / args.steps
            assert torch.equal(out_g, logL)
            M.mbhl_free(ctx_g)

    # ---- FP64 roofline denominator: DFMA-chain probe timed alone, in this run ----
    sink = torch.zeros(8, dtype=torch.float64, device=dev)
    blocks, threads, iters = 148 * 8, 256, 20000
    M.mbhl_dfma_probe(blocks, threads, 200, sink)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    M.mbhl_dfma_probe(blocks, threads, iters, sink)
    p1.record()
    torch.cuda.synchronize()
    fp64_peak = 2.0 * blocks * threads * iters * 8 / (p0.elapsed_time(p1) * 1e-3) / 1e12

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms_step = ms_total / args.steps
    n_job = B if strong else world * B                      # walkers the whole job evaluates per step
    n_rank = (hi - lo) if strong else B
    value = n_job * args.steps / (ms_total * 1e-3)
    dense_ms = stage[3] / args.steps
    flops, flops_table, flops_exec = dense_numerator(pairs, bins, counts)
    achieved = flops / (dense_ms * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm_bytes = 80.0 * bins          # weighted data + weights + frequency, if nothing were reused across walkers
    traffic, traffic_src = DENSE_TRAFFIC.get(args.config, (None, None)) if not strong else (None, None)
    out = {
        "metric": METRIC, "value": value, "unit": "logL/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, B, N, S), "walkers_per_gpu": n_rank,
                   "sharding": ("one batch, rows sharded by shard.sharded_loglike (all_gather of logL over NCCL)" if strong
                                else "every rank its own batch, data replicated, no data-path collective"),
                   "l2": "inputs larger than L2 (0.34 GB weighted data + 1.6 GB spline coefficients per step vs 126 MB L2)",
                   "active_pairs_per_step": pairs, "active_bins_per_step": bins,
                   "stage_ms": _stage_dict(stage / args.steps)},
        "e2e": {"value": n_job * args.steps / e2e_s, "unit": "logL/s", "h2d_bytes_per_step": int(n_rank * 11 * 8),
                "d2h_bytes_per_step": int(n_rank * 8)},
        "gpu_launches": int(launches),
        "cuda_graph": {"ms_per_step": graph_ms, "note": "the same step captured once and replayed from a CUDA graph (timed separately, not the headline)"},
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_dense", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                     "frac": achieved / fp64_peak, "peak_nominal": NOMINAL_FP64_TFLOPS, "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": "DFMA-chain probe measured in this run (nominal 148 SM x 64 lanes x 2 x 1.965 GHz = %.1f)" % NOMINAL_FP64_TFLOPS,
                     "algorithmic_flops_per_launch": flops, "flops_table": flops_table, "flops_executed": flops_exec,
                     "dense_work_counts": dict(zip(("uniform_calls", "gated_calls", "perbin_record_calls", "lane_evals", "epilogues"), counts)),
                     "numerator": "lesser of the SURVEY 8(d) table count and the count executed (k_dense's own tallies, this run)",
                     "dense_ms": dense_ms,
                     "hbm_bound_ms_if_no_reuse": hbm_bytes / (peaks.get("hbm_gbs", 6650.0) * 1e9) * 1e3},
    }
    if cpu is not None:
        out["cpu_baseline"] = cpu
    M.mbhl_free(ctx)
    if world == 1 and args.config == 2 and args.also:
        out["also"] = _also_points(args, torch, M, dev, local, fp64_peak)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args):
    """python bench.py --gpus N without a launcher: re-run this file under torch.distributed.run, one rank per GPU."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")            # the communicator lines (ranks, NVLS) are evidence the driver reads
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd, env=env))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=(0, 1, 2, 3, 4),
                    help="BASELINE.json config; 0-2 are likelihood workloads (2 = default bench line), 3 = sparse-stage isolation, "
                         "4 = dense N x B sweep (one JSON line per point)")
    ap.add_argument("--variant", default="brute", choices=("brute", "het"),
                    help="het: error-vs-speed table of the heterodyned likelihood variant (SURVEY 8(f).4) on the config-2 data")
    ap.add_argument("--sampler", action="store_true", help="time the parallel-tempered stretch-move ensemble (SURVEY 8(f).2) on the config-2 data")
    ap.add_argument("--batch", type=int, default=0, help="config 3: number of parameter sets (default 16384); config 4: only this batch size")
    ap.add_argument("--logn", type=int, default=0, help="config 4: only the grid with N = 2^logn bins")
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--scaling", default="weak", choices=("weak", "strong"),
                    help="N > 1: weak = every rank its own batch of B walkers; strong = ONE batch sharded across the ranks (shard.py)")
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--no-also", dest="also", action="store_false",
                    help="default run only: skip the short extra configs (3, 0, one config-4 point) reported under the key `also`")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.config > 2:
            raise SystemExit("--impl reference times the likelihood configs 0-2")
        run_reference(args)
    elif args.variant == "het":
        run_het(args)
    elif args.sampler:
        run_sampler(args)
    elif args.config == 3:
        run_sparse_isolation(args)
    elif args.config == 4:
        run_dense_sweep(args)
    else:
        if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
            spawn_ranks(args)
        run_ours(args)


if __name__ == "__main__":
    main()
