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
# the roofline numerator is the LESSER of the table count and what ncu counts as executed.  Since the
# linear phase term is folded into the spline records and a knot inside a warp tile costs one pass, the kernel executes
# fewer FP64 operations than the table: ncu (profiles/r01_dense_c2_final_ncu.txt) counts 2 x 6.683e11 DFMA + 6.16e10 DADD
# + 6.15e10 DMUL = 1.4598e12 FLOPs per config-2 launch against 1.6038e12 from the table.
EXECUTED_OVER_TABLE_FLOPS = 1.4598e12 / 1.6038e12
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 lanes x 2 x max SM clock


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


def oracle_sample(cfg, n_bins=None):
    """Builds the workload with the oracle's injections and returns (workload, sample walker indices)."""
    from oracle import likelihood as L
    from oracle.constants import load_model_table
    from paper_2005_01827_b200 import workloads as W
    table = load_model_table()
    wl = W.build(cfg, lambda p, f, S: L.template(table, p, f, S), n_bins=n_bins)
    B = wl["params"].shape[0]
    idx = [0, B // 2, B - 1] if cfg == 2 else ([0, 1] if cfg == 0 else [0])
    return table, wl, idx


def time_oracle(table, wl, idx):
    from oracle import likelihood as L
    t0 = time.perf_counter()
    for b in idx:
        L.loglike_parts(table, wl["params"][b], wl["freqs"], wl["data"], wl["psd"], wl["S"], wl["t0"])
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the oracle, as it stands, on this box's host cores (one process, numpy)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    table, wl, idx = oracle_sample(args.config)
    B, N, S = wl["params"].shape[0], wl["freqs"].size, wl["S"]
    for _ in range(args.warmup):
        time_oracle(table, wl, idx[:1])
    t = sum(time_oracle(table, wl, idx) for _ in range(args.steps))
    value = len(idx) * args.steps / t
    sample = f"walkers {idx} of the batch per step (one per injection group), full grid, single numpy process"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "logL/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, B, N, S), "sample": sample},
        "cpu_baseline": {"value": value, "unit": "logL/s", "cores": 1, "kind": "oracle", "sample": sample},
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


def run_sparse_isolation(args):
    """BASELINE.json configs[3]: B = 16384 parameter sets, steps a1-a5 only (mbhl_sparse), no dense stage."""
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
    # algorithmic HBM bytes per parameter set: knots + y written once and read once by the
    # spline kernel, coefficient records written once
    bytes_set = 6 * S * (8 + 64) * 2 + 6 * (S - 1) * 256
    hbm, hbm_src = _hbm_peak()
    spline_bytes = B * (6 * S * (8 + 64) + 6 * (S - 1) * 256)       # what k_spline itself reads and writes
    achieved = spline_bytes / (stage[2] * 1e-3) / 1e9
    fp64_peak = _fp64_probe(torch, M, dev)
    flops_set = 1730.0 * 6 * S                                       # ~1600 + 130 FLOPs per knot
    print(json.dumps({
        "metric": "parameter sets/sec (sparse stage only)", "value": B / (ms * 1e-3), "unit": "sets/s", "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[3]: B={B} parameter sets (config-0 priors, M_T log-uniform 1e5-1e8), 6 modes x S={S} knots; "
                               "per-walker constants + PhenomHM + response + spline coefficients, no dense stage",
                   "l2": "outputs larger than L2 (coefficient records %.1f GB per step)" % (B * 6 * (S - 1) * 256 / 1e9),
                   "stage_ms": {k: float(v) for k, v in zip(("consts", "sparse", "spline"), stage[:3])}},
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_spline", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
                     "traffic": None, "peak_source": hbm_src, "algorithmic_bytes_per_launch": spline_bytes,
                     "whole_stage": {"hbm_bound_ms": B * bytes_set / (hbm * 1e9) * 1e3, "fp64_bound_ms": B * flops_set / (fp64_peak * 1e12) * 1e3,
                                     "measured_ms": ms, "fp64_peak_tflops": fp64_peak}}}))
    M.mbhl_free(ctx)


def run_dense_sweep(args):
    """BASELINE.json configs[4]: dense grid N x batch B sweep, random priors with M_T log-uniform [1e5, 1e8]; one line per point."""
    torch, M, dev, local = _device_setup()
    from paper_2005_01827_b200 import workloads as W
    S = 1024
    fp64_peak = _fp64_probe(torch, M, dev)
    hbm, _ = _hbm_peak()
    all_params = W.sparse_batch(4096, seed_offset=4)
    rng = np.random.default_rng(W.SEED0 + 4)
    for logn in (16, 18, 20, 22, 23):
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
        for B in (1, 16, 256, 1024, 4096):
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
            flops = (FLOP_PER_PAIR * pairs + FLOP_PER_BIN * bins) * min(1.0, EXECUTED_OVER_TABLE_FLOPS)
            fp64_ms = flops / (fp64_peak * 1e12) * 1e3
            hbm_ms = (80.0 * N * max(1, (B + 7) // 8) + B * 6 * (S - 1) * 256) / (hbm * 1e9) * 1e3
            print(json.dumps({"metric": METRIC, "value": B / (ms * 1e-3), "unit": "logL/s", "n_gpus": 1, "steps": steps, "ms_per_step": ms,
                              "dtype": "f64", "data": "synthetic",
                              "config": {"workload": f"BASELINE.json configs[4] point: N=2^{logn} bins ending at 0.1 Hz, B={B}, S={S}",
                                         "active_pairs_per_step": pairs, "active_bins_per_step": bins,
                                         "stage_ms": {k: float(v) for k, v in zip(("consts", "sparse", "spline", "dense", "reduce"), stage)}},
                              "roofline": {"bound": "alu" if fp64_ms >= hbm_ms else "hbm", "dense_fp64_bound_ms": fp64_ms, "dense_hbm_bound_ms": hbm_ms,
                                           "frac": max(fp64_ms, hbm_ms) / stage[3], "frac_of_step": max(fp64_ms, hbm_ms) / ms,
                                           "fp64_peak_tflops": fp64_peak},
                              "finite": bool(torch.isfinite(logL).all().item())}), flush=True)
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


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2005_01827_b200 import binding as M
    from paper_2005_01827_b200 import build as mbuild
    from paper_2005_01827_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
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
    if rank > 0:   # each rank gets its own walkers around the same injections (weak scaling)
        rng = np.random.default_rng(W.SEED0 + 1000 + rank)
        params_np = params_np * (1.0 + 1e-4 * rng.standard_normal(params_np.shape) * (np.arange(11) == 0))
    t = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=dev)
    ctx = M.mbhl_init(t(wl["freqs"]), t(wl["data"]), t(wl["psd"]), sparse_points=S, t0=wl["t0"], max_batch=B, device=local)
    params = t(params_np)
    logL = torch.empty(B, dtype=torch.float64, device=dev)
    params_pin = torch.from_numpy(params_np.copy()).pin_memory()
    logL_pin = torch.empty(B, dtype=torch.float64).pin_memory()

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
        M.mbhl_loglike(ctx, params, logL)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = M.mbhl_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    M.mbhl_stage_times(ctx)                 # resets the per-call event ring: the mean below covers the timed steps only
    barrier()
    e0.record()
    for _ in range(args.steps):
        M.mbhl_loglike(ctx, params, logL)
    e1.record()
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    launches = M.mbhl_launch_count(ctx) - launches0
    stage = np.array(M.mbhl_stage_times(ctx)) * args.steps       # mean over the timed steps (CUDA events on the launch stream)
    pairs, bins = M.mbhl_last_work(ctx)
    # ---- end to end: host buffers, H2D + D2H inside the timed region ----
    M.mbhl_loglike_host(ctx, params_pin, logL_pin)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        M.mbhl_loglike_host(ctx, params_pin, logL_pin)     # synchronous: returns after the D2H copy landed
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    clocks = sampler.stop()
    assert np.array_equal(logL_pin.numpy(), logL.cpu().numpy())

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
    value = world * B * args.steps / (ms_total * 1e-3)
    dense_ms = stage[3] / args.steps
    flops = (FLOP_PER_PAIR * pairs + FLOP_PER_BIN * bins) * min(1.0, EXECUTED_OVER_TABLE_FLOPS)
    achieved = flops / (dense_ms * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm_bytes = 80.0 * bins          # weighted data + weights + frequency, if nothing were reused across walkers
    out = {
        "metric": METRIC, "value": value, "unit": "logL/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, B, N, S), "walkers_per_gpu": B,
                   "l2": "inputs larger than L2 (0.34 GB weighted data + 1.6 GB spline coefficients per step vs 126 MB L2)",
                   "active_pairs_per_step": pairs, "active_bins_per_step": bins,
                   "stage_ms": {k: float(v / args.steps) for k, v in zip(("consts", "sparse", "spline", "dense", "reduce"), stage)}},
        "e2e": {"value": world * B * args.steps / e2e_s, "unit": "logL/s", "h2d_bytes_per_step": int(B * 11 * 8),
                "d2h_bytes_per_step": int(B * 8)},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_dense", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                     "frac": achieved / fp64_peak, "peak_nominal": NOMINAL_FP64_TFLOPS, "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                     # dram__bytes_read.sum + dram__bytes_write.sum of one k_dense launch, from the committed ncu --set full capture
                     "traffic": 2.04e9 if args.config == 2 else None, "traffic_source": "profiles/r01_dense_c2_final_ncu.txt (bytes per launch)",
                     "peak_source": "DFMA-chain probe measured in this run (nominal 148 SM x 64 lanes x 2 x 1.965 GHz = %.1f)" % NOMINAL_FP64_TFLOPS,
                     "algorithmic_flops_per_launch": flops, "dense_ms": dense_ms,
                     "hbm_bound_ms_if_no_reuse": hbm_bytes / (peaks.get("hbm_gbs", 6650.0) * 1e9) * 1e3},
    }
    if args.cpu_baseline:
        table, owl, idx = oracle_sample(args.config)
        tcpu = time_oracle(table, owl, idx)
        out["cpu_baseline"] = {"value": len(idx) / tcpu, "unit": "logL/s", "cores": 1, "kind": "oracle",
                               "sample": f"walkers {idx} of the batch (one per injection group), full grid, {tcpu:.1f} s"}
    print(json.dumps(out))
    M.mbhl_free(ctx)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=(0, 1, 2, 3, 4),
                    help="BASELINE.json config; 0-2 are likelihood workloads (2 = default bench line), 3 = sparse-stage isolation, "
                         "4 = dense N x B sweep (one JSON line per point)")
    ap.add_argument("--sampler", action="store_true", help="time the parallel-tempered stretch-move ensemble (SURVEY 8(f).2) on the config-2 data")
    ap.add_argument("--batch", type=int, default=0, help="config 3 only: number of parameter sets (default 16384)")
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.config > 2:
            raise SystemExit("--impl reference times the likelihood configs 0-2")
        run_reference(args)
    elif args.sampler:
        run_sampler(args)
    elif args.config == 3:
        run_sparse_isolation(args)
    elif args.config == 4:
        run_dense_sweep(args)
    else:
        if int(os.environ.get("WORLD_SIZE", "1")) > 1 or args.gpus > 1:
            args.cpu_baseline = args.cpu_baseline and int(os.environ.get("RANK", "0")) == 0 and int(os.environ.get("WORLD_SIZE", "1")) == 1
        run_ours(args)


if __name__ == "__main__":
    main()
