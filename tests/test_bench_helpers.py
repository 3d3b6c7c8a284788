"""Host-side logic of bench.py (no GPU): roofline numerator bookkeeping, oracle sample choice, rank spawning arguments."""
import importlib.util
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_numerator_is_the_lesser_of_table_and_executed():
    b = load_bench()
    pairs, bins = 1000 * 128, 300 * 128
    # everything on the fast path, no wasted lanes: executed = 98 per pair + 29.75 per bin < table 113 / 40
    counts = (1000, 0, 0, 0, 300)
    flops, table, execd = b.dense_numerator(pairs, bins, counts)
    assert table == 113.0 * pairs + 40.0 * bins
    assert execd == 128.0 * (98.0 * 1000 + 29.75 * 300)
    assert flops == execd < table
    # a kernel that evaluated many out-of-band lanes (gated calls) cannot inflate the numerator beyond the table
    wasteful = (1000, 5000, 0, 0, 300)
    flops2, table2, execd2 = b.dense_numerator(pairs, bins, wasteful)
    assert execd2 > table2 and flops2 == table2
    # single-bin evaluations count one bin on one lane
    assert b.executed_flops((0, 0, 0, 10, 0)) == 105.0 * 10


def test_traffic_table_points_at_committed_profiles():
    b = load_bench()
    for cfg, (nbytes, src) in b.DENSE_TRAFFIC.items():
        assert nbytes > 0 and os.path.exists(os.path.join(ROOT, src.split(" ")[0])), src


def test_host_core_count_and_workload_name():
    b = load_bench()
    assert 1 <= b.host_cores() <= (os.cpu_count() or 1)
    assert "configs[2]" in b.workload_name(2, 1024, 4197160, 1024)


def test_stage_dict_names_the_fused_kernel_and_drops_the_retired_slot():
    # mbhl_stage_times keeps five slots for layout; slot 2 (the former stand-alone spline kernel) is a zero-length interval
    import bench
    d = bench._stage_dict([0.06, 0.88, 0.007, 58.5, 0.008])
    assert d == {"consts": 0.06, "sparse_spline_fused": 0.88, "dense": 58.5, "reduce": 0.008}
