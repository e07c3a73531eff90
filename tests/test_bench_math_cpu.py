"""The arithmetic bench.py reports with (-m "not gpu"): the FP32 issue roofline, the mix-weighted ceilings of SURVEY.md §8(d), the
DRAM traffic table it reads from profiles/, and the whole-job throughput formula. Numbers retyped from DESIGN.md §8 / BASELINE.md."""
import importlib.util
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_under_test", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_fp32_issue_peak_is_the_documented_roofline(bench):
    # 148 SMs x 4 schedulers x 32 lanes x 1965 MHz = 37.22 T lane-instructions/s
    assert bench.fp32_issue_peak(1965.0, 148) == pytest.approx(37.22496e12, rel=1e-9)
    assert bench.fp32_issue_peak(1000.0, 1) == 128e9
    # north_star's 40 % on config 3 (19.77 G GP ops) is a call of 1.327 ms
    assert 19_766_828_032 / (0.40 * bench.fp32_issue_peak(1965.0, 148)) * 1e3 == pytest.approx(1.3275, abs=1e-3)
    # and the numbers of BASELINE.md §4: 1.503 ms -> 35.3 %, k_eval 1.119 ms -> 47.5 %
    assert 19_766_828_032 / 1.503e-3 / bench.fp32_issue_peak(1965.0, 148) == pytest.approx(0.353, abs=1e-3)
    assert 19_766_828_032 / 1.119e-3 / bench.fp32_issue_peak(1965.0, 148) == pytest.approx(0.475, abs=1e-3)


def test_mix_ceilings_by_hand(bench):
    # only additions on two variables: "x0 x1 ADD": 3 tokens, 3 issue slots, no MUFU, 2 shared-memory words
    c = bench.mix_ceilings({"LOAD": 2, "ADD": 1})
    assert c["issue_slots_per_gp_op"] == 1.0 and c["issue_ceiling"] == 1.0
    assert c["mufu_ceiling"] is None and c["smem_ceiling"] == pytest.approx(1 / (4 * 2 / 3))
    assert c["ceiling"] == pytest.approx(0.375)
    # one SIN per three tokens: a MUFU instruction on a third of the GP ops: 16 MUFU lanes against 128 -> 3 / 8
    c = bench.mix_ceilings({"CONST": 2, "SIN": 1})
    assert c["mufu_per_gp_op"] == pytest.approx(1 / 3) and c["mufu_ceiling"] == pytest.approx(0.375)
    assert c["issue_ceiling"] == pytest.approx(3 / 4) and c["ceiling"] == pytest.approx(0.375)
    # commands the table has no weight for are left out and counted
    c = bench.mix_ceilings({"ADD": 4, "POW": 3, "TANH": 1})
    assert c["tokens_without_weight"] == 4 and c["issue_ceiling"] == 1.0
    assert bench.mix_ceilings({"POW": 3}) is None
    # every command of the hot path and of the f1 mix has a weight
    for name in ("LOAD", "CONST", "ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP", "DUP", "SWAP", "DEL", "SIGN", "SQUARE", "CUBE"):
        assert name in bench.MIX_WEIGHTS


def test_mix_ceiling_of_config3_is_the_documented_one(bench):
    from paper_2607_06731_b200 import colonies as C
    cfg = C.CONFIGS[3]
    tokens, lengths, _ = C.generate_programs(cfg, 100_000)
    import numpy as np
    ops = tokens.view(np.uint32) & 0xFF
    hist = {C.OP_NAME[int(k)]: int(v) for k, v in zip(*np.unique(ops, return_counts=True))}
    c = bench.mix_ceilings(hist)
    # 1.555 issue slots, 0.238 MUFU, 0.372 words per GP op: ceilings 64.3 % / 52.4 % / 67.1 %, MUFU binds
    assert c["issue_slots_per_gp_op"] == pytest.approx(1.555, abs=0.01)
    assert c["mufu_per_gp_op"] == pytest.approx(0.238, abs=0.003)
    assert c["smem_words_per_gp_op"] == pytest.approx(0.372, abs=0.004)
    assert c["ceiling"] == c["mufu_ceiling"] == pytest.approx(0.524, abs=0.006)


def test_dram_traffic_table_is_read_from_profiles(bench):
    t = bench.dram_traffic_table()
    assert t[(3, "mse", "k_eval")] == 358883840 + 31895040          # profiles/r2_dram_traffic.csv, r2_ncu_config3.md
    assert t[(3, "mse", "k_compile")] == 367928576 + 265106432
    assert (4, "mse", "k_eval") in t and (3, "correlation", "k_eval") in t


def test_job_throughput_is_units_over_the_slowest_rank(bench):
    # one rank, 2 steps of 10 units in 4 ms: 5 units per ms = 5000 per second
    value, ms_max = bench.job_throughput(10, 2, 4.0, 1)
    assert value == pytest.approx(5000.0) and ms_max == 4.0
