"""Host arithmetic of bench.py (no GPU): the algorithmic work per token that the roofline fractions divide by, the
whole-config roofline, and the job-level throughput formula.  Expected values are SURVEY.md section 8(d)'s table
(flop/token, B/token per call and config), which follows from PAPER.md:73-78 Eq. 1-2 and P:94."""
import sys, os
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import pytest

import bench
from paper_2606_05484_b200 import inputs as I

# (config, call) -> (flop/token, B/token); backward is the headline one: full, dB off (2*d*ra less than with dB)
TABLE = {
    ("c1", "encode"): (262144, 2304), ("c1", "decode"): (393216, 2308), ("c1", "backward"): (1310720 - 2 * 1024 * 64, 6660),
    ("c2", "encode"): (655360, 2064), ("c2", "decode"): (262144, 2068), ("c2", "backward"): (786432 - 2 * 1024 * 64, 6292),
    ("c3", "encode"): (5242880, 4104), ("c3", "decode"): (1572864, 4108), ("c3", "backward"): (5242880 - 2 * 2048 * 128, 12812),
}


@pytest.mark.parametrize("name,call", sorted(TABLE))
def test_algorithmic_work_per_token(name, call):
    cfg = I.CONFIGS[name]
    flops, nbytes = TABLE[(name, call)]
    assert bench.alg_flops_per_token(cfg)[call] == flops
    assert bench.alg_bytes_per_token(cfg)[call] == nbytes


def test_roofline_step_arithmetic():
    cfg = I.CONFIGS["c1"]
    peaks = {"hbm": 8000.0, "bf16": 2250.0, "src": "test"}
    calls = {"mapl_encode": 10.0, "mapl_decode": 10.0, "mapl_codec_backward": 30.0, "mapl_codec_backward_decode_side": 20.0}
    out = bench.roofline_step(cfg, peaks, 0.15, 3, calls)
    N = cfg.n_tokens
    t = [max(b * N / 8000e9, f * N / 2250e12) * 1e6 for f, b in (TABLE[("c1", c)] for c in ("encode", "decode", "backward"))]
    assert out["t_roof_us_per_boundary"] == pytest.approx(sum(t), abs=0.01)
    assert out["measured_us_per_boundary"] == 50.0            # the decode-side-only variant is not part of the sum
    assert out["frac"] == pytest.approx(sum(t) / 50.0, abs=1e-3)
    assert out["nominal"]["frac"] == out["frac"]              # same peaks here
    assert 22.5 < sum(t) < 23.5                               # c1 total 23.1 us at nominal peaks


def test_job_tokens_per_second_is_whole_job():
    # 3 boundaries x 16384 tokens per rank-step, 4 ranks, 10 steps in 2 ms
    assert bench.job_tokens_per_second(3 * 16384, 4, 10, 2.0) == pytest.approx(3 * 16384 * 4 * 10 / 2e-3)
