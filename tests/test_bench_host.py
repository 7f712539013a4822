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
    out = bench.roofline_step(cfg, peaks, calls)
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


def test_kernel_work_counts_every_backward_stream_once():
    """g is read by k_tc_bwd_gz and re-read by k_tc_bwd_du; the call's algorithmic bytes count it once,
    so the two kernels' byte counts must add up to the call's plus the gz re-read that only exists between them."""
    for name in ("c1", "c2", "c3"):
        cfg = I.CONFIGS[name]
        s = 2
        gzb, _ = bench.kernel_alg_work("k_tc_bwd_gz", cfg)
        dub, _ = bench.kernel_alg_work("k_tc_bwd_du", cfg)
        call = bench.alg_bytes_per_token(cfg)["backward"] * cfg.n_tokens
        assert gzb + dub == call
        _, f1 = bench.kernel_alg_work("k_tc_bwd_gz", cfg)
        _, f2 = bench.kernel_alg_work("k_tc_bwd_du", cfg)
        assert f1 + f2 == bench.alg_flops_per_token(cfg)["backward"] * cfg.n_tokens


def test_stiefel_flops_and_step_stats():
    d = 2048
    # NS-5 24 d r^2 -> 0.20 / 0.81 / 3.22 / 12.9 GFLOP at r = 64 / 128 / 256 / 512
    for r, gf in ((64, 0.20), (128, 0.81), (256, 3.22), (512, 12.9)):
        assert bench.stiefel_alg_flops(d, r, "ns5") / 1e9 == pytest.approx(gf, rel=0.02)
    assert bench.stiefel_alg_flops(d, 64, "qr") == pytest.approx(7 * d * 64 * 64 + 64 ** 3 / 3.0)
    st = bench.step_time_stats([1.0, 3.0, 2.0])
    assert st == {"median": 2.0, "max": 3.0, "min": 1.0}
    assert bench.FFMA_TFLOPS == pytest.approx(74.4, abs=0.1)


def test_default_headline_is_the_rvq_config():
    cfg, desc = bench.workload(bench.HEADLINE)
    assert desc.startswith("c3:") and cfg.rvq_levels == 2 and cfg.rvq_k == 4096 and cfg.d == 2048
