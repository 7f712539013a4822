"""GPU parity: the CUDA codec (through the C ABI) against the fp64 oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's: codes bit-exact outside near ties (S5),
relative Frobenius error <= 1e-5 (fp32) / 2e-2 (bf16)."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

from _util import TOL, Dev, compare, desc_of, rel_fro, run_gpu, run_oracle, to_dev, to_np

pytestmark = pytest.mark.gpu


def _roundtrip(bi, **kw):
    gpu = run_gpu(bi, **kw)
    ora, stats = run_oracle(bi, gpu_codes=gpu["codes"], with_H=kw.get("with_H", True))
    errs = compare(gpu, ora, stats, TOL[bi.cfg.act_dtype])
    return gpu, ora, stats, errs


def test_c0_full():
    """configs[0]: tiny codec, fp32, N=4096, RVQ 2x256, anchors V=1024 ra=16."""
    bi = I.make_boundary(I.CONFIGS["c0"], 0)
    gpu, ora, stats, errs = _roundtrip(bi)
    assert stats["excepted"] < 0.02 * 4096 * 2
    print("c0", errs, stats)


@pytest.mark.parametrize("name,n", [("c1", 1000), ("c1", 2048 + 77), ("c2", 1024 + 13), ("c3", 512 + 5)])
def test_reduced_configs(name, n):
    """configs[1..3] at reduced token counts: several tiles plus a ragged tail."""
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n), 0)
    gpu, ora, stats, errs = _roundtrip(bi)
    print(name, n, errs, stats)


@pytest.mark.parametrize("name,n", [("c1", 700), ("c2", 300), ("c0", 999)])
def test_anchor_visible(name, n):
    """A std 1.0 so the anchor term is well above the bf16 spacing of Hhat (S9)."""
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n).with_anchor_std(1.0), 1)
    _roundtrip(bi)


@pytest.mark.parametrize("act", ["f32", "bf16"])
def test_anchor_only(act):
    """Z = 0 => Hhat rows are A[tok] B (S9 anchor-only case)."""
    bi = I.make_generic(3, 333, 128, 32, 0, 0, 500, 24, act, a_std=1.0)
    dev = Dev(bi)
    desc = desc_of(bi)
    dt = mb.act_torch_dtype(desc)
    Z = torch.zeros((333, 32), dtype=dt, device="cuda")
    Hhat = torch.empty((333, 128), dtype=dt, device="cuda")
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    mb.mapl_decode(desc, Z, None, dev.U, None, dev.tok, dev.A, dev.B, Hhat, ws)
    ref = o.decode(np.zeros((333, 32)), bi.U.f64, bi.tok, bi.A.f64, bi.B.f64)
    assert rel_fro(to_np(Hhat), ref) <= TOL[act]


@pytest.mark.parametrize("act", ["f32", "bf16"])
@pytest.mark.parametrize("shape", [
    # (N, d, r, L, K, V, ra)
    (1, 64, 8, 0, 0, 10, 8),
    (65, 72, 24, 2, 37, 50, 16),
    (257, 200, 40, 3, 100, 300, 0),
    (130, 256, 256, 0, 0, 64, 8),     # r == d
    (70, 128, 16, 1, 1, 20, 8),       # K == 1: all codes 0
    (513, 384, 96, 2, 257, 1000, 40),
])
def test_ragged_shapes(act, shape):
    N, d, r, L, K, V, ra = shape
    bi = I.make_generic(N % 97, N, d, r, L, K, V, ra, act)
    gpu, ora, stats, errs = _roundtrip(bi)
    if L and K == 1:
        assert (gpu["codes"] == 0).all()


@pytest.mark.parametrize("shape", [
    # (N, d, r, L, K, V, ra) -- corners of the tensor-core envelope (bf16, d % 128 == 0, r in {64,128,256}, ra in {0,64,128})
    (600, 8192, 256, 2, 8192, 1000, 128),   # longest projection chain, largest codebook
    (300, 128, 64, 0, 0, 100, 0),           # smallest d, no anchor, no RVQ
    (1000, 4096, 128, 4, 128, 500, 64),     # smallest codebook the path takes, four levels
    (150, 1024, 64, 8, 256, 200, 128),      # eight levels (the maximum), anchor wider than the payload
    (259, 2048, 256, 0, 0, 300, 64),        # two ragged tiles, RVQ off at r = 256
])
def test_tc_envelope_corners(shape):
    N, d, r, L, K, V, ra = shape
    bi = I.make_generic(40 + N % 13, N, d, r, L, K, V, ra, "bf16")
    _roundtrip(bi)


def test_identity_at_full_rank_no_anchor():
    """r = d, RVQ off, no anchor: Hhat = H up to rounding."""
    bi = I.make_generic(5, 200, 64, 64, 0, 0, 1, 0, "f32")
    gpu = run_gpu(bi)
    assert rel_fro(gpu["Hhat"], bi.H.f64) <= 1e-5


def test_empty_batch():
    bi = I.make_generic(7, 0, 64, 16, 2, 8, 10, 8, "f32")
    gpu = run_gpu(bi)
    assert gpu["Hhat"].shape == (0, 64)
    assert np.all(gpu["dU"] == 0.0) and np.all(gpu["dA"] == 0.0)


@pytest.mark.parametrize("act", ["f32", "bf16"])
def test_accumulate_and_decode_side_only(act):
    bi = I.make_generic(11, 300, 128, 32, 2, 64, 100, 16, act)
    base = run_gpu(bi)
    acc = run_gpu(bi, accumulate=True)          # outputs pre-filled with 1.0
    for k in ("dU", "dA", "dB"):
        assert rel_fro(acc[k] - 1.0, base[k]) <= 5 * TOL[act], k
    # H = NULL: decode-side term only (S8)
    gpu = run_gpu(bi, with_H=False)
    ora, stats = run_oracle(bi, gpu_codes=gpu["codes"], with_H=False)
    compare(gpu, ora, stats, TOL[act])
    assert gpu["dH"] is None


def test_decode_from_z_equals_decode_from_codes():
    bi = I.make_generic(13, 400, 256, 64, 3, 128, 200, 32, "bf16")
    a = run_gpu(bi, use_codes_for_decode=True)
    b = run_gpu(bi, use_codes_for_decode=False)   # uses the bf16-rounded zhat
    assert np.array_equal(a["codes"], b["codes"])
    assert rel_fro(b["Hhat"], a["Hhat"]) <= 2e-2


def test_c1_full_size_one_boundary():
    """configs[1] at full size (N=16384): every output against the oracle."""
    bi = I.make_boundary(I.CONFIGS["c1"], 0)
    gpu, ora, stats, errs = _roundtrip(bi, want_dB=False)
    print("c1 full", errs)


# ---------------------------------------------------------------- fused tcgen05 projection + RVQ kernel

def _with_codebook(bi, C64):
    return dataclasses.replace(bi, C=I.store(C64, "f32"))


def test_tc_rvq_duplicate_codewords_take_the_lowest_index():
    """Tensor-core envelope (bf16, d=256, r=64, K=256).  Level 0: every codeword identical (each k is
    a candidate: the exhaustive fp32 fallback must return index 0).  Level 1: the codebook holds each
    codeword twice (k and k+128): the lower copy must win (S4)."""
    bi = I.make_generic(21, 300, 256, 64, 2, 256, 100, 0, "bf16")
    C = bi.C.f64.copy()
    C[0, :, :] = C[0, 0, :]
    C[1, 128:, :] = C[1, :128, :]
    bi = _with_codebook(bi, C)
    gpu = run_gpu(bi)
    assert (gpu["codes"][:, 0] == 0).all()
    assert (gpu["codes"][:, 1] < 128).all()
    ora, stats = run_oracle(bi, gpu_codes=gpu["codes"])
    compare(gpu, ora, stats, TOL["bf16"])


def test_tc_rvq_planted_codewords_are_recovered():
    """z = C0[k0] + C1[k1] exactly representable on the span of U: codes = (k0, k1), no near ties."""
    bi = I.make_generic(22, 256, 256, 64, 2, 128, 50, 0, "bf16", cb_std=(4.0, 0.25))
    rng = np.random.default_rng(5)
    k0, k1 = rng.integers(0, 128, 256), rng.integers(0, 128, 256)
    Z = bi.C.f64[0][k0] + bi.C.f64[1][k1]
    H = I.store(Z @ bi.U.f64.T, "bf16")           # bf16 rounding of H perturbs z by ~2^-9 relative
    bi = dataclasses.replace(bi, H=H)
    gpu = run_gpu(bi)
    assert np.array_equal(gpu["codes"][:, 0], k0)
    assert np.array_equal(gpu["codes"][:, 1], k1)


def test_tc_rvq_candidate_list_full_only_under_the_early_threshold():
    """One near-copy of a vector w + 2u in every 32-codeword piece (64 pieces, so every scan warp sees more
    pieces within the margin of the running minimum than its candidate list holds), and w itself in the
    LAST piece.  Tokens near w: the list is full until the last piece tightens the threshold, the pieces
    left out lie above the final threshold, and the answer is K-5 without the exhaustive pass.  Tokens
    near w + 2u: the near-copies really are within the final margin (exhaustive pass).  Both against the
    oracle under the near-tie rule S5.  Found at c3: one such token after 8 Stiefel steps made one warp
    re-score all K=4096 codewords (encode 260 -> 2990 us)."""
    K, r, n = 2048, 64, 336
    bi = I.make_generic(29, n, 256, r, 1, K, 100, 0, "bf16", cb_std=(1.0,))
    rng = np.random.default_rng(11)
    C = bi.C.f64.copy()
    w = rng.standard_normal(r)
    u = rng.standard_normal(r)
    u /= np.linalg.norm(u)
    for j in range(K // 32):
        C[0, 32 * j + 3] = w + 2.0 * u + 2e-2 * rng.standard_normal(r)   # score spread ~1e-2: far above fp32 noise, far below the margin (~0.15)
    C[0, K - 5] = w
    Z = np.where((np.arange(n) % 3 == 0)[:, None], w + 2.0 * u, w)[:, :] + 0.02 * rng.standard_normal((n, r))
    bi = dataclasses.replace(_with_codebook(bi, C), H=I.store(Z @ bi.U.f64.T, "bf16"))
    gpu, ora, stats, errs = _roundtrip(bi)
    near_w = np.arange(n) % 3 != 0
    assert (gpu["codes"][near_w, 0] == K - 5).all()
    assert (gpu["codes"][~near_w, 0] % 32 == 3).all()


@pytest.mark.parametrize("r,K,L", [(64, 128, 1), (128, 512, 3), (256, 1024, 2), (64, 4096, 2)])
def test_tc_rvq_envelope_shapes(r, K, L):
    bi = I.make_generic(23 + r % 7, 200 + r, 512, r, L, K, 300, 64, "bf16")
    gpu, ora, stats, errs = _roundtrip(bi)
    assert stats["forced"] <= stats["excepted"]


def test_c2_full_size_one_boundary():
    """configs[2] at full size (N=16384, the launch configuration bench.py times): every output
    against the oracle, RVQ codes under the near-tie rule S5."""
    bi = I.make_boundary(I.CONFIGS["c2"], 0)
    gpu, ora, stats, errs = _roundtrip(bi, want_dB=False)
    print("c2 full", errs, stats)


def _sample_idx(N, seed=7):
    rng = np.random.default_rng(seed)
    return np.unique(np.concatenate([np.arange(0, 40), np.arange(N - 40, N), np.arange(100, 130),
                                     np.arange(N // 2 - 4, N // 2 + 36), rng.integers(0, N, 150)]))


def _check_sampled_tokens(bi, gpu, U64, idx):
    """per-token outputs (codes under S5, Zhat, Hhat, gz, dH) of the sampled tokens against the oracle run on those
    tokens with projector U64; whole-sample Frobenius norm AND worst row."""
    from _util import ROW_TOL, max_row_err
    H, g = bi.H.f64[idx], bi.g.f64[idx]
    Z = o.project(H, U64)
    res, n_exc, n_forced, bad = o.follow_codes(Z, bi.C.f64, gpu["codes"][idx])
    assert int(bad.sum()) == 0, f"non-admissible RVQ codes: {int(bad.sum())} (excepted {n_exc}, forced {n_forced})"
    assert np.array_equal(gpu["codes"][idx], res["codes"])
    Hhat = o.decode(res["Zhat"], U64, bi.tok[idx], bi.A.f64, bi.B.f64)
    bw = o.backward(g, H, res["Zhat"], U64, bi.tok[idx], bi.A.f64, bi.B.f64, want_dB=False)
    for k, ref in (("Zq", res["Zhat"]), ("Hhat", Hhat), ("gz", bw["gz"]), ("dH", bw["dH"])):
        e, er = rel_fro(gpu[k][idx], ref), max_row_err(gpu[k][idx], ref)
        assert np.isfinite(gpu[k]).all() and e <= TOL["bf16"], f"{k}: {e:.3e}"
        assert er <= ROW_TOL["bf16"], f"{k}: worst row {er:.3e}"
    return n_exc, n_forced


def test_c3_full_size_every_output():
    """configs[3] at full size (N=32768: two waves of CTA pairs, as bench.py launches it), EVERY output against the
    oracle run on all 32768 tokens: the per-token ones (codes under S5, Zhat, Hhat, gz, dH; whole tensor and worst
    row) and the N-reductions dU and dA through the launch geometry bench.py times (k_tc_bwd_du<pair>, 144-CTA
    token split, TMA reduce-add).  The oracle pass is ~6e11 fp64 flop: tens of seconds on the box's cores."""
    cfg = I.CONFIGS["c3"]
    bi = I.make_boundary(cfg, 0)
    gpu, ora, stats, errs = _roundtrip(bi, want_dB=False)
    print("c3 full", errs, stats)
    assert errs["dU"] <= TOL["bf16"] and errs["dA"] <= TOL["bf16"]
    # tokens absent from tok have zero dA rows, at any size
    absent = np.setdiff1d(np.arange(cfg.vocab), bi.tok)
    assert not gpu["dA"][absent].any()


def test_c3_shaped_rvq_off_full_size_dU_dA():
    """The c3 shape with RVQ off (L = 0, r = 256, d = 2048, N = 32768): dU and dA of the plain projection codec through
    the same backward launch geometry, against the oracle (the decode-side term then uses the bf16 wire payload Z)."""
    import dataclasses as dc
    cfg = dc.replace(I.CONFIGS["c3"], rvq_levels=0, rvq_k=0, cb_std=())
    bi = I.make_boundary(cfg, 1)
    gpu, ora, stats, errs = _roundtrip(bi, want_dB=False)
    print("c3 L=0 full", errs)


@pytest.mark.parametrize("name", ["c3", "c2"])
@pytest.mark.parametrize("boundary", [1, 2])
def test_sampled_parity_after_ten_gpu_stiefel_steps(name, boundary):
    """Data-dependent paths on NON-pristine state: boundaries 1 and 2 at full size, after the projector has taken 10
    GPU training steps (encode, decode, backward, Stiefel step with G = dU / N, reading S12, re-pack) -- the state in
    which the RVQ candidate-list cliff of round 1 appeared.  Then codes (S5), Zhat, Hhat, gz, dH of sampled tokens
    against the oracle run with the GPU's projector U_10; the projector must still be orthonormal to 1e-5."""
    cfg = I.CONFIGS[name]
    bi = I.make_boundary(cfg, boundary)
    dev = Dev(bi)
    desc = desc_of(bi)
    N, d, r, L = cfg.n_tokens, cfg.d, cfg.r, cfg.rvq_levels
    act = torch.bfloat16
    pack = mb.alloc_workspace(mb.mapl_param_pack_bytes(desc))
    desc.param_pack = pack.data_ptr()
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    st_ws = mb.alloc_workspace(mb.mapl_stiefel_workspace_bytes(d, r, 1))
    U = dev.U.clone().unsqueeze(0).contiguous()
    codes = torch.empty((N, L), dtype=torch.int32, device="cuda")
    Zq = torch.empty((N, r), dtype=act, device="cuda")
    Hhat = torch.empty((N, d), dtype=act, device="cuda")
    gz = torch.empty((N, r), dtype=act, device="cuda")
    dH = torch.empty((N, d), dtype=act, device="cuda")
    dU = torch.empty((1, d, r), dtype=torch.float32, device="cuda")
    dA = torch.empty((cfg.vocab, cfg.anchor_rank), dtype=torch.float32, device="cuda")
    mb.mapl_pack_params(desc, U[0], dev.B, dev.C, pack)

    def fwd_bwd():
        mb.mapl_encode(desc, dev.H, U[0], dev.C, Zq, codes, ws)
        mb.mapl_decode(desc, None, codes, U[0], dev.C, dev.tok, dev.A, dev.B, Hhat, ws)
        mb.mapl_codec_backward(desc, dev.g, dev.H, None, codes, U[0], dev.C, dev.tok, dev.A, dev.B, gz, dU[0], dA,
                               None, dH, False, ws)
    for _ in range(10):
        fwd_bwd()
        mb.mapl_stiefel_step(U, dU, 1e-2 / N, mb.MAPL_RETRACT_NS, 5, None, st_ws)
        mb.mapl_pack_params(desc, U[0], None, None, pack)
    fwd_bwd()
    torch.cuda.synchronize()
    U10 = to_np(U[0])
    assert np.linalg.norm(U10.T @ U10 - np.eye(r)) <= 1e-5
    assert rel_fro(U10, bi.U.f64) > 1e-4           # the projector did move
    gpu = dict(codes=to_np(codes), Zq=to_np(Zq), Hhat=to_np(Hhat), gz=to_np(gz), dH=to_np(dH))
    n_exc, n_forced = _check_sampled_tokens(bi, gpu, U10, _sample_idx(N, seed=11 + boundary))
    print(name, boundary, "excepted", n_exc, "forced", n_forced)


def test_tc_rvq_eight_levels_with_halving_codebooks():
    """L = 8 (the ABI's maximum) with the codebook scale halving per level: the residual shrinks ~2x per level while
    the absolute error of z stays, so the last levels are where a z that is not fp32-accurate (a two-term bf16 split of
    U is 2^-17) would leave the S5 tolerance.  Every level's code must stay admissible."""
    bi = I.make_generic(33, 900, 1024, 64, 8, 256, 100, 0, "bf16", cb_std=tuple(2.0 ** (-l) for l in range(8)))
    gpu, ora, stats, errs = _roundtrip(bi)
    print("L=8", stats, errs)


def test_tc_rvq_tight_codebook():
    """A k-means-like tight codebook: codewords = a common large offset plus small spread, so that D << ||c||^2 and
    the expanded form 0.5||c||^2 - rho.c cancels heavily: the exact re-scoring must still decide like the
    direct form sum (rho - c)^2 of the oracle."""
    bi = I.make_generic(34, 700, 512, 128, 2, 512, 100, 0, "bf16", cb_std=(1.0, 0.5))
    rng = np.random.default_rng(12)
    C = bi.C.f64.copy()
    # the projected activations have entries of size ~sqrt(d/r...) ~ O(1); give both the data and the codewords a
    # common offset 40x larger than the spread
    off = 40.0 * rng.standard_normal(128)
    C[0] = off[None, :] + C[0]
    Z = off[None, :] + 1.5 * rng.standard_normal((700, 128))
    bi = dataclasses.replace(_with_codebook(bi, C), H=I.store(Z @ bi.U.f64.T, "bf16"))
    gpu, ora, stats, errs = _roundtrip(bi)
    print("tight", stats, errs)


def test_projector_only_repack_equals_full_repack():
    """mapl_pack_params with codebooks == NULL re-packs U/B only and keeps the codebook section: after a
    projector update the encode / decode results equal those of a complete re-pack, bit for bit."""
    bi = I.make_generic(31, 700, 512, 128, 2, 512, 300, 64, "bf16")
    dev = Dev(bi)
    desc = desc_of(bi)
    pack = mb.alloc_workspace(mb.mapl_param_pack_bytes(desc))
    desc.param_pack = pack.data_ptr()
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    N, d, r, L = bi.cfg.n_tokens, bi.cfg.d, bi.cfg.r, bi.cfg.rvq_levels
    mb.mapl_pack_params(desc, dev.U, dev.B, dev.C, pack)
    U2 = to_dev(I.make_generic(32, 8, 512, 128, 0, 0, 10, 0, "bf16").U)      # another orthonormal projector

    def run():
        codes = torch.empty((N, L), dtype=torch.int32, device="cuda")
        Hhat = torch.empty((N, d), dtype=torch.bfloat16, device="cuda")
        mb.mapl_encode(desc, dev.H, U2, dev.C, None, codes, ws)
        mb.mapl_decode(desc, None, codes, U2, dev.C, dev.tok, dev.A, dev.B, Hhat, ws)
        torch.cuda.synchronize()
        return codes.cpu().numpy(), Hhat.float().cpu().numpy()

    mb.mapl_pack_params(desc, U2, None, None, pack)           # projector-only re-pack
    a = run()
    mb.mapl_pack_params(desc, U2, dev.B, dev.C, pack)         # complete re-pack
    b = run()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    # and the projector did change the result
    mb.mapl_pack_params(desc, dev.U, dev.B, dev.C, pack)
    codes0 = torch.empty((N, L), dtype=torch.int32, device="cuda")
    mb.mapl_encode(desc, dev.H, dev.U, dev.C, None, codes0, ws)
    torch.cuda.synchronize()
    assert not np.array_equal(codes0.cpu().numpy(), a[0])


@pytest.mark.parametrize("name,n", [("c1", 5000), ("c2", 3000), ("c3", 4000)])
def test_repeatability_of_atomic_free_outputs(name, n):
    """Every output that involves no atomics (codes, Zhat, Hhat, gz, dH) must be bit-identical from run to
    run: a race between the TMA / MMA / epilogue roles or between the two CTAs of a pair would show up here."""
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n), 2)
    dev = Dev(bi)
    ref = run_gpu(bi, dev=dev, want_dB=False)
    for _ in range(8):
        out = run_gpu(bi, dev=dev, want_dB=False)
        for k in ("codes", "Zq", "Hhat", "gz", "dH"):
            if ref[k] is not None:
                assert np.array_equal(ref[k], out[k]), f"{k} differs between runs"
        # the atomically accumulated gradients may differ in the last bits only
        for k in ("dU", "dA"):
            assert rel_fro(out[k], ref[k]) <= 1e-5


def test_cluster_of_two_pairs_multicast_path():
    """MAPL_NQ=2: decode and backward-gz run as clusters of two CTA pairs that share every parameter tile by TMA
    multicast (opt-in).  The switch is read once per process, so this runs in a subprocess:
    reduced c1 / c3 against the oracle."""
    import os, subprocess, sys
    code = ("import sys; sys.path.insert(0, 'tests'); import test_parity_codec as T; "
            "T.test_reduced_configs('c1', 2125); T.test_reduced_configs('c3', 517); T.test_anchor_visible('c2', 300); print('ok')")
    env = dict(os.environ, MAPL_NQ="2")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and "ok" in out.stdout, out.stdout[-2000:] + out.stderr[-2000:]


def test_tc_rvq_candidate_list_spills_to_the_overflow_area():
    """12 near-copies of w in 12 different 32-codeword pieces of ONE scan thread's share (even pieces): more groups
    inside the final margin than the shared-memory list holds (8 at r = 64), fewer than list + overflow area (16), so
    the answer comes from the overflow entries without the exhaustive pass.  Codes against the oracle under S5; the
    true nearest copy is decided by the exact pass."""
    K, r, n = 2048, 64, 336
    bi = I.make_generic(36, n, 256, r, 1, K, 100, 0, "bf16", cb_std=(1.0,))
    rng = np.random.default_rng(13)
    C = bi.C.f64.copy()
    w = rng.standard_normal(r) * 1.5
    spots = [64 * j + 5 for j in range(3, 15)]                 # pieces 6, 8, ..., 28: all even
    for k in spots:
        C[0, k] = w + 2e-3 * rng.standard_normal(r)            # spread far below the margin (~0.1), far above fp32 noise
    Z = w[None, :] + 0.02 * rng.standard_normal((n, r))
    bi = dataclasses.replace(_with_codebook(bi, C), H=I.store(Z @ bi.U.f64.T, "bf16"))
    gpu, ora, stats, errs = _roundtrip(bi)
    assert np.isin(gpu["codes"][:, 0], spots).all()


@pytest.mark.parametrize("scale", [1e-6, 3e3])
def test_tc_rvq_extreme_activation_scale(scale):
    """Residuals far smaller / larger than the codebook: the per-token power-of-two scale of the fp16 operand leaves the
    range in which the norm step's a' is an fp16 power of two (tiny h: `hard` tokens, exhaustive exact pass) or sits at
    its other end (large h).  Codes must still be the oracle's."""
    bi = I.make_generic(37, 200, 256, 64, 2, 256, 100, 0, "bf16", cb_std=(1.0, 0.5))
    H = I.store(bi.H.f64 * scale, "bf16")
    bi = dataclasses.replace(bi, H=H)
    gpu = run_gpu(bi)
    ora, stats = run_oracle(bi, gpu_codes=gpu["codes"])
    assert stats["bad"] == 0, stats
    assert np.array_equal(gpu["codes"], ora["codes"])
