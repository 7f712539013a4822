"""Host logic of the seeded input generators (no method arithmetic lives there)."""
import numpy as np

from paper_2606_05484_b200 import inputs as I


def test_bf16_rounding_rne():
    x = np.array([1.0, 1.0 + 2 ** -8, 1.0 + 2 ** -7, 1.0 + 3 * 2 ** -8, -2.5, 0.0, 3.3895314e38], np.float32)
    b = I.f32_to_bf16_bits(x)
    back = I.bf16_bits_to_f32(b)
    # 1 + 2^-8 is a tie -> even (1.0); 1 + 3*2^-8 is a tie -> even (1 + 2^-6)
    assert back[0] == 1.0 and back[1] == 1.0 and back[2] == np.float32(1.0 + 2 ** -7)
    assert back[3] == np.float32(1.0 + 2 ** -6) and back[4] == -2.5 and back[5] == 0.0
    import torch
    t = torch.from_numpy(x).to(torch.bfloat16).view(torch.uint16).numpy()
    assert np.array_equal(t[:6], b[:6])
    r = np.random.default_rng(0).standard_normal(10000).astype(np.float32)
    assert np.array_equal(I.f32_to_bf16_bits(r), torch.from_numpy(r).to(torch.bfloat16).view(torch.uint16).numpy())


def test_boundary_recipe_shapes_and_determinism():
    cfg = I.CONFIGS["c0"].with_tokens(512)
    a = I.make_boundary(cfg, 0); b = I.make_boundary(cfg, 0); c = I.make_boundary(cfg, 1)
    assert np.array_equal(a.H.data, b.H.data) and not np.array_equal(a.H.data, c.H.data)
    assert a.H.data.dtype == np.float32 and a.H.shape == (512, 256)
    assert a.U.shape == (256, 32) and a.C.shape == (2, 256, 32) and a.A.shape == (1024, 16)
    assert np.abs(a.U.f64.T @ a.U.f64 - np.eye(32)).max() < 1e-6
    assert a.tok.min() >= 0 and a.tok.max() < 1024
    # oracle view is the exact promotion of the stored bits
    assert np.array_equal(a.H.f64.astype(np.float32), a.H.data)
    c1 = I.make_boundary(I.CONFIGS["c1"].with_tokens(256), 0)
    assert c1.H.data.dtype == np.uint16 and c1.C is None
    assert np.array_equal(I.f32_to_bf16_bits(c1.H.f64.astype(np.float32)), c1.H.data)
    assert np.abs(c1.B.f64 @ c1.B.f64.T - np.eye(64)).max() < 1e-6     # orthonormal rows


def test_zipf_shares():
    """Zipf(1.1) over 32000 ids: top-1 ~ 14%, top-10 ~ 38% of positions (DESIGN.md input recipe)."""
    tok = I.zipf_tokens(np.random.default_rng(1), 200000, 32000)
    cnt = np.bincount(tok, minlength=32000) / tok.size
    assert 0.13 < cnt[0] < 0.155 and 0.36 < cnt[:10].sum() < 0.40 and 0.58 < cnt[:100].sum() < 0.64
    assert tok.max() < 32000


def test_h_spectrum_is_low_rank_plus_noise():
    b = I.make_boundary(I.CONFIGS["c0"].with_tokens(1024), 0)
    s = np.linalg.svd(b.H.f64, compute_uv=False)
    energy = np.cumsum(s ** 2) / np.sum(s ** 2)
    assert energy[31] > 0.99 and energy[15] < 0.99


def test_stiefel_inputs():
    s = I.make_stiefel(64, d=256, batch=2)
    assert s.U.shape == (2, 256, 64) and s.G.shape == (2, 256, 64)
    assert np.abs(s.U.f64[1].T @ s.U.f64[1] - np.eye(64)).max() < 1e-6
    s2 = I.make_stiefel(64, d=256, batch=2, step=3)
    assert np.array_equal(s.U.data, s2.U.data) and not np.array_equal(s.G.data, s2.G.data)
