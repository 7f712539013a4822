"""Sender-side anchor centring (Eq. 1 in full): mapl_center_table +
mapl_encode_centered through the C ABI against the fp64 oracle (oracle.project with A_s, B_s, then the
same RVQ / near-tie rule as the hot path)."""
import numpy as np
import pytest
import torch

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

from _util import TOL, desc_of, rel_fro, to_dev, to_np

pytestmark = pytest.mark.gpu


def _centered_encode(bi, a_std=1.0):
    """GPU: T = A_s (B_s U), then encode_centered.  The sender's anchor factors are the boundary's A, B
    rescaled so that the centring term is comparable to h (an error in it cannot hide)."""
    c = bi.cfg
    desc = desc_of(bi)
    act = mb.act_torch_dtype(desc)
    A_s = (bi.A.f64 * (a_std / max(bi.A.f64.std(), 1e-30))).astype(np.float32)
    B_s = bi.B.f64.astype(np.float32)
    dA, dB, dU, dH, dtok = to_dev(A_s), to_dev(B_s), to_dev(bi.U), to_dev(bi.H), to_dev(bi.tok)
    dC = to_dev(bi.C) if bi.C is not None else None
    T = torch.empty((c.vocab, c.r), dtype=torch.float32, device="cuda")
    cws = mb.alloc_workspace(mb.mapl_center_workspace_bytes(desc))
    mb.mapl_center_table(desc, dA, dB, dU, T, cws)
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    N, r, L = c.n_tokens, c.r, c.rvq_levels
    Zq = torch.empty((N, r), dtype=act, device="cuda")
    codes = torch.empty((N, L), dtype=torch.int32, device="cuda") if L > 0 else None
    mb.mapl_encode_centered(desc, dH, dtok, T, dU, dC, Zq, codes, ws)
    torch.cuda.synchronize()
    return A_s.astype(np.float64), B_s.astype(np.float64), to_np(T), to_np(Zq), (to_np(codes) if L > 0 else None)


@pytest.mark.parametrize("name,n", [("c0", 999), ("c1", 1500), ("c2", 1037), ("c3", 517)])
def test_centered_encode_matches_oracle(name, n):
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n), 3)
    A_s, B_s, T, Zq, codes = _centered_encode(bi)
    U = bi.U.f64
    # the table itself: T = A_s (B_s U) (fp32 GEMMs)
    assert rel_fro(T, A_s @ (B_s @ U)) <= 1e-5
    Z = o.project(bi.H.f64, U, bi.tok, A_s, B_s)
    # centring really changes z
    assert rel_fro(o.project(bi.H.f64, U), Z) > 1e-2
    tol = TOL[bi.cfg.act_dtype]
    if bi.cfg.rvq_levels == 0:
        assert rel_fro(Zq, Z) <= tol
        return
    res, n_exc, n_forced, bad = o.follow_codes(Z, bi.C.f64, codes)
    assert int(bad.sum()) == 0, f"non-admissible codes: {int(bad.sum())} (excepted {n_exc}, forced {n_forced})"
    assert np.array_equal(codes, res["codes"])
    assert rel_fro(Zq, res["Zhat"]) <= tol


def test_centered_encode_bf16_ragged_shape_rounds_once():
    """bf16 activations at a shape outside the tensor-core envelope (fp32 SIMT kernels), RVQ off, with an anchor much
    larger than the centred z: T[tok] must be subtracted from the fp32 accumulator BEFORE the single bf16 rounding
    (mapl.h); rounding U^T h to bf16 first would leave an error of 2^-9 |U^T h|, far above the centred z's own
    rounding."""
    bi = I.make_generic(35, 333, 200, 40, 0, 0, 300, 24, "bf16", a_std=1.0)
    c = bi.cfg
    desc = desc_of(bi)
    # H = A_s[tok] B_s + small: the centred z is ~50x smaller than U^T h
    A_s = (30.0 * bi.A.f64).astype(np.float32)
    B_s = bi.B.f64.astype(np.float32)
    small = bi.H.f64 * 0.1
    H = I.store(A_s.astype(np.float64)[bi.tok] @ B_s.astype(np.float64) + small, "bf16")
    dA, dB, dU, dH, dtok = to_dev(A_s), to_dev(B_s), to_dev(bi.U), to_dev(H), to_dev(bi.tok)
    T = torch.empty((c.vocab, c.r), dtype=torch.float32, device="cuda")
    cws = mb.alloc_workspace(mb.mapl_center_workspace_bytes(desc))
    mb.mapl_center_table(desc, dA, dB, dU, T, cws)
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    Zq = torch.empty((c.n_tokens, c.r), dtype=torch.bfloat16, device="cuda")
    mb.mapl_encode_centered(desc, dH, dtok, T, dU, None, Zq, None, ws)
    torch.cuda.synchronize()
    Z = o.project(H.f64, bi.U.f64, bi.tok, A_s.astype(np.float64), B_s.astype(np.float64))
    Zu = o.project(H.f64, bi.U.f64)
    assert np.linalg.norm(Zu) > 10 * np.linalg.norm(Z)          # the offset dominates the uncentred projection
    assert rel_fro(to_np(Zq), Z) <= 4e-3                        # one bf16 rounding of the centred z (2^-9 per entry)


def test_zero_anchor_reduces_to_plain_encode():
    bi = I.make_boundary(I.CONFIGS["c2"].with_tokens(700), 4)
    desc = desc_of(bi)
    c = bi.cfg
    dU, dH, dtok, dC = to_dev(bi.U), to_dev(bi.H), to_dev(bi.tok), to_dev(bi.C)
    T = torch.zeros((c.vocab, c.r), dtype=torch.float32, device="cuda")
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    a = torch.empty((c.n_tokens, c.rvq_levels), dtype=torch.int32, device="cuda")
    b = torch.empty_like(a)
    mb.mapl_encode_centered(desc, dH, dtok, T, dU, dC, None, a, ws)
    mb.mapl_encode(desc, dH, dU, dC, None, b, ws)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


@pytest.mark.parametrize("name,n", [("c0", 999), ("c1", 1500), ("c2", 1037), ("c3", 517)])
def test_center_backward_matches_oracle(name, n):
    """dA_s, dB_s and the dU correction of the centring term against oracle.center_backward, for a Gaussian
    gz in the activation dtype; then the accumulate variant."""
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n), 5)
    c = bi.cfg
    desc = desc_of(bi)
    act = mb.act_torch_dtype(desc)
    rng = np.random.default_rng(99)
    gz64 = rng.standard_normal((n, c.r))
    gz = torch.from_numpy(gz64).to(act).cuda()
    gz64 = gz.double().cpu().numpy()                       # the stored (rounded) values
    A_s = (bi.A.f64 / max(bi.A.f64.std(), 1e-30)).astype(np.float32)
    B_s = bi.B.f64.astype(np.float32)
    dA_s, dB_s = to_dev(A_s), to_dev(B_s)
    dU_t, dtok = to_dev(bi.U), to_dev(bi.tok)
    ws = mb.alloc_workspace(mb.mapl_center_backward_workspace_bytes(desc))
    dA = torch.full((c.vocab, c.anchor_rank), float("nan"), dtype=torch.float32, device="cuda")
    dB = torch.full((c.anchor_rank, c.d), float("nan"), dtype=torch.float32, device="cuda")
    dU0 = torch.from_numpy(rng.standard_normal((c.d, c.r)).astype(np.float32)).cuda()
    dU = dU0.clone()
    mb.mapl_center_backward(desc, gz, dtok, dA_s, dB_s, dU_t, dA, dB, dU, False, ws)
    torch.cuda.synchronize()
    ref = o.center_backward(gz64, bi.tok, A_s.astype(np.float64), B_s.astype(np.float64), bi.U.f64)
    tol = 1e-5                                             # fp32 arithmetic whatever the activation dtype
    assert rel_fro(to_np(dA), ref["dA_s"]) <= tol
    assert rel_fro(to_np(dB), ref["dB_s"]) <= tol
    assert rel_fro(to_np(dU) - to_np(dU0), ref["dU_corr"]) <= 1e-4   # difference of fp32 numbers of size ~1
    absent = np.setdiff1d(np.arange(c.vocab), bi.tok)
    assert not to_np(dA)[absent].any()
    # accumulate: a second call adds the same amounts
    mb.mapl_center_backward(desc, gz, dtok, dA_s, dB_s, dU_t, dA, dB, dU, True, ws)
    torch.cuda.synchronize()
    assert rel_fro(to_np(dA), 2 * ref["dA_s"]) <= tol
    assert rel_fro(to_np(dB), 2 * ref["dB_s"]) <= tol
