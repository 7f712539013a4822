"""Grouped multi-codebook VQ of a wire payload (reading S3):
mapl_mcvq_quantize / mapl_mcvq_dequantize through the C ABI against oracle.mcvq on the same stored values."""
import numpy as np
import pytest
import torch

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

from _util import TOL, rel_fro, to_np

pytestmark = pytest.mark.gpu


def _payload(n, r, act, seed):
    """A payload with the statistics of a projected activation: Z = H U of the seeded generic boundary, stored in act."""
    bi = I.make_generic(seed, n, 512, r, 0, 0, 100, 0, act)
    Z = o.project(bi.H.f64, bi.U.f64)
    t = torch.from_numpy(Z).to(torch.bfloat16 if act == "bf16" else torch.float32).cuda()
    return t, t.double().cpu().numpy()


@pytest.mark.parametrize("act", ["bf16", "f32"])
@pytest.mark.parametrize("n,r,L,K", [(1000, 256, 2, 256), (777, 64, 3, 37), (129, 128, 1, 256), (5, 8, 2, 4)])
def test_mcvq_matches_oracle(act, n, r, L, K):
    X, X64 = _payload(n, r, act, 60 + r + L)
    rng = np.random.default_rng(61 + K)
    scale = X64.std() * (0.6 ** np.arange(L))[:, None, None]
    Cb = (rng.standard_normal((L, K, r)) * scale).astype(np.float32)
    dC = torch.from_numpy(Cb).cuda()
    codes = torch.empty((n, L, r // 2), dtype=torch.uint8, device="cuda")
    Xq = torch.empty_like(X)
    mb.mapl_mcvq_quantize(X, dC, codes, Xq)
    torch.cuda.synchronize()
    gc = codes.cpu().numpy().astype(np.int32)
    ref = o.mcvq(X64, Cb.astype(np.float64), 2, other_codes=gc)
    assert ref["bad"] == 0, f"non-admissible codes: {ref['bad']} (excepted {ref['excepted']}, forced {ref['forced']})"
    assert np.array_equal(gc, ref["codes"])
    tol = TOL[act]
    assert rel_fro(to_np(Xq), ref["Xq"]) <= tol
    # receiver side: dequantise from the bytes alone
    Xq2 = torch.empty_like(X)
    mb.mapl_mcvq_dequantize(codes, dC, Xq2)
    torch.cuda.synchronize()
    assert torch.equal(Xq, Xq2)
    # payload: (r/2) L bytes per token
    assert codes.numel() * codes.element_size() == n * (r // 2) * L


def test_mcvq_payload_feeds_decode():
    """Forward wire with MCVQ: encode (RVQ off) -> quantise Z -> dequantise -> decode; the reconstruction equals the
    oracle's decode of the oracle-dequantised payload."""
    from _util import Dev, desc_of
    bi = I.make_boundary(I.CONFIGS["c1"].with_tokens(900), 6)
    dev = Dev(bi)
    desc = desc_of(bi)
    c = bi.cfg
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    Z = torch.empty((c.n_tokens, c.r), dtype=torch.bfloat16, device="cuda")
    mb.mapl_encode(desc, dev.H, dev.U, None, Z, None, ws)
    rng = np.random.default_rng(70)
    Cb = (rng.standard_normal((2, 256, c.r)) * np.array([2.0, 0.7])[:, None, None]).astype(np.float32)
    dC = torch.from_numpy(Cb).cuda()
    codes = torch.empty((c.n_tokens, 2, c.r // 2), dtype=torch.uint8, device="cuda")
    mb.mapl_mcvq_quantize(Z, dC, codes, None)
    Zq = torch.empty_like(Z)
    mb.mapl_mcvq_dequantize(codes, dC, Zq)
    Hhat = torch.empty((c.n_tokens, c.d), dtype=torch.bfloat16, device="cuda")
    mb.mapl_decode(desc, Zq, None, dev.U, None, dev.tok, dev.A, dev.B, Hhat, ws)
    torch.cuda.synchronize()
    ref = o.mcvq(Z.double().cpu().numpy(), Cb.astype(np.float64), 2, other_codes=codes.cpu().numpy().astype(np.int32))
    assert ref["bad"] == 0
    Hh = o.decode(ref["Xq"], bi.U.f64, bi.tok, bi.A.f64, bi.B.f64)
    assert rel_fro(to_np(Hhat), Hh) <= TOL["bf16"]
