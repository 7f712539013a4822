"""Two independent CUDA implementations of the RVQ encode against each other on seeded random shapes: the tcgen05 kernel
(fp16 coarse scores, candidate lists, exact fp32 pass; `mapl_encode` on bf16 boundaries inside the tensor-core envelope)
and the fp32 SIMT kernel (`mapl_encode_rvq_static`: exact arithmetic throughout).  They may differ only where the paper's
arg-min (S4, S5) is decided by rounding: at the first level where a token's codes differ, the two chosen
codewords must be at the same distance from the residual up to fp32 rounding, measured here in fp64.  This is a
consistency check between kernels, not oracle parity (tests/test_parity_codec.py is that); it covers shapes, level counts
and codebook scales the fixed configurations do not."""
import random

import pytest
import torch

from paper_2606_05484_b200 import binding as mb

pytestmark = pytest.mark.gpu

NEAR_TIE = 2e-5          # relative gap of squared distances; fp32 rounding of a 64..256-term sum is ~1e-7..1e-6


def _case(rng, gen):
    d = rng.choice([256, 512, 1024, 2048])
    r = min(rng.choice([64, 128, 256]), d)
    K = rng.choice([128, 256, 512, 1024, 2048, 4096])
    L = rng.choice([1, 2, 3, 4, 6, 8])
    if L * K > mb.mapl_static_scratch_rows():
        L = max(1, mb.mapl_static_scratch_rows() // K)
    N = rng.choice([1, 7, 100, 517, 1000, 4096, 5000, 16384 + 3])
    std = rng.choice([1.0, 0.3, 0.05])
    scale = rng.choice([0.1, 1.0, 30.0])
    H = (torch.randn(N, d, device="cuda", generator=gen) * scale).to(torch.bfloat16)
    U = torch.linalg.qr(torch.randn(d, r, device="cuda", generator=gen))[0].contiguous()
    z_rms = float(H.float().norm(dim=1).mean()) / d ** 0.5
    Cb = torch.stack([torch.randn(K, r, device="cuda", generator=gen) * (std * 0.5 ** l * z_rms) for l in range(L)]).contiguous()
    return d, r, K, L, N, H, U, Cb


@pytest.mark.parametrize("seed", range(12))
def test_tensor_core_and_simt_rvq_differ_only_at_near_ties(seed):
    rng = random.Random(seed)
    gen = torch.Generator(device="cuda").manual_seed(seed)
    for _ in range(3):
        d, r, K, L, N, H, U, Cb = _case(rng, gen)
        desc = mb.make_desc(N, d, r, torch.bfloat16, L, K, 0, 0)
        ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
        ca = torch.full((N, L), -1, dtype=torch.int32, device="cuda")
        cb = ca.clone()
        mb.mapl_encode(desc, H, U, Cb, None, ca, ws)
        mb.mapl_encode_rvq_static(desc, H, U, Cb, None, cb)
        torch.cuda.synchronize()
        what = f"d={d} r={r} K={K} L={L} N={N}"
        assert 0 <= int(ca.min()) and int(ca.max()) < K, what
        assert 0 <= int(cb.min()) and int(cb.max()) < K, what
        differ = (ca != cb).any(dim=1).nonzero().flatten()
        assert differ.numel() <= max(2, N // 500), f"{what}: {differ.numel()} tokens differ"      # near ties are rare
        z = H.double() @ U.double()
        for t in differ.tolist():
            rho = z[t].clone()
            for l in range(L):
                ka, kb = int(ca[t, l]), int(cb[t, l])
                if ka != kb:
                    da = float((rho - Cb[l, ka].double()).pow(2).sum())
                    db = float((rho - Cb[l, kb].double()).pow(2).sum())
                    assert abs(da - db) <= NEAR_TIE * max(da, db), f"{what}: token {t} level {l}: {ka} ({da}) vs {kb} ({db})"
                    break
                rho -= Cb[l, ka].double()
