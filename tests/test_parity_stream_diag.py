"""device side of the streaming codebook synchronisation (App. F) and the
retained-energy diagnostic of Fig. 4(b), through the C ABI against the oracle."""
import numpy as np
import pytest
import torch

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

from _util import Dev, desc_of, to_dev

pytestmark = pytest.mark.gpu


def test_streaming_sync_converges_to_the_senders_codebook():
    L, K, r = 2, 256, 128
    rng = np.random.default_rng(90)
    sender64 = rng.standard_normal((L, K, r)).astype(np.float32)
    sender = torch.from_numpy(sender64).cuda()
    receiver = torch.zeros_like(sender)
    ref = np.zeros((L, K, r))
    parts = I.codebook_stream_parts(L * K, interval=5, seed=1)
    for t in range(5):
        idx = torch.from_numpy(parts[t]).cuda()
        rows = torch.empty((idx.numel(), r), dtype=torch.float32, device="cuda")
        mb.mapl_codebook_delta_pack(sender, idx, rows)                 # what travels with micro-batch t
        mb.mapl_codebook_delta_apply(receiver, idx, rows)
        torch.cuda.synchronize()
        ref = o.codebook_delta_apply(ref, parts[t], sender64.reshape(-1, r)[parts[t]])
        assert np.array_equal(receiver.cpu().numpy().astype(np.float64), ref)      # bit-exact copies
        assert rows.numel() * 4 <= (L * K * r * 4) // 5 + r * 4                   # a fifth of the table per micro-batch
    assert torch.equal(receiver, sender)


@pytest.mark.parametrize("name,n", [("c0", 999), ("c1", 3000)])
def test_energy_retained_matches_oracle(name, n):
    bi = I.make_boundary(I.CONFIGS[name].with_tokens(n), 7)
    dev = Dev(bi)
    c = bi.cfg
    desc = desc_of(bi)
    desc.rvq_levels = 0; desc.rvq_k = 0; desc.rvq_group_dim = 0
    act = mb.act_torch_dtype(desc)
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    Z = torch.empty((n, c.r), dtype=act, device="cuda")
    mb.mapl_encode(desc, dev.H, dev.U, None, Z, None, ws)
    sums = torch.zeros(2, dtype=torch.float64, device="cuda")
    mb.mapl_energy_retained(dev.H, Z, sums)
    torch.cuda.synchronize()
    s = sums.cpu().numpy()
    E = s[0] / s[1]
    E_ref = o.energy_retained(bi.H.f64, o.project(bi.H.f64, bi.U.f64))
    assert abs(s[1] - (bi.H.f64 ** 2).sum()) <= 1e-6 * s[1]           # ||H||^2 of the stored values
    assert abs(E - E_ref) <= (1e-5 if name == "c0" else 5e-3) and 0.0 < E <= 1.0 + 1e-6
