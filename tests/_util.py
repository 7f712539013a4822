"""Shared helpers of the parity tests: move seeded inputs to the GPU, call the C ABI through the
Python binding, run the oracle on the same stored values, compare."""
from __future__ import annotations

import numpy as np
import torch

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

TOL = {"f32": 1e-5, "bf16": 2e-2}     # BASELINE.json north_star: relative Frobenius error
# Per-token outputs (Zq, Hhat, gz, dH) are additionally checked ROW BY ROW, so that a single wrong token fails at any N
# (a whole-tensor norm at N = 16384 lets six garbage rows through).  Bounds: bf16 -- the north_star bound applied to every
# row on its own (a row carries one bf16 rounding of its result, 2^-9, plus the bf16 operand roundings of the
# contraction, a few 2^-9 in all); fp32 -- 5x the tensor bound (a row has no averaging over N).  Rows whose oracle
# norm is below 1e-3 of the RMS row norm are measured against that floor instead (a zero row has no relative error).
ROW_TOL = {"f32": 5e-5, "bf16": 2e-2}
PER_TOKEN = ("Zq", "Hhat", "gz", "dH")


def to_dev(s):
    if isinstance(s, np.ndarray):
        return torch.from_numpy(np.ascontiguousarray(s)).cuda()
    if s.dtype == "bf16":
        return torch.from_numpy(s.data.copy()).cuda().view(torch.bfloat16)
    return torch.from_numpy(s.data.copy()).cuda()


def to_np(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().numpy().astype(np.float64) if t.is_floating_point() else t.cpu().numpy()


def rel_fro(a: np.ndarray, b: np.ndarray) -> float:
    """||a - b||_F / ||b||_F  (b = oracle)."""
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def max_row_err(a: np.ndarray, b: np.ndarray) -> float:
    """max over rows n of ||a_n - b_n|| / max(||b_n||, 1e-3 rms_n ||b_n||)  (b = oracle)."""
    if b.shape[0] == 0:
        return 0.0
    nb = np.linalg.norm(b, axis=1)
    floor = 1e-3 * float(np.sqrt(np.mean(nb * nb)))
    den = np.maximum(nb, floor if floor > 0 else 1.0)
    return float(np.max(np.linalg.norm(a - b, axis=1) / den))


def desc_of(bi: I.BoundaryInputs, anchor=True):
    c = bi.cfg
    act = torch.bfloat16 if c.act_dtype == "bf16" else torch.float32
    return mb.make_desc(c.n_tokens, c.d, c.r, act, c.rvq_levels, c.rvq_k if c.rvq_levels else 0,
                        c.vocab if anchor else 0, c.anchor_rank if anchor else 0)


class Dev:
    """device copies of one boundary's inputs"""

    def __init__(self, bi: I.BoundaryInputs):
        self.H, self.U, self.g = to_dev(bi.H), to_dev(bi.U), to_dev(bi.g)
        self.C = to_dev(bi.C) if bi.C is not None else None
        self.tok, self.A, self.B = to_dev(bi.tok), to_dev(bi.A), to_dev(bi.B)


def run_gpu(bi: I.BoundaryInputs, dev: Dev = None, want_dB=True, want_dH=True, use_codes_for_decode=True,
            want_zq=True, accumulate=False, with_H=True):
    """encode -> decode -> backward through the C ABI; returns numpy outputs."""
    c = bi.cfg
    dev = dev or Dev(bi)
    desc = desc_of(bi, anchor=c.anchor_rank > 0)
    act = mb.act_torch_dtype(desc)
    N, d, r, L = c.n_tokens, c.d, c.r, c.rvq_levels
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    Zq = torch.empty((N, r), dtype=act, device="cuda") if (L == 0 or want_zq) else None
    codes = torch.empty((N, L), dtype=torch.int32, device="cuda") if L > 0 else None
    mb.mapl_encode(desc, dev.H, dev.U, dev.C, Zq, codes, ws)
    Hhat = torch.empty((N, d), dtype=act, device="cuda")
    anchor = c.anchor_rank > 0
    tok, A, B = (dev.tok, dev.A, dev.B) if anchor else (None, None, None)
    if L > 0 and use_codes_for_decode:
        mb.mapl_decode(desc, None, codes, dev.U, dev.C, tok, A, B, Hhat, ws)
    else:
        mb.mapl_decode(desc, Zq, None, dev.U, dev.C, tok, A, B, Hhat, ws)
    gz = torch.empty((N, r), dtype=act, device="cuda")
    fill = 1.0 if accumulate else float("nan")
    dU = torch.full((d, r), fill, dtype=torch.float32, device="cuda")
    dA = torch.full((c.vocab, c.anchor_rank), fill, dtype=torch.float32, device="cuda") if anchor else None
    dB = torch.full((c.anchor_rank, d), fill, dtype=torch.float32, device="cuda") if (anchor and want_dB) else None
    dH = torch.empty((N, d), dtype=act, device="cuda") if (want_dH and with_H) else None
    if L > 0 and use_codes_for_decode:
        mb.mapl_codec_backward(desc, dev.g, dev.H if with_H else None, None, codes, dev.U, dev.C, tok, A, B,
                               gz, dU, dA, dB, dH, accumulate, ws)
    else:
        mb.mapl_codec_backward(desc, dev.g, dev.H if with_H else None, Zq, None, dev.U, dev.C, tok, A, B,
                               gz, dU, dA, dB, dH, accumulate, ws)
    torch.cuda.synchronize()
    out = dict(Zq=Zq, codes=codes, Hhat=Hhat, gz=gz, dU=dU, dA=dA, dB=dB, dH=dH)
    return {k: (to_np(v) if v is not None else None) for k, v in out.items()}


def run_oracle(bi: I.BoundaryInputs, gpu_codes=None, want_dB=True, with_H=True, zhat_override=None):
    """oracle on the same stored values; with RVQ the oracle follows admissible near-tie choices of
    the CUDA path (S5).  Returns (outputs, stats)."""
    c = bi.cfg
    H, U, g = bi.H.f64, bi.U.f64, bi.g.f64
    stats = dict(excepted=0, forced=0, bad=0)
    Z = o.project(H, U)
    codes = None
    if c.rvq_levels > 0:
        if gpu_codes is not None:
            res, n_exc, n_forced, bad = o.follow_codes(Z, bi.C.f64, gpu_codes)
            stats = dict(excepted=n_exc, forced=n_forced, bad=int(bad.sum()))
        else:
            res = o.rvq(Z, bi.C.f64)
        Zhat, codes = res["Zhat"], res["codes"]
    else:
        Zhat = Z
    if zhat_override is not None:
        Zhat = zhat_override
    anchor = c.anchor_rank > 0
    tok, A, B = (bi.tok, bi.A.f64, bi.B.f64) if anchor else (None, None, None)
    Hhat = o.decode(Zhat, U, tok, A, B)
    bw = o.backward(g, H if with_H else None, Zhat, U, tok, A, B, want_dB=want_dB)
    out = dict(Zq=Zhat, codes=codes, Hhat=Hhat, **bw)
    return out, stats


def compare(gpu: dict, ora: dict, stats: dict, tol: float, keys=("Zq", "Hhat", "gz", "dU", "dA", "dB", "dH")):
    errs = {}
    row_tol = ROW_TOL["f32"] if tol <= TOL["f32"] else ROW_TOL["bf16"]
    assert stats["bad"] == 0, f"non-admissible RVQ code differences: {stats}"
    if ora.get("codes") is not None:
        assert np.array_equal(gpu["codes"], ora["codes"]), "codes differ after near-tie forcing"
    for k in keys:
        if gpu.get(k) is None or ora.get(k) is None:
            continue
        errs[k] = rel_fro(gpu[k], ora[k])
        assert np.isfinite(gpu[k]).all(), f"{k}: non-finite values"
        assert errs[k] <= tol, f"{k}: rel Frobenius error {errs[k]:.3e} > {tol:.1e} ({errs})"
        if k in PER_TOKEN:
            e = max_row_err(gpu[k], ora[k])
            errs[k + "_row"] = e
            assert e <= row_tol, f"{k}: worst row relative error {e:.3e} > {row_tol:.1e}"
    return errs
