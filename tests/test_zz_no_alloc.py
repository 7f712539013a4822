"""mapl_encode_rvq_static (include/mapl.h, csrc/static_scratch.cu): the RVQ encode whose scratch is a device array of the
library -- no workspace argument, no allocation -- against the existing path (mapl_encode with a caller workspace), on
two calls in a row that share the array.  Collected last on purpose (the suite runs with `pytest -x`)."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2606_05484_b200 import binding as mb
from paper_2606_05484_b200 import inputs as I

from _util import ROW_TOL, Dev, desc_of, to_np


def _both_paths(bi):
    """(codes, zq) of mapl_encode with a workspace, and of the static-scratch entry point, on the same device inputs"""
    c = bi.cfg
    dev = Dev(bi)
    desc = desc_of(bi, anchor=False)
    act = mb.act_torch_dtype(desc)
    N, r, L = c.n_tokens, c.r, c.rvq_levels
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    codes_a = torch.full((N, L), -1, dtype=torch.int32, device="cuda")
    zq_a = torch.full((N, r), float("nan"), dtype=act, device="cuda")
    mb.mapl_encode(desc, dev.H, dev.U, dev.C, zq_a, codes_a, ws)
    codes_b = torch.full((N, L), -1, dtype=torch.int32, device="cuda")
    zq_b = torch.full((N, r), float("nan"), dtype=act, device="cuda")
    mb.mapl_encode_rvq_static(desc, dev.H, dev.U, dev.C, zq_b, codes_b)
    torch.cuda.synchronize()
    return (to_np(codes_a), to_np(zq_a).astype(np.float64)), (to_np(codes_b), to_np(zq_b).astype(np.float64))


def _check_equal(bi):
    (codes_a, zq_a), (codes_b, zq_b) = _both_paths(bi)
    assert np.array_equal(codes_a, codes_b)                     # integer work: bit-exact
    tol = ROW_TOL[bi.cfg.act_dtype]                             # the per-row bound the parity tests use
    scale = np.maximum(np.linalg.norm(zq_a, axis=1), 1e-30)
    assert np.isfinite(zq_b).all()
    assert (np.linalg.norm(zq_a - zq_b, axis=1) / scale).max() <= tol


@pytest.mark.gpu
def test_static_scratch_encode_matches_the_workspace_path_on_two_calls_in_a_row():
    """fp32 boundaries (both entry points run the fp32 SIMT kernels).  The second call uses other codebooks with FEWER
    rows (3 x 128 < 2 x 256): the array still holds the first call's half norms behind the new ones, which must not
    matter; the third call returns to the first shape."""
    first = I.make_boundary(I.CONFIGS["c0"], 0)
    second_cfg = dataclasses.replace(I.CONFIGS["c0"].with_tokens(1000), rvq_levels=3, rvq_k=128, cb_std=(0.5, 0.25, 0.125))
    second = I.make_boundary(second_cfg, 1)
    _check_equal(first)
    _check_equal(second)
    _check_equal(first)


@pytest.mark.gpu
def test_static_scratch_encode_without_zq_and_with_zero_tokens():
    bi = I.make_boundary(I.CONFIGS["c0"].with_tokens(517), 2)
    dev = Dev(bi)
    desc = desc_of(bi, anchor=False)
    ws = mb.alloc_workspace(mb.mapl_workspace_bytes(desc))
    codes_a = torch.full((517, 2), -1, dtype=torch.int32, device="cuda")
    codes_b = torch.full((517, 2), -1, dtype=torch.int32, device="cuda")
    mb.mapl_encode(desc, dev.H, dev.U, dev.C, None, codes_a, ws)
    mb.mapl_encode_rvq_static(desc, dev.H, dev.U, dev.C, None, codes_b)
    assert torch.equal(codes_a, codes_b)
    empty = desc_of(I.make_boundary(I.CONFIGS["c0"].with_tokens(8), 0), anchor=False)
    empty.n_tokens = 0
    mb.mapl_encode_rvq_static(empty, None, None, None, None, None)      # nothing to do: NULL tensors are fine


def test_static_scratch_limit_is_an_error_not_a_fault():
    """L*K beyond the array -> MAPL_ERR_WORKSPACE before anything is launched.  Needs no GPU: with n_tokens == 0 the
    pointers are never read and no CUDA call is made, so this goes through the raw C ABI (the binding asks torch for
    the current CUDA stream)."""
    import ctypes as C
    lib = mb.raw_lib()
    rows = mb.mapl_static_scratch_rows()
    assert rows == 16384

    def call(desc):
        status = lib.mapl_encode_rvq_static(C.byref(desc), None, None, None, None, None, None)
        return lib.mapl_status_string(status).decode()

    assert call(mb.make_desc(0, 256, 32, torch.float32, 4, rows // 4, 0, 0)) == "MAPL_OK"
    assert call(mb.make_desc(0, 256, 32, torch.float32, 4, rows // 4 + 1, 0, 0)) == "MAPL_ERR_WORKSPACE"
    assert call(mb.make_desc(64, 256, 32, torch.float32, 8, rows, 0, 0)) == "MAPL_ERR_WORKSPACE"     # checked before the pointers
    assert call(mb.make_desc(0, 256, 32, torch.float32, 0, 0, 0, 0)) == "MAPL_ERR_INVALID_ARG"       # RVQ off: use mapl_encode
