"""C-ABI surface checks that need no GPU: the library loads, exports every symbol include/mapl.h
declares, rejects bad arguments before touching CUDA, and has no CPU fallback."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2606_05484_b200 import binding as mb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "mapl.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mapl_[a-z_0-9]+)\s*\(", src)))


def test_exports_every_declared_symbol():
    lib = C.CDLL(mb.LIB_PATH)
    syms = _declared_symbols()
    for must in ("mapl_encode", "mapl_decode", "mapl_codec_backward", "mapl_stiefel_step",
                 "mapl_workspace_bytes", "mapl_stiefel_workspace_bytes", "mapl_status_string"):
        assert must in syms
    for s in syms:
        assert hasattr(lib, s), s


def test_binding_names_match_c_names():
    for s in ("mapl_encode", "mapl_decode", "mapl_codec_backward", "mapl_stiefel_step"):
        assert callable(getattr(mb, s))


def test_status_strings_and_version():
    lib = mb.raw_lib()
    assert lib.mapl_status_string(0) == b"MAPL_OK"
    assert lib.mapl_status_string(-4) == b"MAPL_ERR_WORKSPACE"
    assert b"sm_100a" in lib.mapl_version()


def test_workspace_queries():
    d = mb.make_desc(16384, 1024, 128, torch.bfloat16, 0, 0, 32000, 64)
    assert mb.mapl_workspace_bytes(d) > 0
    bad = mb.make_desc(16, 1024, 12, torch.bfloat16)          # r % 8 != 0
    assert mb.raw_lib().mapl_workspace_bytes(C.byref(bad)) == 0
    assert mb.mapl_stiefel_workspace_bytes(2048, 512, 3) >= 3 * (2 * 2048 * 512 + 3 * 512 * 512) * 4
    assert mb.raw_lib().mapl_stiefel_workspace_bytes(64, 128, 1) == 0     # r > d


def test_argument_errors_are_reported_before_any_cuda_call():
    lib = mb.raw_lib()
    d = mb.make_desc(64, 64, 16, torch.float32, 0, 0, 0, 0)
    buf = (C.c_char * 4096)()
    p = C.addressof(buf)
    p = (p + 15) & ~15
    # NULL H
    assert lib.mapl_encode(C.byref(d), None, p, None, p, None, p, 4096, None) == -1
    # RVQ off but Zq_out NULL
    assert lib.mapl_encode(C.byref(d), p, p, None, None, None, p, 4096, None) == -1
    # misaligned pointer
    assert lib.mapl_encode(C.byref(d), p + 4, p, None, p, None, p, 4096, None) == -3
    # workspace too small / NULL
    assert lib.mapl_encode(C.byref(d), p, p, None, p, None, p, 0, None) == -4
    assert lib.mapl_encode(C.byref(d), p, p, None, p, None, None, 1 << 20, None) == -4
    # decode: both Z and codes, or neither
    assert lib.mapl_decode(C.byref(d), p, p, p, None, None, None, None, p, p, 4096, None) == -1
    assert lib.mapl_decode(C.byref(d), None, None, p, None, None, None, None, p, p, 4096, None) == -1
    # backward: dH without H
    assert lib.mapl_codec_backward(C.byref(d), p, None, p, None, p, None, None, None, None, p, p, None, None, p,
                                   0, p, 4096, None) == -1
    # grouped MCVQ is not on the hot path yet
    g = mb.make_desc(64, 64, 16, torch.float32, 2, 8, 0, 0)
    g.rvq_group_dim = 2
    assert lib.mapl_encode(C.byref(g), p, p, p, p, p, p, 4096, None) == -2
    # stiefel
    assert lib.mapl_stiefel_step(64, 16, 1, None, p, C.c_float(0.1), 0, 5, None, p, 1 << 20, None) == -1
    assert lib.mapl_stiefel_step(64, 16, 1, p, p, C.c_float(0.1), 7, 5, None, p, 1 << 20, None) == -1
    assert lib.mapl_stiefel_step(64, 16, 1, p, p, C.c_float(0.1), 1, 0, None, p, 1 << 20, None) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback():
    """Without a CUDA device a valid compute call fails with MAPL_ERR_CUDA; the binding refuses CPU tensors."""
    lib = mb.raw_lib()
    d = mb.make_desc(64, 64, 16, torch.float32, 0, 0, 0, 0)
    n = mb.mapl_workspace_bytes(d) + 64 * 64 * 4 * 4
    buf = (C.c_char * (n + 64))()
    p = (C.addressof(buf) + 15) & ~15
    assert lib.mapl_encode(C.byref(d), p, p, None, p, None, p, n, None) == -5
    with pytest.raises(mb.MaplError):
        t = torch.zeros(64, 64)
        mb.mapl_encode(d, t, t, None, t, None, torch.zeros(n, dtype=torch.uint8))


def test_centering_entry_points_check_arguments():
    lib = mb.raw_lib()
    d = mb.make_desc(64, 64, 16, torch.float32, 0, 0, 100, 8)
    assert mb.mapl_center_workspace_bytes(d) >= 8 * 16 * 4
    no_anchor = mb.make_desc(64, 64, 16, torch.float32, 0, 0, 0, 0)
    assert mb.mapl_center_workspace_bytes(no_anchor) == 0
    buf = (C.c_char * 8192)()
    p = (C.addressof(buf) + 15) & ~15
    # tok / table missing
    assert lib.mapl_encode_centered(C.byref(d), p, None, p, p, None, p, None, p, 8192, None) == -1
    assert lib.mapl_encode_centered(C.byref(d), p, p, None, p, None, p, None, p, 8192, None) == -1
    # table_out NULL
    assert lib.mapl_center_table(C.byref(d), p, p, p, None, p, 8192, None) == -1
    # workspace too small
    assert lib.mapl_center_table(C.byref(d), p, p, p, p, p, 16, None) == -4


def test_mcvq_entry_points_check_arguments():
    lib = mb.raw_lib()
    buf = (C.c_char * 8192)()
    p = (C.addressof(buf) + 15) & ~15
    assert lib.mapl_mcvq_quantize(16, 64, 1, 2, 300, p, p, p, None, None) == -1       # K > 256: no byte index
    assert lib.mapl_mcvq_quantize(16, 64, 1, 2, 256, None, p, p, None, None) == -1    # X NULL
    assert lib.mapl_mcvq_quantize(16, 12, 1, 2, 256, p, p, p, None, None) == -1       # r % 8 != 0
    assert lib.mapl_mcvq_dequantize(16, 64, 1, 2, 256, p, p, None, None) == -1        # Xq_out NULL
    assert lib.mapl_mcvq_quantize(0, 64, 1, 2, 256, None, None, None, None, None) == 0  # empty batch: no-op
