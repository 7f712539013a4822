"""Thin Python face of libmapl.so (include/mapl.h): argument marshalling only -- every step of the
codec runs in the CUDA kernels behind the C ABI.  torch is used for device memory and the stream.

The functions carry the C names (mapl_encode, mapl_decode, mapl_codec_backward,
mapl_stiefel_step).  Importing this module fails loudly when libmapl.so is missing; calling a
compute function without a CUDA device raises (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmapl.so")

MAPL_F32, MAPL_BF16 = 0, 1
MAPL_RETRACT_QR, MAPL_RETRACT_NS = 0, 1


class MaplError(RuntimeError):
    pass


class BoundaryDesc(C.Structure):
    """mapl_boundary_desc (include/mapl.h)."""
    _fields_ = [("n_tokens", C.c_int64), ("d", C.c_int32), ("r", C.c_int32), ("act_dtype", C.c_int32),
                ("rvq_levels", C.c_int32), ("rvq_k", C.c_int32), ("rvq_group_dim", C.c_int32),
                ("vocab", C.c_int32), ("anchor_rank", C.c_int32), ("param_pack", C.c_void_p)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_05484_b200.build` "
                          "(nvcc, sm_100a).  There is no fallback path.")
    lib = C.CDLL(LIB_PATH)
    vp, sz, i32, f32 = C.c_void_p, C.c_size_t, C.c_int32, C.c_float
    dp = C.POINTER(BoundaryDesc)
    lib.mapl_status_string.restype = C.c_char_p
    lib.mapl_status_string.argtypes = [C.c_int]
    lib.mapl_version.restype = C.c_char_p
    lib.mapl_last_cuda_error.restype = C.c_int
    lib.mapl_workspace_bytes.restype = sz
    lib.mapl_workspace_bytes.argtypes = [dp]
    lib.mapl_stiefel_workspace_bytes.restype = sz
    lib.mapl_stiefel_workspace_bytes.argtypes = [i32, i32, i32]
    lib.mapl_param_pack_bytes.restype = sz
    lib.mapl_param_pack_bytes.argtypes = [dp]
    lib.mapl_pack_params.restype = C.c_int
    lib.mapl_pack_params.argtypes = [dp, vp, vp, vp, vp, vp]
    lib.mapl_encode.argtypes = [dp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.mapl_static_scratch_rows.restype = sz
    lib.mapl_static_scratch_rows.argtypes = []
    lib.mapl_encode_rvq_static.restype = C.c_int
    lib.mapl_encode_rvq_static.argtypes = [dp, vp, vp, vp, vp, vp, vp]
    lib.mapl_center_workspace_bytes.restype = sz
    lib.mapl_center_workspace_bytes.argtypes = [dp]
    lib.mapl_center_table.restype = C.c_int
    lib.mapl_center_table.argtypes = [dp, vp, vp, vp, vp, vp, sz, vp]
    lib.mapl_center_backward_workspace_bytes.restype = sz
    lib.mapl_center_backward_workspace_bytes.argtypes = [dp]
    lib.mapl_center_backward.restype = C.c_int
    lib.mapl_center_backward.argtypes = [dp, vp, vp, vp, vp, vp, vp, vp, vp, C.c_int, vp, sz, vp]
    lib.mapl_encode_centered.restype = C.c_int
    lib.mapl_encode_centered.argtypes = [dp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.mapl_decode.argtypes = [dp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.mapl_codec_backward.argtypes = [dp] + [vp] * 14 + [C.c_int, vp, sz, vp]
    lib.mapl_stiefel_step.argtypes = [i32, i32, i32, vp, vp, f32, i32, i32, vp, vp, sz, vp]
    lib.mapl_mcvq_quantize.restype = C.c_int
    lib.mapl_mcvq_quantize.argtypes = [C.c_int64, i32, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.mapl_mcvq_dequantize.restype = C.c_int
    lib.mapl_mcvq_dequantize.argtypes = [C.c_int64, i32, i32, i32, i32, vp, vp, vp, vp]
    lib.mapl_codebook_delta_pack.restype = C.c_int
    lib.mapl_codebook_delta_pack.argtypes = [vp, i32, vp, i32, vp, vp]
    lib.mapl_codebook_delta_apply.restype = C.c_int
    lib.mapl_codebook_delta_apply.argtypes = [vp, i32, vp, i32, vp, vp]
    lib.mapl_energy_retained.restype = C.c_int
    lib.mapl_energy_retained.argtypes = [C.c_int64, i32, i32, i32, vp, vp, vp, vp]
    lib.mapl_spel_workspace_bytes.restype = sz
    lib.mapl_spel_workspace_bytes.argtypes = [i32, i32, i32]
    lib.mapl_spel_step.restype = C.c_int
    lib.mapl_spel_step.argtypes = [i32, i32, i32, vp, vp, vp, f32, f32, i32, i32, vp, sz, vp]
    lib.mapl_profile_kernel_count.restype = C.c_int
    lib.mapl_profile_kernel_name.restype = C.c_char_p
    lib.mapl_profile_kernel_name.argtypes = [C.c_int]
    lib.mapl_profile_enable.restype = None
    lib.mapl_profile_enable.argtypes = [C.c_int]
    lib.mapl_profile_reset.restype = None
    lib.mapl_profile_read.restype = C.c_int
    lib.mapl_profile_read.argtypes = [C.c_int, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong),
                                      C.POINTER(C.c_double)]
    for n in ("mapl_encode", "mapl_decode", "mapl_codec_backward", "mapl_stiefel_step"):
        getattr(lib, n).restype = C.c_int
    return lib


_lib = _load()


def _check(status: int, what: str):
    if status != 0:
        msg = _lib.mapl_status_string(status).decode()
        extra = f" (cudaError {_lib.mapl_last_cuda_error()})" if status == -5 else ""
        raise MaplError(f"{what}: {msg}{extra}")


def _ptr(t: Optional[torch.Tensor], dtype=None, name: str = "") -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise MaplError(f"{name}: expected a CUDA tensor (no CPU path exists)")
    if not t.is_contiguous():
        raise MaplError(f"{name}: tensor must be contiguous row-major")
    if dtype is not None and t.dtype != dtype:
        raise MaplError(f"{name}: expected {dtype}, got {t.dtype}")
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def version() -> str:
    return _lib.mapl_version().decode()


def make_desc(n_tokens: int, d: int, r: int, act_dtype: torch.dtype, rvq_levels: int = 0, rvq_k: int = 0,
              vocab: int = 0, anchor_rank: int = 0) -> BoundaryDesc:
    act = {torch.float32: MAPL_F32, torch.bfloat16: MAPL_BF16}[act_dtype]
    return BoundaryDesc(n_tokens, d, r, act, rvq_levels, rvq_k, r if rvq_levels > 0 else 0, vocab, anchor_rank,
                        None)


def act_torch_dtype(desc: BoundaryDesc) -> torch.dtype:
    return torch.bfloat16 if desc.act_dtype == MAPL_BF16 else torch.float32


def mapl_workspace_bytes(desc: BoundaryDesc) -> int:
    n = int(_lib.mapl_workspace_bytes(C.byref(desc)))
    if n == 0:
        raise MaplError("mapl_workspace_bytes: invalid descriptor")
    return n


def mapl_stiefel_workspace_bytes(d: int, r: int, batch: int) -> int:
    n = int(_lib.mapl_stiefel_workspace_bytes(d, r, batch))
    if n == 0:
        raise MaplError("mapl_stiefel_workspace_bytes: invalid shape")
    return n


def mapl_param_pack_bytes(desc: BoundaryDesc) -> int:
    return int(_lib.mapl_param_pack_bytes(C.byref(desc)))


def mapl_pack_params(desc: BoundaryDesc, U, B, codebooks, pack_out) -> None:
    """Write the prepared parameter pack for (U, B, codebooks) into `pack_out` (uint8 device tensor of
    mapl_param_pack_bytes(desc) bytes).  Reference it with `desc.param_pack = pack_out.data_ptr()`."""
    f = torch.float32
    _check(_lib.mapl_pack_params(C.byref(desc), _ptr(U, f, "U"), _ptr(B, f, "B"), _ptr(codebooks, f, "codebooks"),
                                 _ptr(pack_out, None, "pack_out"), _stream()), "mapl_pack_params")


def alloc_workspace(nbytes: int, device="cuda") -> torch.Tensor:
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def mapl_encode(desc: BoundaryDesc, H, U, codebooks, Zq_out, codes_out, workspace) -> None:
    act = act_torch_dtype(desc)
    _check(_lib.mapl_encode(C.byref(desc), _ptr(H, act, "H"), _ptr(U, torch.float32, "U"),
                            _ptr(codebooks, torch.float32, "codebooks"), _ptr(Zq_out, act, "Zq_out"),
                            _ptr(codes_out, torch.int32, "codes_out"), _ptr(workspace, None, "workspace"),
                            workspace.numel() * workspace.element_size(), _stream()), "mapl_encode")


def mapl_static_scratch_rows() -> int:
    return int(_lib.mapl_static_scratch_rows())


def mapl_encode_rvq_static(desc: BoundaryDesc, H, U, codebooks, Zq_out, codes_out) -> None:
    """mapl_encode with RVQ on the fp32 SIMT kernels, scratch in a device array of the library: no workspace, no
    allocation (include/mapl.h).  levels * K > mapl_static_scratch_rows() raises MAPL_ERR_WORKSPACE."""
    act = act_torch_dtype(desc)
    _check(_lib.mapl_encode_rvq_static(C.byref(desc), _ptr(H, act, "H"), _ptr(U, torch.float32, "U"),
                                       _ptr(codebooks, torch.float32, "codebooks"), _ptr(Zq_out, act, "Zq_out"),
                                       _ptr(codes_out, torch.int32, "codes_out"), _stream()), "mapl_encode_rvq_static")


def mapl_center_workspace_bytes(desc: BoundaryDesc) -> int:
    return int(_lib.mapl_center_workspace_bytes(C.byref(desc)))


def mapl_center_table(desc: BoundaryDesc, A_s, B_s, U, table_out, workspace) -> None:
    """T = A_s (B_s U), [V,r] fp32: the per-token-id centring rows of mapl_encode_centered (Eq. 1)."""
    f = torch.float32
    _check(_lib.mapl_center_table(C.byref(desc), _ptr(A_s, f, "A_s"), _ptr(B_s, f, "B_s"), _ptr(U, f, "U"),
                                  _ptr(table_out, f, "table_out"), _ptr(workspace, None, "workspace"),
                                  workspace.numel() * workspace.element_size(), _stream()), "mapl_center_table")


def mapl_encode_centered(desc: BoundaryDesc, H, tok, center_table, U, codebooks, Zq_out, codes_out, workspace) -> None:
    act = act_torch_dtype(desc)
    _check(_lib.mapl_encode_centered(
        C.byref(desc), _ptr(H, act, "H"), _ptr(tok, torch.int32, "tok"), _ptr(center_table, torch.float32, "center_table"),
        _ptr(U, torch.float32, "U"), _ptr(codebooks, torch.float32, "codebooks"), _ptr(Zq_out, act, "Zq_out"),
        _ptr(codes_out, torch.int32, "codes_out"), _ptr(workspace, None, "workspace"),
        workspace.numel() * workspace.element_size(), _stream()), "mapl_encode_centered")


def mapl_center_backward_workspace_bytes(desc: BoundaryDesc) -> int:
    return int(_lib.mapl_center_backward_workspace_bytes(C.byref(desc)))


def mapl_center_backward(desc: BoundaryDesc, gz, tok, A_s, B_s, U, dA_s_out, dB_s_out, dU_inout, accumulate: bool,
                         workspace) -> None:
    """Backward of the centring term (include/mapl.h): dA_s, optional dB_s, and dU += -B_s^T A_s[tok]^T gz."""
    act = act_torch_dtype(desc)
    f = torch.float32
    _check(_lib.mapl_center_backward(
        C.byref(desc), _ptr(gz, act, "gz"), _ptr(tok, torch.int32, "tok"), _ptr(A_s, f, "A_s"), _ptr(B_s, f, "B_s"),
        _ptr(U, f, "U"), _ptr(dA_s_out, f, "dA_s_out"), _ptr(dB_s_out, f, "dB_s_out"), _ptr(dU_inout, f, "dU_inout"),
        int(bool(accumulate)), _ptr(workspace, None, "workspace"), workspace.numel() * workspace.element_size(),
        _stream()), "mapl_center_backward")


def mapl_decode(desc: BoundaryDesc, Z, codes, U, codebooks, tok, A, B, Hhat_out, workspace) -> None:
    act = act_torch_dtype(desc)
    f = torch.float32
    _check(_lib.mapl_decode(C.byref(desc), _ptr(Z, act, "Z"), _ptr(codes, torch.int32, "codes"), _ptr(U, f, "U"),
                            _ptr(codebooks, f, "codebooks"), _ptr(tok, torch.int32, "tok"), _ptr(A, f, "A"),
                            _ptr(B, f, "B"), _ptr(Hhat_out, act, "Hhat_out"), _ptr(workspace, None, "workspace"),
                            workspace.numel() * workspace.element_size(), _stream()), "mapl_decode")


def mapl_codec_backward(desc: BoundaryDesc, g, H, Z, codes, U, codebooks, tok, A, B, gz_out, dU_out, dA_out,
                        dB_out, dH_out, accumulate: bool, workspace) -> None:
    act = act_torch_dtype(desc)
    f = torch.float32
    _check(_lib.mapl_codec_backward(
        C.byref(desc), _ptr(g, act, "g"), _ptr(H, act, "H"), _ptr(Z, act, "Z"), _ptr(codes, torch.int32, "codes"),
        _ptr(U, f, "U"), _ptr(codebooks, f, "codebooks"), _ptr(tok, torch.int32, "tok"), _ptr(A, f, "A"),
        _ptr(B, f, "B"), _ptr(gz_out, act, "gz_out"), _ptr(dU_out, f, "dU_out"), _ptr(dA_out, f, "dA_out"),
        _ptr(dB_out, f, "dB_out"), _ptr(dH_out, act, "dH_out"), int(bool(accumulate)),
        _ptr(workspace, None, "workspace"), workspace.numel() * workspace.element_size(), _stream()),
        "mapl_codec_backward")


def mapl_stiefel_step(U_inout, G, lr: float, retraction: int, ns_iters: int, info_out, workspace) -> None:
    f = torch.float32
    if U_inout.dim() == 2:
        batch, (d, r) = 1, U_inout.shape
    else:
        batch, d, r = U_inout.shape
    if tuple(G.shape) != tuple(U_inout.shape):
        raise MaplError("mapl_stiefel_step: G must have the shape of U")
    _check(_lib.mapl_stiefel_step(d, r, batch, _ptr(U_inout, f, "U_inout"), _ptr(G, f, "G"), float(lr),
                                  int(retraction), int(ns_iters), _ptr(info_out, f, "info_out"),
                                  _ptr(workspace, None, "workspace"),
                                  workspace.numel() * workspace.element_size(), _stream()), "mapl_stiefel_step")


def _act_code(t: torch.Tensor) -> int:
    return {torch.float32: MAPL_F32, torch.bfloat16: MAPL_BF16}[t.dtype]


def mapl_mcvq_quantize(X, codebooks, codes_out, Xq_out=None) -> None:
    """Grouped (G = 2) multi-codebook VQ of a payload X [N,r]; codebooks [L,K,r] fp32; codes_out [N,L,r/2] uint8."""
    N, r = X.shape
    L, K, _ = codebooks.shape
    _check(_lib.mapl_mcvq_quantize(N, r, _act_code(X), L, K, _ptr(X, None, "X"), _ptr(codebooks, torch.float32, "codebooks"),
                                   _ptr(codes_out, torch.uint8, "codes_out"), _ptr(Xq_out, X.dtype, "Xq_out"), _stream()),
           "mapl_mcvq_quantize")


def mapl_mcvq_dequantize(codes, codebooks, Xq_out) -> None:
    N, r = Xq_out.shape
    L, K, _ = codebooks.shape
    _check(_lib.mapl_mcvq_dequantize(N, r, _act_code(Xq_out), L, K, _ptr(codes, torch.uint8, "codes"),
                                     _ptr(codebooks, torch.float32, "codebooks"), _ptr(Xq_out, None, "Xq_out"), _stream()),
           "mapl_mcvq_dequantize")


def mapl_codebook_delta_pack(codebooks, idx, rows_out) -> None:
    """rows_out[i] = codebooks.view(-1, r)[idx[i]]: the codewords a micro-batch carries (streaming sync)."""
    r = codebooks.shape[-1]
    _check(_lib.mapl_codebook_delta_pack(_ptr(codebooks, torch.float32, "codebooks"), r, _ptr(idx, torch.int32, "idx"),
                                         idx.numel(), _ptr(rows_out, torch.float32, "rows_out"), _stream()),
           "mapl_codebook_delta_pack")


def mapl_codebook_delta_apply(codebooks_inout, idx, rows) -> None:
    r = codebooks_inout.shape[-1]
    _check(_lib.mapl_codebook_delta_apply(_ptr(codebooks_inout, torch.float32, "codebooks"), r, _ptr(idx, torch.int32, "idx"),
                                          idx.numel(), _ptr(rows, torch.float32, "rows"), _stream()),
           "mapl_codebook_delta_apply")


def mapl_energy_retained(H, Z, sums_inout) -> None:
    """sums_inout (float64[2], zeroed by the caller) += (||Z||_F^2, ||H||_F^2); E = sums[0] / sums[1] (Fig. 4b)."""
    N, d = H.shape
    _check(_lib.mapl_energy_retained(N, d, Z.shape[1], _act_code(H), _ptr(H, None, "H"), _ptr(Z, H.dtype, "Z"),
                                     _ptr(sums_inout, torch.float64, "sums_inout"), _stream()), "mapl_energy_retained")


def mapl_spel_workspace_bytes(d: int, r: int, batch: int) -> int:
    return int(_lib.mapl_spel_workspace_bytes(d, r, batch))


def mapl_spel_step(U_inout, G, M_inout, lr: float, beta: float, lmo_iters: int, retr_iters: int, workspace) -> None:
    """Full SPEL update (include/mapl.h): tangent projection, momentum, LMO direction, retraction."""
    f = torch.float32
    if U_inout.dim() == 2:
        batch, (d, r) = 1, U_inout.shape
    else:
        batch, d, r = U_inout.shape
    if tuple(G.shape) != tuple(U_inout.shape) or tuple(M_inout.shape) != tuple(U_inout.shape):
        raise MaplError("mapl_spel_step: G and M must have the shape of U")
    _check(_lib.mapl_spel_step(d, r, batch, _ptr(U_inout, f, "U_inout"), _ptr(G, f, "G"), _ptr(M_inout, f, "M_inout"),
                               float(lr), float(beta), int(lmo_iters), int(retr_iters), _ptr(workspace, None, "workspace"),
                               workspace.numel() * workspace.element_size(), _stream()), "mapl_spel_step")


def raw_lib():
    """The ctypes handle (tests use it to exercise error returns without a GPU)."""
    return _lib
