"""ctypes/numpy face of oracle/mapl_oracle.c (fp64, host memory).  TEST INFRASTRUCTURE.

Every function promotes its inputs to contiguous float64 / int32 and returns fresh numpy arrays.
No arithmetic of the method lives here except the bookkeeping of the near-tie rule (reading S5 in
DESIGN.md), which is stated in `near_tie_mask` / `admissible_codes`.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def _d(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_ip)


def _f64(a) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


_lib.mapl_oracle_threads.restype = C.c_int
_lib.mapl_oracle_sqdist.restype = C.c_double
_lib.mapl_oracle_sqdist.argtypes = [C.c_int, _dp, _dp]
_lib.mapl_oracle_project.argtypes = [C.c_int64, C.c_int, C.c_int, _dp, _dp, _ip, _dp, _dp, C.c_int, _dp]
_lib.mapl_oracle_rvq.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, _dp, _dp, _ip, _ip, _dp, _dp, _dp, _dp]
_lib.mapl_oracle_dequant.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, _ip, _dp, _dp]
_lib.mapl_oracle_decode.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, _dp, _dp, _ip, _dp, _dp, _dp]
_lib.mapl_oracle_backward.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _dp,
                                      _ip, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
_lib.mapl_oracle_tangent.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]
_lib.mapl_oracle_qr.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]
_lib.mapl_oracle_newton_schulz.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp]
_lib.mapl_oracle_stiefel_step.argtypes = [C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_int, C.c_int, _dp, _dp]

RETRACT_QR, RETRACT_NS = 0, 1


def threads() -> int:
    return int(_lib.mapl_oracle_threads())


def project(H, U, tok=None, A_s=None, B_s=None) -> np.ndarray:
    """Z = (H - A_s[tok] B_s) U  (Eq. 1); hot path: A_s None -> Z = H U."""
    H, U = _f64(H), _f64(U)
    N, d = H.shape
    r = U.shape[1]
    assert U.shape[0] == d
    Z = np.empty((N, r), np.float64)
    if A_s is None:
        _lib.mapl_oracle_project(N, d, r, _d(H), _d(U), None, None, None, 0, _d(Z))
    else:
        tok, A_s, B_s = _i32(tok), _f64(A_s), _f64(B_s)
        _lib.mapl_oracle_project(N, d, r, _d(H), _d(U), _i(tok), _d(A_s), _d(B_s), A_s.shape[1], _d(Z))
    return Z


def rvq(Z, Cb, forced=None):
    """Residual VQ of each row of Z with codebooks Cb [L,K,r].
    Returns dict(codes [N,L] int32, Zhat [N,r], rho [N,r] final residual, d1, d2 [N,L])."""
    Z, Cb = _f64(Z), _f64(Cb)
    N, r = Z.shape
    L, K, r2 = Cb.shape
    assert r2 == r
    codes = np.empty((N, L), np.int32)
    Zhat = np.empty((N, r), np.float64)
    rho = np.empty((N, r), np.float64)
    d1 = np.empty((N, L), np.float64)
    d2 = np.empty((N, L), np.float64)
    forced = _i32(forced)
    _lib.mapl_oracle_rvq(N, r, L, K, _d(Z), _d(Cb), _i(forced), _i(codes), _d(Zhat), _d(rho), _d(d1), _d(d2))
    return dict(codes=codes, Zhat=Zhat, rho=rho, d1=d1, d2=d2)


def dequant(codes, Cb) -> np.ndarray:
    codes, Cb = _i32(codes), _f64(Cb)
    N, L = codes.shape
    _, K, r = Cb.shape
    Zhat = np.empty((N, r), np.float64)
    _lib.mapl_oracle_dequant(N, r, L, K, _i(codes), _d(Cb), _d(Zhat))
    return Zhat


def encode(H, U, Cb=None, forced=None):
    """mapl_encode: Z = H U, then RVQ if codebooks are given.  Zhat = Z when RVQ is off."""
    Z = project(H, U)
    if Cb is None:
        return dict(Z=Z, Zhat=Z, codes=None)
    out = rvq(Z, Cb, forced)
    out["Z"] = Z
    return out


def decode(Zhat, U, tok=None, A=None, B=None) -> np.ndarray:
    """Hhat = Zhat U^T + A[tok] B  (Eq. 2, Eq. 3)."""
    Zhat, U = _f64(Zhat), _f64(U)
    N, r = Zhat.shape
    d = U.shape[0]
    assert U.shape[1] == r
    Hhat = np.empty((N, d), np.float64)
    if A is None or np.shape(A)[1] == 0:
        _lib.mapl_oracle_decode(N, d, r, 0, _d(Zhat), _d(U), None, None, None, _d(Hhat))
    else:
        tok, A, B = _i32(tok), _f64(A), _f64(B)
        assert tok.min() >= 0 and tok.max() < A.shape[0]
        _lib.mapl_oracle_decode(N, d, r, A.shape[1], _d(Zhat), _d(U), _i(tok), _d(A), _d(B), _d(Hhat))
    return Hhat


def backward(g, H, Zhat, U, tok=None, A=None, B=None, want_dB=True, want_dH=True):
    """gz, dU, dA, dB, dH of <g, Hhat> (STE reading S7).  H None ->
    decode-side term of dU only, no dH."""
    g, Zhat, U = _f64(g), _f64(Zhat), _f64(U)
    H = _f64(H)
    N, d = g.shape
    r = U.shape[1]
    has_anchor = A is not None and np.shape(A)[1] > 0
    gz = np.empty((N, r), np.float64)
    dU = np.empty((d, r), np.float64)
    dH = np.empty((N, d), np.float64) if (want_dH and H is not None) else None
    dA = dB = None
    ra = V = 0
    if has_anchor:
        tok, A, B = _i32(tok), _f64(A), _f64(B)
        V, ra = A.shape
        dA = np.empty((V, ra), np.float64)
        dB = np.empty((ra, d), np.float64) if want_dB else None
    _lib.mapl_oracle_backward(N, d, r, ra, V, _d(g), _d(H), _d(Zhat), _d(U),
                              _i(tok) if has_anchor else None, _d(A) if has_anchor else None,
                              _d(B) if has_anchor else None, _d(gz), _d(dU), _d(dA), _d(dB), _d(dH))
    return dict(gz=gz, dU=dU, dA=dA, dB=dB, dH=dH)


def center_backward(gz, tok, A_s, B_s, U, want_dB=True):
    """Backward of the sender-side centring term of PAPER.md:73 Eq. 1, Z = (H - A_s[tok] B_s) U, for an
    upstream gradient gz = dL/dZ (plain loops over the definition; library matmuls as steps):
        dL/dA_s[v,:] = - sum_{n: tok_n = v} (B_s U) gz_n           [V,ra]
        dL/dB_s      = - (sum_n A_s[tok_n]^T gz_n^T) U^T           [ra,d]
        dU_corr      = - B_s^T (sum_n A_s[tok_n] gz_n^T)           [d,r]   (added to H^T gz: the U-gradient of Eq. 1
                                                                           is (H - A_s[tok] B_s)^T gz)"""
    gz, A_s, B_s, U = _f64(gz), _f64(A_s), _f64(B_s), _f64(U)
    tok = _i32(tok)
    V, ra = A_s.shape
    N, r = gz.shape
    Wc = B_s @ U                                   # [ra,r]
    dA = np.zeros((V, ra), np.float64)
    Q = np.zeros((ra, r), np.float64)              # sum_n A_s[tok_n] (outer) gz_n
    for n in range(N):
        dA[tok[n], :] -= Wc @ gz[n]
        Q += np.outer(A_s[tok[n]], gz[n])
    dU = -(B_s.T @ Q)
    dB = -(Q @ U.T) if want_dB else None
    return dict(dA_s=dA, dB_s=dB, dU_corr=dU)


def tangent(U, G) -> np.ndarray:
    """xi = G - U sym(U^T G)  (Eq. 4)."""
    U, G = _f64(U), _f64(G)
    d, r = U.shape
    xi = np.empty((d, r), np.float64)
    _lib.mapl_oracle_tangent(d, r, _d(U), _d(G), _d(xi))
    return xi


def qr_retract(Y):
    """(Q, R) thin Householder QR with diag(R) > 0."""
    Y = _f64(Y)
    d, r = Y.shape
    Q = np.empty((d, r), np.float64)
    R = np.empty((r, r), np.float64)
    _lib.mapl_oracle_qr(d, r, _d(Y), _d(Q), _d(R))
    return Q, R


def newton_schulz(Y, iters: int = 5) -> np.ndarray:
    Y = _f64(Y)
    d, r = Y.shape
    X = np.empty((d, r), np.float64)
    _lib.mapl_oracle_newton_schulz(d, r, int(iters), _d(Y), _d(X))
    return X


def stiefel_step(U, G, lr: float, retraction: int, ns_iters: int = 5):
    """(U_plus, xi).  retraction: RETRACT_QR | RETRACT_NS."""
    U, G = _f64(U), _f64(G)
    d, r = U.shape
    Uo = np.empty((d, r), np.float64)
    xi = np.empty((d, r), np.float64)
    _lib.mapl_oracle_stiefel_step(d, r, _d(U), _d(G), float(lr), int(retraction), int(ns_iters), _d(Uo), _d(xi))
    return Uo, xi


# ---------------------------------------------------------------- near-tie rule (reading S5)

REL_GAP = 1e-4


def mcvq(X, Cb, G: int, other_codes=None, rel: float = REL_GAP):
    """Grouped multi-codebook VQ (reading S3): the r channels are cut into r/G groups
    of G consecutive channels; group g is residual-vector-quantised on its own, over L rounds, with the G-dimensional
    codewords Cb[l, k, gG:(g+1)G].  Every group is exactly the full-vector RVQ of this module applied to that slice.
    other_codes [N,L,r/G] (optional): follow admissible near-tie choices of another implementation (rule S5, per group).
    Returns dict(codes [N,L,r/G] int32, Xq [N,r], excepted, forced, bad)."""
    X, Cb = _f64(X), _f64(Cb)
    N, r = X.shape
    L, K, _ = Cb.shape
    assert r % G == 0
    ng = r // G
    codes = np.empty((N, L, ng), np.int32)
    Xq = np.empty((N, r), np.float64)
    n_exc = n_forced = n_bad = 0
    for g in range(ng):
        sl = slice(g * G, (g + 1) * G)
        Xg = np.ascontiguousarray(X[:, sl])
        Cg = np.ascontiguousarray(Cb[:, :, sl])
        if other_codes is None:
            res = rvq(Xg, Cg)
        else:
            res, e, f, bad = follow_codes(Xg, Cg, np.ascontiguousarray(other_codes[:, :, g]), rel)
            n_exc += e; n_forced += f; n_bad += int(bad.sum())
        codes[:, :, g] = res["codes"]
        Xq[:, sl] = res["Zhat"]
    return dict(codes=codes, Xq=Xq, excepted=n_exc, forced=n_forced, bad=n_bad)


def mcvq_dequant(codes, Cb, G: int) -> np.ndarray:
    """Xq[n, gG:(g+1)G] = sum_l Cb[l, codes[n,l,g], gG:(g+1)G]."""
    codes, Cb = np.asarray(codes), _f64(Cb)
    N, L, ng = codes.shape
    Xq = np.zeros((N, ng * G), np.float64)
    for g in range(ng):
        for l in range(L):
            Xq[:, g * G:(g + 1) * G] += Cb[l, codes[:, l, g], g * G:(g + 1) * G]
    return Xq


def energy_retained(H, Z) -> float:
    """Fig. 4(b): ||X A||_F^2 / ||X||_F^2 with Z = X A."""
    H, Z = _f64(H), _f64(Z)
    return float((Z * Z).sum() / (H * H).sum())


def codebook_delta_apply(Cb, idx, rows) -> np.ndarray:
    """Receiver side of the streaming codebook synchronisation: the rows idx of the [L*K, r] table are
    replaced by `rows`; returns the patched copy."""
    Cb = _f64(Cb).copy()
    flat = Cb.reshape(-1, Cb.shape[-1])
    flat[np.asarray(idx)] = _f64(rows)
    return Cb


def spel_step(U, G, m, lr: float, beta: float, lmo_iters: int = 5, retr_iters: int = 7):
    """Full SPEL update, Eq. 4-7, step by step in the paper's order; PolarExpress is read as the
    cubic Newton-Schulz iteration (reading S11), for Eq. 6 from m / ||m||_F.  Returns (U_new, m_new, d)."""
    U, G, m = _f64(U), _f64(G), _f64(m)
    xi = tangent(U, G)                                    # Eq. 4
    m_new = beta * m + (1.0 - beta) * xi                  # Eq. 5
    nrm = float(np.sqrt((m_new * m_new).sum()))
    X0 = m_new / nrm if nrm > 0 else np.zeros_like(m_new)
    d = newton_schulz(X0, lmo_iters)                      # Eq. 6
    U_new = newton_schulz(U - lr * d, retr_iters)         # Eq. 7
    return U_new, m_new, d


def near_tie_mask(d1: np.ndarray, d2: np.ndarray, rel: float = REL_GAP) -> np.ndarray:
    """(token, level) pairs whose top-2 squared-distance gap is below `rel` relative:
    (D2 - D1)/D1 < rel  (north_star: codes bit-exact "except where the oracle's top-2 distance gap is
    below 1e-4 relative")."""
    return (d2 - d1) < rel * d1


def follow_codes(Z, Cb, other_codes, rel: float = REL_GAP):
    """Run the oracle RVQ, adopting `other_codes` at excepted (token, level) pairs when that choice
    is admissible (its distance <= D1 (1 + rel)); everywhere else the oracle's own argmin stands.
    Levels are resolved one by one because a forced choice changes later residuals.
    Returns (result dict, n_excepted, n_forced, mismatch mask [N,L] of NON-admissible differences)."""
    Z, Cb = _f64(Z), _f64(Cb)
    other = _i32(other_codes)
    N, r = Z.shape
    L, K, _ = Cb.shape
    forced = np.full((N, L), -1, np.int32)
    bad = np.zeros((N, L), bool)
    n_exc = 0
    res = None
    for l in range(L):
        res = rvq(Z, Cb, forced)
        diff = res["codes"][:, l] != other[:, l]
        exc = near_tie_mask(res["d1"][:, l], res["d2"][:, l], rel)
        n_exc += int(exc.sum())
        for n in np.nonzero(diff)[0]:
            ok = False
            if exc[n] and 0 <= other[n, l] < K:
                # residual entering level l = Z - sum of codewords chosen so far (forced run)
                rho = Z[n] - sum(Cb[q, res["codes"][n, q]] for q in range(l))
                rho = np.ascontiguousarray(rho)
                c = np.ascontiguousarray(Cb[l, other[n, l]])
                D = _lib.mapl_oracle_sqdist(r, _d(rho), _d(c))
                ok = D <= res["d1"][n, l] * (1.0 + rel)
            if ok:
                forced[n, l] = other[n, l]
            else:
                bad[n, l] = True
    res = rvq(Z, Cb, forced)
    return res, n_exc, int((forced >= 0).sum()), bad
