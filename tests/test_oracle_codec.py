"""Pins of the fp64 oracle's codec functions (project / rvq / decode / backward) against things
other than itself: closed forms, invariants, brute force, finite differences, hand-worked values.
Citations: P:NN = /root/reference/PAPER.md line NN; S# = DESIGN.md reading."""
import itertools
import os

import numpy as np
import pytest

from oracle import mapl_oracle as o
from paper_2606_05484_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _orth(rng, d, r):
    q, rr = np.linalg.qr(rng.standard_normal((d, r)))
    return q * np.sign(np.diag(rr))


# ------------------------------------------------------------------ projection / reconstruction

def test_exact_inverse_at_full_rank():
    """P:78 'A_p^T is the exact inverse of A_p': r = d, RVQ off, no anchor => Hhat = H."""
    rng = np.random.default_rng(1)
    H = rng.standard_normal((37, 24))
    U = _orth(rng, 24, 24)
    Hhat = o.decode(o.project(H, U), U)
    assert np.abs(Hhat - H).max() < 1e-12


def test_encode_of_decode_is_identity():
    """U^T U = I => project(decode(z)) = z for any z (P:78 isometric on the column space)."""
    rng = np.random.default_rng(2)
    U = _orth(rng, 40, 7)
    Z = rng.standard_normal((19, 7))
    assert np.abs(o.project(o.decode(Z, U), U) - Z).max() < 1e-12


def test_projection_is_contraction_and_isometry_on_span():
    rng = np.random.default_rng(3)
    U = _orth(rng, 32, 5)
    H = rng.standard_normal((50, 32))
    assert np.linalg.norm(o.project(H, U)) < np.linalg.norm(H)
    Z0 = rng.standard_normal((50, 5))
    Hs = Z0 @ U.T
    assert abs(np.linalg.norm(o.project(Hs, U)) - np.linalg.norm(Hs)) < 1e-12


def test_projection_closed_form_selector():
    """U = [I_r; 0] => Z = first r columns of H; catches a transposed operand."""
    rng = np.random.default_rng(4)
    H = rng.standard_normal((11, 9))
    U = np.zeros((9, 4))
    U[:4, :4] = np.eye(4)
    assert np.array_equal(o.project(H, U), H[:, :4])
    # non-square, non-symmetric: single nonzero entry U[i0,j0]
    U2 = np.zeros((9, 4)); U2[6, 1] = 2.0
    Z = o.project(H, U2)
    expect = np.zeros((11, 4)); expect[:, 1] = 2.0 * H[:, 6]
    assert np.array_equal(Z, expect)


def test_projection_matches_library_matmul():
    rng = np.random.default_rng(5)
    H = rng.standard_normal((33, 20)); U = rng.standard_normal((20, 6))
    assert np.abs(o.project(H, U) - H @ U).max() < 1e-12


def test_sender_centring_eq1():
    """P:73 Eq. 1: Z = (X - E_small[t] P) A."""
    rng = np.random.default_rng(6)
    H = rng.standard_normal((21, 12)); U = _orth(rng, 12, 3)
    A = rng.standard_normal((7, 2)); B = rng.standard_normal((2, 12))
    tok = rng.integers(0, 7, 21).astype(np.int32)
    Z = o.project(H, U, tok, A, B)
    assert np.abs(Z - (H - A[tok] @ B) @ U).max() < 1e-12


def test_payload_bytes_per_token_golden():
    """Payload accounting printed by the paper (tests/golden/payload_bytes.txt: P:19)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "payload_bytes.txt")) if l.strip() and not l.startswith("#")]
    for kind, a, b, c, expect in rows:
        a, b, c, expect = int(a), int(b), int(c), int(expect)
        if kind == "proj":      # r channels x 2 bytes (bf16)
            assert a * 2 == expect
        elif kind == "raw":     # d channels x 2 bytes
            assert a * 2 == expect
        elif kind == "mcvq":    # (r/G) groups x R rounds x log2(K)/8 bytes  (reading S3)
            r, G, R = a, b, c
            assert (r // G) * R * 1 == expect


# ------------------------------------------------------------------ RVQ

def _brute_rvq(Z, Cb):
    """independent per-level exhaustive search (numpy broadcasting, direct distances)."""
    L, K, r = Cb.shape
    rho = Z.copy()
    codes = np.zeros((Z.shape[0], L), np.int64)
    for l in range(L):
        D = ((rho[:, None, :] - Cb[l][None, :, :]) ** 2).sum(-1)
        codes[:, l] = np.argmin(D, axis=1)       # first occurrence = lowest index
        rho = rho - Cb[l][codes[:, l]]
    return codes, rho


@pytest.mark.parametrize("seed,N,r,K,L", [(0, 64, 4, 8, 3), (1, 50, 3, 5, 2), (2, 33, 1, 7, 1), (3, 40, 6, 16, 4)])
def test_rvq_matches_exhaustive_search(seed, N, r, K, L):
    rng = np.random.default_rng(seed)
    Z = rng.standard_normal((N, r))
    Cb = np.stack([rng.standard_normal((K, r)) * 2.0 ** (-l) for l in range(L)])
    out = o.rvq(Z, Cb)
    codes, rho = _brute_rvq(Z, Cb)
    assert np.array_equal(out["codes"], codes)
    assert np.abs(out["rho"] - rho).max() < 1e-12
    # Zhat = sum of chosen codewords and Z - Zhat = final residual
    Zs = sum(Cb[l][codes[:, l]] for l in range(L))
    assert np.abs(out["Zhat"] - Zs).max() < 1e-12
    assert np.abs((Z - out["Zhat"]) - out["rho"]).max() < 1e-12
    assert np.abs(o.dequant(out["codes"], Cb) - Zs).max() < 1e-12
    # d1 <= d2 and d1 is the distance to the chosen word at level 0
    assert (out["d1"] <= out["d2"]).all()
    assert np.abs(out["d1"][:, 0] - ((Z - Cb[0][codes[:, 0]]) ** 2).sum(-1)).max() < 1e-12
    # second-best: brute force
    D0 = np.sort(((Z[:, None, :] - Cb[0][None]) ** 2).sum(-1), axis=1)
    if K > 1:
        assert np.abs(out["d2"][:, 0] - D0[:, 1]).max() < 1e-12


def test_rvq_hand_worked_2d():
    """Hand-worked case (tests/golden/rvq_hand_2d.txt): 2-D, K=4, L=2."""
    vals = [list(map(float, l.split())) for l in open(os.path.join(GOLD, "rvq_hand_2d.txt"))
            if l.strip() and not l.startswith("#")]
    C0 = np.array(vals[0:4]); C1 = np.array(vals[4:8])
    cases = vals[8:]
    Cb = np.stack([C0, C1])
    Z = np.array([c[:2] for c in cases])
    out = o.rvq(Z, Cb)
    for i, c in enumerate(cases):
        assert tuple(out["codes"][i]) == (int(c[2]), int(c[3])), (i, out["codes"][i])
        assert np.abs(out["rho"][i] - np.array(c[4:6])).max() < 1e-12


def test_rvq_degenerate_cases():
    rng = np.random.default_rng(7)
    Z = rng.standard_normal((10, 3))
    # K = 1: all codes 0
    Cb = rng.standard_normal((2, 1, 3))
    assert (o.rvq(Z, Cb)["codes"] == 0).all()
    # duplicate codewords: the lower index wins (S4)
    C0 = rng.standard_normal((6, 3)); C0[4] = C0[1]; C0[5] = C0[0]
    out = o.rvq(Z, C0[None])
    assert not np.isin(out["codes"], [4, 5]).any()
    # exact composition z = C0[k0] + C1[k1], well separated scales => codes (k0,k1), residual 0
    C0 = 10.0 * np.eye(4)[:, :3] + 0.0
    C0 = np.array([[10, 0, 0], [0, 10, 0], [0, 0, 10], [-10, 0, 0]], float)
    C1 = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [0, -1, 0]], float)
    pairs = list(itertools.product(range(4), range(4)))
    Zc = np.array([C0[a] + C1[b] for a, b in pairs])
    out = o.rvq(Zc, np.stack([C0, C1]))
    assert [tuple(c) for c in out["codes"]] == pairs
    assert np.abs(out["rho"]).max() == 0.0


def test_rvq_forced_codes_and_follow():
    rng = np.random.default_rng(8)
    Z = rng.standard_normal((30, 4))
    Cb = np.stack([rng.standard_normal((8, 4)), 0.5 * rng.standard_normal((8, 4))])
    base = o.rvq(Z, Cb)
    # craft a near tie at level 0 of token 0: codeword 7 = codeword k* mirrored through z in a tiny way
    k = base["codes"][0, 0]
    Cb2 = Cb.copy()
    other = (k + 1) % 8
    Cb2[0, other] = Cb[0, k] + 1e-9        # almost identical distance
    b2 = o.rvq(Z, Cb2)
    alt = b2["codes"].copy()
    alt[0, 0] = other if b2["codes"][0, 0] == k else k
    # after taking the alternative, later level is whatever greedy gives from the alt residual
    rho_alt = Z[0] - Cb2[0, alt[0, 0]]
    alt[0, 1] = np.argmin(((rho_alt[None] - Cb2[1]) ** 2).sum(-1))
    res, n_exc, n_forced, bad = o.follow_codes(Z, Cb2, alt)
    assert n_exc >= 1 and n_forced == 1 and not bad.any()
    assert np.array_equal(res["codes"], alt)
    # a NON-admissible difference is flagged, not forced
    alt2 = b2["codes"].copy()
    far = int(np.argmax(((Z[3][None] - Cb2[0]) ** 2).sum(-1)))
    alt2[3, 0] = far
    _, _, n_forced2, bad2 = o.follow_codes(Z, Cb2, alt2)
    assert bad2[3, 0] and n_forced2 == 0


# ------------------------------------------------------------------ decode / anchor

def test_decode_linearity_and_anchor_only():
    """P:75 Eq. 2 / P:106 Eq. 3: decode(Z,A) - decode(0,A) = Z U^T ; Z = 0 => row n = A[tok_n] B."""
    rng = np.random.default_rng(9)
    U = _orth(rng, 18, 4)
    Z = rng.standard_normal((25, 4))
    A = rng.standard_normal((6, 3)); B = rng.standard_normal((3, 18))
    tok = rng.integers(0, 6, 25).astype(np.int32)
    full = o.decode(Z, U, tok, A, B)
    anchor = o.decode(np.zeros_like(Z), U, tok, A, B)
    assert np.abs((full - anchor) - Z @ U.T).max() < 1e-12
    assert np.abs(anchor - A[tok] @ B).max() < 1e-12
    for a, b in itertools.combinations(range(25), 2):
        if tok[a] == tok[b]:
            assert np.array_equal(anchor[a], anchor[b])
    # ra = 0 => pure reconstruction
    assert np.abs(o.decode(Z, U) - Z @ U.T).max() < 1e-12
    # single-entry anchor pins index order of A[tok] and B
    A1 = np.zeros((6, 3)); A1[2, 1] = 3.0
    B1 = np.zeros((3, 18)); B1[1, 5] = 0.5
    out = o.decode(np.zeros_like(Z), U, tok, A1, B1)
    exp = np.zeros((25, 18)); exp[tok == 2, 5] = 1.5
    assert np.array_equal(out, exp)


# ------------------------------------------------------------------ backward

def _loss(g, H, U, tok, A, B, c=None):
    """<g, Hhat> with Hhat = (H U + c) U^T + A[tok] B; c = frozen STE offset (S7)."""
    Z = H @ U
    if c is not None:
        Z = Z + c
    return float(np.sum(g * (Z @ U.T + A[tok] @ B)))


def _fd(fun, X, idx, h=1e-6):
    Xp = X.copy(); Xm = X.copy()
    Xp[idx] += h; Xm[idx] -= h
    return (fun(Xp) - fun(Xm)) / (2 * h)


@pytest.mark.parametrize("with_rvq", [False, True])
def test_backward_matches_finite_differences(with_rvq):
    rng = np.random.default_rng(10 + with_rvq)
    N, d, r, V, ra = 14, 10, 3, 5, 2
    H = rng.standard_normal((N, d)); U = _orth(rng, d, r)
    A = rng.standard_normal((V, ra)); B = rng.standard_normal((ra, d))
    tok = rng.integers(0, V, N).astype(np.int32)
    g = rng.standard_normal((N, d))
    Z = H @ U
    if with_rvq:
        Cb = np.stack([rng.standard_normal((6, r)), 0.3 * rng.standard_normal((6, r))])
        Zhat = o.rvq(Z, Cb)["Zhat"]
        c = Zhat - Z                      # frozen: STE surrogate Hhat = (H U + c) U^T + ...
    else:
        Zhat, c = Z, None
    out = o.backward(g, H, Zhat, U, tok, A, B)
    for idx in [(0, 0), (3, 1), (9, 2), (5, 0)]:
        fd = _fd(lambda X: _loss(g, H, X, tok, A, B, c), U, idx)
        assert abs(fd - out["dU"][idx]) < 1e-6 * max(1.0, abs(fd)), ("dU", idx)
    for idx in [(0, 0), (4, 1), (2, 0)]:
        fd = _fd(lambda X: _loss(g, H, U, tok, X, B, c), A, idx)
        assert abs(fd - out["dA"][idx]) < 1e-6 * max(1.0, abs(fd)), ("dA", idx)
    for idx in [(0, 0), (1, 7)]:
        fd = _fd(lambda X: _loss(g, H, U, tok, A, X, c), B, idx)
        assert abs(fd - out["dB"][idx]) < 1e-6 * max(1.0, abs(fd)), ("dB", idx)
    for idx in [(0, 0), (13, 9), (6, 4)]:
        fd = _fd(lambda X: _loss(g, X, U, tok, A, B, c), H, idx)
        assert abs(fd - out["dH"][idx]) < 1e-6 * max(1.0, abs(fd)), ("dH", idx)
    # gz = dL/dZhat: perturb the offset c
    c0 = np.zeros_like(Z) if c is None else c
    for idx in [(0, 0), (7, 2)]:
        fd = _fd(lambda X: _loss(g, H, U, tok, A, B, X), c0, idx)
        assert abs(fd - out["gz"][idx]) < 1e-6 * max(1.0, abs(fd)), ("gz", idx)


def test_backward_adjoint_identities_and_split():
    rng = np.random.default_rng(12)
    N, d, r, V, ra = 40, 16, 5, 9, 3
    H = rng.standard_normal((N, d)); U = _orth(rng, d, r)
    A = rng.standard_normal((V, ra)); B = rng.standard_normal((ra, d))
    tok = rng.integers(0, V - 2, N).astype(np.int32)     # tokens V-2, V-1 never occur
    g = rng.standard_normal((N, d)); Zhat = rng.standard_normal((N, r))
    out = o.backward(g, H, Zhat, U, tok, A, B)
    # <g, Zhat U^T> = <g U, Zhat>
    assert abs(np.sum(g * (Zhat @ U.T)) - np.sum(out["gz"] * Zhat)) < 1e-10
    # <g, A[tok] B> = <dA, A> = <dB, B>
    lhs = np.sum(g * (A[tok] @ B))
    assert abs(lhs - np.sum(out["dA"] * A)) < 1e-10
    assert abs(lhs - np.sum(out["dB"] * B)) < 1e-10
    # absent tokens: zero rows; duplicates add
    assert np.all(out["dA"][V - 2:] == 0.0)
    gA = g @ B.T
    ref = np.zeros((V, ra)); np.add.at(ref, tok, gA)
    assert np.abs(out["dA"] - ref).max() < 1e-11
    # H = None split (S8): dU_full - dU_decode_only = H^T gz
    dec = o.backward(g, None, Zhat, U, tok, A, B)
    assert dec["dH"] is None
    assert np.abs((out["dU"] - dec["dU"]) - H.T @ out["gz"]).max() < 1e-10
    assert np.abs(dec["dU"] - g.T @ Zhat).max() < 1e-10
    assert np.abs(out["dH"] - out["gz"] @ U.T).max() < 1e-12
    assert np.abs(out["gz"] - g @ U).max() < 1e-12
    # no anchor
    na = o.backward(g, H, Zhat, U)
    assert na["dA"] is None and np.abs(na["dU"] - out["dU"]).max() == 0.0


def test_centring_backward_matches_finite_differences():
    """center_backward is the gradient of L = <gz, (H - A_s[tok] B_s) U> w.r.t. A_s, B_s, and its dU_corr completes
    H^T gz to the U-gradient of Eq. 1 (central differences in fp64 on every entry class)."""
    rng = np.random.default_rng(16)
    N, d, r, V, ra = 23, 10, 4, 6, 3
    H = rng.standard_normal((N, d)); U = _orth(rng, d, r)
    A = rng.standard_normal((V, ra)); B = rng.standard_normal((ra, d))
    tok = rng.integers(0, V - 1, N).astype(np.int32)          # id V-1 never occurs
    gz = rng.standard_normal((N, r))
    L = lambda A_, B_, U_: float((gz * o.project(H, U_, tok, A_, B_)).sum())
    bw = o.center_backward(gz, tok, A, B, U)
    eps = 1e-6

    def fd(X, which):
        G = np.zeros_like(X)
        for idx in np.ndindex(*X.shape):
            Xp, Xm = X.copy(), X.copy()
            Xp[idx] += eps; Xm[idx] -= eps
            args = {"A": (Xp, B, U), "B": (A, Xp, U), "U": (A, B, Xp)}[which], {"A": (Xm, B, U), "B": (A, Xm, U), "U": (A, B, Xm)}[which]
            G[idx] = (L(*args[0]) - L(*args[1])) / (2 * eps)
        return G

    assert np.abs(bw["dA_s"] - fd(A, "A")).max() < 1e-7
    assert np.abs(bw["dB_s"] - fd(B, "B")).max() < 1e-7
    assert np.abs((H.T @ gz + bw["dU_corr"]) - fd(U, "U")).max() < 1e-7
    assert not bw["dA_s"][V - 1].any()                          # absent id: zero row
    # closed form of the U term: (H - A_s[tok] B_s)^T gz
    assert np.abs((H - A[tok] @ B).T @ gz - (H.T @ gz + bw["dU_corr"])).max() < 1e-12


# ------------------------------------------------------------------ grouped MCVQ (reading S3)

def test_mcvq_groups_match_brute_force_and_reduce_to_rvq():
    rng = np.random.default_rng(50)
    N, r, G, K, L = 37, 8, 2, 9, 3
    X = rng.standard_normal((N, r))
    Cb = rng.standard_normal((L, K, r)) * (0.5 ** np.arange(L))[:, None, None]
    out = o.mcvq(X, Cb, G)
    # independent brute force: per token, per group, per round, every codeword, direct distances
    for n in range(N):
        for g in range(r // G):
            rho = X[n, g * G:(g + 1) * G].copy()
            for l in range(L):
                D = [float(((rho - Cb[l, k, g * G:(g + 1) * G]) ** 2).sum()) for k in range(K)]
                k_star = int(np.argmin(D))
                assert out["codes"][n, l, g] == k_star
                rho -= Cb[l, k_star, g * G:(g + 1) * G]
    assert np.abs(out["Xq"] - o.mcvq_dequant(out["codes"], Cb, G)).max() < 1e-12
    # one group of r channels is the full-vector RVQ
    full = o.mcvq(X, Cb, r)
    ref = o.rvq(X, Cb)
    assert np.array_equal(full["codes"][:, :, 0], ref["codes"]) and np.abs(full["Xq"] - ref["Zhat"]).max() < 1e-12
    # groups do not talk to each other: changing the channels of one group changes that group's codes only
    X2 = X.copy(); X2[:, 2:4] += 5.0
    out2 = o.mcvq(X2, Cb, G)
    assert np.array_equal(np.delete(out2["codes"], 1, axis=2), np.delete(out["codes"], 1, axis=2))


def test_mcvq_payload_is_256_bytes_at_the_papers_setting():
    """P:181 / P:403: r=256, G=2, K=256, R=2 -> 128 groups x 2 rounds x 1 byte."""
    r, G, R, K = 256, 2, 2, 256
    codes_per_token = (r // G) * R
    assert codes_per_token * int(np.ceil(np.log2(K) / 8)) == 256


# ------------------------------------------------------------------ streaming codebook sync + retained energy (row 4)

def test_energy_retained_closed_forms():
    """E = ||X A||^2 / ||X||^2: 1 when the rows of X lie in span(A); sum of the top-r squared singular values over all of them
    when A holds the top-r right singular vectors (P:55 energy formula); at most 1 for any orthonormal A."""
    rng = np.random.default_rng(80)
    X = rng.standard_normal((50, 12)) * np.linspace(3, 0.1, 12)
    A = _orth(rng, 12, 4)
    assert o.energy_retained(X, o.project(X, A)) <= 1.0 + 1e-12
    Xin = rng.standard_normal((50, 4)) @ A.T
    assert abs(o.energy_retained(Xin, o.project(Xin, A)) - 1.0) < 1e-12
    _, s, Vt = np.linalg.svd(X, full_matrices=False)
    assert abs(o.energy_retained(X, o.project(X, Vt[:4].T)) - (s[:4] ** 2).sum() / (s ** 2).sum()) < 1e-12


def test_codebook_stream_schedule_refreshes_every_row_once_per_interval():
    parts = I.codebook_stream_parts(2 * 256, interval=5, seed=3)
    allidx = np.concatenate(parts)
    assert len(parts) == 5 and sorted(allidx.tolist()) == list(range(512))        # a partition of the rows
    assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1             # a fifth each
    rng = np.random.default_rng(81)
    sender = rng.standard_normal((2, 256, 8)); receiver = np.zeros_like(sender)
    for t in range(5):                                                              # static sender: converged after 5
        rows = sender.reshape(-1, 8)[parts[t]]
        receiver = o.codebook_delta_apply(receiver, parts[t], rows)
    assert np.array_equal(receiver, sender)
