"""Seeded synthetic inputs for the MAPL boundary codec (shared by oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only draws the random tensors of the
BASELINE.json configs (recipe: DESIGN.md "Input recipe") and rounds them once
(round-to-nearest-even) to their storage dtype.  The oracle receives the rounded values promoted
to fp64; the CUDA path receives them as stored.  Stand-ins for the paper's workload
(LLaMA 150M/1B boundary activations, 32 000-entry vocabulary, context 2048, bf16 -- PAPER.md:159,
PAPER.md:381-391); no dataset, tokenizer or trained weight is used.

Every draw comes from numpy default_rng(SeedSequence([260605484, cfg, boundary, tensor_id])).
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

ROOT_SEED = 260605484

# tensor ids inside a SeedSequence
_T_H, _T_U, _T_C, _T_TOK, _T_A, _T_B, _T_G, _T_GSTIEFEL, _T_S, _T_W = range(10)


@dataclasses.dataclass(frozen=True)
class CodecConfig:
    """One BASELINE.json codec workload (configs[0..3])."""
    name: str
    cfg_id: int
    n_tokens: int          # N = micro-batch x seq
    d: int
    r: int
    rvq_levels: int        # L (0 = RVQ off)
    rvq_k: int             # K
    vocab: int             # V
    anchor_rank: int       # ra
    act_dtype: str         # "f32" | "bf16"
    k0: int                # rank of the low-rank part of H
    n_boundaries: int
    cb_std: tuple = ()     # per-level codebook std
    tok_dist: str = "zipf"  # "uniform" | "zipf"
    b_kind: str = "orth"   # "gauss" (std 0.02) | "orth" (orthonormal rows)
    a_std: float = 0.02

    def with_tokens(self, n_tokens: int) -> "CodecConfig":
        return dataclasses.replace(self, n_tokens=int(n_tokens))

    def with_anchor_std(self, a_std: float) -> "CodecConfig":
        return dataclasses.replace(self, a_std=float(a_std))


CONFIGS = {
    "c0": CodecConfig("c0", 0, 4096, 256, 32, 2, 256, 1024, 16, "f32", 32, 1,
                      cb_std=(0.5, 0.5), tok_dist="uniform", b_kind="gauss"),
    "c1": CodecConfig("c1", 1, 8 * 2048, 1024, 128, 0, 0, 32000, 64, "bf16", 128, 3),
    "c2": CodecConfig("c2", 2, 8 * 2048, 1024, 64, 4, 1024, 32000, 64, "bf16", 128, 1,
                      cb_std=(1.0, 0.5, 0.25, 0.125)),
    "c3": CodecConfig("c3", 3, 16 * 2048, 2048, 256, 2, 4096, 32000, 128, "bf16", 256, 3,
                      cb_std=(1.0, 0.5)),
}

# configs[4]: Stiefel sweep (d fixed, 3 projectors per r)
STIEFEL_D = 2048
STIEFEL_RS = (64, 128, 256, 512)
STIEFEL_BATCH = 3
STIEFEL_LR = 1e-2
STIEFEL_NS_ITERS = 5


def _rng(cfg_id: int, boundary: int, tensor_id: int, extra: int = 0) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([ROOT_SEED, cfg_id, boundary, tensor_id, extra]))


# ---------------------------------------------------------------- storage rounding

def round_to_f32(x64: np.ndarray) -> np.ndarray:
    """fp64 -> fp32, round-to-nearest-even (numpy's cast)."""
    return np.asarray(x64, dtype=np.float64).astype(np.float32)


def f32_to_bf16_bits(x32: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even, NaN-free inputs."""
    u = np.ascontiguousarray(x32, dtype=np.float32).view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def round_to_bf16_bits(x64: np.ndarray) -> np.ndarray:
    """fp64 -> bf16 bit pattern.  Rounds once: fp64 -> fp32 (RNE) -> bf16 (RNE).  (The double
    rounding can differ from a direct fp64->bf16 RNE only on exact fp32 half-way cases; both
    sides of every parity test consume the SAME stored bits, so it is immaterial.)"""
    return f32_to_bf16_bits(round_to_f32(x64))


@dataclasses.dataclass
class Stored:
    """A tensor as stored for the CUDA path plus its exact fp64 promotion for the oracle."""
    dtype: str             # "f32" | "bf16" | "i32"
    data: np.ndarray       # float32 / uint16 (bf16 bits) / int32
    f64: Optional[np.ndarray]  # exact promotion (None for ints)

    @property
    def shape(self):
        return self.data.shape


def store(x64: np.ndarray, dtype: str) -> Stored:
    if dtype == "f32":
        d = round_to_f32(x64)
        return Stored("f32", d, d.astype(np.float64))
    if dtype == "bf16":
        b = round_to_bf16_bits(x64)
        return Stored("bf16", b, bf16_bits_to_f32(b).astype(np.float64))
    raise ValueError(dtype)


# ---------------------------------------------------------------- tensors

def orthonormal_columns(rng: np.random.Generator, d: int, r: int) -> np.ndarray:
    """Q of the thin QR (diag(R) > 0) of a seeded [d,r] Gaussian, fp64."""
    q, rr = np.linalg.qr(rng.standard_normal((d, r)))
    return q * np.sign(np.diag(rr))[None, :]


def zipf_tokens(rng: np.random.Generator, n: int, vocab: int, s: float = 1.1) -> np.ndarray:
    """ids with p(k) ~ k^-s, k = 1..vocab, id = k-1, by inverse CDF on seeded uniforms."""
    w = np.arange(1, vocab + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    ids = np.searchsorted(cdf, rng.random(n), side="left")
    return np.minimum(ids, vocab - 1).astype(np.int32)


def low_rank_plus_noise(rng_s, rng_w, rng_n, n: int, d: int, k0: int) -> np.ndarray:
    """H = S.W + 0.1.N with S[:, j] ~ N(0, 1/(j+1)), W ~ N(0,1), N ~ N(0,1)  (BASELINE.json configs[0])."""
    s = rng_s.standard_normal((n, k0)) / np.sqrt(np.arange(1, k0 + 1, dtype=np.float64))[None, :]
    w = rng_w.standard_normal((k0, d))
    return s @ w + 0.1 * rng_n.standard_normal((n, d))


@dataclasses.dataclass
class BoundaryInputs:
    cfg: CodecConfig
    boundary: int
    H: Stored        # [N,d] act dtype
    U: Stored        # [d,r] f32
    C: Optional[Stored]   # [L,K,r] f32 or None
    tok: np.ndarray  # [N] int32
    A: Stored        # [V,ra] f32
    B: Stored        # [ra,d] f32
    g: Stored        # [N,d] act dtype


def make_boundary(cfg: CodecConfig, boundary: int = 0) -> BoundaryInputs:
    n, d, r = cfg.n_tokens, cfg.d, cfg.r
    c, b = cfg.cfg_id, boundary
    H = store(low_rank_plus_noise(_rng(c, b, _T_S), _rng(c, b, _T_W), _rng(c, b, _T_H), n, d, cfg.k0),
              cfg.act_dtype)
    U = store(orthonormal_columns(_rng(c, b, _T_U), d, r), "f32")
    C = None
    if cfg.rvq_levels > 0:
        rc = _rng(c, b, _T_C)
        cb = np.stack([std * rc.standard_normal((cfg.rvq_k, r)) for std in cfg.cb_std[:cfg.rvq_levels]])
        C = store(cb, "f32")
    rt = _rng(c, b, _T_TOK)
    if cfg.tok_dist == "uniform":
        tok = rt.integers(0, cfg.vocab, size=n, dtype=np.int64).astype(np.int32)
    else:
        tok = zipf_tokens(rt, n, cfg.vocab)
    A = store(cfg.a_std * _rng(c, b, _T_A).standard_normal((cfg.vocab, cfg.anchor_rank)), "f32")
    if cfg.b_kind == "gauss":
        Bm = 0.02 * _rng(c, b, _T_B).standard_normal((cfg.anchor_rank, d))
    else:
        Bm = orthonormal_columns(_rng(c, b, _T_B), d, cfg.anchor_rank).T.copy()
    B = store(Bm, "f32")
    g = store(_rng(c, b, _T_G).standard_normal((n, d)), cfg.act_dtype)
    return BoundaryInputs(cfg, boundary, H, U, C, tok, A, B, g)


def make_generic(seed: int, n: int, d: int, r: int, L: int, K: int, vocab: int, ra: int,
                 act_dtype: str, k0: Optional[int] = None, a_std: float = 1.0,
                 cb_std: Optional[tuple] = None) -> BoundaryInputs:
    """Same recipe at arbitrary (ragged / edge) shapes, for parity tests.  cfg_id 100+ keeps the
    streams disjoint from the named configs."""
    k0 = k0 if k0 is not None else max(1, min(d, r))
    cb = cb_std if cb_std is not None else tuple(2.0 ** (-l) for l in range(L))
    cfg = CodecConfig(f"generic{seed}", 100 + seed, n, d, r, L, K, vocab, ra, act_dtype, k0, 1,
                      cb_std=cb, tok_dist="zipf", b_kind="gauss" if ra > d else "orth", a_std=a_std)
    return make_boundary(cfg, 0)


@dataclasses.dataclass
class StiefelInputs:
    d: int
    r: int
    batch: int
    U: Stored   # [batch,d,r] f32
    G: Stored   # [batch,d,r] f32


def make_stiefel(r: int, d: int = STIEFEL_D, batch: int = STIEFEL_BATCH, step: int = 0,
                 g_scale: float = 1.0) -> StiefelInputs:
    """configs[4]: `batch` independent projectors (orthonormal, seeded QR) and Gaussian Euclidean
    gradients.  step > 0 draws the "fresh G per step" variant (reading S13)."""
    Us = np.stack([orthonormal_columns(_rng(4, i, _T_U, r), d, r) for i in range(batch)])
    Gs = np.stack([g_scale * _rng(4, i, _T_GSTIEFEL, r * 100003 + step).standard_normal((d, r))
                   for i in range(batch)])
    return StiefelInputs(d, r, batch, store(Us, "f32"), store(Gs, "f32"))


def codebook_stream_parts(n_rows: int, interval: int = 5, seed: int = 0):
    """Streaming codebook synchronisation schedule ("streaming interval 5"; reading S15): a seeded
    permutation of the n_rows = L*K codeword rows cut into `interval` parts; micro-batch t carries part t % interval.
    Protocol bookkeeping only (no arithmetic of the method); returns a list of int32 index arrays."""
    perm = np.random.default_rng(np.random.SeedSequence([260605484, 15, seed])).permutation(n_rows).astype(np.int32)
    return [np.ascontiguousarray(p) for p in np.array_split(perm, interval)]
