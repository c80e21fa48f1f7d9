"""Seeded synthetic input generators shared by the tests, the bench and the oracle checks.

This module holds NONE of the method's arithmetic (no packing, no addressing): it only draws
page-ID lists, request lengths and session schedules with ``numpy.random.default_rng(seed)``
(PCG64) in the order written, following the recipes of SURVEY.md 8(d) / DESIGN.md "Input
recipe".  The shapes stand in for the paper's Qwen3-Omni sessions; the
datasets and weights themselves are not needed by a bitwise copy path.

Neither ``oracle/`` nor the CUDA path imports the other; both are driven from here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List

import numpy as np


@dataclass(frozen=True)
class PoolShape:
    """Geometry of one paged KV pool (layers, K/V slices, page size, shape, dtype)."""

    L: int  # layers
    C: int  # K/V slices (2)
    H: int  # KV heads held by this rank
    D: int  # head dim
    e: int  # element bytes (2 = bf16)
    T: int  # tokens per page
    P: int  # pages in the pool

    @property
    def tokrow_bytes(self) -> int:
        return self.H * self.D * self.e

    @property
    def row_bytes(self) -> int:
        return self.T * self.tokrow_bytes

    @property
    def page_bytes(self) -> int:
        return self.L * self.C * self.row_bytes

    @property
    def tok_bytes(self) -> int:
        return self.L * self.C * self.tokrow_bytes

    def with_(self, **kw) -> "PoolShape":
        d = dict(L=self.L, C=self.C, H=self.H, D=self.D, e=self.e, T=self.T, P=self.P)
        d.update(kw)
        return PoolShape(**d)


# BASELINE.json:configs[0] and configs[1..4]
TINY = PoolShape(L=4, C=2, H=2, D=64, e=2, T=16, P=256)
QWEN3_OMNI = PoolShape(L=48, C=2, H=4, D=128, e=2, T=16, P=65536)


def random_bits_u16(rng: np.random.Generator, n_elems: int) -> np.ndarray:
    """Random 16-bit patterns (include NaN payloads, -0, subnormals when read as bf16)."""
    return rng.integers(0, 65536, size=n_elems, dtype=np.uint16)


# --------------------------------------------------------------------------------------------
# config 1 -- Tiny
# --------------------------------------------------------------------------------------------
@dataclass
class TinyCase:
    shape: PoolShape
    src_ids: np.ndarray
    dst_ids: np.ndarray


def tiny_case(seed: int = 0, n: int = 37, shape: PoolShape = TINY) -> TinyCase:
    rng = np.random.default_rng(seed)
    src_ids = rng.choice(shape.P, n, replace=False).astype(np.int32)
    dst_ids = rng.permutation(shape.P)[:n].astype(np.int32)
    return TinyCase(shape, src_ids, dst_ids)


# --------------------------------------------------------------------------------------------
# config 2 -- single-request prefix offload
# --------------------------------------------------------------------------------------------
@dataclass
class PrefixCase:
    shape: PoolShape
    src_ids: np.ndarray  # fragmented: a random sample of the pool, unsorted
    dst_ids: np.ndarray  # other free pages, disjoint from src_ids


def prefix_case(seed: int = 0, n_tokens: int = 8192, shape: PoolShape = QWEN3_OMNI) -> PrefixCase:
    rng = np.random.default_rng(seed)
    n = -(-n_tokens // shape.T)
    src_ids = rng.choice(shape.P, n, replace=False).astype(np.int32)
    free = np.setdiff1d(np.arange(shape.P, dtype=np.int32), src_ids, assume_unique=True)
    dst_ids = rng.choice(free, n, replace=False).astype(np.int32)
    return PrefixCase(shape, src_ids, dst_ids)


# --------------------------------------------------------------------------------------------
# config 3 -- 50-turn multimodal session
# --------------------------------------------------------------------------------------------
@dataclass
class Turn:
    k: int  # 1-based turn index
    delta: int  # tokens appended this turn
    cum_tokens: int  # c_k
    n_matched_pages: int  # floor(c_{k-1} / T): full pages of history reloaded this turn
    spans: List[tuple] = field(default_factory=list)  # (kind, length) placeholder spans


def session_turns(seed: int = 0, turns: int = 50, T: int = 16) -> List[Turn]:
    """Per turn: delta_k = rng.integers(300, 1501); image/audio placeholder spans of 256-1024
    tokens accepted while they fit in delta_k - 8; the rest is text (BASELINE.json:configs[2])."""
    rng = np.random.default_rng(seed)
    out: List[Turn] = []
    c = 0
    for k in range(1, turns + 1):
        delta = int(rng.integers(300, 1501))
        used = 0
        spans = []
        while True:
            s = int(rng.integers(256, 1025))
            if used + s > delta - 8:
                break
            kind = "image" if rng.random() < 0.5 else "audio"
            spans.append((kind, s))
            used += s
        spans.append(("text", delta - used))
        matched = c // T
        c += delta
        out.append(Turn(k, delta, c, matched, spans))
    return out


class FreeList:
    """Permuted free list of page ids; pop from the end, return at random positions."""

    def __init__(self, num_pages: int, rng: np.random.Generator):
        self.rng = rng
        self.free = list(rng.permutation(num_pages).astype(np.int32))

    def pop(self, n: int) -> np.ndarray:
        if n > len(self.free):
            raise RuntimeError("free list exhausted")
        if n == 0:
            return np.zeros(0, dtype=np.int32)
        out = np.array(self.free[-n:][::-1], dtype=np.int32)
        del self.free[-n:]
        return out

    def give_back(self, ids) -> None:
        for g in ids:
            pos = int(self.rng.integers(0, len(self.free) + 1))
            self.free.insert(pos, int(g))


# --------------------------------------------------------------------------------------------
# config 4 -- concurrent offload batch
# --------------------------------------------------------------------------------------------
@dataclass
class BatchCase:
    shape: PoolShape
    lens: np.ndarray  # prompt lengths in tokens, per request
    req_offsets: np.ndarray  # CSR offsets into src_ids / dst_ids, int64[R+1]
    src_ids: np.ndarray
    dst_ids: np.ndarray


def batch_case(seed: int = 0, n_req: int = 64, lo: int = 512, hi: int = 16384,
               shape: PoolShape = QWEN3_OMNI) -> BatchCase:
    rng = np.random.default_rng(seed)
    lens = np.floor(np.exp(rng.uniform(math.log(lo), math.log(hi), size=n_req))).astype(np.int64)
    n_pages = -(-lens // shape.T)
    off = np.zeros(n_req + 1, dtype=np.int64)
    off[1:] = np.cumsum(n_pages)
    total = int(off[-1])
    if 2 * total > shape.P:
        raise ValueError("pool too small for this batch")
    perm = rng.permutation(shape.P).astype(np.int32)
    return BatchCase(shape, lens, off, perm[:total].copy(), perm[total:2 * total].copy())


# --------------------------------------------------------------------------------------------
# config 5 -- cross-role prefix reuse (re-paging Ts -> Td)
# --------------------------------------------------------------------------------------------
@dataclass
class CrossRoleCase:
    src_shape: PoolShape
    dst_shape: PoolShape
    n_tokens: np.ndarray  # per request
    src_offsets: np.ndarray
    dst_offsets: np.ndarray
    src_ids: np.ndarray
    dst_ids: np.ndarray


def crossrole_case(seed: int = 0, n_req: int = 32, prefix_tokens: int = 2048, ragged: bool = False,
                   src_shape: PoolShape = QWEN3_OMNI.with_(P=32768),
                   dst_shape: PoolShape = QWEN3_OMNI.with_(T=64, P=8192)) -> CrossRoleCase:
    rng = np.random.default_rng(seed)
    ntok = np.full(n_req, prefix_tokens, dtype=np.int64)
    if ragged:  # SURVEY.md 8(c) reading 9: 2048 - r_i, r_i in [1, 64)
        ntok = ntok - rng.integers(1, 64, size=n_req)
    ns = -(-ntok // src_shape.T)
    nd = -(-ntok // dst_shape.T)
    so = np.zeros(n_req + 1, dtype=np.int64)
    so[1:] = np.cumsum(ns)
    do = np.zeros(n_req + 1, dtype=np.int64)
    do[1:] = np.cumsum(nd)
    src_ids = rng.choice(src_shape.P, int(so[-1]), replace=False).astype(np.int32)
    dst_ids = rng.choice(dst_shape.P, int(do[-1]), replace=False).astype(np.int32)
    return CrossRoleCase(src_shape, dst_shape, ntok, so, do, src_ids, dst_ids)


def sweep_sizes_pages(max_bytes: int = 8 << 30) -> List[int]:
    """1 MiB ... 8 GiB doubling with layer_count = 32 (page = exactly 1 MiB at the Qwen3-Omni
    shape); SURVEY.md 8(c) reading 14."""
    out = []
    n = 1
    while n * (1 << 20) <= max_bytes:
        out.append(n)
        n *= 2
    return out


# --------------------------------------------------------------------------------------------
# content identities for chained paged hashing
# --------------------------------------------------------------------------------------------
VOCAB = 151_936  # text token ids are drawn below this (a Qwen-sized vocabulary; only the range matters)


@dataclass
class IdentityBatch:
    ident: np.ndarray        # uint64[total tokens]: one content identity per token position
    tok_offsets: np.ndarray  # int64[S+1] CSR over sessions
    shared_prefix: np.ndarray  # int64[S]: tokens each session shares with session 0 (0 for session 0)


def identity_batch(seed: int = 0, lens=None, n_sessions: int = 64, lo: int = 512, hi: int = 16384,
                   share: float = 0.5) -> IdentityBatch:
    """One 64-bit identity per token: a text position carries its token id, every position of an image /
    audio placeholder span carries that item's (random 64-bit) content hash id.  Span structure as in
    config 3 (spans of 256-1,024 positions, half the mass text).  With probability `share` a session
    starts with a copy of a random-length prefix of session 0 (cross-session reuse: equal page-aligned
    prefixes must get equal page ids); the copy length is recorded, not consumed by the hash."""
    rng = np.random.default_rng(seed)
    if lens is None:
        lens = np.floor(np.exp(rng.uniform(math.log(lo), math.log(hi), size=n_sessions))).astype(np.int64)
    lens = np.asarray(lens, dtype=np.int64)
    off = np.zeros(len(lens) + 1, dtype=np.int64)
    np.cumsum(lens, out=off[1:])
    ident = np.zeros(int(off[-1]), dtype=np.uint64)
    shared = np.zeros(len(lens), dtype=np.int64)
    for s, n in enumerate(lens):
        a = ident[off[s]:off[s + 1]]
        pos = 0
        while pos < n:
            if rng.random() < 0.5:  # a multimodal item
                ln = min(int(rng.integers(256, 1025)), int(n) - pos)
                a[pos:pos + ln] = rng.integers(0, 2**64, dtype=np.uint64)
            else:
                ln = min(int(rng.integers(8, 513)), int(n) - pos)
                a[pos:pos + ln] = rng.integers(0, VOCAB, size=ln).astype(np.uint64)
            pos += ln
        if s > 0 and rng.random() < share:
            k = int(rng.integers(1, min(int(n), int(lens[0])) + 1))
            a[:k] = ident[off[0]:off[0] + k]
            shared[s] = k
    return IdentityBatch(ident, off, shared)
