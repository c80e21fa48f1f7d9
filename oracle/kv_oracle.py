"""oracle/kv_oracle.py -- CPU ORACLE binding.  TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` leg may import this module.  It imports nothing from ``paper_2606_31093_b200``
and the CUDA path imports nothing from here.

Two implementations of the same definitions (written from PAPER.md:L207
addressing, PAPER.md:L214 migration, BASELINE.json:configs[0] page-first layout and
BASELINE.json:configs[4] re-paging with a zero-padded tail):

* ``*_py``  -- the definition as literal Python loops over (page, layer, K/V, token, head, dim);
               only for tiny cases.
* ``pack`` / ``unpack`` / ``repage`` / ``*_batched`` / ``cow_append`` -- the same loops compiled from
               ``kv_oracle.c`` (plain C, gcc -O2), called through ctypes.  This is the oracle
               used for parity at scale and the one ``bench.py`` times as ``cpu_baseline``.

Both are pinned by tests/test_oracle_pins.py (worked examples W1/W2 in tests/golden/, numpy
take/transpose/reshape special cases, a separately written pull formulation, invariants).
Parity status: PINNED.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kv_oracle.c")
_LIB = os.path.join(_HERE, "libkvoracle.so")

PAGE_FIRST = 0
LAYER_FIRST = 1
NHD = 0  # in-page order [token][head][dim] ("NHD block stacks")
HND = 1  # in-page order [head][token][dim]


def build(force: bool = False) -> str:
    """Compile kv_oracle.c with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC]
        )
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


@dataclass
class HostPool:
    """A paged KV pool in host memory: ``slabs[l*C + c]`` is a uint8 array of
    ``num_pages * page_stride_bytes`` bytes; in-page order is [token][head][dim]."""

    slabs: List[np.ndarray]
    L: int
    C: int
    num_pages: int
    T: int
    H: int
    D: int
    e: int
    page_stride_bytes: int
    order: int = 0  # in-page order: 0 NHD [token][head][dim], 1 HND [head][token][dim]

    @property
    def row_bytes(self) -> int:
        return self.T * self.H * self.D * self.e

    @property
    def page_bytes(self) -> int:  # bytes of one page in the transfer buffer
        return self.L * self.C * self.row_bytes

    @staticmethod
    def empty(L, C, num_pages, T, H, D, e, page_stride_bytes=None, fill=0, order=0) -> "HostPool":
        row = T * H * D * e
        stride = row if page_stride_bytes is None else int(page_stride_bytes)
        assert stride >= row
        slabs = [np.full(num_pages * stride, fill, dtype=np.uint8) for _ in range(L * C)]
        return HostPool(slabs, L, C, num_pages, T, H, D, e, stride, order)

    def copy(self) -> "HostPool":
        return HostPool([s.copy() for s in self.slabs], self.L, self.C, self.num_pages, self.T,
                        self.H, self.D, self.e, self.page_stride_bytes, self.order)

    def _ptrs(self):
        arr = (ctypes.c_void_p * (self.L * self.C))()
        for i, s in enumerate(self.slabs):
            assert s.dtype == np.uint8 and s.flags["C_CONTIGUOUS"]
            arr[i] = s.ctypes.data
        return arr


def _ids(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _check(rc: int):
    if rc == -2:
        raise IndexError("oracle: page id out of range")
    if rc != 0:
        raise ValueError(f"oracle: bad argument (rc={rc})")


def _assert_distinct(ids: np.ndarray):
    # SURVEY.md 8(c) reading 5: unpack destination ids must be distinct (write race otherwise).
    if len(np.unique(ids)) != len(ids):
        raise ValueError("oracle: duplicate destination page ids")


# ----------------------------------------------------------------------------------------------
# compiled loops
# ----------------------------------------------------------------------------------------------
def pack(pool: HostPool, ids, layer_count: int | None = None, layout: int = PAGE_FIRST,
         threads: int = 1) -> np.ndarray:
    """O-pack.  Returns the transfer buffer as a uint8 array of n * L * C * row bytes."""
    L = pool.L if layer_count is None else int(layer_count)
    assert 0 < L <= pool.L
    ids = _ids(ids)
    n = len(ids)
    buf = np.zeros(n * L * pool.C * pool.row_bytes, dtype=np.uint8)
    # first `L` layers of the descriptor (SURVEY.md 8(c) reading 12): base[l*C+c], l < L
    rc = _load().kvo_pack(pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                          ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.T),
                          ctypes.c_uint32(pool.H), ctypes.c_uint32(pool.D), ctypes.c_uint32(pool.e),
                          ctypes.c_uint64(pool.page_stride_bytes), ctypes.c_int(pool.order),
                          ids.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint64(n),
                          ctypes.c_int(layout), buf.ctypes.data_as(ctypes.c_void_p),
                          ctypes.c_int(threads))
    _check(rc)
    return buf


def unpack(src: np.ndarray, dst_ids, pool: HostPool, Ts: int, n_tokens: int,
           layer_count: int | None = None, layout: int = PAGE_FIRST, threads: int = 1) -> None:
    """O-unpack into ``pool`` in place.  ``Td = pool.T``; ``len(dst_ids) == ceil(n_tokens/Td)``."""
    L = pool.L if layer_count is None else int(layer_count)
    dst_ids = _ids(dst_ids)
    _assert_distinct(dst_ids)
    src = np.ascontiguousarray(src).view(np.uint8).reshape(-1)
    tokrow = pool.H * pool.D * pool.e
    n_src = -(-int(n_tokens) // Ts)
    if src.size < n_src * L * pool.C * Ts * tokrow:
        raise ValueError("oracle: source buffer too small")
    rc = _load().kvo_unpack(src.ctypes.data_as(ctypes.c_void_p),
                            dst_ids.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint64(len(dst_ids)),
                            pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                            ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.H),
                            ctypes.c_uint32(pool.D), ctypes.c_uint32(pool.e),
                            ctypes.c_uint64(pool.page_stride_bytes), ctypes.c_int(pool.order),
                            ctypes.c_uint32(Ts), ctypes.c_uint32(pool.T), ctypes.c_uint64(int(n_tokens)),
                            ctypes.c_int(layout), ctypes.c_int(threads))
    _check(rc)


def pack_batched(pool: HostPool, ids, off, layer_count: int | None = None,
                 layout: int = PAGE_FIRST, threads: int = 1) -> List[np.ndarray]:
    """O-batched pack: one buffer per request r over ids[off[r]:off[r+1]]."""
    L = pool.L if layer_count is None else int(layer_count)
    ids = _ids(ids)
    off = np.ascontiguousarray(np.asarray(off, dtype=np.int64))
    R = len(off) - 1
    bufs = [np.zeros(int(off[r + 1] - off[r]) * L * pool.C * pool.row_bytes, dtype=np.uint8)
            for r in range(R)]
    dsts = (ctypes.c_void_p * max(R, 1))()
    for r in range(R):
        dsts[r] = bufs[r].ctypes.data
    rc = _load().kvo_pack_batched(pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                                  ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.T),
                                  ctypes.c_uint32(pool.H), ctypes.c_uint32(pool.D),
                                  ctypes.c_uint32(pool.e), ctypes.c_uint64(pool.page_stride_bytes),
                                  ctypes.c_int(pool.order), ids.ctypes.data_as(ctypes.c_void_p),
                                  off.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(R),
                                  ctypes.c_int(layout), dsts, ctypes.c_int(threads))
    _check(rc)
    return bufs


def unpack_batched(srcs: Sequence[np.ndarray], dst_ids, off, n_tokens, pool: HostPool, Ts: int,
                   layer_count: int | None = None, layout: int = PAGE_FIRST,
                   threads: int = 1) -> None:
    """O-batched unpack into ``pool`` in place."""
    L = pool.L if layer_count is None else int(layer_count)
    dst_ids = _ids(dst_ids)
    _assert_distinct(dst_ids)
    off = np.ascontiguousarray(np.asarray(off, dtype=np.int64))
    ntok = np.ascontiguousarray(np.asarray(n_tokens, dtype=np.uint64))
    R = len(off) - 1
    keep = [np.ascontiguousarray(s).view(np.uint8).reshape(-1) for s in srcs]
    tokrow = pool.H * pool.D * pool.e
    for r in range(R):
        if keep[r].size < -(-int(ntok[r]) // Ts) * L * pool.C * Ts * tokrow:
            raise ValueError("oracle: source buffer too small")
    ptrs = (ctypes.c_void_p * max(R, 1))()
    for r in range(R):
        ptrs[r] = keep[r].ctypes.data
    rc = _load().kvo_unpack_batched(ptrs, dst_ids.ctypes.data_as(ctypes.c_void_p),
                                    off.ctypes.data_as(ctypes.c_void_p),
                                    ntok.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(R),
                                    pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                                    ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.H),
                                    ctypes.c_uint32(pool.D), ctypes.c_uint32(pool.e),
                                    ctypes.c_uint64(pool.page_stride_bytes), ctypes.c_int(pool.order),
                                    ctypes.c_uint32(Ts), ctypes.c_uint32(pool.T), ctypes.c_int(layout),
                                    ctypes.c_int(threads))
    _check(rc)


def cow_append(pool: HostPool, old_id: int, new_id: int, n_old: int, app: np.ndarray,
               n_app: int, layer_count: int | None = None) -> None:
    """Copy-on-write partial-page append, in place."""
    L = pool.L if layer_count is None else int(layer_count)
    app = np.ascontiguousarray(app).view(np.uint8).reshape(-1)
    if app.size < L * pool.C * n_app * pool.H * pool.D * pool.e:
        raise ValueError("oracle: append buffer too small")
    rc = _load().kvo_cow_append(pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                                ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.T),
                                ctypes.c_uint32(pool.H), ctypes.c_uint32(pool.D),
                                ctypes.c_uint32(pool.e), ctypes.c_uint64(pool.page_stride_bytes),
                                ctypes.c_int(pool.order), ctypes.c_int32(old_id), ctypes.c_int32(new_id),
                                ctypes.c_uint32(n_old), app.ctypes.data_as(ctypes.c_void_p),
                                ctypes.c_uint32(n_app))
    _check(rc)


def cow_append_batched(pool: HostPool, old_ids, new_ids, n_old, n_app, apps: Sequence[np.ndarray],
                       layer_count: int | None = None) -> None:
    """Batched copy-on-write append, in place.
    ``apps[s]`` is session s's dense [layer][K,V][token][head][dim] block of n_app[s] tokens."""
    L = pool.L if layer_count is None else int(layer_count)
    old_ids, new_ids = _ids(old_ids), _ids(new_ids)
    n_old = np.ascontiguousarray(np.asarray(n_old, dtype=np.uint32))
    n_app = np.ascontiguousarray(np.asarray(n_app, dtype=np.uint32))
    S = len(old_ids)
    assert len(new_ids) == S and len(n_old) == S and len(n_app) == S and len(apps) == S
    _assert_distinct(new_ids)
    if np.intersect1d(old_ids, new_ids).size:
        raise ValueError("oracle: a new page id is also an old page id")
    keep = [np.ascontiguousarray(a).view(np.uint8).reshape(-1) for a in apps]
    tokrow = pool.H * pool.D * pool.e
    ptrs = (ctypes.c_void_p * max(S, 1))()
    for s in range(S):
        if keep[s].size < L * pool.C * int(n_app[s]) * tokrow:
            raise ValueError("oracle: append buffer too small")
        ptrs[s] = keep[s].ctypes.data if keep[s].size else None
    rc = _load().kvo_cow_append_batched(pool._ptrs(), ctypes.c_uint32(L), ctypes.c_uint32(pool.C),
                                        ctypes.c_uint32(pool.num_pages), ctypes.c_uint32(pool.T),
                                        ctypes.c_uint32(pool.H), ctypes.c_uint32(pool.D),
                                        ctypes.c_uint32(pool.e),
                                        ctypes.c_uint64(pool.page_stride_bytes),
                                        ctypes.c_int(pool.order),
                                        old_ids.ctypes.data_as(ctypes.c_void_p),
                                        new_ids.ctypes.data_as(ctypes.c_void_p),
                                        n_old.ctypes.data_as(ctypes.c_void_p),
                                        n_app.ctypes.data_as(ctypes.c_void_p), ptrs,
                                        ctypes.c_uint32(S))
    _check(rc)


def _same_geometry(src: HostPool, dst: HostPool, L: int):
    if (src.C, src.H, src.D, src.e) != (dst.C, dst.H, dst.D, dst.e) or L > src.L or L > dst.L:
        raise ValueError("oracle: source and destination pools differ in C/H/D/e or have too few layers")


def repage(src: HostPool, src_ids, dst: HostPool, dst_ids, n_tokens: int,
           layer_count: int | None = None, threads: int = 1) -> None:
    """O-repage pool -> pool (SURVEY.md 8(c) reading 11, 8(f) NEXT-2), into ``dst`` in place."""
    L = min(src.L, dst.L) if layer_count is None else int(layer_count)
    _same_geometry(src, dst, L)
    src_ids, dst_ids = _ids(src_ids), _ids(dst_ids)
    _assert_distinct(dst_ids)
    rc = _load().kvo_repage(src._ptrs(), ctypes.c_uint32(src.num_pages),
                            ctypes.c_uint64(src.page_stride_bytes), ctypes.c_int(src.order),
                            ctypes.c_uint32(src.T),
                            src_ids.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint64(len(src_ids)),
                            dst._ptrs(), ctypes.c_uint32(dst.num_pages),
                            ctypes.c_uint64(dst.page_stride_bytes), ctypes.c_int(dst.order),
                            ctypes.c_uint32(dst.T),
                            dst_ids.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint64(len(dst_ids)),
                            ctypes.c_uint32(L), ctypes.c_uint32(src.C), ctypes.c_uint32(src.H),
                            ctypes.c_uint32(src.D), ctypes.c_uint32(src.e),
                            ctypes.c_uint64(int(n_tokens)), ctypes.c_int(threads))
    _check(rc)


def repage_batched(src: HostPool, src_ids, src_off, dst: HostPool, dst_ids, dst_off, n_tokens,
                   layer_count: int | None = None, threads: int = 1) -> None:
    """Batched O-repage pool -> pool, into ``dst`` in place."""
    L = min(src.L, dst.L) if layer_count is None else int(layer_count)
    _same_geometry(src, dst, L)
    src_ids, dst_ids = _ids(src_ids), _ids(dst_ids)
    _assert_distinct(dst_ids)
    src_off = np.ascontiguousarray(np.asarray(src_off, dtype=np.int64))
    dst_off = np.ascontiguousarray(np.asarray(dst_off, dtype=np.int64))
    ntok = np.ascontiguousarray(np.asarray(n_tokens, dtype=np.uint64))
    R = len(ntok)
    assert len(src_off) == R + 1 and len(dst_off) == R + 1
    rc = _load().kvo_repage_batched(src._ptrs(), ctypes.c_uint32(src.num_pages),
                                    ctypes.c_uint64(src.page_stride_bytes), ctypes.c_int(src.order),
                                    ctypes.c_uint32(src.T),
                                    src_ids.ctypes.data_as(ctypes.c_void_p),
                                    src_off.ctypes.data_as(ctypes.c_void_p), dst._ptrs(),
                                    ctypes.c_uint32(dst.num_pages),
                                    ctypes.c_uint64(dst.page_stride_bytes), ctypes.c_int(dst.order),
                                    ctypes.c_uint32(dst.T),
                                    dst_ids.ctypes.data_as(ctypes.c_void_p),
                                    dst_off.ctypes.data_as(ctypes.c_void_p),
                                    ntok.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(R),
                                    ctypes.c_uint32(L), ctypes.c_uint32(src.C),
                                    ctypes.c_uint32(src.H), ctypes.c_uint32(src.D),
                                    ctypes.c_uint32(src.e), ctypes.c_int(threads))
    _check(rc)


# ----------------------------------------------------------------------------------------------
# the definitions as literal Python loops (tiny cases only)
# ----------------------------------------------------------------------------------------------
def _pool_off(pool: HostPool, g, t, h, d) -> int:
    # PAPER.md:L207 region (layer, page_idx, K|V) + in-page order: NHD or HND
    if pool.order == NHD:
        return g * pool.page_stride_bytes + ((t * pool.H + h) * pool.D + d) * pool.e
    return g * pool.page_stride_bytes + ((h * pool.T + t) * pool.D + d) * pool.e


def _buf_index(layout, p, n, l, L, c, C, t, T, h, H, d, D) -> int:
    if layout == PAGE_FIRST:  # BASELINE.json:configs[0]
        return ((((p * L + l) * C + c) * T + t) * H + h) * D + d
    return ((((l * C + c) * n + p) * T + t) * H + h) * D + d


def pack_py(pool: HostPool, ids, layer_count=None, layout=PAGE_FIRST) -> np.ndarray:
    L = pool.L if layer_count is None else int(layer_count)
    C, T, H, D, e = pool.C, pool.T, pool.H, pool.D, pool.e
    ids = [int(i) for i in ids]
    n = len(ids)
    for g in ids:
        if not (0 <= g < pool.num_pages):
            raise IndexError("oracle: page id out of range")
    buf = np.zeros(n * L * C * T * H * D * e, dtype=np.uint8)
    for p in range(n):
        for l in range(L):
            for c in range(C):
                for t in range(T):
                    for h in range(H):
                        for d in range(D):
                            s = _pool_off(pool, ids[p], t, h, d)
                            o = _buf_index(layout, p, n, l, L, c, C, t, T, h, H, d, D) * e
                            buf[o:o + e] = pool.slabs[l * C + c][s:s + e]
    return buf


def unpack_py(src, dst_ids, pool: HostPool, Ts: int, n_tokens: int, layer_count=None,
              layout=PAGE_FIRST) -> None:
    L = pool.L if layer_count is None else int(layer_count)
    C, Td, H, D, e = pool.C, pool.T, pool.H, pool.D, pool.e
    src = np.ascontiguousarray(src).view(np.uint8).reshape(-1)
    dst_ids = [int(i) for i in dst_ids]
    if len(set(dst_ids)) != len(dst_ids):
        raise ValueError("oracle: duplicate destination page ids")
    n_dst = -(-n_tokens // Td)
    n_src = -(-n_tokens // Ts)
    if len(dst_ids) != n_dst:
        raise ValueError("oracle: len(dst_ids) != ceil(n_tokens / Td)")
    for g in dst_ids:
        if not (0 <= g < pool.num_pages):
            raise IndexError("oracle: page id out of range")
    for q in range(n_dst):
        for l in range(L):
            for c in range(C):
                for u in range(Td):
                    for h in range(H):
                        for d in range(D):
                            j = q * Td + u
                            o = _pool_off(pool, dst_ids[q], u, h, d)
                            if j < n_tokens:
                                s = _buf_index(layout, j // Ts, n_src, l, L, c, C, j % Ts, Ts,
                                               h, H, d, D) * e
                                pool.slabs[l * C + c][o:o + e] = src[s:s + e]
                            else:
                                pool.slabs[l * C + c][o:o + e] = 0
