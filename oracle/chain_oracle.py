"""oracle/chain_oracle.py -- CPU ORACLE for chained paged hashing.  TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` leg may import this
module; it imports nothing from ``paper_2606_31093_b200`` and the CUDA path imports nothing from here.

PAPER.md:L276 (Sec. 5.1): "each page ID hashes its predecessor together with the current page's content
identities, thereby representing the complete page-aligned prefix."  The paper names neither the hash
nor the encoding; readings H1-H4 are stated in
``chain_oracle.c``.  Two implementations of the same definition:

* ``fnv1a64_py`` / ``chain_py``  -- literal Python integer arithmetic (mod 2**64), small cases;
* ``fnv1a64`` / ``chain`` / ``chain_batched`` -- the loops of ``chain_oracle.c`` (gcc -O2) via ctypes.

Pins (tests/test_chain_oracle_pins.py): the published FNV-1a 64-bit test vectors (tests/golden/
H1_fnv1a64_vectors.txt), the two implementations against each other, prefix / sensitivity / root /
tail invariants of the chain.  The HASH FUNCTION ITSELF IS A READING (the paper specifies none):
parity is pinned to FNV-1a's published definition, not to anything the paper prints.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chain_oracle.c")
_LIB = os.path.join(_HERE, "libchainoracle.so")

FNV_BASIS = 0xCBF29CE484222325
FNV_PRIME = 0x100000001B3
DEFAULT_ROOT = FNV_BASIS  # chains start from the FNV offset basis unless the caller names a root
_M64 = (1 << 64) - 1


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.cho_fnv1a64.restype = ctypes.c_uint64
        _lib.cho_fnv1a64.argtypes = [ctypes.c_void_p, ctypes.c_uint64]
        _lib.cho_chain.restype = ctypes.c_uint64
        _lib.cho_chain.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_void_p]
        _lib.cho_chain_batched.restype = ctypes.c_int64
        _lib.cho_chain_batched.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32,
                                           ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p,
                                           ctypes.c_int]
    return _lib


# ---- literal Python definition -------------------------------------------------------------------
def fnv1a64_py(msg: bytes) -> int:
    h = FNV_BASIS
    for b in msg:
        h = ((h ^ b) * FNV_PRIME) & _M64
    return h


def chain_py(ident, T: int, root: int = DEFAULT_ROOT) -> list:
    """Page ids of one session: id_k = FNV1a(LE64(id_{k-1}) || LE64(FNV1a(LE64 identities of page k)))."""
    ident = [int(x) for x in ident]
    ids, prev = [], int(root)
    for k in range(len(ident) // T):
        page = b"".join(x.to_bytes(8, "little") for x in ident[k * T:(k + 1) * T])
        d = fnv1a64_py(page)
        prev = fnv1a64_py(prev.to_bytes(8, "little") + d.to_bytes(8, "little"))
        ids.append(prev)
    return ids


# ---- C oracle ------------------------------------------------------------------------------------
def fnv1a64(msg: bytes) -> int:
    buf = np.frombuffer(bytes(msg), dtype=np.uint8)
    return int(_load().cho_fnv1a64(buf.ctypes.data if buf.size else None, buf.size))


def chain(ident, T: int, root: int = DEFAULT_ROOT) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(ident, dtype=np.uint64))
    out = np.zeros(a.size // T, dtype=np.uint64)
    n = _load().cho_chain(a.ctypes.data, a.size, int(T), int(root), out.ctypes.data)
    assert n == out.size
    return out


def chain_batched(ident, tok_off, T: int, roots=None, default_root: int = DEFAULT_ROOT, threads: int = 1):
    """(ids, page_off): ids of all sessions back to back, page_off[s] = index of session s's first id."""
    a = np.ascontiguousarray(np.asarray(ident, dtype=np.uint64))
    off = np.ascontiguousarray(np.asarray(tok_off, dtype=np.int64))
    S = off.size - 1
    lens = np.diff(off)
    if S < 0 or (lens < 0).any() or (S and off[0] < 0):
        raise ValueError("token offsets must be non-negative and non-decreasing")
    out = np.zeros(int((lens // T).sum()), dtype=np.uint64)
    page_off = np.zeros(S + 1, dtype=np.int64)
    r = None if roots is None else np.ascontiguousarray(np.asarray(roots, dtype=np.uint64))
    n = _load().cho_chain_batched(a.ctypes.data, off.ctypes.data, S, int(T), None if r is None else r.ctypes.data,
                                  int(default_root), out.ctypes.data, page_off.ctypes.data, int(threads))
    assert n == out.size
    return out, page_off
