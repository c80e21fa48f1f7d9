"""Pins of the chained-paged-hashing oracle (oracle/chain_oracle.{c,py}, DESIGN.md
readings H1-H4).  Nothing here comes from the CUDA path.

What fixes the oracle besides itself:
* the published 64-bit FNV-1a vectors (tests/golden/H1_fnv1a64_vectors.txt);
* a closed form tied to those vectors: for a message whose bytes after the first are all zero the XOR
  steps are identities, so FNV1a(b, 0, ..., 0) = FNV1a(b) * prime**(n-1) mod 2**64 -- this checks the
  little-endian encoding of identities and ids (a big-endian or 4-byte encoding fails it);
* two separately written implementations (literal Python integers vs the C loops);
* the properties the paper asks of the ids: an id stands for the complete page-aligned prefix (equal
  prefixes <=> equal ids up to the first differing page, all later ids differ), only whole pages get
  ids, sessions are independent, the root separates namespaces.
"""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from oracle import chain_oracle as co
from paper_2606_31093_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "H1_fnv1a64_vectors.txt")
P = 0x100000001B3
M = 1 << 64


def vectors():
    out = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        msg, h = line.split()
        out.append((msg.strip('"').encode(), int(h, 16)))
    return out


def test_published_fnv1a64_vectors():
    vs = vectors()
    assert len(vs) == 5
    for msg, h in vs:
        assert co.fnv1a64_py(msg) == h, msg
        assert co.fnv1a64(msg) == h, msg


def test_zero_tail_closed_form_pins_the_little_endian_encoding():
    """identity 0x61 as LE64 is 'a' followed by seven zero bytes: digest = FNV1a('a') * prime**7."""
    fa = dict(vectors())[b"a"]
    digest = fa * pow(P, 7, M) % M
    assert co.fnv1a64_py((0x61).to_bytes(8, "little")) == digest
    # T = 1, root = 0: message = LE64(0) || LE64(digest); eight leading zero bytes only multiply the basis
    h = co.FNV_BASIS * pow(P, 8, M) % M
    for b in digest.to_bytes(8, "little"):
        h = (h ^ b) * P % M
    assert co.chain_py([0x61], 1, root=0) == [h]
    assert co.chain([0x61], 1, root=0).tolist() == [h]
    # two identities per page: the second identity's bytes follow the first's (order matters)
    assert co.chain_py([0x61, 0x62], 2, root=0) != co.chain_py([0x62, 0x61], 2, root=0)
    d2 = co.fnv1a64_py((0x61).to_bytes(8, "little") + (0x62).to_bytes(8, "little"))
    assert co.chain([0x61, 0x62], 2, root=5)[0] == co.fnv1a64_py((5).to_bytes(8, "little") + d2.to_bytes(8, "little"))


@settings(max_examples=60, deadline=None)
@given(st.lists(st.integers(0, M - 1), min_size=0, max_size=70), st.integers(1, 9), st.integers(0, M - 1))
def test_c_loops_equal_python_integers(ident, T, root):
    want = co.chain_py(ident, T, root)
    got = co.chain(ident, T, root)
    assert got.tolist() == want
    assert len(want) == len(ident) // T  # H4: only whole pages


def test_fnv_c_equals_python_on_random_messages():
    rng = np.random.default_rng(3)
    for n in [0, 1, 7, 8, 9, 16, 127, 128, 1000]:
        msg = rng.integers(0, 256, size=n, dtype=np.uint8).tobytes()
        assert co.fnv1a64(msg) == co.fnv1a64_py(msg)


def test_id_stands_for_the_whole_page_aligned_prefix():
    rng = np.random.default_rng(5)
    T, n = 16, 16 * 40 + 11
    a = rng.integers(0, W.VOCAB, size=n).astype(np.uint64)
    ids = co.chain(a, T)
    assert ids.size == 40 and len(set(ids.tolist())) == 40
    # a longer session with the same beginning has the same first 40 ids
    b = np.concatenate([a[:16 * 40], rng.integers(0, W.VOCAB, size=100).astype(np.uint64)])
    assert np.array_equal(co.chain(b, T)[:40], ids)
    # the partial tail page has no id and does not influence any id
    assert np.array_equal(co.chain(a[:16 * 40], T), ids)
    # changing one identity in page k leaves ids < k and changes every id >= k
    for k, t in [(0, 0), (17, 5), (39, 15)]:
        c = a.copy()
        c[k * T + t] ^= np.uint64(1)
        ic = co.chain(c, T)
        assert np.array_equal(ic[:k], ids[:k])
        assert (ic[k:] != ids[k:]).all()
    # swapping two pages changes both (the chain is order-sensitive, not a set hash)
    c = a.copy()
    c[0:16], c[16:32] = a[16:32], a[0:16]
    assert (co.chain(c, T)[:2] != ids[:2]).all()
    # another root, another namespace: no id in common
    assert not set(co.chain(a, T, root=1).tolist()) & set(ids.tolist())
    # the page size is part of the convention ("consistent page conventions")
    assert co.chain(a, 32)[0] != ids[1]


def test_batched_equals_per_session_and_shared_prefixes_share_ids():
    wb = W.identity_batch(seed=1, n_sessions=12, lo=40, hi=900, share=0.7)
    T = 16
    roots = None
    ids, poff = co.chain_batched(wb.ident, wb.tok_offsets, T, roots)
    ids4, poff4 = co.chain_batched(wb.ident, wb.tok_offsets, T, roots, threads=4)
    assert np.array_equal(ids, ids4) and np.array_equal(poff, poff4)
    lens = np.diff(wb.tok_offsets)
    assert np.array_equal(np.diff(poff), lens // T)
    first = ids[poff[0]:poff[1]]
    assert (wb.shared_prefix[1:] > 0).any()
    for s in range(12):
        mine = ids[poff[s]:poff[s + 1]]
        assert np.array_equal(mine, co.chain(wb.ident[wb.tok_offsets[s]:wb.tok_offsets[s + 1]], T))
        k = int(wb.shared_prefix[s]) // T  # whole pages copied from session 0
        k = min(k, mine.size, first.size)
        assert np.array_equal(mine[:k], first[:k])
        if s and mine.size > k and first.size > k:  # the first page past the copy differs
            assert mine[k] != first[k]
    # per-session roots
    r = np.arange(12, dtype=np.uint64) + np.uint64(100)
    ids_r, _ = co.chain_batched(wb.ident, wb.tok_offsets, T, r)
    for s in range(12):
        assert np.array_equal(ids_r[poff[s]:poff[s + 1]],
                              co.chain(wb.ident[wb.tok_offsets[s]:wb.tok_offsets[s + 1]], T, root=int(r[s])))


def test_empty_and_degenerate_sessions():
    assert co.chain([], 16).size == 0
    assert co.chain([1, 2, 3], 16).size == 0  # shorter than a page
    ids, poff = co.chain_batched(np.arange(40, dtype=np.uint64), [0, 0, 15, 15, 40], 16)
    assert poff.tolist() == [0, 0, 0, 0, 1]
    assert ids.tolist() == co.chain_py(list(range(15, 31)), 16)
    ids, poff = co.chain_batched(np.zeros(0, dtype=np.uint64), [0], 16)
    assert ids.size == 0 and poff.tolist() == [0]
    with pytest.raises(ValueError):
        co.chain_batched(np.zeros(4, dtype=np.uint64), [0, 3, 2], 1)


def test_a_chain_continues_from_its_last_id():
    """Turn k+1 hashes only its new pages: the ids of [old pages | new pages] equal the old ids followed by a
    chain over the new pages rooted at the last old id (what `roots` is for; "hashes its
    predecessor")."""
    rng = np.random.default_rng(11)
    T = 16
    a = rng.integers(0, W.VOCAB, size=T * 50).astype(np.uint64)
    full = co.chain(a, T)
    for cut in (1, 17, 49):
        head = co.chain(a[:cut * T], T)
        tail = co.chain(a[cut * T:], T, root=int(head[-1]))
        assert np.array_equal(np.concatenate([head, tail]), full)
    assert co.chain_py(a[:64].tolist(), T) + co.chain_py(a[64:128].tolist(), T, root=int(full[3])) == full[:8].tolist()
