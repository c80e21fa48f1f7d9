"""Pins for the CPU oracle (oracle/kv_oracle.{c,py}) -- nothing here calls the CUDA path.

Each pin is something OTHER than the oracle's own formula: values derived by hand from the
paper's addressing (tests/golden/), numpy library routines (take / transpose / reshape) for the
special cases the definition reduces to, a separately written pull formulation, and invariants
(bijectivity, untouched bytes, zero-pad count, 64-bit offsets).  Citations: PAPER.md:L207
(sec. 4.1.1 addressing), PAPER.md:L214 (sec. 4.1.2 migration), PAPER.md:L238 (valid token length,
CoW), BASELINE.json:configs[0] (page-first layout), configs[4] (re-paging), SURVEY.md 8(c).
"""
import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings
from hypothesis import strategies as st

from oracle import kv_oracle as ko

IMPLS = {
    "c": (ko.pack, ko.unpack),
    "py": (ko.pack_py, ko.unpack_py),
}
DT = {1: np.uint8, 2: np.uint16, 4: np.uint32}


# ---------------------------------------------------------------------------------------------
# helpers: pools as a stacked numpy array A[L,C,P,T,H,D] (dense stride) <-> HostPool
# ---------------------------------------------------------------------------------------------
def pool_from_array(A: np.ndarray, pad: int = 0, pad_fill: int = 0xA5, order: int = 0) -> ko.HostPool:
    """A is the LOGICAL pool A[L,C,P,T,H,D]; order 1 (HND) stores every page as [H][T][D]."""
    L, C, P, T, H, D = A.shape
    e = A.dtype.itemsize
    row = T * H * D * e
    stride = row + pad
    phys = A if order == 0 else np.ascontiguousarray(A.transpose(0, 1, 2, 4, 3, 5))
    slabs = []
    for l in range(L):
        for c in range(C):
            s = np.full((P, stride), pad_fill, dtype=np.uint8)
            s[:, :row] = np.ascontiguousarray(phys[l, c]).reshape(P, -1).view(np.uint8)
            slabs.append(s.reshape(-1))
    return ko.HostPool(slabs, L, C, P, T, H, D, e, stride, order)


def array_from_pool(pool: ko.HostPool) -> np.ndarray:
    """The LOGICAL pool A[L,C,P,T,H,D], whatever the in-page order."""
    row = pool.row_bytes
    out = np.empty((pool.L, pool.C, pool.num_pages, pool.T, pool.H, pool.D), dtype=DT[pool.e])
    for l in range(pool.L):
        for c in range(pool.C):
            s = pool.slabs[l * pool.C + c].reshape(pool.num_pages, pool.page_stride_bytes)[:, :row]
            v = np.ascontiguousarray(s).view(DT[pool.e])
            if pool.order == 0:
                out[l, c] = v.reshape(pool.num_pages, pool.T, pool.H, pool.D)
            else:
                out[l, c] = v.reshape(pool.num_pages, pool.H, pool.T, pool.D).transpose(0, 2, 1, 3)
    return out


def w1_array():
    L, C, P, T, H, D = 2, 2, 4, 2, 1, 2
    A = np.zeros((L, C, P, T, H, D), dtype=np.uint16)
    for l in range(L):
        for c in range(C):
            for g in range(P):
                for t in range(T):
                    for d in range(D):
                        A[l, c, g, t, 0, d] = 1000 * (2 * l + c) + 4 * g + 2 * t + d
    return A


# ---------------------------------------------------------------------------------------------
# 1. hand-computed worked examples (tests/golden)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("impl", IMPLS)
def test_W1_pack_page_first(impl, golden):
    pack, _ = IMPLS[impl]
    buf = pack(pool_from_array(w1_array()), [3, 0]).view(np.uint16)
    assert buf.tolist() == golden("W1_pack_page_first.txt")


@pytest.mark.parametrize("impl", IMPLS)
def test_W1_pack_layer_first(impl, golden):
    pack, _ = IMPLS[impl]
    buf = pack(pool_from_array(w1_array()), [3, 0], layout=ko.LAYER_FIRST).view(np.uint16)
    assert buf.tolist() == golden("W1_pack_layer_first.txt")


@pytest.mark.parametrize("impl", IMPLS)
def test_W2_repage_padded_tail(impl, golden):
    _, unpack = IMPLS[impl]
    src = np.array(golden("W1_pack_page_first.txt"), dtype=np.uint16)
    dst = pool_from_array(np.full((2, 2, 3, 4, 1, 2), 7777, dtype=np.uint16))
    unpack(src, [2], dst, Ts=2, n_tokens=3)
    got = np.concatenate([s.view(np.uint16) for s in dst.slabs]).tolist()
    assert got == golden("W2_repage_padded_tail.txt")


# ---------------------------------------------------------------------------------------------
# 2. special cases that reduce to library routines
# ---------------------------------------------------------------------------------------------
SHAPES = [  # L, C, P, T, H, D, e
    (1, 1, 5, 1, 1, 1, 1),
    (2, 2, 9, 3, 2, 4, 2),
    (3, 2, 17, 4, 3, 5, 4),
    (4, 2, 32, 16, 2, 8, 2),
    (2, 1, 7, 2, 1, 3, 1),
]


def rand_array(rng, L, C, P, T, H, D, e):
    return rng.integers(0, 256 ** e, size=(L, C, P, T, H, D), dtype=np.uint64).astype(DT[e])


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("pad", [0, 8])
def test_pack_is_numpy_take_transpose(impl, shape, pad):
    pack, _ = IMPLS[impl]
    rng = np.random.default_rng(hash(shape) & 0xFFFF)
    A = rand_array(rng, *shape)
    P = shape[2]
    ids = rng.integers(0, P, size=P + 3)  # duplicates allowed for pack (reading 5)
    pool = pool_from_array(A, pad=pad)
    got = pack(pool, ids).view(A.dtype)
    want = np.take(A, ids, axis=2).transpose(2, 0, 1, 3, 4, 5)  # [page][layer][kv][t][h][d]
    assert np.array_equal(got, want.reshape(-1))
    got_lf = pack(pool, ids, layout=ko.LAYER_FIRST).view(A.dtype)
    assert np.array_equal(got_lf, np.take(A, ids, axis=2).reshape(-1))  # [layer][kv][page]...


@pytest.mark.parametrize("impl", IMPLS)
def test_pack_sequential_single_slab_is_memcpy(impl):
    pack, _ = IMPLS[impl]
    rng = np.random.default_rng(3)
    A = rand_array(rng, 1, 1, 11, 4, 2, 3, 2)
    pool = pool_from_array(A)
    buf = pack(pool, np.arange(11))
    assert buf.tobytes() == pool.slabs[0].tobytes()


@pytest.mark.parametrize("impl", IMPLS)
def test_pack_layer_subset_uses_first_layers(impl):
    pack, _ = IMPLS[impl]
    rng = np.random.default_rng(4)
    A = rand_array(rng, 3, 2, 6, 2, 2, 2, 2)
    ids = [5, 1, 2]
    got = pack(pool_from_array(A), ids, layer_count=2).view(A.dtype)
    want = np.take(A[:2], ids, axis=2).transpose(2, 0, 1, 3, 4, 5)
    assert np.array_equal(got, want.reshape(-1))


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("Ts,Td,ntok", [(2, 4, 8), (2, 4, 7), (4, 2, 9), (3, 5, 11), (16, 64, 130),
                                        (4, 4, 12), (4, 4, 10), (6, 4, 1), (1, 7, 20)])
def test_repage_sequential_is_reshape_plus_zero_fill(impl, Ts, Td, ntok):
    """Sequence tensor S[L,C,ntok,H,D] cut into Ts-token pages IS the page-first buffer; unpacking
    into pages 0..n_dst-1 of a pool must give S re-cut into Td-token pages, zero padded."""
    _, unpack = IMPLS[impl]
    L, C, H, D, e = 2, 2, 2, 3, 2
    rng = np.random.default_rng(Ts * 100 + Td)
    S = rng.integers(1, 65536, size=(L, C, ntok, H, D), dtype=np.uint64).astype(np.uint16)
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    Spad = np.full((L, C, n_src * Ts, H, D), 0xBEEF, dtype=np.uint16)  # stale tail tokens: ignored
    Spad[:, :, :ntok] = S
    buf = Spad.reshape(L, C, n_src, Ts, H, D).transpose(2, 0, 1, 3, 4, 5).copy().reshape(-1)
    P = n_dst + 2
    dst = pool_from_array(np.full((L, C, P, Td, H, D), 0x7777, dtype=np.uint16))
    unpack(buf, np.arange(n_dst), dst, Ts=Ts, n_tokens=ntok)
    B = array_from_pool(dst)
    seq = B[:, :, :n_dst].reshape(L, C, n_dst * Td, H, D)
    assert np.array_equal(seq[:, :, :ntok], S)
    assert np.all(seq[:, :, ntok:] == 0)
    assert np.all(B[:, :, n_dst:] == 0x7777)  # untouched pages
    # layer-first source: [layer][kv][page][t][h][d] is Spad's own order
    dst2 = pool_from_array(np.full((L, C, P, Td, H, D), 0x7777, dtype=np.uint16))
    unpack(Spad.reshape(-1), np.arange(n_dst), dst2, Ts=Ts, n_tokens=ntok, layout=ko.LAYER_FIRST)
    assert np.array_equal(array_from_pool(dst2), B)


# ---------------------------------------------------------------------------------------------
# 3. separately written pull formulation: de-linearise every OUTPUT byte offset by div/mod
# ---------------------------------------------------------------------------------------------
def pull_pack(pool: ko.HostPool, ids, L, layout=0):
    C, T, H, D, e = pool.C, pool.T, pool.H, pool.D, pool.e
    n = len(ids)
    out = np.zeros(n * L * C * T * H * D * e, dtype=np.uint8)
    for o in range(out.size):
        b = o % e; r = o // e
        d = r % D; r //= D
        h = r % H; r //= H
        t = r % T; r //= T
        if layout == 0:
            c = r % C; r //= C
            l = r % L; p = r // L
        else:
            p = r % n; r //= n
            c = r % C; l = r // C
        out[o] = pool.slabs[l * C + c][int(ids[p]) * pool.page_stride_bytes
                                      + ((t * H + h) * D + d) * e + b]
    return out


def pull_unpack(src, dst_ids, pool: ko.HostPool, Ts, n_tokens, L):
    """Returns the expected slabs: for every byte of every destination slab decide where it
    comes from (page-first source only)."""
    C, Td, H, D, e = pool.C, pool.T, pool.H, pool.D, pool.e
    row = Td * H * D * e
    where = {int(g): q for q, g in enumerate(dst_ids)}
    src = np.ascontiguousarray(src).view(np.uint8).reshape(-1)
    out = [s.copy() for s in pool.slabs]
    for lc in range(L * C):
        l, c = divmod(lc, C)
        for o in range(out[lc].size):
            g, within = divmod(o, pool.page_stride_bytes)
            if g not in where or within >= row:
                continue  # untouched page, or stride padding
            b = within % e; r = within // e
            d = r % D; r //= D
            h = r % H; u = r // H
            j = where[g] * Td + u
            if j >= n_tokens:
                out[lc][o] = 0
            else:
                p, t = divmod(j, Ts)
                out[lc][o] = src[(((((p * L + l) * C + c) * Ts + t) * H + h) * D + d) * e + b]
    return out


tiny_dims = st.tuples(st.integers(1, 3), st.integers(1, 2), st.integers(1, 6), st.integers(1, 4),
                      st.integers(1, 2), st.integers(1, 3), st.sampled_from([1, 2, 4]))


@settings(max_examples=40, deadline=None, suppress_health_check=list(HealthCheck))
@given(dims=tiny_dims, pad=st.sampled_from([0, 4]), seed=st.integers(0, 2 ** 16),
       layout=st.sampled_from([0, 1]))
def test_pack_push_equals_pull(dims, pad, seed, layout):
    L, C, P, T, H, D, e = dims
    rng = np.random.default_rng(seed)
    pool = pool_from_array(rand_array(rng, L, C, P, T, H, D, e), pad=pad)
    ids = rng.integers(0, P, size=rng.integers(0, P + 2))
    want = pull_pack(pool, ids, L, layout)
    assert np.array_equal(ko.pack(pool, ids, layout=layout), want)
    assert np.array_equal(ko.pack_py(pool, ids, layout=layout), want)


@settings(max_examples=40, deadline=None, suppress_health_check=list(HealthCheck))
@given(dims=tiny_dims, Ts=st.integers(1, 5), pad=st.sampled_from([0, 4]),
       seed=st.integers(0, 2 ** 16), data=st.data())
def test_unpack_push_equals_pull(dims, Ts, pad, seed, data):
    L, C, P, Td, H, D, e = dims
    rng = np.random.default_rng(seed)
    n_tokens = data.draw(st.integers(0, P * Td))
    n_dst, n_src = -(-n_tokens // Td), -(-n_tokens // Ts)
    src = rng.integers(0, 256, size=n_src * L * C * Ts * H * D * e, dtype=np.uint8)
    dst_ids = rng.permutation(P)[:n_dst]
    base = pool_from_array(rand_array(rng, L, C, P, Td, H, D, e), pad=pad)
    want = pull_unpack(src, dst_ids, base, Ts, n_tokens, L)
    for unpack in (ko.unpack, ko.unpack_py):
        pool = base.copy()
        unpack(src, dst_ids, pool, Ts=Ts, n_tokens=n_tokens)
        for a, b in zip(pool.slabs, want):
            assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# 4. invariants (BASELINE.json:north_star): round trip, bijectivity, untouched bytes, pad count
# ---------------------------------------------------------------------------------------------
def tagged_array(L, C, P, T, H, D):
    n = L * C * P * T * H * D
    return (np.arange(1, n + 1, dtype=np.uint32)).reshape(L, C, P, T, H, D)  # tag 0 = "unwritten"


def test_pack_is_a_bijection_onto_touched_elements():
    A = tagged_array(3, 2, 12, 4, 2, 3)
    ids = np.random.default_rng(5).permutation(12)[:7]
    buf = ko.pack(pool_from_array(A), ids).view(np.uint32)
    assert buf.size == A[:, :, ids].size
    assert np.all(buf != 0), "some buffer element was never written"
    assert len(np.unique(buf)) == buf.size, "some pool element was copied twice"
    assert set(buf.tolist()) == set(A[:, :, ids].reshape(-1).tolist())


@pytest.mark.parametrize("Ts,Td,ntok", [(4, 4, 28), (2, 8, 50), (8, 2, 13), (3, 4, 17)])
def test_unpack_writes_each_touched_element_once_and_nothing_else(Ts, Td, ntok):
    L, C, H, D, P = 2, 2, 2, 3, 20
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    src = np.arange(1, n_src * L * C * Ts * H * D + 1, dtype=np.uint32)
    SENT = 0xFFFFFFFF
    pool = pool_from_array(np.full((L, C, P, Td, H, D), SENT, dtype=np.uint32), pad=16, pad_fill=0x5A)
    dst_ids = np.random.default_rng(6).permutation(P)[:n_dst]
    ko.unpack(src, dst_ids, pool, Ts=Ts, n_tokens=ntok)
    B = array_from_pool(pool)
    touched = B[:, :, dst_ids].reshape(-1)
    data = touched[touched != 0]
    assert np.all(data != SENT), "a slot of a touched page was left unwritten"
    assert len(np.unique(data)) == data.size == ntok * L * C * H * D
    # valid source elements = tokens < ntok of every (page, layer, kv)
    S = src.reshape(n_src, L, C, Ts, H, D).transpose(1, 2, 0, 3, 4, 5).reshape(L, C, n_src * Ts, H, D)
    assert set(data.tolist()) == set(S[:, :, :ntok].reshape(-1).tolist())
    # zero-pad count: (n_dst*Td - n_tokens) * L*C*H*D elements
    assert int((touched == 0).sum()) == (n_dst * Td - ntok) * L * C * H * D
    # untouched pages and stride padding byte-identical
    mask = np.ones(P, bool); mask[dst_ids] = False
    assert np.all(B[:, :, mask] == SENT)
    for s in pool.slabs:
        assert np.all(s.reshape(P, -1)[:, pool.row_bytes:] == 0x5A)


@pytest.mark.parametrize("shape", SHAPES[1:])
def test_round_trip_identity(shape):
    L, C, P, T, H, D, e = shape
    rng = np.random.default_rng(7)
    A = rand_array(rng, *shape)
    Bfill = rand_array(rng, *shape)
    n = P // 2
    ids = rng.permutation(P)[:n]
    ids2 = rng.permutation(P)[:n]
    poolB = pool_from_array(Bfill)
    buf = ko.pack(pool_from_array(A), ids)
    ko.unpack(buf, ids2, poolB, Ts=T, n_tokens=n * T)
    B = array_from_pool(poolB)
    assert np.array_equal(B[:, :, ids2], A[:, :, ids])
    mask = np.ones(P, bool); mask[ids2] = False
    assert np.array_equal(B[:, :, mask], Bfill[:, :, mask])
    # and packing B at ids2 gives the same buffer back
    assert np.array_equal(ko.pack(poolB, ids2), buf)


def test_bit_patterns_survive():
    """bf16 NaN payloads, -0, subnormals, inf: copy is bitwise."""
    pats = np.array([0x7FC1, 0xFFFF, 0x8000, 0x0001, 0x7F80, 0xFF80, 0x0000, 0x7F81], dtype=np.uint16)
    A = np.resize(pats, (1, 2, 3, 2, 2, 4)).astype(np.uint16)
    buf = ko.pack(pool_from_array(A), [2, 0]).view(np.uint16)
    assert np.array_equal(buf, A[:, :, [2, 0]].transpose(2, 0, 1, 3, 4, 5).reshape(-1))


def test_offsets_beyond_4GiB():
    """SURVEY.md 8(c) reading 18: one slab of 262,145 pages x 16 KiB; ids=[262144, 0] must return
    the last page first.  The slab is calloc-backed; only two pages are ever touched."""
    P, T, H, D, e = 262145, 16, 4, 128, 2
    row = T * H * D * e
    slab = np.zeros(P * row, dtype=np.uint8)
    slab[:row] = 0x11
    slab[(P - 1) * row:] = 0xEE
    pool = ko.HostPool([slab], 1, 1, P, T, H, D, e, row)
    buf = ko.pack(pool, [P - 1, 0])
    assert np.all(buf[:row] == 0xEE) and np.all(buf[row:] == 0x11)
    ko.unpack(buf, [P - 2, 1], pool, Ts=T, n_tokens=2 * T)
    assert np.all(slab[(P - 2) * row:(P - 1) * row] == 0xEE) and np.all(slab[row:2 * row] == 0x11)
    assert not slab[2 * row:3 * row].any()


# ---------------------------------------------------------------------------------------------
# 5. batched, threads, errors, CoW
# ---------------------------------------------------------------------------------------------
def test_batched_equals_per_request_and_threads_change_nothing():
    rng = np.random.default_rng(8)
    A = rand_array(rng, 3, 2, 40, 4, 2, 4, 2)
    pool = pool_from_array(A)
    off = np.array([0, 5, 5, 12, 20])
    ids = rng.permutation(40)[:20]
    bufs = ko.pack_batched(pool, ids, off, threads=3)
    for r in range(4):
        want = np.take(A, ids[off[r]:off[r + 1]], axis=2).transpose(2, 0, 1, 3, 4, 5).reshape(-1)
        assert np.array_equal(bufs[r].view(np.uint16), want)
        assert np.array_equal(bufs[r], ko.pack(pool, ids[off[r]:off[r + 1]], threads=1))
    # batched re-paging unpack == per-request unpack
    Td = 8
    ntok = np.array([5 * 4, 0, 7 * 4 - 3, 8 * 4 - 1])
    nd = -(-ntok // Td)
    doff = np.concatenate([[0], np.cumsum(nd)])
    dids = rng.permutation(30)[:doff[-1]]
    base = pool_from_array(rand_array(rng, 3, 2, 30, Td, 2, 4, 2))
    p1, p2 = base.copy(), base.copy()
    ko.unpack_batched(bufs, dids, doff, ntok, p1, Ts=4, threads=4)
    for r in range(4):
        ko.unpack(bufs[r], dids[doff[r]:doff[r + 1]], p2, Ts=4, n_tokens=int(ntok[r]))
    for a, b in zip(p1.slabs, p2.slabs):
        assert np.array_equal(a, b)


def test_errors():
    pool = pool_from_array(w1_array())
    for pack in (ko.pack, ko.pack_py):
        with pytest.raises(IndexError):
            pack(pool, [4])
        with pytest.raises(IndexError):
            pack(pool, [-1])
    buf = ko.pack(pool, [0, 1])
    for unpack in (ko.unpack, ko.unpack_py):
        with pytest.raises(ValueError):
            unpack(buf, [1, 1], pool.copy(), Ts=2, n_tokens=4)  # duplicate destination
        with pytest.raises(ValueError):
            unpack(buf, [1], pool.copy(), Ts=2, n_tokens=4)  # wrong page count
        with pytest.raises(IndexError):
            unpack(buf, [1, 9], pool.copy(), Ts=2, n_tokens=4)


def test_empty_calls_touch_nothing():
    pool = pool_from_array(w1_array())
    before = [s.copy() for s in pool.slabs]
    assert ko.pack(pool, []).size == 0
    ko.unpack(np.zeros(0, np.uint8), [], pool, Ts=2, n_tokens=0)
    for a, b in zip(pool.slabs, before):
        assert np.array_equal(a, b)


def test_cow_append_is_slice_assignment():
    """copy the retained partial page into a writable slot, append there."""
    rng = np.random.default_rng(9)
    L, C, P, T, H, D = 3, 2, 6, 8, 2, 4
    A = rand_array(rng, L, C, P, T, H, D, 2)
    pool = pool_from_array(A, pad=32)
    n_old, n_app = 3, 4
    app = rng.integers(0, 65536, size=(L, C, n_app, H, D), dtype=np.uint64).astype(np.uint16)
    ko.cow_append(pool, old_id=4, new_id=1, n_old=n_old, app=app, n_app=n_app)
    B = array_from_pool(pool)
    want = A.copy()
    want[:, :, 1, :n_old] = A[:, :, 4, :n_old]
    want[:, :, 1, n_old:n_old + n_app] = app
    assert np.array_equal(B, want)  # old page, other pages and slots >= n_old+n_app untouched
    with pytest.raises(ValueError):
        ko.cow_append(pool, 4, 1, 6, app, 4)  # overflow of the page
    with pytest.raises(ValueError):
        ko.cow_append(pool, 2, 2, 1, app, 1)  # in place is not copy-on-write


def w4_pool():
    L, C, P, T, H, D = 2, 2, 3, 4, 1, 2
    A = np.zeros((L, C, P, T, H, D), dtype=np.uint16)
    for l in range(L):
        for c in range(C):
            for g in range(P):
                for t in range(T):
                    for d in range(D):
                        A[l, c, g, t, 0, d] = 1000 * (2 * l + c) + 8 * g + 2 * t + d
    app = np.zeros((L, C, 2, H, D), dtype=np.uint16)
    for l in range(L):
        for c in range(C):
            for t in range(2):
                for d in range(D):
                    app[l, c, t, 0, d] = 500 + 100 * (2 * l + c) + 2 * t + d
    return A, app


def test_W4_cow_append_hand_computed(golden):
    A, app = w4_pool()
    for batched in (False, True):
        pool = pool_from_array(A)
        if batched:
            ko.cow_append_batched(pool, [1], [2], [1], [2], [app])
        else:
            ko.cow_append(pool, old_id=1, new_id=2, n_old=1, app=app, n_app=2)
        got = np.concatenate([s.view(np.uint16) for s in pool.slabs]).tolist()
        assert got == golden("W4_cow_append.txt")


def test_cow_append_batched_is_slice_assignment_per_session():
    """PAPER.md:L238, batched over sessions: every session's new page = its old page's first n_old
    tokens followed by its append block; old pages, other pages and later slots untouched."""
    rng = np.random.default_rng(19)
    L, C, P, T, H, D = 3, 2, 24, 8, 2, 4
    A = rand_array(rng, L, C, P, T, H, D, 2)
    pool = pool_from_array(A, pad=16)
    perm = rng.permutation(P)
    S = 7
    old, new = perm[:S], perm[S:2 * S]
    n_old = np.array([0, 3, 7, 8, 1, 5, 0])
    n_app = np.array([8, 4, 1, 0, 0, 2, 0])  # fresh page, mid, exactly full, pure copy, ..., no-op
    apps = [rng.integers(0, 65536, size=(L, C, int(a), H, D), dtype=np.uint64).astype(np.uint16)
            for a in n_app]
    ko.cow_append_batched(pool, old, new, n_old, n_app, apps)
    want = A.copy()
    for s in range(S):
        want[:, :, new[s], :n_old[s]] = A[:, :, old[s], :n_old[s]]
        want[:, :, new[s], n_old[s]:n_old[s] + n_app[s]] = apps[s]
    assert np.array_equal(array_from_pool(pool), want)
    for s in pool.slabs:  # stride padding untouched
        assert np.all(s.reshape(P, -1)[:, T * H * D * 2:] == 0xA5)
    with pytest.raises(ValueError):
        ko.cow_append_batched(pool, [1, 2], [3, 3], [1, 1], [1, 1], apps[:2])  # duplicate new page
    with pytest.raises(ValueError):
        ko.cow_append_batched(pool, [1, 2], [2, 3], [1, 1], [1, 1], apps[:2])  # new page is an old page
    with pytest.raises(IndexError):
        ko.cow_append_batched(pool, [1], [P], [1], [1], apps[:1])
    # layer subset: only the first layer_count layers are touched
    pool2 = pool_from_array(A)
    ko.cow_append_batched(pool2, old[:2], new[:2], n_old[:2], n_app[:2],
                          [a[:2] for a in apps[:2]], layer_count=2)
    B = array_from_pool(pool2)
    assert np.array_equal(B[2], A[2]) and not np.array_equal(B[:2], A[:2])


# ---------------------------------------------------------------------------------------------
# 6. fused pool -> pool re-paging (SURVEY.md 8(c) reading 11, 8(f) NEXT-2)
# ---------------------------------------------------------------------------------------------
def test_W3_repage_pool_to_pool_hand_computed(golden):
    src = pool_from_array(w1_array())
    dst = pool_from_array(np.full((2, 2, 3, 4, 1, 2), 7777, dtype=np.uint16))
    ko.repage(src, [1, 2, 0], dst, [0, 2], n_tokens=5)
    got = np.concatenate([s.view(np.uint16) for s in dst.slabs]).tolist()
    assert got == golden("W3_repage_pool_to_pool.txt")
    # W2's values again, reached without the buffer: src_ids=[3,0], n_tokens=3, dst_ids=[2]
    dst = pool_from_array(np.full((2, 2, 3, 4, 1, 2), 7777, dtype=np.uint16))
    ko.repage(src, [3, 0], dst, [2], n_tokens=3)
    got = np.concatenate([s.view(np.uint16) for s in dst.slabs]).tolist()
    assert got == golden("W2_repage_padded_tail.txt")


@pytest.mark.parametrize("Ts,Td,ntok", [(4, 16, 61), (16, 4, 64), (3, 5, 31), (8, 8, 40), (2, 7, 1)])
def test_repage_is_numpy_token_stream_reshape(Ts, Td, ntok):
    """Library-routine pin: gather source pages with take, flatten the token axis, cut to n_tokens,
    zero-fill to whole destination pages, reshape, scatter by fancy-index assignment."""
    rng = np.random.default_rng(23)
    L, C, H, D, e = 2, 2, 3, 4, 2
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    A = rand_array(rng, L, C, n_src + 5, Ts, H, D, e)
    B0 = rand_array(rng, L, C, n_dst + 4, Td, H, D, e)
    src_ids = rng.permutation(n_src + 5)[:n_src]
    dst_ids = rng.permutation(n_dst + 4)[:n_dst]
    src, dst = pool_from_array(A, pad=8), pool_from_array(B0, pad=24)
    ko.repage(src, src_ids, dst, dst_ids, n_tokens=ntok, threads=3)
    stream = np.take(A, src_ids, axis=2).reshape(L, C, n_src * Ts, H, D)[:, :, :ntok]
    padded = np.zeros((L, C, n_dst * Td, H, D), dtype=A.dtype)
    padded[:, :, :ntok] = stream
    want = B0.copy()
    want[:, :, dst_ids] = padded.reshape(L, C, n_dst, Td, H, D)
    assert np.array_equal(array_from_pool(dst), want)
    assert np.array_equal(array_from_pool(src), A)  # the source pool is never written
    for s in dst.slabs:  # stride padding untouched
        assert np.all(s.reshape(n_dst + 4, -1)[:, Td * H * D * e:] == 0xA5)


def test_repage_equals_pack_then_unpack_and_batched_equals_per_request():
    rng = np.random.default_rng(29)
    L, C, H, D, e, Ts, Td = 3, 2, 2, 4, 2, 4, 16
    A = rand_array(rng, L, C, 64, Ts, H, D, e)
    B0 = rand_array(rng, L, C, 20, Td, H, D, e)
    src = pool_from_array(A)
    ntok = np.array([37, 0, 64, 5])
    ns, nd = -(-ntok // Ts), -(-ntok // Td)
    soff, doff = np.concatenate([[0], np.cumsum(ns)]), np.concatenate([[0], np.cumsum(nd)])
    sids = rng.permutation(64)[:soff[-1]]
    dids = rng.permutation(20)[:doff[-1]]
    d1, d2, d3 = (pool_from_array(B0) for _ in range(3))
    ko.repage_batched(src, sids, soff, d1, dids, doff, ntok, threads=2)
    for r in range(4):
        a, b = slice(soff[r], soff[r + 1]), slice(doff[r], doff[r + 1])
        ko.repage(src, sids[a], d2, dids[b], n_tokens=int(ntok[r]))
        ko.unpack(ko.pack(src, sids[a]), dids[b], d3, Ts=Ts, n_tokens=int(ntok[r]))
    for x, y, z in zip(d1.slabs, d2.slabs, d3.slabs):
        assert np.array_equal(x, y) and np.array_equal(x, z)
    with pytest.raises(ValueError):
        ko.repage(src, sids[:2], d1, [1, 1], n_tokens=8)  # wrong destination count / duplicates
    with pytest.raises(IndexError):
        ko.repage(src, [64], d1, [1], n_tokens=4)
    with pytest.raises(ValueError):
        ko.repage(src, [1], pool_from_array(rand_array(rng, L, C, 4, Td, H, D + 1, e)), [1], n_tokens=4)


# ---------------------------------------------------------------------------------------------
# 7. HND pools: in-page order [head][token][dim] ("including")
# ---------------------------------------------------------------------------------------------
def w5_pool():
    """Slab c is the word sequence 1000*c + i, i = physical word index; pages are HND."""
    L, C, P, T, H, D = 1, 2, 3, 2, 2, 2
    slabs = [(1000 * c + np.arange(P * T * H * D)).astype(np.uint16).view(np.uint8) for c in range(C)]
    return ko.HostPool(slabs, L, C, P, T, H, D, 2, T * H * D * 2, ko.HND)


@pytest.mark.parametrize("impl", IMPLS)
def test_W5_hnd_pool_hand_computed(impl, golden):
    pack, unpack = IMPLS[impl]
    buf = pack(w5_pool(), [2, 0])
    assert buf.view(np.uint16).tolist() == golden("W5_hnd_pack.txt")
    # the inverse: unpacking that buffer into pages [1, 2] of a zeroed HND pool puts page 2's
    # physical words into page 1 and page 0's into page 2
    dst = w5_pool()
    for s in dst.slabs:
        s[:] = 0
    unpack(buf, [1, 2], dst, Ts=2, n_tokens=4)
    for c in range(2):
        w = dst.slabs[c].view(np.uint16)
        assert w[:8].tolist() == [0] * 8
        assert w[8:16].tolist() == [1000 * c + 16 + i for i in range(8)]
        assert w[16:24].tolist() == [1000 * c + i for i in range(8)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("pad", [0, 8])
def test_hnd_pack_unpack_are_numpy_take_transpose(shape, pad):
    L, C, P, T, H, D, e = shape
    rng = np.random.default_rng(31)
    A = rand_array(rng, L, C, P, T, H, D, e)
    pool = pool_from_array(A, pad=pad, order=ko.HND)
    ids = rng.permutation(P)[:max(1, P // 2)]
    want = np.take(A, ids, axis=2).transpose(2, 0, 1, 3, 4, 5).reshape(-1)
    for f in (ko.pack, ko.pack_py) if P * T * H * D <= 4096 else (ko.pack,):
        assert np.array_equal(f(pool, ids).view(DT[e]), want)
    # unpack into an HND pool == fancy-index assignment on the logical array
    B0 = rand_array(rng, L, C, P, T, H, D, e)
    dst_ids = rng.permutation(P)[:len(ids)]
    dst = pool_from_array(B0, pad=pad, order=ko.HND)
    ko.unpack(want.view(np.uint8), dst_ids, dst, Ts=T, n_tokens=len(ids) * T)
    wantB = B0.copy()
    wantB[:, :, dst_ids] = np.take(A, ids, axis=2)
    assert np.array_equal(array_from_pool(dst), wantB)
    for s in dst.slabs:
        assert np.all(s.reshape(P, -1)[:, T * H * D * e:] == 0xA5)


@pytest.mark.parametrize("so,do", [(0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("Ts,Td,ntok", [(4, 16, 61), (16, 4, 64), (3, 5, 31)])
def test_hnd_repage_and_cow(so, do, Ts, Td, ntok):
    rng = np.random.default_rng(37)
    L, C, H, D, e = 2, 2, 3, 4, 2
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    A = rand_array(rng, L, C, n_src + 5, Ts, H, D, e)
    B0 = rand_array(rng, L, C, n_dst + 4, Td, H, D, e)
    src_ids = rng.permutation(n_src + 5)[:n_src]
    dst_ids = rng.permutation(n_dst + 4)[:n_dst]
    src, dst = pool_from_array(A, pad=8, order=so), pool_from_array(B0, order=do)
    ko.repage(src, src_ids, dst, dst_ids, n_tokens=ntok)
    stream = np.take(A, src_ids, axis=2).reshape(L, C, n_src * Ts, H, D)[:, :, :ntok]
    padded = np.zeros((L, C, n_dst * Td, H, D), dtype=A.dtype)
    padded[:, :, :ntok] = stream
    want = B0.copy()
    want[:, :, dst_ids] = padded.reshape(L, C, n_dst, Td, H, D)
    assert np.array_equal(array_from_pool(dst), want)
    # the same through the NHD buffer
    dst2 = pool_from_array(B0, order=do)
    ko.unpack(ko.pack(src, src_ids), dst_ids, dst2, Ts=Ts, n_tokens=ntok)
    assert np.array_equal(array_from_pool(dst2), want)
    # copy-on-write append in an HND pool: slice assignment on the logical array
    if Td >= 4:
        pool = pool_from_array(B0, order=ko.HND)
        n_old, n_app = 1, Td - 2
        app = rng.integers(0, 65536, size=(L, C, n_app, H, D), dtype=np.uint64).astype(np.uint16)
        ko.cow_append(pool, 0, 1, n_old, app, n_app)
        w = B0.copy()
        w[:, :, 1, :n_old] = B0[:, :, 0, :n_old]
        w[:, :, 1, n_old:n_old + n_app] = app
        assert np.array_equal(array_from_pool(pool), w)
