"""GPU parity: the CUDA path (through the C ABI) vs the CPU oracle, byte for byte.

Same seeded inputs on both sides; integer/byte work => bit-exact is the bar.  Sizes span several
segments/tiles and ragged tails.  Citations: SURVEY.md 8(a) rows a1-a8, BASELINE.json:configs.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import kv_oracle as ko  # noqa: E402
from paper_2606_31093_b200 import workloads as W  # noqa: E402
from tests.kvhelpers import assert_pool_equal, host_pool, to_device  # noqa: E402


@pytest.fixture(scope="module")
def kv():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_31093_b200 import kvtier
    return kvtier


@pytest.fixture()
def ctx(kv):
    c = kv.Ctx(0, staging_bytes=8 << 20)
    yield c
    torch.cuda.synchronize()
    c.close()


KERNELS = {"bulk": 1, "vec": 2, "elem": 3, "shot": 4}

# L, C, P, T, H, D, e, pad
SHAPES = [
    (4, 2, 256, 16, 2, 64, 2, 0),     # BASELINE.json:configs[0] Tiny
    (3, 2, 64, 16, 4, 128, 2, 0),     # Qwen3-Omni row (16 KiB), few layers
    (2, 2, 40, 64, 4, 128, 2, 0),     # 64 KiB rows: split into sub-segments
    (2, 1, 33, 5, 3, 24, 2, 0),       # odd sizes, kv_count 1, tokrow 144 B
    (3, 2, 50, 16, 2, 64, 2, 256),    # padded stride (reading 22)
    (2, 2, 30, 8, 1, 40, 4, 0),       # fp32 elements
    (2, 2, 30, 8, 2, 24, 1, 0),       # fp8-sized elements
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", SHAPES)
def test_pack_unpack_same_page_size(kv, ctx, kernel, shape):
    L, C, P, T, H, D, e, pad = shape
    rng = np.random.default_rng(abs(hash(shape)) % 2**31)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    A = host_pool(rng, L, C, P, T, H, D, e, pad)
    B = host_pool(rng, L, C, P, T, H, D, e, pad)
    n = min(37, P - 3)
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    buf = torch.full((n * dA.page_bytes() + 256,), 0xCD, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, L, ids, buf, dst_bytes=n * dA.page_bytes())
    want = ko.pack(A, ids)
    got = buf.cpu().numpy()
    assert np.array_equal(got[:want.size], want)
    assert np.all(got[want.size:] == 0xCD), "wrote past the end of the buffer"
    assert_pool_equal(tA, A)  # source pool untouched
    kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, src_bytes=n * dA.page_bytes())
    ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
    assert_pool_equal(tB, B)  # touched pages equal, untouched pages + stride padding identical
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS[kernel]


@pytest.mark.parametrize("shape", [SHAPES[0], SHAPES[1], SHAPES[2], SHAPES[4]])
@pytest.mark.parametrize("variant", ["plain", "plain_capped", "general_l2hint", "plain_batched_1", "plain_batched_2",
                                     "plain_batched_5_capped"])
def test_plain_kernel_and_general_kernel_agree_with_the_oracle(kv, ctx, shape, variant):
    """The plain case (equal page sizes, page-first, nothing to zero-fill, host ids; one request or a batch of such
    requests, whose pieces the kernel then finds by binary search) runs the short kernel kv_move_shot_plain; anything
    else -- here an L2 hint, or a ragged tail in one request of the batch -- the general kv_move_shot.  Both must give
    the oracle's bytes; a capped grid makes every CTA of the plain kernel walk several items (the stage and its
    mbarrier phase are reused, and consecutive items fall into different pieces)."""
    L, C, P, T, H, D, e, pad = shape
    rng = np.random.default_rng(7 + abs(hash((shape, variant))) % 2**31)
    if variant == "general_l2hint":
        ctx.set_option(kv.KV_OPT_L2_HINT, 1)
    if variant.endswith("capped"):
        ctx.set_option(kv.KV_OPT_MAX_CTAS, 5)
    A = host_pool(rng, L, C, P, T, H, D, e, pad)
    B = host_pool(rng, L, C, P, T, H, D, e, pad)
    n = min(29, P - 3)
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    page = dA.page_bytes()
    buf = torch.full((n * page + 256,), 0xCD, dtype=torch.uint8, device="cuda")
    want_plain = 0 if variant.startswith("general") else 1
    if "batched" in variant:
        n_req = int(variant.split("_")[2])
        cut = {1: [0, n], 2: [0, n // 3, n], 5: [0, 1, 1, n // 2, n - 2, n]}[n_req]  # (5: with an empty request)
        off = np.asarray(cut, dtype=np.int64)
        bufs = [buf[cut[r] * page:cut[r + 1] * page] for r in range(n_req)]
        kv.kv_pack_batched(ctx, dA, L, ids, off, bufs)
    else:
        kv.kv_pack(ctx, dA, L, ids, buf, dst_bytes=n * page)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT and ctx.stat(kv.KV_STAT_LAST_PLAIN) == want_plain
    want = ko.pack(A, ids)
    got = buf.cpu().numpy()
    assert np.array_equal(got[:want.size], want)
    assert np.all(got[want.size:] == 0xCD), "wrote past the end of the buffer"
    if "batched" in variant:
        ntok = np.asarray([(cut[r + 1] - cut[r]) * T for r in range(n_req)], dtype=np.uint64)
        kv.kv_unpack_batched(ctx, bufs, dst, off, ntok, dB, L, T, T)
    else:
        kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, src_bytes=n * page)
    assert ctx.stat(kv.KV_STAT_LAST_PLAIN) == want_plain
    ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
    assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)
    # a ragged tail is not the plain case: the last page's unused slots are zero-filled by the general kernel
    if variant == "plain":
        kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T - 1, src_bytes=n * page)
        assert ctx.stat(kv.KV_STAT_LAST_PLAIN) == 0
        ko.unpack(want, dst, B, Ts=T, n_tokens=n * T - 1)
        assert_pool_equal(tB, B)
    if variant == "plain_batched_2":  # ... nor is a batch one of whose requests has one
        ntok = np.asarray([(cut[1] - cut[0]) * T - 3, (cut[2] - cut[1]) * T], dtype=np.uint64)
        kv.kv_unpack_batched(ctx, bufs, dst, off, ntok, dB, L, T, T)
        assert ctx.stat(kv.KV_STAT_LAST_PLAIN) == 0
        ko.unpack_batched([want[cut[r] * page:cut[r + 1] * page] for r in range(2)], dst, off, ntok, B, Ts=T)
        assert_pool_equal(tB, B)


@pytest.mark.parametrize("kernel", ["bulk", "vec", "shot", "auto"])
@pytest.mark.parametrize("Ts,Td,ntok", [(16, 64, 2048), (16, 64, 2048 - 37), (64, 16, 1000),
                                        (16, 24, 500), (3, 5, 77), (16, 16, 16 * 9 - 5), (8, 64, 1)])
def test_repage_unpack(kv, ctx, kernel, Ts, Td, ntok):
    """SURVEY.md 8(a) a5; BASELINE.json:configs[4]: sequence order preserved, zero-padded tail.  "shot" is the general
    form of the kernel AUTO picks at the paper's shapes (kv_move_shot: gcd chunking, zero tail); "auto" is whatever the
    library chooses for the shape (0 = KV_OPT_KERNEL's default)."""
    L, C, H, D, e = 3, 2, 4, 128, 2
    rng = np.random.default_rng(Ts * 1000 + Td)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS.get(kernel, 0))
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    P = n_dst + 7
    src = rng.integers(0, 256, size=n_src * L * C * Ts * H * D * e, dtype=np.uint8)
    B = host_pool(rng, L, C, P, Td, H, D, e)
    tB, dB = to_device(B, kv, torch)
    dst = rng.permutation(P)[:n_dst].astype(np.int32)
    kv.kv_unpack(ctx, torch.from_numpy(src).cuda(), dst, dB, L, Ts, Td, ntok)
    ko.unpack(src, dst, B, Ts=Ts, n_tokens=ntok)
    assert_pool_equal(tB, B)


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("kernel", ["bulk", "vec", "elem", "shot", "auto"])
def test_batched_csr_with_empty_requests_and_layouts(kv, ctx, kernel, layout):
    """SURVEY.md 8(a) a8; BASELINE.json:configs[3] (variable-length, CSR-encoded).  With "shot" / "auto" the pack is the
    plain kernel's batched form (pieces by binary search) when page-first and the general kv_move_shot when layer-first;
    the ragged re-paging unpack is the general kernel either way."""
    L, C, P, T, H, D, e = 4, 2, 300, 16, 2, 64, 2
    rng = np.random.default_rng(11 + layout)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS.get(kernel, 0))
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    counts = np.array([5, 0, 33, 1, 0, 17, 64])
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    ids = rng.permutation(P)[:off[-1]].astype(np.int32)
    bufs = [torch.zeros(max(int(c) * dA.page_bytes(), 16), dtype=torch.uint8, device="cuda") for c in counts]
    kv.kv_pack_batched(ctx, dA, L, ids, off, bufs, dst_bytes=[int(c) * dA.page_bytes() for c in counts], layout=layout)
    want = ko.pack_batched(A, ids, off, layout=layout)
    for r, c in enumerate(counts):
        assert np.array_equal(bufs[r].cpu().numpy()[:want[r].size], want[r]), f"request {r}"
    # reverse: batched re-paging unpack 16 -> 8 with ragged token counts
    Td = 8
    ntok = np.array([5 * 16 - 3, 0, 33 * 16, 1, 0, 17 * 16 - 15, 64 * 16 - 9])
    nd = -(-ntok // Td)
    doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
    P2 = int(doff[-1]) + 11
    B = host_pool(rng, L, C, P2, Td, H, D, e)
    tB, dB = to_device(B, kv, torch)
    dids = rng.permutation(P2)[:doff[-1]].astype(np.int32)
    kv.kv_unpack_batched(ctx, bufs, dids, doff, ntok, dB, L, T, Td, layout=layout)
    ko.unpack_batched(want, dids, doff, ntok, B, Ts=T, layout=layout)
    assert_pool_equal(tB, B)


def test_layer_subset(kv, ctx):
    rng = np.random.default_rng(12)
    A = host_pool(rng, 6, 2, 64, 16, 2, 64, 2)
    tA, dA = to_device(A, kv, torch)
    ids = rng.permutation(64)[:20].astype(np.int32)
    buf = torch.zeros(20 * dA.page_bytes(4), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, 4, ids, buf)
    assert np.array_equal(buf.cpu().numpy(), ko.pack(A, ids, layer_count=4))


@pytest.mark.parametrize("off_bytes,pad", [(2, 0), (0, 2), (4, 8), (8, 0)])
def test_misaligned_pointers_take_the_elem_path(kv, ctx, off_bytes, pad):
    """SURVEY.md 8(c) reading 13: never reject on 16-byte misalignment."""
    L, C, P, T, H, D, e = 2, 2, 40, 16, 2, 64, 2
    rng = np.random.default_rng(13)
    A = host_pool(rng, L, C, P, T, H, D, e, pad)
    B = host_pool(rng, L, C, P, T, H, D, e, pad)
    tA, dA = to_device(A, kv, torch, offset_bytes=off_bytes)
    tB, dB = to_device(B, kv, torch, offset_bytes=off_bytes)
    ids = rng.permutation(P)[:21].astype(np.int32)
    dst = rng.permutation(P)[:21].astype(np.int32)
    raw = torch.zeros(21 * dA.page_bytes() + 64, dtype=torch.uint8, device="cuda")
    buf = raw[off_bytes:off_bytes + 21 * dA.page_bytes()]
    kv.kv_pack(ctx, dA, L, ids, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_ELEM
    want = ko.pack(A, ids)
    assert np.array_equal(buf.cpu().numpy(), want)
    kv.kv_unpack(ctx, buf, dst, dB, L, T, T, 21 * T - 5)
    ko.unpack(want, dst, B, Ts=T, n_tokens=21 * T - 5)
    assert_pool_equal(tB, B)


@pytest.mark.parametrize("mode", ["direct", "staged", "auto"])
@pytest.mark.parametrize("Td", [16, 64])
def test_offload_reload_host_tier(kv, ctx, mode, Td):
    """the mode must not change a byte.  Staging is 8 MiB => several chunks."""
    m = {"direct": kv.KV_HOST_DIRECT, "staged": kv.KV_HOST_STAGED, "auto": kv.KV_HOST_AUTO}[mode]
    L, C, P, T, H, D, e = 6, 2, 256, 16, 4, 128, 2   # page = 192 KiB
    rng = np.random.default_rng(14)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n = 100
    ids = rng.permutation(P)[:n].astype(np.int32)
    nbytes = n * dA.page_bytes()
    hp = kv.kv_host_alloc(nbytes + 4096)
    try:
        hv = kv.host_view(hp, nbytes + 4096)
        hv[:] = 0xEE
        kv.kv_offload(ctx, dA, L, ids, hp, nbytes, mode=m)
        torch.cuda.synchronize()
        want = ko.pack(A, ids)
        assert np.array_equal(hv[:nbytes], want)
        assert np.all(hv[nbytes:] == 0xEE)
        ntok = n * T - 11
        n_dst = -(-ntok // Td)
        B = host_pool(rng, L, C, n_dst + 9, Td, H, D, e)
        tB, dB = to_device(B, kv, torch)
        dst = rng.permutation(n_dst + 9)[:n_dst].astype(np.int32)
        kv.kv_reload(ctx, hp, nbytes, dst, dB, L, T, Td, ntok, mode=m)
        torch.cuda.synchronize()
        ko.unpack(want, dst, B, Ts=T, n_tokens=ntok)
        assert_pool_equal(tB, B)
        if mode != "auto":
            assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == m
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


def test_auto_runs_direct_when_the_staging_cannot_be_allocated(kv):
    """A serving engine's KV pools fill HBM, so the staging that the first KV_HOST_AUTO transfer of 4 MiB or more
    allocates may not be there to get.  AUTO must then move the bytes with DIRECT (which needs no staging) instead of
    failing, and must not ask again on every call; an explicit KV_HOST_STAGED reports the failure; reserving a staging
    that does fit brings the staged pipeline back.  The failure is forced with a 64 TiB staging size."""
    L, C, P, T, H, D, e = 6, 2, 256, 16, 4, 128, 2   # page = 192 KiB
    rng = np.random.default_rng(41)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n = 100                                           # 18.75 MiB: AUTO wants STAGED
    ids = rng.permutation(P)[:n].astype(np.int32)
    nbytes = n * dA.page_bytes()
    want = ko.pack(A, ids)
    hp = kv.kv_host_alloc(nbytes)
    c = kv.Ctx(0, staging_bytes=1 << 46)
    try:
        hv = kv.host_view(hp, nbytes)
        for attempt in range(2):  # the second call finds the denial recorded and goes straight to DIRECT
            hv[:] = 0xEE
            kv.kv_offload(c, dA, L, ids, hp, nbytes, mode=kv.KV_HOST_AUTO)
            torch.cuda.synchronize()
            assert np.array_equal(hv, want)
            assert c.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_DIRECT
            assert c.last_cuda_error() == 2  # cudaErrorMemoryAllocation, kept for the caller to see
        hv[:] = 0xEE
        with pytest.raises(kv.KvError) as ei:
            kv.kv_offload(c, dA, L, ids, hp, nbytes, mode=kv.KV_HOST_STAGED)
        assert ei.value.status == kv.KV_ERR_CUDA
        torch.cuda.synchronize()
        assert np.all(hv == 0xEE), "a failed call wrote to the host buffer"
        hv[:] = want
        B = host_pool(rng, L, C, n + 5, T, H, D, e)
        tB, dB = to_device(B, kv, torch)
        dst = rng.permutation(n + 5)[:n].astype(np.int32)
        kv.kv_reload(c, hp, nbytes, dst, dB, L, T, T, n * T, mode=kv.KV_HOST_AUTO)
        torch.cuda.synchronize()
        assert c.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_DIRECT
        ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
        assert_pool_equal(tB, B)
        c.set_option(kv.KV_OPT_RESERVE_STAGING, 8 << 20)  # a size that fits: the staged pipeline is back
        hv[:] = 0xEE
        kv.kv_offload(c, dA, L, ids, hp, nbytes, mode=kv.KV_HOST_AUTO)
        torch.cuda.synchronize()
        assert c.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_STAGED
        assert np.array_equal(hv, want)
    finally:
        torch.cuda.synchronize()
        c.close()
        kv.kv_host_free(hp)


@pytest.mark.parametrize("mode", ["direct", "staged"])
def test_offload_reload_batched(kv, ctx, mode):
    m = {"direct": kv.KV_HOST_DIRECT, "staged": kv.KV_HOST_STAGED}[mode]
    L, C, P, T, H, D, e = 6, 2, 400, 16, 4, 128, 2
    rng = np.random.default_rng(15)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    counts = np.array([30, 0, 75, 3, 50])   # 192 KiB pages; 8 MiB staging => chunks span requests
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    ids = rng.permutation(P)[:off[-1]].astype(np.int32)
    sizes = [max(int(c) * dA.page_bytes(), 4096) for c in counts]
    hps = [kv.kv_host_alloc(s) for s in sizes]
    try:
        kv.kv_offload_batched(ctx, dA, L, ids, off, hps, host_bytes=sizes, mode=m)
        torch.cuda.synchronize()
        want = ko.pack_batched(A, ids, off)
        for r in range(len(counts)):
            assert np.array_equal(kv.host_view(hps[r], sizes[r])[:want[r].size], want[r]), f"req {r}"
        Td = 64
        ntok = np.array([30 * 16 - 1, 0, 75 * 16 - 40, 3 * 16, 50 * 16 - 63])
        nd = -(-ntok // Td)
        doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
        P2 = int(doff[-1]) + 5
        B = host_pool(rng, L, C, P2, Td, H, D, e)
        tB, dB = to_device(B, kv, torch)
        dids = rng.permutation(P2)[:doff[-1]].astype(np.int32)
        kv.kv_reload_batched(ctx, hps, dids, doff, ntok, dB, L, T, Td, host_bytes=sizes, mode=m)
        torch.cuda.synchronize()
        ko.unpack_batched(want, dids, doff, ntok, B, Ts=T)
        assert_pool_equal(tB, B)
    finally:
        torch.cuda.synchronize()
        for p in hps:
            kv.kv_host_free(p)


def test_errors_write_nothing(kv, ctx):
    L, C, P, T, H, D, e = 2, 2, 32, 16, 2, 64, 2
    rng = np.random.default_rng(16)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    buf = torch.full((8 * dA.page_bytes(),), 0x77, dtype=torch.uint8, device="cuda")

    def status(fn):
        with pytest.raises(kv.KvError) as ei:
            fn()
        return ei.value.status

    assert status(lambda: kv.kv_pack(ctx, dA, L, [1, 2, P], buf)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_pack(ctx, dA, L, [1, -1], buf)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_pack(ctx, dA, L, np.arange(9), buf)) == kv.KV_ERR_SIZE
    assert status(lambda: kv.kv_pack(ctx, dA, L + 1, [1], buf)) == kv.KV_ERR_DESC
    assert status(lambda: kv.kv_pack(ctx, dA, L, [1], buf, layout=7)) == kv.KV_ERR_LAYOUT
    assert status(lambda: kv.kv_unpack(ctx, buf, [1, 1], dA, L, T, T, 2 * T, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    assert status(lambda: kv.kv_unpack(ctx, buf, [1, 2], dA, L, T, T, 3 * T)) == kv.KV_ERR_SIZE
    assert status(lambda: kv.kv_unpack(ctx, buf, [1, 2], dA, L, T, 2 * T, 2 * T)) == kv.KV_ERR_SIZE
    pageable = np.zeros(8 * dA.page_bytes(), dtype=np.uint8)
    assert status(lambda: kv.kv_offload(ctx, dA, L, [1, 2], pageable, pageable.nbytes, mode=kv.KV_HOST_DIRECT)) == kv.KV_ERR_HOST_MEM
    assert status(lambda: kv.kv_offload(ctx, dA, L, [1, 2], pageable, pageable.nbytes, mode=kv.KV_HOST_STAGED)) == kv.KV_ERR_HOST_MEM
    torch.cuda.synchronize()
    assert torch.all(buf == 0x77)
    assert_pool_equal(tA, A)
    # n == 0 is OK with no launch
    before = ctx.stat(kv.KV_STAT_LAUNCHES)
    kv.kv_pack(ctx, dA, L, [], buf)
    kv.kv_unpack(ctx, buf, [], dA, L, T, T, 0)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == before


def test_ids_on_device_and_status_word(kv, ctx):
    L, C, P, T, H, D, e = 2, 2, 64, 16, 2, 64, 2
    rng = np.random.default_rng(17)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    ids = rng.permutation(P)[:10].astype(np.int32)
    dids = torch.from_numpy(ids).cuda()
    buf = torch.zeros(10 * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, L, dids, buf, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert np.array_equal(buf.cpu().numpy(), ko.pack(A, ids))
    assert ctx.device_status() == 0
    bad = ids.copy(); bad[3] = P + 5
    buf.fill_(0x55)
    kv.kv_pack(ctx, dA, L, torch.from_numpy(bad).cuda(), buf, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert ctx.device_status() & 1
    got = buf.cpu().numpy().reshape(10, -1)
    want = ko.pack(A, ids).reshape(10, -1)
    assert np.array_equal(np.delete(got, 3, 0), np.delete(want, 3, 0))
    assert np.all(got[3] == 0x55)  # the bad page was skipped


def test_duplicate_source_ids_allowed_in_pack(kv, ctx):
    rng = np.random.default_rng(18)
    A = host_pool(rng, 2, 2, 16, 16, 2, 64, 2)
    tA, dA = to_device(A, kv, torch)
    ids = np.array([3, 3, 0, 3, 15], dtype=np.int32)
    buf = torch.zeros(5 * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, 2, ids, buf)
    assert np.array_equal(buf.cpu().numpy(), ko.pack(A, ids))


def test_tuning_options_do_not_change_bytes(kv, ctx):
    L, C, P, T, H, D, e = 4, 2, 128, 16, 4, 128, 2
    rng = np.random.default_rng(19)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    ids = rng.permutation(P)[:77].astype(np.int32)
    want = ko.pack(A, ids)
    for stage, stages, warps, lag, hint in [(16384, 3, 4, 1, 0), (8192, 6, 4, 2, 0), (4096, 8, 2, 3, 1),
                                            (16384, 12, 1, 3, 0), (32768, 2, 3, 1, 1), (1024, 16, 8, 2, 0)]:
        ctx.set_option(kv.KV_OPT_STAGE_BYTES, stage)
        ctx.set_option(kv.KV_OPT_STAGES_PER_WARP, stages)
        ctx.set_option(kv.KV_OPT_WARPS, warps)
        ctx.set_option(kv.KV_OPT_STORE_LAG, lag)
        ctx.set_option(kv.KV_OPT_L2_HINT, hint)
        buf = torch.zeros(77 * dA.page_bytes(), dtype=torch.uint8, device="cuda")
        kv.kv_pack(ctx, dA, L, ids, buf)
        assert np.array_equal(buf.cpu().numpy(), want), (stage, stages, warps, lag, hint)


def test_medium_qwen_shape_parity(kv, ctx):
    """Qwen3-Omni-shaped pool (48 L, 4 H, 128 D, bf16, T 16) with 1,024 pages (1.5 GiB):
    pack 300 fragmented pages (450 MiB) and scatter them back; full byte compare."""
    s = W.QWEN3_OMNI.with_(P=1024)
    rng = np.random.default_rng(20)
    A = host_pool(rng, s.L, s.C, s.P, s.T, s.H, s.D, s.e)
    tA, dA = to_device(A, kv, torch)
    ids = rng.choice(s.P, 300, replace=False).astype(np.int32)
    buf = torch.zeros(300 * s.page_bytes, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, s.L, ids, buf)
    want = ko.pack(A, ids, threads=8)
    assert np.array_equal(buf.cpu().numpy(), want)
    dst = rng.permutation(s.P)[:300].astype(np.int32)
    kv.kv_unpack(ctx, buf, dst, dA, s.L, s.T, s.T, 300 * s.T)
    ko.unpack(want, dst, A, Ts=s.T, n_tokens=300 * s.T, threads=8)
    assert_pool_equal(tA, A)


@pytest.mark.parametrize("mode", ["direct", "staged"])
def test_offload_and_reload_at_once_on_two_contexts(kv, ctx, mode):
    """The schedule bench.py's e2e leg times: one ctx offloads on one stream while a second ctx reloads
    another buffer into other pages of the SAME pool on a second stream (reading R21: calls on
    different streams are independent if their destination pages are disjoint; one ctx per stream).
    Several rounds back to back, no synchronisation in between beyond each stream's own order."""
    m = {"direct": kv.KV_HOST_DIRECT, "staged": kv.KV_HOST_STAGED}[mode]
    L, C, P, T, H, D, e = 6, 2, 768, 16, 4, 128, 2   # page = 192 KiB
    rng = np.random.default_rng(141)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n, rounds = 90, 4
    page = dA.page_bytes()
    perm = rng.permutation(P).astype(np.int32)
    src = [perm[r * n:(r + 1) * n] for r in range(rounds)]                 # pages offloaded in round r
    dst = [perm[(rounds + r) * n:(rounds + r + 1) * n] for r in range(rounds - 1)]  # pages restored in round r+1
    hps = [kv.kv_host_alloc(n * page) for _ in range(rounds)]
    ctx2 = kv.Ctx(0, staging_bytes=8 << 20)
    s_off, s_rel = torch.cuda.Stream(), torch.cuda.Stream()
    done = [torch.cuda.Event() for _ in range(rounds)]
    try:
        for r in range(rounds):
            kv.kv_offload(ctx, dA, L, src[r], hps[r], n * page, mode=m, stream=s_off)
            done[r].record(s_off)
            if r:  # restore what round r-1 offloaded, into fresh pages, while round r's offload runs
                s_rel.wait_event(done[r - 1])
                kv.kv_reload(ctx2, hps[r - 1], n * page, dst[r - 1], dA, L, T, T, n * T, mode=m, stream=s_rel)
        torch.cuda.synchronize()
        for r in range(rounds):
            want = ko.pack(A, src[r])
            assert np.array_equal(kv.host_view(hps[r], n * page), want), f"round {r}: offloaded bytes"
        for r in range(rounds - 1):
            ko.unpack(ko.pack(A, src[r]), dst[r], A, Ts=T, n_tokens=n * T)
        assert_pool_equal(tA, A)
    finally:
        torch.cuda.synchronize()
        ctx2.close()
        for hp in hps:
            kv.kv_host_free(hp)
