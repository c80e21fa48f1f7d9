"""GPU parity for the SURVEY.md 8(f) rows built on top of the hot path: fused pool -> pool
re-paging (NEXT-2, kv_repage) and copy-on-write partial-page append (NEXT-1, kv_cow_append,
PAPER.md:L238), byte for byte against the CPU oracle on the same seeded inputs."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import kv_oracle as ko  # noqa: E402
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


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("Ts,Td,ntok,pad", [(16, 64, 2048, 0), (16, 64, 2048 - 37, 0), (64, 16, 1000, 0),
                                            (16, 24, 500, 0), (3, 5, 77, 0), (16, 16, 16 * 9, 256),
                                            (8, 64, 1, 0), (16, 64, 65, 0)])
def test_repage_pool_to_pool(kv, ctx, kernel, Ts, Td, ntok, pad):
    L, C, H, D, e = 3, 2, 4, 128, 2
    rng = np.random.default_rng(Ts * 977 + Td * 31 + ntok)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    A = host_pool(rng, L, C, n_src + 9, Ts, H, D, e, pad)
    B = host_pool(rng, L, C, n_dst + 7, Td, H, D, e, pad)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    sids = rng.permutation(n_src + 9)[:n_src].astype(np.int32)
    dids = rng.permutation(n_dst + 7)[:n_dst].astype(np.int32)
    launches = ctx.stat(kv.KV_STAT_LAUNCHES)
    kv.kv_repage(ctx, dA, sids, dB, dids, L, ntok, flags=kv.KV_FLAG_VALIDATE)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == launches + 1  # fused: one launch, no buffer
    ko.repage(A, sids, B, dids, n_tokens=ntok)
    assert_pool_equal(tB, B)  # touched pages equal; untouched pages and stride padding identical
    assert_pool_equal(tA, A)  # the source pool is never written
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS[kernel]


def test_repage_batched_and_page_migration_inside_one_pool(kv, ctx):
    L, C, H, D, e, Ts, Td = 4, 2, 2, 64, 2, 16, 64
    rng = np.random.default_rng(41)
    A = host_pool(rng, L, C, 400, Ts, H, D, e)
    B = host_pool(rng, L, C, 120, Td, H, D, e)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    ntok = np.array([2048, 0, 2048 - 61, 17, 64, 1000])
    ns, nd = -(-ntok // Ts), -(-ntok // Td)
    soff = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
    sids = rng.permutation(400)[:soff[-1]].astype(np.int32)
    dids = rng.permutation(120)[:doff[-1]].astype(np.int32)
    kv.kv_repage_batched(ctx, dA, sids, soff, dB, dids, doff, ntok, L)
    ko.repage_batched(A, sids, soff, B, dids, doff, ntok)
    assert_pool_equal(tB, B)
    # layer subset
    kv.kv_repage_batched(ctx, dA, sids[::-1].copy()[-int(soff[1]):], soff[:2], dB, dids[:int(doff[1])], doff[:2], ntok[:1], 2)
    ko.repage_batched(A, sids[::-1].copy()[-int(soff[1]):], soff[:2], B, dids[:int(doff[1])], doff[:2], ntok[:1], layer_count=2)
    assert_pool_equal(tB, B)
    # Ts == Td inside ONE pool: a page migration (defragmentation); disjoint source/destination ids
    perm = rng.permutation(400).astype(np.int32)
    src, dst = perm[:50], perm[50:100]
    A2 = A.copy()
    kv.kv_repage(ctx, dA, src, dA, dst, L, 50 * Ts)
    ko.repage(A, src, A2, dst, n_tokens=50 * Ts)
    assert_pool_equal(tA, A2)


def test_repage_errors_write_nothing(kv, ctx):
    L, C, H, D, e = 2, 2, 2, 64, 2
    rng = np.random.default_rng(43)
    A = host_pool(rng, L, C, 20, 16, H, D, e)
    B = host_pool(rng, L, C, 10, 64, H, D, e)
    Bh = host_pool(rng, L, C, 10, 64, H + 1, D, e)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    _, dBh = to_device(Bh, kv, torch)
    s8 = np.arange(8, dtype=np.int32)

    def status(fn):
        try:
            fn()
        except kv.KvError as ex:
            return ex.status
        return 0

    assert status(lambda: kv.kv_repage(ctx, dA, s8, dB, [1, 2, 3], L, 128)) == kv.KV_ERR_SIZE
    assert status(lambda: kv.kv_repage(ctx, dA, s8[:7], dB, [1, 2], L, 128)) == kv.KV_ERR_SIZE
    assert status(lambda: kv.kv_repage(ctx, dA, [0, 1, 2, 3, 4, 5, 6, 20], dB, [1, 2], L, 128)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_repage(ctx, dA, s8, dB, [1, 10], L, 128)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_repage(ctx, dA, s8, dB, [1, 1], L, 128, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    assert status(lambda: kv.kv_repage(ctx, dA, s8, dBh, [1, 2], L, 128)) == kv.KV_ERR_DESC
    assert status(lambda: kv.kv_repage(ctx, dA, s8, dB, [1, 2], L + 1, 128)) == kv.KV_ERR_DESC
    kv.kv_repage(ctx, dA, [], dB, [], L, 0)  # empty: KV_OK, no launch
    torch.cuda.synchronize()
    assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)


# ------------------------------------------------------------------------------------------------
# copy-on-write partial-page append
# ------------------------------------------------------------------------------------------------
COW_SHAPES = [  # L, C, P, T, H, D, e, pad
    (4, 2, 64, 16, 2, 64, 2, 0),     # Tiny-like
    (3, 2, 40, 16, 4, 128, 2, 0),    # Qwen3-Omni row
    (2, 2, 24, 64, 4, 128, 2, 0),    # 64 KiB rows: parts longer than one stage
    (2, 1, 30, 5, 3, 24, 2, 0),      # odd sizes (tokrow 144 B)
    (2, 2, 30, 16, 2, 64, 2, 256),   # padded stride
    (2, 2, 30, 8, 1, 5, 1, 0),       # 5-byte token rows: elem path with unit 1
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", COW_SHAPES)
def test_cow_append_batched(kv, ctx, kernel, shape):
    L, C, P, T, H, D, e, pad = shape
    rng = np.random.default_rng(abs(hash(shape)) % 2**31)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    A = host_pool(rng, L, C, P, T, H, D, e, pad)
    tA, dA = to_device(A, kv, torch)
    S = 9
    perm = rng.permutation(P).astype(np.int32)
    old, new = perm[:S], perm[S:2 * S]
    n_old = rng.integers(0, T + 1, size=S)
    n_app = np.array([rng.integers(0, T - o + 1) for o in n_old])
    n_old[0], n_app[0] = 0, T      # a fresh page filled by the append alone
    n_old[1], n_app[1] = T, 0      # a plain page copy
    n_old[2], n_app[2] = 0, 0      # nothing to do for this session
    n_old[3], n_app[3] = T - 1, 1  # exactly full after the append
    apps = [rng.integers(0, 256, size=L * C * int(a) * H * D * e, dtype=np.uint8) for a in n_app]
    dev_apps = [torch.from_numpy(a).cuda() if a.size else None for a in apps]
    launches = ctx.stat(kv.KV_STAT_LAUNCHES)
    kv.kv_cow_append_batched(ctx, dA, L, old, new, n_old, n_app, dev_apps, flags=kv.KV_FLAG_VALIDATE)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == launches + 1  # all sessions in one launch
    ko.cow_append_batched(A, old, new, n_old, n_app, apps)
    assert_pool_equal(tA, A)  # new pages equal; old pages, other pages, later slots, padding identical
    want_kernel = KERNELS[kernel] if (H * D * e) % 16 == 0 else KERNELS["elem"]
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == want_kernel


def test_cow_append_single_layer_subset_and_host_append_block(kv, ctx):
    L, C, P, T, H, D, e = 4, 2, 32, 16, 2, 64, 2
    rng = np.random.default_rng(47)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n_old, n_app, Lsub = 5, 7, 3
    app = rng.integers(0, 256, size=Lsub * C * n_app * H * D * e, dtype=np.uint8)
    hp = kv.kv_host_alloc(app.size)  # the new rows may sit in mapped pinned host memory
    try:
        kv.host_view(hp, app.size)[:] = app
        kv.kv_cow_append(ctx, dA, Lsub, 3, 9, n_old, hp, n_app)
        torch.cuda.synchronize()
    finally:
        kv.kv_host_free(hp)
    ko.cow_append(A, 3, 9, n_old, app, n_app, layer_count=Lsub)
    assert_pool_equal(tA, A)


def test_cow_errors_write_nothing(kv, ctx):
    L, C, P, T, H, D, e = 2, 2, 16, 16, 2, 64, 2
    rng = np.random.default_rng(53)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    app = torch.zeros(L * C * T * H * D * e, dtype=torch.uint8, device="cuda")

    def status(fn):
        try:
            fn()
        except kv.KvError as ex:
            return ex.status
        return 0

    assert status(lambda: kv.kv_cow_append(ctx, dA, L, 1, 2, 10, app, 7)) == kv.KV_ERR_SIZE      # overflows the page
    assert status(lambda: kv.kv_cow_append(ctx, dA, L, 2, 2, 1, app, 1)) == kv.KV_ERR_SIZE       # in place is not CoW
    assert status(lambda: kv.kv_cow_append(ctx, dA, L, 1, P, 1, app, 1)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_cow_append(ctx, dA, L, -1, 2, 1, app, 1)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_cow_append(ctx, dA, L, 1, 2, 1, None, 1)) == kv.KV_ERR_NULL
    assert status(lambda: kv.kv_cow_append_batched(ctx, dA, L, [1, 3], [2, 2], [1, 1], [1, 1], [app, app],
                                                   flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    assert status(lambda: kv.kv_cow_append_batched(ctx, dA, L, [1, 2], [2, 3], [1, 1], [1, 1], [app, app],
                                                   flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    kv.kv_cow_append_batched(ctx, dA, L, [], [], [], [], [])  # empty: KV_OK, no launch
    torch.cuda.synchronize()
    assert_pool_equal(tA, A)


# ------------------------------------------------------------------------------------------------
# CUDA graphs: a transfer is one kernel node; device-resident ids are re-read at every replay
# ------------------------------------------------------------------------------------------------
def test_cuda_graph_capture_and_replay_with_device_ids(kv, ctx):
    L, C, P, T, H, D, e = 4, 2, 256, 16, 2, 64, 2
    rng = np.random.default_rng(61)
    A = host_pool(rng, L, C, P, T, H, D, e)
    B = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    n = 37
    d_src = torch.zeros(n, dtype=torch.int32, device="cuda")
    d_dst = torch.zeros(n, dtype=torch.int32, device="cuda")
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    launches = ctx.stat(kv.KV_STAT_LAUNCHES)
    hp = kv.kv_host_alloc(buf.numel())
    with torch.cuda.graph(g, stream=side):
        kv.kv_pack(ctx, dA, L, d_src, buf, flags=kv.KV_FLAG_IDS_ON_DEVICE, stream=side)
        kv.kv_unpack(ctx, buf, d_dst, dB, L, T, T, n * T, flags=kv.KV_FLAG_IDS_ON_DEVICE, stream=side)
        # not replayable: staged host mode -> refused, nothing enqueued
        with pytest.raises(kv.KvError) as ei:
            kv.kv_offload(ctx, dA, L, np.arange(n), hp, buf.numel(), mode=kv.KV_HOST_STAGED, stream=side)
        assert ei.value.status == kv.KV_ERR_CAPTURE
    kv.kv_host_free(hp)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == launches + 2
    for rep in range(3):  # new page ids per replay, no host work besides the id upload
        src = rng.choice(P, n, replace=False).astype(np.int32)
        dst = rng.permutation(P)[:n].astype(np.int32)
        d_src.copy_(torch.from_numpy(src))
        d_dst.copy_(torch.from_numpy(dst))
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        want = ko.pack(A, src)
        assert np.array_equal(buf.cpu().numpy(), want), f"replay {rep}: pack != oracle"
        ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
        assert_pool_equal(tB, B)
    assert ctx.device_status() == 0


def test_cuda_graph_large_transfer_host_ids_and_direct_offload(kv, ctx):
    """Large captured transfers use the static work distribution; host ids are baked into the node;
    KV_HOST_AUTO captured = DIRECT (one kernel storing to mapped pinned memory)."""
    L, C, P, T, H, D, e = 6, 2, 512, 16, 4, 128, 2
    rng = np.random.default_rng(67)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n = 400  # 400 * 12 = 4,800 segments >= 8 per warp: dynamic claiming when launched live
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    nbytes = n * dA.page_bytes()
    buf = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    hp = kv.kv_host_alloc(nbytes)
    try:
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            kv.kv_pack(ctx, dA, L, ids, buf, stream=side)
            kv.kv_offload(ctx, dA, L, ids, hp, nbytes, stream=side)  # AUTO would be STAGED (75 MiB) live
        assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_DIRECT
        want = ko.pack(A, ids)
        for rep in range(2):
            buf.zero_()
            kv.host_view(hp, nbytes)[:] = 0
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            assert np.array_equal(buf.cpu().numpy(), want)
            assert np.array_equal(kv.host_view(hp, nbytes), want)
        # too many ids for the kernel parameters -> cannot be captured
        big_ids = rng.integers(0, P, size=9000).astype(np.int32)
        big = torch.empty(16, dtype=torch.uint8, device="cuda")
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=side):
            kv.kv_pack(ctx, dA, L, ids[:4], buf, stream=side)
            with pytest.raises(kv.KvError) as ei:
                kv.kv_pack(ctx, dA, L, big_ids, big, dst_bytes=1 << 40, stream=side)
            assert ei.value.status == kv.KV_ERR_CAPTURE
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


# ------------------------------------------------------------------------------------------------
# availability flag after a transfer, peer mapping (one GPU here: the flag and
# error paths; the data path of a peer pool is the same kernels on UVA addresses)
# ------------------------------------------------------------------------------------------------
def test_signal_follows_the_transfer_in_stream_order(kv, ctx):
    L, C, P, T, H, D, e = 4, 2, 256, 16, 4, 128, 2
    rng = np.random.default_rng(89)
    A = host_pool(rng, L, C, P, T, H, D, e)
    B = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    n = 200
    src = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    dflag = torch.zeros(1, dtype=torch.int64, device="cuda")
    hflag_p = kv.kv_host_alloc(64)
    hflag = kv.host_view(hflag_p, 64).view(np.uint64)
    hflag[:] = 0
    try:
        side = torch.cuda.Stream()
        kv.kv_pack(ctx, dA, L, src, buf, stream=side)
        kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, stream=side)
        kv.kv_signal(ctx, dflag, 0x1234_5678_9ABC_DEF0, stream=side)
        kv.kv_signal(ctx, hflag_p, 7, stream=side)
        import time
        t0 = time.time()
        while hflag[0] != 7:  # the host polls the mapped word: no stream synchronisation
            assert time.time() - t0 < 10, "flag never arrived"
        # the flag was stored after the transfer's kernels completed: a copy on ANOTHER stream, started
        # only now, already sees every unpacked page
        other = torch.cuda.Stream()
        with torch.cuda.stream(other):
            snap = [t.clone() for t in tB]
        other.synchronize()
        ko.unpack(ko.pack(A, src), dst, B, Ts=T, n_tokens=n * T)
        assert_pool_equal(snap, B)
        side.synchronize()
        assert int(dflag.item()) == 0x1234_5678_9ABC_DEF0
        pageable = np.zeros(1, dtype=np.uint64)
        with pytest.raises(kv.KvError) as ei:
            kv.kv_signal(ctx, pageable, 1)
        assert ei.value.status == kv.KV_ERR_HOST_MEM
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hflag_p)


def test_peer_enable_errors_on_this_box(kv, ctx):
    with pytest.raises(kv.KvError) as ei:
        kv.kv_peer_enable(ctx, 0)  # the ctx's own device
    assert ei.value.status == kv.KV_ERR_SIZE
    with pytest.raises(kv.KvError) as ei:
        kv.kv_peer_enable(ctx, -1)
    assert ei.value.status == kv.KV_ERR_SIZE
    n = torch.cuda.device_count()
    with pytest.raises(kv.KvError) as ei:
        kv.kv_peer_enable(ctx, n)  # no such device
    assert ei.value.status == kv.KV_ERR_CUDA
    if n > 1 and torch.cuda.can_device_access_peer(0, 1):  # exercised only where a second GPU is visible
        kv.kv_peer_enable(ctx, 1)
        kv.kv_peer_enable(ctx, 1)  # twice is fine
        L, C, P, T, H, D, e = 2, 2, 64, 16, 4, 128, 2
        rng = np.random.default_rng(97)
        A = host_pool(rng, L, C, P, T, H, D, e)
        B = host_pool(rng, L, C, P, T, H, D, e)
        tA, dA = to_device(A, kv, torch)
        tB = [torch.from_numpy(x).to("cuda:1") for x in B.slabs]
        dB = kv.PoolDesc(tB, L, C, P, T, H, D, e)
        ids = rng.choice(P, 20, replace=False).astype(np.int32)
        buf = torch.zeros(20 * dA.page_bytes(), dtype=torch.uint8, device="cuda:0")
        kv.kv_pack(ctx, dA, L, ids, buf)
        kv.kv_unpack(ctx, buf, ids, dB, L, T, T, 20 * T)  # push into the peer's pool over NVLink
        torch.cuda.synchronize(0)
        ko.unpack(ko.pack(A, ids), ids, B, Ts=T, n_tokens=20 * T)
        assert_pool_equal(tB, B)


def test_cuda_graph_capture_of_hnd_transfer_uses_cached_tensor_maps(kv, ctx):
    """Tensor maps are built in device memory (an allocation + a blocking copy) on a pool's first use, which a
    capturing stream cannot do.  A first-ever captured HND call therefore carries its maps INSIDE its kernel
    parameters (encoding a map is pure host work); a warmed-up one uses the cached device copies.  Both replay the
    oracle's bytes: pack, unpack, HND -> HND re-page and a staged offload, each captured before any live call."""
    L, C, P, T, H, D, e = 3, 2, 128, 16, 4, 128, 2
    rng = np.random.default_rng(101)
    A = host_pool(rng, L, C, P, T, H, D, e, order=ko.HND)
    B = host_pool(rng, L, C, P, T, H, D, e, order=ko.HND)
    Cq = host_pool(rng, L, C, 40, 64, H, D, e, order=ko.HND)  # re-page destination: 64-token pages
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    tC, dC = to_device(Cq, kv, torch)
    n = 60
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    dst64 = rng.permutation(40)[:n * T // 64].astype(np.int32)
    nbytes = n * dA.page_bytes()
    buf = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    hp = kv.kv_host_alloc(nbytes)
    try:
        kv.host_view(hp, nbytes)[:] = 0
        ctx.set_option(kv.KV_OPT_RESERVE_STAGING, 0)  # a captured STAGED transfer needs the staging to exist
        want = ko.pack(A, ids)
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            kv.kv_pack(ctx, dA, L, ids, buf, stream=side)
            assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1  # maps in the parameters
            kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, stream=side)
            assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
            kv.kv_repage(ctx, dA, ids, dC, dst64, L, n * T, stream=side)
            assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
            kv.kv_offload(ctx, dA, L, ids, hp, nbytes, mode=kv.KV_HOST_STAGED, stream=side)
            assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(buf.cpu().numpy(), want)
        assert np.array_equal(kv.host_view(hp, nbytes), want)
        ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
        assert_pool_equal(tB, B)
        ko.unpack(want, dst64, Cq, Ts=T, n_tokens=n * T)
        assert_pool_equal(tC, Cq)
        assert_pool_equal(tA, A)
        kv.kv_pack(ctx, dA, L, ids, buf)  # live call builds and caches the maps in device memory
        assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
        torch.cuda.synchronize()
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=side):
            kv.kv_pack(ctx, dA, L, ids, buf, stream=side)
        assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
        buf.zero_()
        g2.replay()
        torch.cuda.synchronize()
        assert np.array_equal(buf.cpu().numpy(), want)
        # tensor maps switched off: a captured call takes the lane paths, as a live one does
        ctx2 = kv.Ctx(0)
        try:
            ctx2.set_option(kv.KV_OPT_TENSOR_MAPS, 0)
            g3 = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g3, stream=side):
                kv.kv_pack(ctx2, dA, L, ids, buf, stream=side)
            assert ctx2.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 0
            buf.zero_()
            g3.replay()
            torch.cuda.synchronize()
            assert np.array_equal(buf.cpu().numpy(), want)
        finally:
            torch.cuda.synchronize()
            ctx2.close()
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


# ------------------------------------------------------------------------------------------------
# SURVEY.md 8(c) reading 18 on the device: id * page_stride beyond 2^32 inside ONE slab
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", [1, 2, 3])
def test_page_offsets_beyond_4_gib_in_one_slab(kv, ctx, kernel):
    """One (layer, K) slab of 262,145 pages x 16 KiB = 4 GiB + 16 KiB: ids [262144, 0, 262143, 131072] must
    come back in that order (the oracle's pin, tests/test_oracle_pins.py, on the device), and unpacking
    into the far end must touch only those pages.  Expected bytes come from the slab's closed-form fill
    (64-bit word i holds i * 0x9E3779B97F4A7C15 mod 2^64), nothing from the library."""
    free, _ = torch.cuda.mem_get_info()
    if free < 10 << 30:
        pytest.skip("needs 10 GiB of free device memory")
    P, T, H, D, e = 262145, 16, 4, 128, 2
    row = T * H * D * e
    wpp = row // 8  # 64-bit words per page
    ctx.set_option(kv.KV_OPT_KERNEL, kernel)
    slab = torch.arange(P * wpp, dtype=torch.int64, device="cuda")
    slab.mul_(-7046029254386353131)  # 0x9E3779B97F4A7C15 as a signed 64-bit value; wraps mod 2^64
    desc = kv.PoolDesc([slab], 1, 1, P, T, H, D, e)

    def page_words(g):
        i = np.arange(g * wpp, (g + 1) * wpp, dtype=np.uint64)
        return i * np.uint64(0x9E3779B97F4A7C15)

    ids = np.array([262144, 0, 262143, 131072], dtype=np.int32)
    buf = torch.zeros(len(ids) * row, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, desc, 1, ids, buf)
    torch.cuda.synchronize()
    got = buf.cpu().numpy().view(np.uint64).reshape(len(ids), wpp)
    for p, g in enumerate(ids):
        assert np.array_equal(got[p], page_words(int(g))), f"buffer page {p} is not pool page {g}"
    # scatter the buffer into four other pages, two of them past the 4 GiB line
    dst = np.array([262142, 1, 200000, 262141], dtype=np.int32)
    kv.kv_unpack(ctx, buf, dst, desc, 1, T, T, len(ids) * T, flags=kv.KV_FLAG_VALIDATE)
    torch.cuda.synchronize()
    view = slab.view(P, wpp)
    for p, g in enumerate(dst):
        assert np.array_equal(view[int(g)].cpu().numpy().view(np.uint64), page_words(int(ids[p])))
    for g in (262143, 262144, 262140, 0, 2, 199999, 200001):  # neighbours untouched
        assert np.array_equal(view[g].cpu().numpy().view(np.uint64), page_words(g))
    # every other page: 64-bit checksum per page against the closed form, on the device
    sums = view.sum(dim=1)
    i0 = torch.arange(P, dtype=torch.int64, device="cuda") * wpp
    want = (i0 * wpp + wpp * (wpp - 1) // 2) * (-7046029254386353131)
    mask = torch.ones(P, dtype=torch.bool, device="cuda")
    mask[torch.as_tensor(dst.astype(np.int64), device="cuda")] = False
    assert torch.equal(sums[mask], want[mask]), "a page outside the destination set changed"
    del slab, view, sums, i0, want
    torch.cuda.empty_cache()


@pytest.mark.parametrize("tensor_maps", [1, 0])
def test_hnd_page_offsets_beyond_4_gib(kv, ctx, tensor_maps):
    """The same slab read as an HND pool: the tensor-map path addresses page 262,144 through the map's
    page coordinate (stride 16 KiB, 4 GiB from the base), the lane paths through 64-bit arithmetic."""
    free, _ = torch.cuda.mem_get_info()
    if free < 10 << 30:
        pytest.skip("needs 10 GiB of free device memory")
    P, T, H, D, e = 262145, 16, 4, 128, 2
    row = T * H * D * e
    wpp, wpr = row // 8, D * e // 8
    ctx.set_option(kv.KV_OPT_TENSOR_MAPS, tensor_maps)
    slab = torch.arange(P * wpp, dtype=torch.int64, device="cuda")
    slab.mul_(-7046029254386353131)
    desc = kv.PoolDesc([slab], 1, 1, P, T, H, D, e, order=kv.KV_ORDER_HND)

    def nhd_words(g):  # the HND page g re-ordered to [token][head][dim]
        i = np.arange(g * wpp, (g + 1) * wpp, dtype=np.uint64) * np.uint64(0x9E3779B97F4A7C15)
        return i.reshape(H, T, wpr).transpose(1, 0, 2).reshape(-1)

    ids = np.array([262144, 0, 262143, 131072], dtype=np.int32)
    buf = torch.zeros(len(ids) * row, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, desc, 1, ids, buf)
    torch.cuda.synchronize()
    assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == tensor_maps
    got = buf.cpu().numpy().view(np.uint64).reshape(len(ids), wpp)
    for p, g in enumerate(ids):
        assert np.array_equal(got[p], nhd_words(int(g))), f"buffer page {p} is not pool page {g} transposed"
    dst = np.array([262142, 1, 200000, 262141], dtype=np.int32)
    kv.kv_unpack(ctx, buf, dst, desc, 1, T, T, len(ids) * T)
    torch.cuda.synchronize()
    view = slab.view(P, wpp)
    for p, g in enumerate(dst):  # HND -> NHD buffer -> HND page: the source page's words, in place
        src = np.arange(int(ids[p]) * wpp, (int(ids[p]) + 1) * wpp, dtype=np.uint64) * np.uint64(0x9E3779B97F4A7C15)
        assert np.array_equal(view[int(g)].cpu().numpy().view(np.uint64), src)
    del slab, view
    torch.cuda.empty_cache()


@pytest.mark.parametrize("orders", [(0, 0), (1, 0), (0, 1)])
def test_repage_with_device_resident_ids(kv, ctx, orders):
    """kv_repage_batched with KV_FLAG_IDS_ON_DEVICE: both id lists are device arrays (say, written by a
    GPU-side slot allocator); an out-of-range id of either list skips its piece and raises the status word."""
    L, C, H, D, e, Ts, Td = 3, 2, 4, 128, 2, 16, 64
    rng = np.random.default_rng(131 + orders[0] * 2 + orders[1])
    ntok = [2048 - 37, 0, 100, 64]
    ns, nd = [-(-t // Ts) for t in ntok], [-(-t // Td) for t in ntok]
    A = host_pool(rng, L, C, sum(ns) + 9, Ts, H, D, e, order=orders[0])
    B = host_pool(rng, L, C, sum(nd) + 7, Td, H, D, e, order=orders[1])
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    soff = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
    sids = rng.permutation(sum(ns) + 9)[:soff[-1]].astype(np.int32)
    dids = rng.permutation(sum(nd) + 7)[:doff[-1]].astype(np.int32)
    d_s, d_d = torch.from_numpy(sids).cuda(), torch.from_numpy(dids).cuda()
    kv.kv_repage_batched(ctx, dA, d_s, soff, dB, d_d, doff, ntok, L, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    torch.cuda.synchronize()
    ko.repage_batched(A, sids, soff, B, dids, doff, ntok)
    assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)
    assert ctx.device_status() == 0
    # a bad SOURCE id: the pieces that would read it are skipped, everything else is as the oracle says
    bad = sids.copy()
    bad[3] = A.num_pages + 5
    d_s.copy_(torch.from_numpy(bad))
    kv.kv_repage_batched(ctx, dA, d_s, soff, dB, d_d, doff, ntok, L, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert ctx.device_status() == 1
    assert ctx.device_status() == 0  # reading clears it
    # the single-request entry takes device tensors too
    one_s, one_d = d_s[:0], d_d[:0]
    kv.kv_repage(ctx, dA, one_s, dB, one_d, L, 0, flags=kv.KV_FLAG_IDS_ON_DEVICE)  # empty: KV_OK


# ------------------------------------------------------------------------------------------------
# layer-first host buffers through the staged pipeline, and the layer-by-layer reload
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("staging_mib,Ts,Td", [(8, 16, 16), (2, 16, 16), (1, 16, 64), (2, 64, 16), (8, 16, 24)])
def test_layer_first_host_tier_staged_equals_direct_equals_oracle(kv, order, staging_mib, Ts, Td):
    """KV_HOST_STAGED with a layer-first buffer: chunks of whole layers (8 MiB staging), layers cut by page
    ranges (1-2 MiB staging: one layer of the widest request does not fit a slot), re-paging, batched with
    an empty request, NHD and HND pools.  Host bytes and pool bytes equal the oracle's in both modes."""
    L, C, H, D, e = 5, 2, 4, 128, 2
    rng = np.random.default_rng(151 + staging_mib + Ts + Td + order)
    ctx = kv.Ctx(0, staging_bytes=staging_mib << 20)
    counts_tok = [Ts * 90 - 7, 0, Ts * 3, 1, Ts * 41]
    ns = [-(-t // Ts) for t in counts_tok]
    nd = [-(-t // Td) for t in counts_tok]
    A = host_pool(rng, L, C, sum(ns) + 11, Ts, H, D, e, order=order)
    B = host_pool(rng, L, C, sum(nd) + 13, Td, H, D, e, order=order)
    tA, dA = to_device(A, kv, torch)
    soff = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
    sids = rng.permutation(sum(ns) + 11)[:soff[-1]].astype(np.int32)
    dids = rng.permutation(sum(nd) + 13)[:doff[-1]].astype(np.int32)
    page_s = dA.page_bytes()
    hps = [kv.kv_host_alloc(max(n * page_s, 16)) for n in ns]
    try:
        want = ko.pack_batched(A, sids, soff, layout=ko.LAYER_FIRST)
        for m in (kv.KV_HOST_STAGED, kv.KV_HOST_DIRECT):
            for hp, n in zip(hps, ns):
                kv.host_view(hp, max(n * page_s, 16))[:] = 0x5A
            kv.kv_offload_batched(ctx, dA, L, sids, soff, hps, [n * page_s for n in ns], mode=m,
                                  layout=kv.KV_LAYOUT_LAYER_FIRST)
            torch.cuda.synchronize()
            assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == m
            for r, n in enumerate(ns):
                assert np.array_equal(kv.host_view(hps[r], n * page_s)[:n * page_s], want[r]), f"mode {m} request {r}"
            Bm = ko.HostPool([s.copy() for s in B.slabs], L, C, B.num_pages, Td, H, D, e, B.page_stride_bytes, order)
            tB, dB = to_device(Bm, kv, torch)
            kv.kv_reload_batched(ctx, hps, dids, doff, counts_tok, dB, L, Ts, Td,
                                 host_bytes=[n * page_s for n in ns], mode=m, layout=kv.KV_LAYOUT_LAYER_FIRST,
                                 flags=kv.KV_FLAG_VALIDATE)
            torch.cuda.synchronize()
            ko.unpack_batched(want, dids, doff, counts_tok, Bm, Ts=Ts, layout=ko.LAYER_FIRST)
            assert_pool_equal(tB, Bm)
    finally:
        torch.cuda.synchronize()
        ctx.close()
        for hp in hps:
            kv.kv_host_free(hp)


@pytest.mark.parametrize("mode", ["staged", "direct"])
def test_reload_layerwise_publishes_layers_in_order(kv, mode):
    """kv_reload_layerwise: flag l is stored only after layer l's pages are in the pool, and (staged) long
    before the whole transfer ends.  A second stream waits for each flag ON THE DEVICE and snapshots that
    layer at once; every snapshot must already equal the oracle's layer."""
    m = {"staged": kv.KV_HOST_STAGED, "direct": kv.KV_HOST_DIRECT}[mode]
    L, C, P, T, H, D, e = 12, 2, 700, 16, 4, 128, 2   # 1 MiB... per (layer, K|V): 600 pages x 16 KiB = 9.4 MiB
    rng = np.random.default_rng(157)
    ctx = kv.Ctx(0, staging_bytes=48 << 20)   # 24 MiB slots: one layer (18.75 MiB) per chunk
    B = host_pool(rng, L, C, P, T, H, D, e)
    tB, dB = to_device(B, kv, torch)
    n = 600
    dst = rng.permutation(P)[:n].astype(np.int32)
    nbytes = n * dB.page_bytes()
    hp = kv.kv_host_alloc(nbytes)
    fl_p = kv.kv_host_alloc(L * 8)
    try:
        src = rng.integers(0, 256, size=nbytes, dtype=np.uint8)
        kv.host_view(hp, nbytes)[:] = src
        flags_h = kv.host_view(fl_p, L * 8).view(np.uint64)
        flags_h[:] = 0
        ko.unpack(src, dst, B, Ts=T, n_tokens=n * T, layout=ko.LAYER_FIRST)  # B is now the expected pool
        side = torch.cuda.Stream()
        main = torch.cuda.Stream()
        seen_order = []
        kv.kv_reload_layerwise(ctx, hp, nbytes, dst, dB, L, T, T, n * T, fl_p, 42, mode=m, stream=main)
        assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == m
        snaps = []
        import time
        t0 = time.time()
        for l in range(L):  # the host polls the mapped flags; the snapshot of layer l starts the moment flag l is seen
            while flags_h[l] != 42:
                assert time.time() - t0 < 20, f"flag {l} never arrived"
            seen_order.append([int(x) for x in flags_h])
            with torch.cuda.stream(side):
                snaps.append([tB[l * C + c].clone() for c in range(C)])
        side.synchronize()
        main.synchronize()
        for l in range(L):
            assert all(x == 42 for x in seen_order[l][:l + 1]), "flags are stored in ascending layer order"
            for c in range(C):
                assert np.array_equal(snaps[l][c].cpu().numpy(), B.slabs[l * C + c]), f"layer {l} was published early"
        import os
        if mode == "staged" and os.environ.get("CUDA_LAUNCH_BLOCKING") != "1":  # (blocking launches: the call returns when all is done)
            # streaming: when flag 0 was seen the last layer had not been published yet
            streamed = seen_order[0][L - 1] == 0
            for _ in range(3):  # a descheduled polling thread can miss the window: look again (timing only)
                if streamed:
                    break
                flags_h[:] = 0
                main.synchronize()
                kv.kv_reload_layerwise(ctx, hp, nbytes, dst, dB, L, T, T, n * T, fl_p, 42, mode=m, stream=main)
                t0 = time.time()
                while flags_h[0] != 42:
                    assert time.time() - t0 < 20
                streamed = flags_h[L - 1] == 0
                main.synchronize()
            assert streamed, "layer 0 was never published before the last layer"
        assert_pool_equal(tB, B)
        # no pages: the flags are still stored
        flags_h[:] = 0
        kv.kv_reload_layerwise(ctx, hp, 0, [], dB, L, T, T, 0, fl_p, 7, mode=m, stream=main)
        main.synchronize()
        assert (flags_h == 7).all()
    finally:
        torch.cuda.synchronize()
        ctx.close()
        kv.kv_host_free(hp)
        kv.kv_host_free(fl_p)


def test_reload_layerwise_errors_and_capture(kv, ctx):
    """Flag array in pageable memory is refused before anything is enqueued; under stream capture the call is one
    DIRECT launch plus the flag stores, replayable."""
    L, C, P, T, H, D, e = 4, 2, 64, 16, 2, 64, 2
    rng = np.random.default_rng(163)
    B = host_pool(rng, L, C, P, T, H, D, e)
    tB, dB = to_device(B, kv, torch)
    n = 20
    dst = rng.permutation(P)[:n].astype(np.int32)
    nbytes = n * dB.page_bytes()
    hp = kv.kv_host_alloc(nbytes)
    try:
        src = rng.integers(0, 256, size=nbytes, dtype=np.uint8)
        kv.host_view(hp, nbytes)[:] = src
        pageable = np.zeros(L, dtype=np.uint64)
        with pytest.raises(kv.KvError) as ei:
            kv.kv_reload_layerwise(ctx, hp, nbytes, dst, dB, L, T, T, n * T, pageable, 1)
        assert ei.value.status == kv.KV_ERR_HOST_MEM
        torch.cuda.synchronize()
        assert_pool_equal(tB, B)  # nothing moved
        dflags = torch.zeros(L, dtype=torch.int64, device="cuda")
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            kv.kv_reload_layerwise(ctx, hp, nbytes, dst, dB, L, T, T, n * T, dflags, 9, stream=side)
        assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_DIRECT
        ko.unpack(src, dst, B, Ts=T, n_tokens=n * T, layout=ko.LAYER_FIRST)
        for rep in range(2):
            dflags.zero_()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            assert (dflags == 9).all()
            assert_pool_equal(tB, B)
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


def test_layer_ranges_offload_behind_producer_events(kv, ctx):
    """Offload that follows the producer layer by layer WITHOUT any device-side waiting: a layer range is
    just a descriptor whose base array starts at that layer, written to that layer's place in the
    layer-first host buffer; ordering comes from cudaStreamWaitEvent on the producer's per-layer events.
    (A kernel or stream operation that waits for a flag another stream raises is not used anywhere in
    this library: nothing guarantees the two run at the same time.)"""
    L, C, P, T, H, D, e = 6, 2, 300, 16, 4, 128, 2
    rng = np.random.default_rng(173)
    final = host_pool(rng, L, C, P, T, H, D, e)
    t_final = [torch.from_numpy(x).cuda() for x in final.slabs]
    t_pool = [torch.full_like(x, 0x11) for x in t_final]  # stale
    n = 200
    ids = rng.permutation(P)[:n].astype(np.int32)
    row = T * H * D * e
    nbytes = n * L * C * row
    hp = kv.kv_host_alloc(nbytes)
    try:
        s_prod, s_off = torch.cuda.Stream(), torch.cuda.Stream()
        evs = []
        with torch.cuda.stream(s_prod):
            for l in range(L):
                torch.cuda._sleep(500_000)
                for c in range(C):
                    t_pool[l * C + c].copy_(t_final[l * C + c])
                ev = torch.cuda.Event()
                ev.record(s_prod)
                evs.append(ev)
        for l0 in range(0, L, 2):  # ranges of two layers
            s_off.wait_event(evs[l0 + 1])
            sub = kv.PoolDesc(t_pool[l0 * C:(l0 + 2) * C], 2, C, P, T, H, D, e)
            kv.kv_offload(ctx, sub, 2, ids, hp + l0 * C * n * row, 2 * C * n * row,
                          layout=kv.KV_LAYOUT_LAYER_FIRST, stream=s_off)
        s_off.synchronize()
        want = ko.pack(final, ids, layout=ko.LAYER_FIRST)
        assert np.array_equal(kv.host_view(hp, nbytes), want)
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


def test_cow_append_with_device_resident_ids(kv, ctx):
    """kv_cow_append_batched with KV_FLAG_IDS_ON_DEVICE: old / new page ids in device arrays; a bad session
    (id out of range, or old == new) is skipped and raises the status word, the others are as the oracle says."""
    L, C, P, T, H, D, e = 3, 2, 64, 16, 4, 128, 2
    rng = np.random.default_rng(179)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    S = 7
    perm = rng.permutation(P).astype(np.int32)
    old, new = perm[:S].copy(), perm[S:2 * S].copy()
    n_old = rng.integers(0, T + 1, size=S)
    n_app = np.array([rng.integers(0, T - o + 1) for o in n_old])
    n_old[0], n_app[0] = 5, 4
    apps = [rng.integers(0, 256, size=L * C * int(a) * H * D * e, dtype=np.uint8) for a in n_app]
    dev = [torch.from_numpy(a).cuda() if a.size else None for a in apps]
    d_old, d_new = torch.from_numpy(old).cuda(), torch.from_numpy(new).cuda()
    kv.kv_cow_append_batched(ctx, dA, L, d_old, d_new, n_old, n_app, dev, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    torch.cuda.synchronize()
    ko.cow_append_batched(A, old, new, n_old, n_app, apps)
    assert_pool_equal(tA, A)
    assert ctx.device_status() == 0
    # session 0 gets an out-of-range new id, session 1 old == new: both skipped, the rest done again (idempotent)
    bad_new = new.copy()
    bad_new[0] = P + 3
    bad_new[1] = old[1]
    d_new.copy_(torch.from_numpy(bad_new))
    kv.kv_cow_append_batched(ctx, dA, L, d_old, d_new, n_old, n_app, dev, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert ctx.device_status() == 1
    assert_pool_equal(tA, A)
    with pytest.raises(kv.KvError) as ei:
        kv.kv_cow_append(ctx, dA, L, 1, 2, 3, None, 0, flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert ei.value.status == kv.KV_ERR_LAYOUT


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("H", [1, 2])
def test_narrow_rows_of_a_head_partition(kv, ctx, H, order):
    """A tensor-parallel rank holds its own head partition of every page: 1 or 2 KV heads =
    4 / 8 KiB rows: one row per single-warp CTA (kv_move_shot); with KV_OPT_KERNEL = bulk and enough segments the ring
    re-shapes itself (8 x 4 or 4 x 4 stages instead of 2 x 4).  Same bytes as the oracle, NHD and HND."""
    L, C, P, T, D, e = 48, 2, 160, 16, 128, 2
    rng = np.random.default_rng(181 + H + 2 * order)
    A = host_pool(rng, L, C, P, T, H, D, e, order=order)
    B = host_pool(rng, L, C, P, T, H, D, e, order=order)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    n = 64 if H == 1 else 40  # x 96 slabs = 6,144 / 3,840 segments: enough for the re-shaped ring
    src = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, L, src, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT and ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 4096 * H
    want = ko.pack(A, src)
    assert np.array_equal(buf.cpu().numpy(), want)
    ctx.set_option(kv.KV_OPT_KERNEL, kv.KV_KERNEL_BULK)  # the re-shaped ring moves the same bytes
    buf.zero_()
    kv.kv_pack(ctx, dA, L, src, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_BULK and ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 4096 * H
    assert np.array_equal(buf.cpu().numpy(), want)
    ctx.set_option(kv.KV_OPT_KERNEL, kv.KV_KERNEL_AUTO)
    kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T - 5, flags=kv.KV_FLAG_VALIDATE)
    ko.unpack(want, dst, B, Ts=T, n_tokens=n * T - 5)
    assert_pool_equal(tB, B)
    kv.kv_repage(ctx, dA, src, dB, dst[::-1].copy(), L, n * T)
    ko.repage(A, src, B, dst[::-1].copy(), n_tokens=n * T)
    assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)


def test_four_threads_four_contexts(kv):
    """'One ctx per calling thread' (kvtier.h): four host threads, each with its own ctx and stream, hammer the same
    source pool into their own destination pools at once (ctypes drops the GIL inside the library, so the C side
    really runs concurrently).  Every thread's result equals the oracle's."""
    import threading
    L, C, P, T, H, D, e = 4, 2, 128, 16, 4, 128, 2
    rng = np.random.default_rng(191)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n, rounds, nthreads = 48, 25, 4
    plans = []
    for t in range(nthreads):
        r = np.random.default_rng(1000 + t)
        B = host_pool(r, L, C, P, T, H, D, e, order=t % 2)
        tB, dB = to_device(B, kv, torch)
        steps = [(r.choice(P, n, replace=False).astype(np.int32), r.permutation(P)[:n].astype(np.int32)) for _ in range(rounds)]
        plans.append((B, tB, dB, steps))
    errors = []

    def worker(t):
        try:
            B, tB, dB, steps = plans[t]
            ctx = kv.Ctx(0, staging_bytes=8 << 20)
            stream = torch.cuda.Stream()
            buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
            for src, dst in steps:
                kv.kv_pack(ctx, dA, L, src, buf, stream=stream)
                kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, stream=stream)
            stream.synchronize()
            ctx.close()
        except Exception as ex:  # noqa: BLE001
            errors.append((t, repr(ex)))

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(nthreads)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    assert not errors, errors
    torch.cuda.synchronize()
    for B, tB, dB, steps in plans:
        for src, dst in steps:
            ko.unpack(ko.pack(A, src), dst, B, Ts=T, n_tokens=n * T)
        assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)
