"""GPU parity, round 2: several transfers in ONE launch (kv_submit: the direction is a property of the piece),
STAGED host transfers captured into CUDA graphs and replayed, staged transfers of ONE ctx on two streams,
and the peer-GPU push (runs where a second GPU is visible).  Everything byte for byte against the CPU oracle
(the mixed call = the oracle's single functions applied in sequence: its operations are independent)."""
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


KERNELS = {"auto": 0, "bulk": 1, "vec": 2, "elem": 3, "shot": 4}


# ------------------------------------------------------------------------------------------------
# kv_submit: a turn's scatter + copy-on-write appends + gather in one launch
# ------------------------------------------------------------------------------------------------
def _turn(kv, rng, A, n_unpack, n_pack, n_cow, ragged, layout):
    """Operations of one submit on host pool A + the oracle's result.  Returns (ops builder, check)."""
    L, C, P, T, H, D, e = A.L, A.C, A.num_pages, A.T, A.H, A.D, A.e
    page = L * C * T * H * D * e
    perm = rng.permutation(P).astype(np.int32)
    k = 0
    un_ids = [perm[k + sum(n_unpack[:i]):k + sum(n_unpack[:i + 1])] for i in range(len(n_unpack))]
    k += sum(n_unpack)
    pk_ids = [perm[k + sum(n_pack[:i]):k + sum(n_pack[:i + 1])] for i in range(len(n_pack))]
    k += sum(n_pack)
    old, new = perm[k:k + n_cow], perm[k + n_cow:k + 2 * n_cow]
    ntoks = [n * T - (int(rng.integers(0, T)) if ragged and n else 0) for n in n_unpack]  # ceil(ntok / T) == n
    srcs = [rng.integers(0, 256, size=max(n * page, 16), dtype=np.uint8) for n in n_unpack]
    n_old = rng.integers(0, T + 1, size=n_cow)
    n_app = np.array([rng.integers(0, T - o + 1) for o in n_old], dtype=np.int64)
    apps = [rng.integers(0, 256, size=L * C * int(a) * H * D * e, dtype=np.uint8) for a in n_app]
    return dict(un_ids=un_ids, pk_ids=pk_ids, old=old, new=new, ntoks=ntoks, srcs=srcs, n_old=n_old, n_app=n_app,
                apps=apps, page=page)


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("kernel", list(KERNELS))
def test_submit_mixed_operations_equal_the_single_calls(kv, ctx, kernel, order, layout):
    L, C, P, T, H, D, e = 3, 2, 96, 16, 4, 64, 2
    rng = np.random.default_rng(1000 + 7 * KERNELS[kernel] + 3 * order + layout)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    A = host_pool(rng, L, C, P, T, H, D, e, pad=(6 if kernel == "elem" else 0), order=order)
    tA, dA = to_device(A, kv, torch)
    t = _turn(kv, rng, A, n_unpack=[9, 0, 5], n_pack=[7, 11], n_cow=4, ragged=True, layout=layout)
    d_srcs = [torch.from_numpy(s).cuda() for s in t["srcs"]]
    d_apps = [torch.from_numpy(a).cuda() if a.size else None for a in t["apps"]]
    d_bufs = [torch.full((len(i) * t["page"],), 0xCD, dtype=torch.uint8, device="cuda") for i in t["pk_ids"]]
    ops = []
    for s_, ids, nt in zip(d_srcs, t["un_ids"], t["ntoks"]):
        ops.append(kv.op_unpack(s_, ids, nt, src_bytes=len(ids) * t["page"]))
    for i in range(len(t["old"])):
        ops.append(kv.op_cow_append(int(t["old"][i]), int(t["new"][i]), int(t["n_old"][i]), d_apps[i], int(t["n_app"][i])))
    for b, ids in zip(d_bufs, t["pk_ids"]):
        ops.append(kv.op_pack(ids, b))
    # the oracle: pack first (it reads the pool as it was), then the writes -- any order gives the same bytes because
    # the operations are independent
    wants = [ko.pack(A, ids, layout=layout) for ids in t["pk_ids"]]
    launches = ctx.stat(kv.KV_STAT_LAUNCHES)
    kv.kv_submit(ctx, dA, L, ops, layout=layout, flags=kv.KV_FLAG_VALIDATE)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == launches + 1, "one launch for the whole list"
    torch.cuda.synchronize()
    for s_, ids, nt in zip(t["srcs"], t["un_ids"], t["ntoks"]):
        if len(ids):
            ko.unpack(s_[:len(ids) * t["page"]], ids, A, Ts=T, n_tokens=nt, layout=layout)
    ko.cow_append_batched(A, t["old"], t["new"], t["n_old"], t["n_app"], t["apps"])
    for b, w in zip(d_bufs, wants):
        assert np.array_equal(b.cpu().numpy(), w), "pack operation != oracle"
    assert_pool_equal(tA, A)


def test_submit_errors_write_nothing(kv, ctx):
    L, C, P, T, H, D, e = 2, 2, 32, 16, 2, 64, 2
    rng = np.random.default_rng(77)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    page = dA.page_bytes()
    buf = torch.full((4 * page,), 0x11, dtype=torch.uint8, device="cuda")
    src = torch.zeros(4 * page, dtype=torch.uint8, device="cuda")
    good = kv.op_unpack(src, [1, 2, 3, 4], 4 * T)
    for bad, status in ((kv.op_pack([5, 6, P], buf), kv.KV_ERR_PAGE_RANGE),
                        (kv.op_pack([5, 6, 7, 8, 9], buf), kv.KV_ERR_SIZE),
                        (kv.op_cow_append(9, 9, 1, src, 1), kv.KV_ERR_SIZE),
                        (kv.op_unpack(src, [1, 2, 3], 4 * T), kv.KV_ERR_SIZE)):
        with pytest.raises(kv.KvError) as ei:
            kv.kv_submit(ctx, dA, L, [good, bad])  # the valid operation before it must not run either
        assert ei.value.status == status
    with pytest.raises(kv.KvError) as ei:
        kv.kv_submit(ctx, dA, L, [good, kv.op_cow_append(9, 4, 1, src, 1)], flags=kv.KV_FLAG_VALIDATE)
    assert ei.value.status == kv.KV_ERR_DUP_PAGE
    torch.cuda.synchronize()
    assert_pool_equal(tA, A)
    assert bool((buf == 0x11).all())


def test_submit_captured_turn_replays(kv, ctx):
    """A whole turn as ONE kernel node of a CUDA graph (host ids baked in)."""
    L, C, P, T, H, D, e = 4, 2, 128, 16, 2, 64, 2
    rng = np.random.default_rng(79)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    t = _turn(kv, rng, A, n_unpack=[20], n_pack=[13], n_cow=2, ragged=False, layout=0)
    d_src = torch.from_numpy(t["srcs"][0]).cuda()
    d_apps = [torch.from_numpy(a).cuda() if a.size else None for a in t["apps"]]
    buf = torch.zeros(13 * t["page"], dtype=torch.uint8, device="cuda")
    ops = [kv.op_unpack(d_src, t["un_ids"][0], t["ntoks"][0]), kv.op_pack(t["pk_ids"][0], buf)]
    ops += [kv.op_cow_append(int(t["old"][i]), int(t["new"][i]), int(t["n_old"][i]), d_apps[i], int(t["n_app"][i]))
            for i in range(2)]
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        kv.kv_submit(ctx, dA, L, ops, stream=side)
    want = ko.pack(A, t["pk_ids"][0])
    ko.unpack(t["srcs"][0], t["un_ids"][0], A, Ts=T, n_tokens=t["ntoks"][0])
    ko.cow_append_batched(A, t["old"], t["new"], t["n_old"], t["n_app"], t["apps"])
    for _ in range(2):
        buf.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(buf.cpu().numpy(), want)
        assert_pool_equal(tA, A)


# ------------------------------------------------------------------------------------------------
# STAGED host transfers inside a CUDA graph: copy nodes on a forked branch + one kernel node
# per chunk with its tables in its parameters; device-resident ids are re-read at every replay
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("dev_ids", [False, True])
def test_staged_offload_and_reload_captured_and_replayed(kv, layout, dev_ids):
    L, C, P, T, H, D, e = 6, 2, 256, 16, 4, 128, 2  # page = 192 KiB
    rng = np.random.default_rng(83 + layout)
    A = host_pool(rng, L, C, P, T, H, D, e)
    B = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    n = 100
    nbytes = n * dA.page_bytes()  # 18.75 MiB through 2 x 4 MiB slots: five chunks each way
    ctx = kv.Ctx(0, staging_bytes=8 << 20)
    hp = kv.kv_host_alloc(nbytes)
    try:
        hv = kv.host_view(hp, nbytes)
        side = torch.cuda.Stream()
        flags = kv.KV_FLAG_IDS_ON_DEVICE if dev_ids else 0
        src0 = rng.choice(P, n, replace=False).astype(np.int32)
        dst0 = rng.permutation(P)[:n].astype(np.int32)
        d_src = torch.from_numpy(src0).cuda()
        d_dst = torch.from_numpy(dst0).cuda()
        # without a staging buffer an explicit STAGED cannot be captured (an allocation would break the capture)
        g0 = torch.cuda.CUDAGraph()
        flag0 = torch.zeros(1, dtype=torch.int64, device="cuda")  # (allocated before the capture: no allocation inside one)
        torch.cuda.synchronize()
        with torch.cuda.graph(g0, stream=side):
            with pytest.raises(kv.KvError) as ei:
                kv.kv_offload(ctx, dA, L, src0, hp, nbytes, mode=kv.KV_HOST_STAGED, layout=layout, stream=side)
            assert ei.value.status == kv.KV_ERR_CAPTURE
            kv.kv_signal(ctx, flag0, 1, stream=side)  # a graph must not be empty
        ctx.set_option(kv.KV_OPT_RESERVE_STAGING, 0)
        memcpys = ctx.stat(kv.KV_STAT_MEMCPYS)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            kv.kv_offload(ctx, dA, L, d_src if dev_ids else src0, hp, nbytes, mode=kv.KV_HOST_AUTO, layout=layout,
                          flags=flags, stream=side)
            assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_STAGED  # AUTO captures what it would run eagerly
            kv.kv_reload(ctx, hp, nbytes, d_dst if dev_ids else dst0, dB, L, T, T, n * T, mode=kv.KV_HOST_STAGED,
                         layout=layout, flags=flags, stream=side)
        assert ctx.stat(kv.KV_STAT_MEMCPYS) - memcpys >= 10  # copy nodes only: no table copy was enqueued
        src, dst = src0, dst0
        for rep in range(3):
            if dev_ids and rep:  # fresh ids per replay, no new capture
                src = rng.choice(P, n, replace=False).astype(np.int32)
                dst = rng.permutation(P)[:n].astype(np.int32)
                d_src.copy_(torch.from_numpy(src))
                d_dst.copy_(torch.from_numpy(dst))
            hv[:] = 0
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            want = ko.pack(A, src, layout=layout)
            assert np.array_equal(hv, want), f"replay {rep}: captured staged offload != oracle"
            ko.unpack(want, dst, B, Ts=T, n_tokens=n * T, layout=layout)
            assert_pool_equal(tB, B)
        # an eager staged call on the same stream after the replays: the graph's slots are ordered by the stream
        with torch.cuda.stream(side):
            kv.kv_reload(ctx, hp, nbytes, dst[::-1].copy(), dB, L, T, T, n * T, mode=kv.KV_HOST_STAGED, layout=layout,
                         stream=side)
        torch.cuda.synchronize()
        ko.unpack(want, dst[::-1].copy(), B, Ts=T, n_tokens=n * T, layout=layout)
        assert_pool_equal(tB, B)
        assert ctx.device_status() == 0
    finally:
        torch.cuda.synchronize()
        ctx.close()
        kv.kv_host_free(hp)


def test_eager_staged_call_while_a_capture_of_the_same_ctx_is_open(kv):
    """Between cudaStreamBeginCapture and EndCapture of a graph that holds a staged transfer, the ctx's side stream is
    part of that capture.  An eager multi-chunk staged transfer of the same ctx on ANOTHER stream must not enqueue onto
    it: explicit KV_HOST_STAGED is refused (KV_ERR_CAPTURE, nothing written), KV_HOST_AUTO moves the bytes with DIRECT,
    and the graph under construction stays valid and replays the oracle's bytes."""
    L, C, P, T, H, D, e = 6, 2, 256, 16, 4, 128, 2  # page = 192 KiB
    rng = np.random.default_rng(97)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n = 100
    nbytes = n * dA.page_bytes()  # 18.75 MiB through 2 x 4 MiB slots: five chunks
    ctx = kv.Ctx(0, staging_bytes=8 << 20)
    h_graph, h_eager = kv.kv_host_alloc(nbytes), kv.kv_host_alloc(nbytes)
    try:
        v_graph, v_eager = kv.host_view(h_graph, nbytes), kv.host_view(h_eager, nbytes)
        v_graph[:] = 0
        v_eager[:] = 0xEE
        ids_g = rng.choice(P, n, replace=False).astype(np.int32)
        ids_e = rng.choice(P, n, replace=False).astype(np.int32)
        ctx.set_option(kv.KV_OPT_RESERVE_STAGING, 0)
        cap_stream, other = torch.cuda.Stream(), torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=cap_stream, capture_error_mode="thread_local"):
            kv.kv_offload(ctx, dA, L, ids_g, h_graph, nbytes, mode=kv.KV_HOST_STAGED, stream=cap_stream)
            # the capture is still open: the side stream is inside it
            with pytest.raises(kv.KvError) as ei:
                kv.kv_offload(ctx, dA, L, ids_e, h_eager, nbytes, mode=kv.KV_HOST_STAGED, stream=other)
            assert ei.value.status == kv.KV_ERR_CAPTURE
            kv.kv_offload(ctx, dA, L, ids_e, h_eager, nbytes, mode=kv.KV_HOST_AUTO, stream=other)
            assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_DIRECT
        other.synchronize()
        assert np.array_equal(v_eager, ko.pack(A, ids_e)), "the eager AUTO call (DIRECT) != oracle"
        assert np.all(v_graph == 0), "a captured transfer ran before its graph was launched"
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(v_graph, ko.pack(A, ids_g)), "the graph captured around the refused call != oracle"
        v_eager[:] = 0xEE  # with the capture closed, the eager staged pipeline is available again
        kv.kv_offload(ctx, dA, L, ids_e, h_eager, nbytes, mode=kv.KV_HOST_STAGED, stream=other)
        other.synchronize()
        assert np.array_equal(v_eager, ko.pack(A, ids_e))
    finally:
        torch.cuda.synchronize()
        ctx.close()
        kv.kv_host_free(h_graph)
        kv.kv_host_free(h_eager)


# ------------------------------------------------------------------------------------------------
# ONE ctx, staged transfers on TWO streams with different chunk sizes: the slots are fixed pieces of the staging
# buffer, so the per-slot events order the two calls whatever their chunking (kvtier.h "A kv_ctx ...")
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lead_mib,repage", [(-1, False), (0, False), (100, False), (-1, True), (8, True)])
def test_staged_transfer_with_a_short_leading_chunk(kv, lead_mib, repage):
    """Staged page-first transfers of 128 MiB or more lead an offload / end a reload with a SHORT chunk
    (KV_OPT_LEAD_CHUNK, default 32 MiB) so that the one kernel no copy hides is a short one: unequal chunks, the
    oracle's bytes (reload also with re-paging 16 -> 64, where a chunk must hold whole pages of both sizes)."""
    L, C, P, T, H, D, e = 16, 2, 330, 16, 4, 128, 2  # page = 512 KiB; 300 pages = 150 MiB
    rng = np.random.default_rng(11 + lead_mib + 7 * repage)
    A = host_pool(rng, L, C, P, T, H, D, e)
    tA, dA = to_device(A, kv, torch)
    n = 300
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    page = dA.page_bytes()
    ctx = kv.Ctx(0, staging_bytes=256 << 20)  # two slots of 128 MiB
    try:
        if lead_mib >= 0:
            ctx.set_option(kv.KV_OPT_LEAD_CHUNK, lead_mib << 20)
        hp = kv.kv_host_alloc(n * page)
        kv.host_view(hp, n * page)[:] = 0xEE
        l0, m0 = ctx.stat(kv.KV_STAT_LAUNCHES), ctx.stat(kv.KV_STAT_MEMCPYS)
        kv.kv_offload(ctx, dA, L, ids, hp, n * page, mode=kv.KV_HOST_STAGED)
        torch.cuda.synchronize()
        chunks = ctx.stat(kv.KV_STAT_LAUNCHES) - l0
        assert chunks == ctx.stat(kv.KV_STAT_MEMCPYS) - m0
        # equal chunks: two of 75 MiB; a 32 MiB lead: 32 + 118; a 100 MiB lead is more than half the payload: refused
        assert chunks == (2 if lead_mib in (0, 100) else 2 if lead_mib == -1 else 3)
        want = ko.pack(A, ids)
        assert np.array_equal(kv.host_view(hp, n * page), want)
        if repage:
            Td, Pd = 64, 90
            B = host_pool(rng, L, C, Pd, Td, H, D, e)
            tB, dB = to_device(B, kv, torch)
            ntok = n * T - 21
            nd = -(-ntok // Td)
            dst = rng.permutation(Pd)[:nd].astype(np.int32)
            kv.kv_reload(ctx, hp, n * page, dst, dB, L, T, Td, ntok, mode=kv.KV_HOST_STAGED)
            ko.unpack(want, dst, B, Ts=T, n_tokens=ntok)
        else:
            B = host_pool(rng, L, C, P, T, H, D, e)
            tB, dB = to_device(B, kv, torch)
            dst = rng.permutation(P)[:n].astype(np.int32)
            kv.kv_reload(ctx, hp, n * page, dst, dB, L, T, T, n * T, mode=kv.KV_HOST_STAGED)
            ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
        torch.cuda.synchronize()
        assert_pool_equal(tB, B)
        assert_pool_equal(tA, A)
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)
        ctx.close()


@pytest.mark.parametrize("rep", range(3))
def test_two_streams_one_ctx_staged_calls_share_the_slots(kv, rep):
    L, C, P, T, H, D, e = 8, 2, 512, 16, 4, 128, 2  # page = 256 KiB
    rng = np.random.default_rng(91 + rep)
    B = host_pool(rng, L, C, P, T, H, D, e)
    tB, dB = to_device(B, kv, torch)
    n1, n2 = 160, 90
    perm = rng.permutation(P).astype(np.int32)
    dst1, dst2 = perm[:n1], perm[n1:n1 + n2]
    nb1, nb2 = n1 * dB.page_bytes(), n2 * dB.page_bytes()  # 40 MiB and 22.5 MiB
    ctx = kv.Ctx(0, staging_bytes=32 << 20)  # two slots of 16 MiB
    h1, h2, fl = kv.kv_host_alloc(nb1), kv.kv_host_alloc(nb2), kv.kv_host_alloc(L * 8)
    try:
        s1 = rng.integers(0, 256, size=nb1, dtype=np.uint8)
        s2 = rng.integers(0, 256, size=nb2, dtype=np.uint8)
        kv.host_view(h1, nb1)[:] = s1
        kv.host_view(h2, nb2)[:] = s2
        kv.host_view(fl, L * 8)[:] = 0
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        # call A: plain reload in 16 MiB chunks on stream sa; call B right behind it on stream sb: a layer-by-layer
        # reload, whose chunks are capped (64 MiB rule, here the 4 MiB option) -> different chunk size, same slots
        kv.kv_reload(ctx, h1, nb1, dst1, dB, L, T, T, n1 * T, mode=kv.KV_HOST_STAGED, stream=sa)
        ctx.set_option(kv.KV_OPT_CHUNK_BYTES, 4 << 20)
        kv.kv_reload_layerwise(ctx, h2, nb2, dst2, dB, L, T, T, n2 * T, fl, 5, mode=kv.KV_HOST_STAGED, stream=sb)
        ctx.set_option(kv.KV_OPT_CHUNK_BYTES, 0)
        # and an offload of the pages call A is writing, on sb, ordered behind A by an event (it reads A's result)
        ev = torch.cuda.Event()
        ev.record(sa)
        sb.wait_event(ev)
        h3 = kv.kv_host_alloc(nb1)
        kv.kv_offload(ctx, dB, L, dst1, h3, nb1, mode=kv.KV_HOST_STAGED, stream=sb)
        torch.cuda.synchronize()
        ko.unpack(s1, dst1, B, Ts=T, n_tokens=n1 * T)
        ko.unpack(s2, dst2, B, Ts=T, n_tokens=n2 * T, layout=ko.LAYER_FIRST)
        assert_pool_equal(tB, B)
        assert np.array_equal(kv.host_view(h3, nb1), s1), "offload behind the reload != what was reloaded"
        assert (kv.host_view(fl, L * 8).view(np.uint64) == 5).all()
        kv.kv_host_free(h3)
    finally:
        torch.cuda.synchronize()
        ctx.close()
        for h in (h1, h2, fl):
            kv.kv_host_free(h)


# ------------------------------------------------------------------------------------------------
# the provider pushes into a pool on ANOTHER GPU.  One process, two devices.
# ------------------------------------------------------------------------------------------------
def _need_two_gpus():
    if torch.cuda.device_count() < 2 or not torch.cuda.can_device_access_peer(0, 1):
        pytest.skip("needs two peer-accessible GPUs in one process (this lease has one)")


@pytest.mark.parametrize("order", [0, 1])
def test_peer_push_unpack_and_repage_into_a_pool_on_gpu1(kv, ctx, order):
    _need_two_gpus()
    kv.kv_peer_enable(ctx, 1)
    L, C, P, T, H, D, e = 4, 2, 128, 16, 4, 128, 2
    rng = np.random.default_rng(97 + order)
    A = host_pool(rng, L, C, P, T, H, D, e)
    B = host_pool(rng, L, C, 64, 64, H, D, e, order=order)  # the peer's pool: page size 64 (cross-role, config 5)
    tA, dA = to_device(A, kv, torch)
    tB = [torch.from_numpy(x).to("cuda:1") for x in B.slabs]
    dB = kv.PoolDesc(tB, L, C, 64, 64, H, D, e, order=order)
    ntok = 40 * T - 9
    src = rng.choice(P, 40, replace=False).astype(np.int32)
    dst = rng.permutation(64)[:-(-ntok // 64)].astype(np.int32)
    flag = torch.zeros(1, dtype=torch.int64, device="cuda:1")
    buf = torch.zeros(40 * dA.page_bytes(), dtype=torch.uint8, device="cuda:0")
    kv.kv_pack(ctx, dA, L, src, buf)
    kv.kv_unpack(ctx, buf, dst, dB, L, T, 64, ntok)  # posted stores over NVLink into GPU 1's pages
    kv.kv_signal(ctx, flag, 7)                       # availability flag in GPU 1's memory, behind the transfer
    torch.cuda.synchronize(0)
    assert int(flag.cpu()[0]) == 7
    ko.unpack(ko.pack(A, src), dst, B, Ts=T, n_tokens=ntok)
    assert_pool_equal(tB, B)
    dst2 = rng.permutation(64)[:len(dst)].astype(np.int32)
    kv.kv_repage(ctx, dA, src, dB, dst2, L, ntok)    # fused: local pages -> peer pages, no buffer
    torch.cuda.synchronize(0)
    ko.repage(A, src, B, dst2, n_tokens=ntok)
    assert_pool_equal(tB, B)
    # pull direction: pack FROM the peer's pool into a local buffer
    back = torch.zeros(len(dst2) * dB.page_bytes(), dtype=torch.uint8, device="cuda:0")
    kv.kv_pack(ctx, dB, L, dst2, back)
    torch.cuda.synchronize(0)
    assert np.array_equal(back.cpu().numpy(), ko.pack(B, dst2))
