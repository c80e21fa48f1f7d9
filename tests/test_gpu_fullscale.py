"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(default ctx options, 96 GiB pool on one B200, page ids drawn by paper_2606_31093_b200.workloads).

The pool lives only on the device.  Touched pages are snapshotted to the host with torch indexing
(nothing of the library), the oracle runs on that compact mini-pool with renumbered ids (the
result depends only on page contents and order), and the comparison is byte for byte.  The
untouched-pages invariant is checked with per-page 64-bit checksums of every slab before/after.
SURVEY.md 8(c) "Scale"; BASELINE.json:configs[1..4].
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import kv_oracle as ko  # noqa: E402
from paper_2606_31093_b200 import workloads as W  # noqa: E402
from tests.kvhelpers import device_pool, page_checksums, snapshot_pages  # noqa: E402

THREADS = 16


@pytest.fixture(scope="module")
def kv():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    free, _ = torch.cuda.mem_get_info()
    if free < 150 << 30:
        pytest.skip("needs a 180 GB B200 (96 GiB pool + 26.5 GiB batch buffers)")
    from paper_2606_31093_b200 import kvtier
    return kvtier


@pytest.fixture(scope="module")
def pool(kv):
    shape = W.QWEN3_OMNI
    slabs, desc = device_pool(torch, kv, shape, seed=0)
    yield shape, slabs, desc
    del slabs
    torch.cuda.empty_cache()


@pytest.fixture()
def ctx(kv):
    c = kv.Ctx(0)
    yield c
    torch.cuda.synchronize()
    c.close()


def assert_untouched(before, after, touched_ids, P):
    mask = torch.ones(P, dtype=torch.bool, device="cuda")
    mask[torch.as_tensor(np.asarray(touched_ids, dtype=np.int64), device="cuda")] = False
    assert torch.equal(before[:, mask], after[:, mask]), "an untouched page changed"


def test_config2_single_prefix_pack_offload_reload(kv, ctx, pool):
    """BASELINE.json:configs[1]: 512 fragmented pages (8,192 tokens, 768 MiB) -> device staging,
    -> pinned host in both modes, then reloaded into 512 other free pages."""
    shape, slabs, desc = pool
    case = W.prefix_case(0)
    n = len(case.src_ids)
    nbytes = n * shape.page_bytes
    mini = snapshot_pages(torch, slabs, case.src_ids, shape)
    want = ko.pack(mini, np.arange(n), threads=THREADS)
    buf = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, desc, shape.L, case.src_ids, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT and ctx.stat(kv.KV_STAT_LAST_GRID) == 512 * 96
    assert np.array_equal(buf.cpu().numpy(), want), "kv_pack != oracle at full scale"
    hp = kv.kv_host_alloc(nbytes)
    try:
        hv = kv.host_view(hp, nbytes)
        for mode in (kv.KV_HOST_DIRECT, kv.KV_HOST_STAGED, kv.KV_HOST_AUTO):
            hv[:] = 0
            kv.kv_offload(ctx, desc, shape.L, case.src_ids, hp, nbytes, mode=mode)
            torch.cuda.synchronize()
            assert np.array_equal(hv, want), f"kv_offload mode {mode} != oracle"
        before = page_checksums(torch, slabs, shape)
        dst_sets = [case.dst_ids, case.dst_ids[::-1].copy(), np.roll(case.dst_ids, 7)]
        for mode, dst in zip((kv.KV_HOST_DIRECT, kv.KV_HOST_STAGED, -1), dst_sets):
            if mode == -1:
                kv.kv_unpack(ctx, buf, dst, desc, shape.L, shape.T, shape.T, n * shape.T)
            else:
                kv.kv_reload(ctx, hp, nbytes, dst, desc, shape.L, shape.T, shape.T, n * shape.T, mode=mode)
            torch.cuda.synchronize()
            got = snapshot_pages(torch, slabs, dst, shape)
            exp = ko.HostPool([np.zeros_like(s) for s in got.slabs], shape.L, shape.C, n, shape.T,
                              shape.H, shape.D, shape.e, shape.row_bytes)
            ko.unpack(want, np.arange(n), exp, Ts=shape.T, n_tokens=n * shape.T, threads=THREADS)
            for a, b in zip(got.slabs, exp.slabs):
                assert np.array_equal(a, b), f"reload/unpack mode {mode} != oracle"
        after = page_checksums(torch, slabs, shape)
        assert_untouched(before, after, case.dst_ids, shape.P)
        # source pages were never written
        assert torch.equal(before[:, torch.as_tensor(case.src_ids.astype(np.int64), device="cuda")],
                           after[:, torch.as_tensor(case.src_ids.astype(np.int64), device="cuda")])
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


def test_config3_50_turn_session(kv, ctx, pool):
    """BASELINE.json:configs[2]: per turn, reload the matched prefix from the session's host
    buffer into freshly popped scattered pages, then offload the turn's new full pages by
    appending to the host buffer (page-first => tail write).  Checked: the final host buffer and
    the reloaded pages at turns 2, 10, 25 and 50 against the oracle."""
    shape, slabs, desc = pool
    turns = W.session_turns(0)
    rng = np.random.default_rng(0)
    fl = W.FreeList(shape.P, rng)
    total_pages = turns[-1].cum_tokens // shape.T
    hp = kv.kv_host_alloc(total_pages * shape.page_bytes)
    hv = kv.host_view(hp, total_pages * shape.page_bytes)
    expected = np.zeros(total_pages * shape.page_bytes, dtype=np.uint8)
    gen = torch.Generator(device="cuda").manual_seed(123)
    in_host = 0
    check_turns = {2, 10, 25, 50}
    try:
        for t in turns:
            ids = fl.pop(t.n_matched_pages)
            assert t.n_matched_pages == in_host
            kv.kv_reload(ctx, hp, in_host * shape.page_bytes, ids, desc, shape.L, shape.T, shape.T,
                         in_host * shape.T)  # turn 1: n = 0, a no-op
            if t.k in check_turns:
                torch.cuda.synchronize()
                got = snapshot_pages(torch, slabs, ids, shape)
                exp = ko.HostPool([np.zeros_like(s) for s in got.slabs], shape.L, shape.C, len(ids),
                                  shape.T, shape.H, shape.D, shape.e, shape.row_bytes)
                ko.unpack(expected[:in_host * shape.page_bytes], np.arange(len(ids)), exp, Ts=shape.T,
                          n_tokens=in_host * shape.T, threads=THREADS)
                for a, b in zip(got.slabs, exp.slabs):
                    assert np.array_equal(a, b), f"turn {t.k}: reloaded pages != oracle"
            # the turn's prefill writes new KV: pages that become full this turn
            n_new = t.cum_tokens // shape.T - in_host
            new_ids = fl.pop(n_new)
            idx = torch.as_tensor(new_ids.astype(np.int64), device="cuda")
            for s in slabs:
                rows = torch.empty(n_new, shape.row_bytes // 2, dtype=torch.bfloat16, device="cuda").normal_(generator=gen)
                s.view(shape.P, shape.row_bytes).index_copy_(0, idx, rows.view(torch.uint8))
            kv.kv_offload(ctx, desc, shape.L, new_ids, hp + in_host * shape.page_bytes,
                          n_new * shape.page_bytes)
            mini = snapshot_pages(torch, slabs, new_ids, shape)
            expected[in_host * shape.page_bytes:(in_host + n_new) * shape.page_bytes] = ko.pack(
                mini, np.arange(n_new), threads=THREADS)
            in_host += n_new
            torch.cuda.synchronize()
            fl.give_back(ids)
            fl.give_back(new_ids)
        assert in_host == total_pages == 2875
        assert np.array_equal(hv, expected), "session host buffer != oracle"
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


def test_config4_concurrent_batch(kv, ctx, pool):
    """BASELINE.json:configs[3] as stated: 64 requests, 18,091 pages, 26.5 GiB in ONE batched call into per-request
    page-first buffers -- in device memory (kv_pack_batched) AND in pinned host memory (a single kv_offload_batched
    over all 64 requests) -- plus the reverse batched unpack (from the device buffers) and reload (from the pinned
    ones) into fresh pages.  EVERY request of all four transfers is compared with the oracle, streaming one request
    at a time so that host RAM holds one request's expectation only."""
    shape, slabs, desc = pool
    b = W.batch_case(0)
    R = len(b.lens)
    counts = np.diff(b.req_offsets)
    page = shape.page_bytes
    total = int(b.req_offsets[-1]) * page
    sizes = [int(c) * page for c in counts]
    big = torch.empty(total, dtype=torch.uint8, device="cuda")
    bufs = [big[int(b.req_offsets[r]) * page:int(b.req_offsets[r + 1]) * page] for r in range(R)]
    hp = kv.kv_host_alloc(total)  # 26.5 GiB pinned: the 64 per-request host buffers
    try:
        hps = [hp + int(b.req_offsets[r]) * page for r in range(R)]
        kv.host_view(hp, total)[::4096] = 0xA5  # touch every page; nothing of the result is there yet
        # third page set for the reload: disjoint from the sources and from the unpack's destinations
        used = np.zeros(shape.P, dtype=bool)
        used[b.src_ids] = True
        used[b.dst_ids] = True
        dst2 = np.random.default_rng(44).permutation(np.flatnonzero(~used))[:len(b.dst_ids)].astype(np.int32)
        ntok = counts * shape.T
        before = page_checksums(torch, slabs, shape)
        kv.kv_pack_batched(ctx, desc, shape.L, b.src_ids, b.req_offsets, bufs, dst_bytes=sizes)
        assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 18091 * 96
        launches, memcpys = ctx.stat(kv.KV_STAT_LAUNCHES), ctx.stat(kv.KV_STAT_MEMCPYS)
        kv.kv_offload_batched(ctx, desc, shape.L, b.src_ids, b.req_offsets, hps, host_bytes=sizes)  # AUTO
        assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_STAGED
        assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == total
        kv.kv_unpack_batched(ctx, bufs, b.dst_ids, b.req_offsets, ntok, desc, shape.L, shape.T, shape.T)
        kv.kv_reload_batched(ctx, hps, dst2, b.req_offsets, ntok, desc, shape.L, shape.T, shape.T, host_bytes=sizes)
        torch.cuda.synchronize()
        after = page_checksums(torch, slabs, shape)
        assert_untouched(before, after, np.concatenate([b.dst_ids, dst2]), shape.P)
        hv = kv.host_view(hp, total)
        for r in range(R):
            lo, hi = int(b.req_offsets[r]), int(b.req_offsets[r + 1])
            ids = b.src_ids[lo:hi]
            mini = snapshot_pages(torch, slabs, ids, shape)
            want = ko.pack(mini, np.arange(len(ids)), threads=THREADS)
            assert np.array_equal(bufs[r].cpu().numpy(), want), f"request {r}: kv_pack_batched != oracle"
            assert np.array_equal(hv[lo * page:hi * page], want), f"request {r}: kv_offload_batched (pinned host) != oracle"
            exp = ko.HostPool([np.zeros_like(s) for s in mini.slabs], shape.L, shape.C, len(ids), shape.T,
                              shape.H, shape.D, shape.e, shape.row_bytes)
            ko.unpack(want, np.arange(len(ids)), exp, Ts=shape.T, n_tokens=len(ids) * shape.T, threads=THREADS)
            for name, dd in (("kv_unpack_batched", b.dst_ids[lo:hi]), ("kv_reload_batched (pinned host)", dst2[lo:hi])):
                got = snapshot_pages(torch, slabs, dd, shape)
                for x, y in zip(got.slabs, exp.slabs):
                    assert np.array_equal(x, y), f"request {r}: {name} != oracle"
            del mini, want, exp, got
        # the DIRECT mode of the same batched call on four of the requests (92 % of the link: 26.5 GiB would take 0.5 s
        # more; the mode must not change a byte)
        sel = [0, 16, 32, 48]
        off = np.concatenate([[0], np.cumsum(counts[sel])]).astype(np.int64)
        ids = np.concatenate([b.src_ids[b.req_offsets[r]:b.req_offsets[r + 1]] for r in sel]).astype(np.int32)
        for r in sel:
            hv[int(b.req_offsets[r]) * page:int(b.req_offsets[r + 1]) * page] = 0
        kv.kv_offload_batched(ctx, desc, shape.L, ids, off, [hps[r] for r in sel], host_bytes=[sizes[r] for r in sel],
                              mode=kv.KV_HOST_DIRECT)
        torch.cuda.synchronize()
        for r in sel:
            assert np.array_equal(hv[int(b.req_offsets[r]) * page:int(b.req_offsets[r + 1]) * page], bufs[r].cpu().numpy()), \
                f"offload_batched DIRECT req {r}"
    finally:
        torch.cuda.synchronize()
        kv.kv_host_free(hp)


@pytest.mark.parametrize("ragged", [False, True])
def test_config5_cross_role_repage(kv, ctx, pool, ragged):
    """BASELINE.json:configs[4]: LLM pool (page 16) -> diffusion-role pool (page 64), 32 requests of
    2,048 tokens (and the ragged variant, SURVEY.md 8(c) reading 9).  The two 48 GiB pools are the
    lower and upper halves of the 96 GiB allocation."""
    shape, slabs, desc = pool
    c5 = W.crossrole_case(0, ragged=ragged)
    s_src, s_dst = c5.src_shape, c5.dst_shape
    half = s_src.P * s_src.row_bytes
    assert half == s_dst.P * s_dst.row_bytes == 512 << 20
    src_slabs = [s[:half] for s in slabs]
    dst_slabs = [s[half:] for s in slabs]
    d_src = kv.PoolDesc(src_slabs, s_src.L, s_src.C, s_src.P, s_src.T, s_src.H, s_src.D, s_src.e)
    d_dst = kv.PoolDesc(dst_slabs, s_dst.L, s_dst.C, s_dst.P, s_dst.T, s_dst.H, s_dst.D, s_dst.e)
    R = len(c5.n_tokens)
    ns = np.diff(c5.src_offsets)
    big = torch.empty(int(c5.src_offsets[-1]) * s_src.page_bytes, dtype=torch.uint8, device="cuda")
    bufs = [big[int(c5.src_offsets[r]) * s_src.page_bytes:int(c5.src_offsets[r + 1]) * s_src.page_bytes] for r in range(R)]
    kv.kv_pack_batched(ctx, d_src, s_src.L, c5.src_ids, c5.src_offsets, bufs)
    before = page_checksums(torch, dst_slabs, s_dst)
    kv.kv_unpack_batched(ctx, bufs, c5.dst_ids, c5.dst_offsets, c5.n_tokens, d_dst, s_dst.L, 16, 64)
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384
    torch.cuda.synchronize()
    after = page_checksums(torch, dst_slabs, s_dst)
    assert_untouched(before, after, c5.dst_ids, s_dst.P)
    for r in range(R):
        ids = c5.src_ids[c5.src_offsets[r]:c5.src_offsets[r + 1]]
        mini = snapshot_pages(torch, src_slabs, ids, s_src)
        want = ko.pack(mini, np.arange(len(ids)), threads=THREADS)
        assert np.array_equal(bufs[r].cpu().numpy(), want), f"request {r}: pack != oracle"
        dids = c5.dst_ids[c5.dst_offsets[r]:c5.dst_offsets[r + 1]]
        got = snapshot_pages(torch, dst_slabs, dids, s_dst)
        exp = ko.HostPool([np.full_like(s, 0x5A) for s in got.slabs], s_dst.L, s_dst.C, len(dids), 64,
                          s_dst.H, s_dst.D, s_dst.e, s_dst.row_bytes)
        ko.unpack(want, np.arange(len(dids)), exp, Ts=16, n_tokens=int(c5.n_tokens[r]), threads=THREADS)
        for x, y in zip(got.slabs, exp.slabs):
            assert np.array_equal(x, y), f"request {r}: re-paged pages != oracle"
    # fused pool -> pool re-paging (kv_repage_batched) into OTHER free
    # destination pages: one launch, no transfer buffer, same bytes as the oracle's O-repage
    free = np.setdiff1d(np.arange(s_dst.P, dtype=np.int32), c5.dst_ids)
    dids2 = np.random.default_rng(5).permutation(free)[:len(c5.dst_ids)].astype(np.int32)
    before = page_checksums(torch, dst_slabs, s_dst)
    launches = ctx.stat(kv.KV_STAT_LAUNCHES)
    kv.kv_repage_batched(ctx, d_src, c5.src_ids, c5.src_offsets, d_dst, dids2, c5.dst_offsets, c5.n_tokens, s_dst.L)
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == launches + 1 and ctx.stat(kv.KV_STAT_LAST_GRID) == 32 * 32 * 4 * 96
    torch.cuda.synchronize()
    assert_untouched(before, page_checksums(torch, dst_slabs, s_dst), dids2, s_dst.P)
    for r in range(0, R, 5):
        ids = c5.src_ids[c5.src_offsets[r]:c5.src_offsets[r + 1]]
        mini = snapshot_pages(torch, src_slabs, ids, s_src)
        dd = dids2[c5.dst_offsets[r]:c5.dst_offsets[r + 1]]
        got = snapshot_pages(torch, dst_slabs, dd, s_dst)
        exp = ko.HostPool([np.full_like(s, 0x5A) for s in got.slabs], s_dst.L, s_dst.C, len(dd), 64,
                          s_dst.H, s_dst.D, s_dst.e, s_dst.row_bytes)
        ko.repage(mini, np.arange(len(ids)), exp, np.arange(len(dd)), n_tokens=int(c5.n_tokens[r]), threads=THREADS)
        for x, y in zip(got.slabs, exp.slabs):
            assert np.array_equal(x, y), f"request {r}: fused re-page != oracle"
    # and it equals what pack + unpack produced, for ALL requests (device-side compare)
    a = torch.as_tensor(c5.dst_ids.astype(np.int64), device="cuda")
    b2 = torch.as_tensor(dids2.astype(np.int64), device="cuda")
    for s in dst_slabs[::5]:
        v = s.view(s_dst.P, s_dst.row_bytes)
        assert torch.equal(v.index_select(0, a), v.index_select(0, b2))


def test_cow_tail_pages_of_64_sessions(kv, ctx, pool):
    """PAPER.md:L238 at the Qwen3-Omni shape: 64 sessions each extend a retained partial tail page
    (copy n_old tokens into a fresh page, append n_app new tokens) in ONE launch."""
    shape, slabs, desc = pool
    rng = np.random.default_rng(64)
    S = 64
    perm = rng.permutation(shape.P).astype(np.int32)
    old, new = perm[:S], perm[S:2 * S]
    n_old = rng.integers(0, shape.T, size=S)
    n_app = np.array([rng.integers(0, shape.T - o + 1) for o in n_old])
    apps_h = [rng.integers(0, 256, size=shape.L * shape.C * int(a) * shape.H * shape.D * shape.e, dtype=np.uint8) for a in n_app]
    apps = [torch.from_numpy(a).cuda() if a.size else None for a in apps_h]
    touched = np.concatenate([old, new])
    mini = snapshot_pages(torch, slabs, touched, shape)
    before = page_checksums(torch, slabs, shape)
    kv.kv_cow_append_batched(ctx, desc, shape.L, old, new, n_old, n_app, apps, flags=kv.KV_FLAG_VALIDATE)
    torch.cuda.synchronize()
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT  # AUTO: one ragged piece per single-warp CTA
    assert_untouched(before, page_checksums(torch, slabs, shape), new, shape.P)
    ko.cow_append_batched(mini, np.arange(S), np.arange(S, 2 * S), n_old, n_app, apps_h)
    got = snapshot_pages(torch, slabs, touched, shape)
    for x, y in zip(got.slabs, mini.slabs):
        assert np.array_equal(x, y), "batched CoW append != oracle"


@pytest.mark.parametrize("n", [1, 2, 16, 64, 683, 8192])
def test_transfer_size_sweep_points(kv, ctx, pool, n):
    """BASELINE.json:configs[4] sweep 1 MiB - 8 GiB (layer_count = 32 => 1 MiB pages; 683 is the
    48-layer cross-check point, ~1 GiB).  Sampled buffer pages vs the oracle + full torch gather."""
    shape, slabs, desc = pool
    L = 48 if n == 683 else 32
    rng = np.random.default_rng(n)
    ids = rng.choice(shape.P, n, replace=False).astype(np.int32)
    page = L * shape.C * shape.row_bytes
    buf = torch.zeros(n * page, dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, desc, L, ids, buf)
    torch.cuda.synchronize()
    sample = np.unique(np.concatenate([[0, n - 1], rng.integers(0, n, size=min(n, 24))]))
    mini = snapshot_pages(torch, slabs, ids[sample], shape, layer_count=L)
    want = ko.pack(mini, np.arange(len(sample)), layer_count=L, threads=THREADS).reshape(len(sample), page)
    got = buf.view(n, page)[torch.as_tensor(sample, device="cuda")].cpu().numpy()
    assert np.array_equal(got, want)
    # property at any size: buffer[p][lc] is slab lc's row ids[p] (torch gather, all pages)
    idx = torch.as_tensor(ids.astype(np.int64), device="cuda")
    v = buf.view(n, L * shape.C, shape.row_bytes)
    for lc in range(0, L * shape.C, 5):
        assert torch.equal(v[:, lc], slabs[lc].view(shape.P, shape.row_bytes).index_select(0, idx))
    del buf
