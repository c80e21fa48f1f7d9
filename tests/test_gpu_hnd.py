"""GPU parity for HND pools (in-page order [head][token][dim]; "compute-oriented
layouts, including NHD block stacks").  The transfer buffer stays NHD, so
every transfer to or from an HND pool transposes [token] and [head].  Byte for byte against the
CPU oracle on the same seeded inputs, all three kernels."""
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


@pytest.fixture(params=[1, 0], ids=["tensormaps", "lanes"])
def ctx(kv, request):
    """Every case runs twice: HND sides moved by cp.async.bulk.tensor through per-slab tensor maps
    (the default), and by the lane paths (cp.async row gather / 16-byte stores) alone."""
    c = kv.Ctx(0, staging_bytes=8 << 20)
    c.set_option(kv.KV_OPT_TENSOR_MAPS, request.param)
    c.tensor_maps = request.param
    yield c
    torch.cuda.synchronize()
    c.close()


KERNELS = {"bulk": 1, "vec": 2, "elem": 3, "shot": 4}
HND = ko.HND

SHAPES = [  # L, C, P, T, H, D, e, pad, n
    (4, 2, 256, 16, 2, 64, 2, 0, 37),     # Tiny (BASELINE.json:configs[0]) with HND pools
    (3, 2, 90, 16, 4, 128, 2, 0, 41),     # Qwen3-Omni row: 16 KiB, 256-byte head_dim rows
    (2, 2, 40, 64, 4, 128, 2, 0, 9),      # 64 KiB rows: 4 items per row
    (2, 2, 50, 16, 8, 128, 1, 256, 13),   # fp8 elements, padded stride
    (2, 1, 30, 5, 3, 24, 2, 0, 11),       # 48-byte rows, odd sizes, single latent pool
    (2, 2, 30, 8, 3, 5, 1, 0, 7),         # 5-byte rows: elem path with unit 1
    (1, 2, 20, 4, 2, 1024, 4, 0, 5),      # 4 KiB head_dim rows: one row per stage
    (1, 1, 12, 2, 2, 2560, 4, 0, 5),      # 10 KiB rows do not fit a stage: vec takes over from bulk
]


def want_kernel(kernel, H, D, e):
    if (D * e) % 16:
        return KERNELS["elem"]
    if kernel == "bulk" and D * e > 4096:  # a head_dim row must fit one (4 KiB) stage of the transposing ring
        return KERNELS["vec"]
    if kernel == "shot" and D * e > 16384:  # ... or the one 16 KiB stage of a shot CTA
        return KERNELS["vec"]
    return KERNELS[kernel]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", SHAPES)
def test_pack_unpack_hnd(kv, ctx, kernel, shape):
    L, C, P, T, H, D, e, pad, n = shape
    rng = np.random.default_rng(abs(hash(shape)) % 2**31)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    A = host_pool(rng, L, C, P, T, H, D, e, pad, order=HND)
    B = host_pool(rng, L, C, P, T, H, D, e, pad, order=HND)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    src = rng.choice(P, n, replace=False).astype(np.int32)
    dst = rng.permutation(P)[:n].astype(np.int32)
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, L, src, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == want_kernel(kernel, H, D, e)
    want = ko.pack(A, src)
    assert np.array_equal(buf.cpu().numpy(), want)
    assert_pool_equal(tA, A)
    kv.kv_unpack(ctx, buf, dst, dB, L, T, T, n * T, flags=kv.KV_FLAG_VALIDATE)
    ko.unpack(want, dst, B, Ts=T, n_tokens=n * T)
    assert_pool_equal(tB, B)
    # HND pool -> buffer -> NHD pool of the same shape: the round trip converts the layout
    N = host_pool(rng, L, C, P, T, H, D, e, pad, order=ko.NHD)
    tN, dN = to_device(N, kv, torch)
    kv.kv_unpack(ctx, buf, dst, dN, L, T, T, n * T)
    ko.unpack(want, dst, N, Ts=T, n_tokens=n * T)
    assert_pool_equal(tN, N)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("Ts,Td,ntok", [(16, 64, 2048 - 37), (64, 16, 1000), (16, 24, 500), (3, 5, 77),
                                        (16, 64, 1), (16, 16, 16 * 7 - 5)])
def test_unpack_repaging_into_hnd(kv, ctx, kernel, layout, Ts, Td, ntok):
    L, C, H, D, e = 3, 2, 4, 128, 2
    rng = np.random.default_rng(Ts * 131 + Td * 7 + ntok + layout)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    B = host_pool(rng, L, C, n_dst + 5, Td, H, D, e, order=HND)
    tB, dB = to_device(B, kv, torch)
    src = rng.integers(0, 256, size=n_src * L * C * Ts * H * D * e, dtype=np.uint8)
    dids = rng.permutation(n_dst + 5)[:n_dst].astype(np.int32)
    kv.kv_unpack(ctx, torch.from_numpy(src).cuda(), dids, dB, L, Ts, Td, ntok, layout=layout)
    ko.unpack(src, dids, B, Ts=Ts, n_tokens=ntok, layout=layout)
    assert_pool_equal(tB, B)  # incl. zero-padded tail slots of every head's run, untouched pages


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("orders", [(0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("Ts,Td,ntok,pad", [(16, 64, 2048 - 37, 0), (64, 16, 1000, 0), (16, 24, 500, 256),
                                            (16, 16, 16 * 9, 0), (16, 16, 16 * 9 - 3, 0), (8, 64, 1, 0)])
def test_repage_across_orders(kv, ctx, kernel, orders, Ts, Td, ntok, pad):
    L, C, H, D, e = 3, 2, 4, 128, 2
    rng = np.random.default_rng(Ts * 977 + Td * 31 + ntok + orders[0] * 2 + orders[1])
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    n_src, n_dst = -(-ntok // Ts), -(-ntok // Td)
    A = host_pool(rng, L, C, n_src + 9, Ts, H, D, e, pad, order=orders[0])
    B = host_pool(rng, L, C, n_dst + 7, Td, H, D, e, pad, order=orders[1])
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    sids = rng.permutation(n_src + 9)[:n_src].astype(np.int32)
    dids = rng.permutation(n_dst + 7)[:n_dst].astype(np.int32)
    kv.kv_repage(ctx, dA, sids, dB, dids, L, ntok, flags=kv.KV_FLAG_VALIDATE)
    ko.repage(A, sids, B, dids, n_tokens=ntok)
    assert_pool_equal(tB, B)
    assert_pool_equal(tA, A)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", [(4, 2, 64, 16, 2, 64, 2, 0), (3, 2, 40, 16, 4, 128, 2, 0),
                                   (2, 2, 24, 64, 4, 128, 2, 256), (2, 1, 30, 5, 3, 24, 2, 0)])
def test_cow_append_hnd(kv, ctx, kernel, shape):
    L, C, P, T, H, D, e, pad = shape
    rng = np.random.default_rng(abs(hash(shape)) % 2**31 + 1)
    ctx.set_option(kv.KV_OPT_KERNEL, KERNELS[kernel])
    A = host_pool(rng, L, C, P, T, H, D, e, pad, order=HND)
    tA, dA = to_device(A, kv, torch)
    S = 9
    perm = rng.permutation(P).astype(np.int32)
    old, new = perm[:S], perm[S:2 * S]
    n_old = rng.integers(0, T + 1, size=S)
    n_app = np.array([rng.integers(0, T - o + 1) for o in n_old])
    n_old[0], n_app[0] = 0, T
    n_old[1], n_app[1] = T, 0
    n_old[2], n_app[2] = 0, 0
    n_old[3], n_app[3] = T - 1, 1
    apps = [rng.integers(0, 256, size=L * C * int(a) * H * D * e, dtype=np.uint8) for a in n_app]
    dev_apps = [torch.from_numpy(a).cuda() if a.size else None for a in apps]
    kv.kv_cow_append_batched(ctx, dA, L, old, new, n_old, n_app, dev_apps, flags=kv.KV_FLAG_VALIDATE)
    ko.cow_append_batched(A, old, new, n_old, n_app, apps)
    assert_pool_equal(tA, A)


@pytest.mark.parametrize("mode", ["direct", "staged"])
def test_host_tier_batched_hnd(kv, ctx, mode):
    """Offload / reload of HND pools, batched, both host modes: the host buffer is the same NHD
    page-first bytes whatever the pool order and the mode."""
    L, C, P, T, H, D, e = 4, 2, 300, 16, 4, 128, 2
    rng = np.random.default_rng(71)
    m = {"direct": kv.KV_HOST_DIRECT, "staged": kv.KV_HOST_STAGED}[mode]
    A = host_pool(rng, L, C, P, T, H, D, e, order=HND)
    B = host_pool(rng, L, C, P, T, H, D, e, order=HND)
    tA, dA = to_device(A, kv, torch)
    tB, dB = to_device(B, kv, torch)
    counts = np.array([40, 0, 1, 77, 13])
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    src = rng.choice(P, off[-1], replace=False).astype(np.int32)
    dst = rng.permutation(P)[:off[-1]].astype(np.int32)
    page = dA.page_bytes()
    hps = [kv.kv_host_alloc(max(int(c) * page, 16)) for c in counts]
    try:
        kv.kv_offload_batched(ctx, dA, L, src, off, hps, [int(c) * page for c in counts], mode=m)
        torch.cuda.synchronize()
        want = ko.pack_batched(A, src, off)
        for r, c in enumerate(counts):
            assert np.array_equal(kv.host_view(hps[r], int(c) * page), want[r]), f"request {r}"
        kv.kv_reload_batched(ctx, hps, dst, off, counts * T, dB, L, T, T,
                             host_bytes=[int(c) * page for c in counts], mode=m)
        torch.cuda.synchronize()
        ko.unpack_batched(want, dst, off, counts * T, B, Ts=T)
        assert_pool_equal(tB, B)
    finally:
        for hp in hps:
            kv.kv_host_free(hp)


def test_hnd_degenerate_orders_are_plain_copies(kv, ctx):
    """One head, or one token per page: [token][head] and [head][token] are the same bytes, and
    the library takes the contiguous path (segment = whole row)."""
    rng = np.random.default_rng(73)
    for (T, H) in [(16, 1), (1, 4)]:
        L, C, P, D, e, n = 2, 2, 40, 128, 2, 9
        A = host_pool(rng, L, C, P, T, H, D, e, order=HND)
        tA, dA = to_device(A, kv, torch)
        ids = rng.choice(P, n, replace=False).astype(np.int32)
        buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
        kv.kv_pack(ctx, dA, L, ids, buf)
        assert np.array_equal(buf.cpu().numpy(), ko.pack(A, ids))


@pytest.mark.parametrize("ctx", [1], indirect=True, ids=["tensormaps"])  # a test ABOUT tensor maps: no "lanes" case is generated
def test_auto_with_tensor_maps_is_one_bulk_kernel(kv, ctx):
    """AUTO with tensor maps (the default): every direction of an HND transfer is one async-copy kernel, whole-token
    boxes moved by cp.async.bulk.tensor; the second call on the same pool reuses the cached maps."""
    L, C, P, T, H, D, e, n = 3, 2, 64, 16, 4, 128, 2, 20
    rng = np.random.default_rng(83)
    A = host_pool(rng, L, C, P, T, H, D, e, order=HND)
    N = host_pool(rng, L, C, P, T, H, D, e, order=ko.NHD)
    tA, dA = to_device(A, kv, torch)
    tN, dN = to_device(N, kv, torch)
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        kv.kv_pack(ctx, dA, L, ids, buf)
        assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
        assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
        assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 8192  # 120 rows of 16 KiB split once to cover the chip
    want = ko.pack(A, ids)
    assert np.array_equal(buf.cpu().numpy(), want)
    kv.kv_unpack(ctx, buf, ids[::-1].copy(), dA, L, T, T, n * T)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"] and ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
    ko.unpack(want, ids[::-1].copy(), A, Ts=T, n_tokens=n * T)
    assert_pool_equal(tA, A)
    kv.kv_repage(ctx, dA, ids, dN, ids, L, n * T)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"] and ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
    ko.repage(A, ids, N, ids, n_tokens=n * T)
    assert_pool_equal(tN, N)
    kv.kv_repage(ctx, dN, ids, dA, ids, L, n * T)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"] and ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
    ko.repage(N, ids, A, ids, n_tokens=n * T)
    assert_pool_equal(tA, A)
    kv.kv_pack(ctx, dN, L, ids, buf)  # NHD pool: nothing to transpose, no maps
    assert ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 0


def test_auto_kernel_choice_per_direction(kv, ctx):
    """AUTO without tensor maps: with segments of 4 KiB or more every direction takes
    kv_move_shot (strided source: cp.async row gathers into the CTA's stage; strided destination: 16-byte stores from
    it); a pool whose whole rows are shorter keeps the earlier choices -- strided source only -> bulk ring, strided
    destination -> vec."""
    L, C, P, T, H, D, e, n = 3, 2, 64, 16, 4, 128, 2, 20
    rng = np.random.default_rng(79)
    ctx.set_option(kv.KV_OPT_TENSOR_MAPS, 0)
    A = host_pool(rng, L, C, P, T, H, D, e, order=HND)
    N = host_pool(rng, L, C, P, T, H, D, e, order=ko.NHD)
    tA, dA = to_device(A, kv, torch)
    tN, dN = to_device(N, kv, torch)
    ids = rng.choice(P, n, replace=False).astype(np.int32)
    buf = torch.zeros(n * dA.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dA, L, ids, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 8192  # 120 rows of 16 KiB split once to cover the chip
    want = ko.pack(A, ids)
    assert np.array_equal(buf.cpu().numpy(), want)
    kv.kv_unpack(ctx, buf, ids[::-1].copy(), dA, L, T, T, n * T)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
    ko.unpack(want, ids[::-1].copy(), A, Ts=T, n_tokens=n * T)
    assert_pool_equal(tA, A)
    kv.kv_repage(ctx, dA, ids, dN, ids, L, n * T)  # HND -> NHD pool: strided source only
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
    ko.repage(A, ids, N, ids, n_tokens=n * T)
    assert_pool_equal(tN, N)
    kv.kv_repage(ctx, dN, ids, dA, ids, L, n * T)  # NHD -> HND pool: strided destination
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
    ko.repage(N, ids, A, ids, n_tokens=n * T)
    assert_pool_equal(tA, A)
    kv.kv_pack(ctx, dN, L, ids, buf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["shot"]
    # short rows (4 tokens x 2 heads x 128 B = 1 KiB per row): the earlier choices
    S = host_pool(rng, L, C, P, 4, 2, 64, 2, order=HND)
    tS, dS = to_device(S, kv, torch)
    sbuf = torch.zeros(n * dS.page_bytes(), dtype=torch.uint8, device="cuda")
    kv.kv_pack(ctx, dS, L, ids, sbuf)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["bulk"]
    wants = ko.pack(S, ids)
    assert np.array_equal(sbuf.cpu().numpy(), wants)
    kv.kv_unpack(ctx, sbuf, ids[::-1].copy(), dS, L, 4, 4, n * 4)
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == KERNELS["vec"]
    ko.unpack(wants, ids[::-1].copy(), S, Ts=4, n_tokens=n * 4)
    assert_pool_equal(tS, S)


@pytest.mark.parametrize("variant", ["plain", "plain_capped", "general_l2hint", "plain_batched_3", "general_ragged"])
@pytest.mark.parametrize("shape", [SHAPES[0], SHAPES[1], SHAPES[2], SHAPES[3]])
def test_hnd_plain_kernel_and_general_kernel_agree_with_the_oracle(kv, variant, shape):
    """HND pools: the plain case (equal page sizes, page-first, nothing to zero-fill, host ids, whole boxes by tensor
    copies) takes the short kernel kv_move_shot_plain<.., kTrans> -- one tensor copy on the pool side, one bulk copy on
    the buffer side, per single-warp CTA; an L2 hint or a ragged tail the general kernel.  Same bytes either way."""
    L, C, P, T, H, D, e, pad, n = shape
    rng = np.random.default_rng(3 + abs(hash((shape, variant))) % 2**31)
    ctx = kv.Ctx(0)
    try:
        if variant == "general_l2hint":
            ctx.set_option(kv.KV_OPT_L2_HINT, 1)
        if variant.endswith("capped"):
            ctx.set_option(kv.KV_OPT_MAX_CTAS, 7)
        A = host_pool(rng, L, C, P, T, H, D, e, pad, order=HND)
        B = host_pool(rng, L, C, P, T, H, D, e, pad, order=HND)
        tA, dA = to_device(A, kv, torch)
        tB, dB = to_device(B, kv, torch)
        src = rng.choice(P, n, replace=False).astype(np.int32)
        dst = rng.permutation(P)[:n].astype(np.int32)
        page = dA.page_bytes()
        buf = torch.full((n * page + 256,), 0xCD, dtype=torch.uint8, device="cuda")
        want_plain = 0 if variant.startswith("general") else 1
        ntok_all = n * T - (5 if variant == "general_ragged" and T > 5 else (1 if variant == "general_ragged" else 0))
        if "batched" in variant:
            cut = [0, n // 4, n // 4, n]  # an empty request in the middle
            off = np.asarray(cut, dtype=np.int64)
            bufs = [buf[cut[r] * page:cut[r + 1] * page] for r in range(3)]
            kv.kv_pack_batched(ctx, dA, L, src, off, bufs)
        else:
            kv.kv_pack(ctx, dA, L, src, buf, dst_bytes=n * page)
        assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT and ctx.stat(kv.KV_STAT_LAST_TENSOR_MAPS) == 1
        assert ctx.stat(kv.KV_STAT_LAST_PLAIN) == (0 if variant == "general_l2hint" else 1)  # a pack has no tail to pad
        want = ko.pack(A, src)
        got = buf.cpu().numpy()
        assert np.array_equal(got[:want.size], want)
        assert np.all(got[want.size:] == 0xCD), "wrote past the end of the buffer"
        if "batched" in variant:
            ntok = np.asarray([(cut[r + 1] - cut[r]) * T for r in range(3)], dtype=np.uint64)
            kv.kv_unpack_batched(ctx, bufs, dst, off, ntok, dB, L, T, T)
        else:
            kv.kv_unpack(ctx, buf, dst, dB, L, T, T, ntok_all, src_bytes=n * page)
        assert ctx.stat(kv.KV_STAT_LAST_PLAIN) == want_plain
        ko.unpack(want, dst, B, Ts=T, n_tokens=ntok_all)
        assert_pool_equal(tB, B)
        assert_pool_equal(tA, A)
    finally:
        torch.cuda.synchronize()
        ctx.close()
