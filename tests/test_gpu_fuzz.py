"""Seeded random cases of every transfer against the CPU oracle, byte for byte: random shapes, page
sizes on both sides, in-page orders, buffer layouts, strides with padding, ragged token counts, CSR
batches with empty requests, every kernel choice (AUTO / bulk ring / vec / elem / shot), tensor maps on and off,
PDL / dynamic claiming / inline tables on and off, stage sizes and warp counts of the bulk ring.
The directed cases live in test_gpu_parity / test_gpu_next / test_gpu_hnd; this file is the net under
them: each seed draws one configuration and runs pack -> unpack (re-paged) -> fused re-page ->
copy-on-write append -> host-tier offload / re-paging reload (random mode and pipeline chunk size) on it."""
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


def draw(rng):
    e = int(rng.choice([1, 2, 2, 2, 4, 8]))
    D = int(rng.choice([8, 16, 24, 64, 128, 128, 256, 40]))
    H = int(rng.choice([1, 2, 3, 4, 4, 8]))
    Ts = int(rng.choice([1, 2, 4, 8, 16, 16, 16, 32, 64, 5, 12]))
    Td = int(rng.choice([Ts, Ts, 16, 64, 4, 8, 32, 7, 24]))
    L = int(rng.integers(1, 5))
    C = int(rng.choice([1, 2, 2]))
    pad_unit = int(rng.choice([0, 0, e, 16, 256]))
    return dict(e=e, D=D, H=H, Ts=Ts, Td=Td, L=L, C=C, pad=pad_unit,
                order_s=int(rng.integers(0, 2)), order_d=int(rng.integers(0, 2)),
                layout=int(rng.integers(0, 2)), kernel=int(rng.choice([0, 0, 1, 2, 3, 4, 4])),
                tensor_maps=int(rng.integers(0, 2)), R=int(rng.integers(1, 5)),
                pdl=int(rng.integers(0, 2)), dynamic=int(rng.integers(0, 2)), inline=int(rng.integers(0, 2)),
                stage=int(rng.choice([16384, 16384, 4096, 1024, 8192])), warps=int(rng.choice([2, 2, 1, 4])),
                max_ctas=int(rng.choice([0, 0, 1, 3])))  # 1 or 3 CTAs: many segments per warp -> guided claiming


@pytest.mark.parametrize("seed", range(300))
def test_random_configuration(kv, seed):
    rng = np.random.default_rng(10_000 + seed)
    c = draw(rng)
    e, D, H, Ts, Td, L, C = c["e"], c["D"], c["H"], c["Ts"], c["Td"], c["L"], c["C"]
    ctx = kv.Ctx(0, staging_bytes=4 << 20)
    try:
        ctx.set_option(kv.KV_OPT_KERNEL, c["kernel"])
        ctx.set_option(kv.KV_OPT_TENSOR_MAPS, c["tensor_maps"])
        ctx.set_option(kv.KV_OPT_PDL, c["pdl"])
        ctx.set_option(kv.KV_OPT_DYNAMIC, c["dynamic"])
        ctx.set_option(kv.KV_OPT_INLINE_TABLES, c["inline"])
        if c["stage"] != 16384 or c["warps"] != 2:  # setting them pins the ring geometry; the defaults leave it automatic
            ctx.set_option(kv.KV_OPT_STAGE_BYTES, c["stage"])
            ctx.set_option(kv.KV_OPT_WARPS, c["warps"])
        ctx.set_option(kv.KV_OPT_MAX_CTAS, c["max_ctas"])
        # requests: token counts, some empty, ragged against both page sizes
        ntok = [int(rng.choice([0, 1, Ts, Td, Ts * 3 + 1, int(rng.integers(1, 400))])) for _ in range(c["R"])]
        ns = [-(-t // Ts) for t in ntok]
        nd = [-(-t // Td) for t in ntok]
        Ps, Pd = sum(ns) + 5, sum(nd) + 6
        A = host_pool(rng, L, C, Ps, Ts, H, D, e, c["pad"], order=c["order_s"])
        B = host_pool(rng, L, C, Pd, Td, H, D, e, c["pad"], order=c["order_d"])
        B2 = ko.HostPool([s.copy() for s in B.slabs], L, C, Pd, Td, H, D, e, B.page_stride_bytes, c["order_d"])
        pristine = [s.copy() for s in B.slabs]  # the destination pool BEFORE any transfer (step 5 starts from it)
        tA, dA = to_device(A, kv, torch)
        tB, dB = to_device(B, kv, torch)
        tB2, dB2 = to_device(B2, kv, torch)
        soff = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
        doff = np.concatenate([[0], np.cumsum(nd)]).astype(np.int64)
        sids = rng.permutation(Ps)[:soff[-1]].astype(np.int32)
        dids = rng.permutation(Pd)[:doff[-1]].astype(np.int32)
        page_s = L * C * Ts * H * D * e
        # 1. batched pack (whole source pages) into per-request buffers
        bufs = [torch.full((max(n * page_s, 16),), 0xAB, dtype=torch.uint8, device="cuda") for n in ns]
        kv.kv_pack_batched(ctx, dA, L, sids, soff, bufs, [n * page_s for n in ns], layout=c["layout"])
        want = ko.pack_batched(A, sids, soff, layout=c["layout"])
        for r, n in enumerate(ns):
            assert np.array_equal(bufs[r].cpu().numpy()[:n * page_s], want[r]), f"{c}: pack, request {r}"
        assert_pool_equal(tA, A)
        # 2. batched unpack with re-paging Ts -> Td and ragged tails
        kv.kv_unpack_batched(ctx, bufs, dids, doff, ntok, dB, L, Ts, Td, layout=c["layout"],
                             flags=kv.KV_FLAG_VALIDATE)
        ko.unpack_batched(want, dids, doff, ntok, B, Ts=Ts, layout=c["layout"])
        assert_pool_equal(tB, B)
        # 3. the same movement fused pool -> pool
        kv.kv_repage_batched(ctx, dA, sids, soff, dB2, dids, doff, ntok, L, flags=kv.KV_FLAG_VALIDATE)
        ko.repage_batched(A, sids, soff, B2, dids, doff, ntok)
        assert_pool_equal(tB2, B2)
        assert_pool_equal(tA, A)
        # 4. copy-on-write append on the destination pool
        S = int(rng.integers(1, 4))
        if Pd >= 2 * S:
            perm = rng.permutation(Pd).astype(np.int32)
            old, new = perm[:S], perm[S:2 * S]
            n_old = rng.integers(0, Td + 1, size=S)
            n_app = np.array([rng.integers(0, Td - o + 1) for o in n_old])
            apps = [rng.integers(0, 256, size=L * C * int(a) * H * D * e, dtype=np.uint8) for a in n_app]
            dev = [torch.from_numpy(a).cuda() if a.size else None for a in apps]
            kv.kv_cow_append_batched(ctx, dB, L, old, new, n_old, n_app, dev, flags=kv.KV_FLAG_VALIDATE)
            ko.cow_append_batched(B, old, new, n_old, n_app, apps)
            assert_pool_equal(tB, B)
        # 5. the host tier on the same requests: offload A's pages, reload them re-paged into a PRISTINE copy of the
        #    destination pool -- taken before steps 2-4, so none of the bytes the reload must deliver is there yet and a
        #    reload that writes nothing fails; random mode, random pipeline chunk size (multi-chunk, layer ranges,
        #    page ranges); a chunk smaller than one lcm(Ts, Td) unit is refused with KV_ERR_SIZE -> direct
        B3 = ko.HostPool([s_.copy() for s_ in pristine], L, C, Pd, Td, H, D, e, B.page_stride_bytes, c["order_d"])
        tB3, dB3 = to_device(B3, kv, torch)  # uploaded BEFORE the oracle touches B3
        if doff[-1]:
            assert not all(np.array_equal(a, b) for a, b in zip(pristine, B2.slabs)), "the transfer would be invisible"
        ko.unpack_batched(want, dids, doff, ntok, B3, Ts=Ts, layout=c["layout"])
        mode = int(rng.choice([kv.KV_HOST_DIRECT, kv.KV_HOST_STAGED, kv.KV_HOST_STAGED]))
        ctx.set_option(kv.KV_OPT_CHUNK_BYTES, int(rng.choice([0, 64 << 10, 256 << 10, 1 << 20])))
        hps = [kv.kv_host_alloc(max(n * page_s, 16)) for n in ns]
        try:
            def both(m):
                kv.kv_offload_batched(ctx, dA, L, sids, soff, hps, [n * page_s for n in ns], mode=m, layout=c["layout"])
                torch.cuda.synchronize()
                for r, n in enumerate(ns):
                    assert np.array_equal(kv.host_view(hps[r], max(n * page_s, 16))[:n * page_s], want[r]), f"{c}: offload {m}, request {r}"
                kv.kv_reload_batched(ctx, hps, dids, doff, ntok, dB3, L, Ts, Td, host_bytes=[n * page_s for n in ns],
                                     mode=m, layout=c["layout"])
                torch.cuda.synchronize()
            try:
                both(mode)
            except kv.KvError as ex:
                assert ex.status == kv.KV_ERR_SIZE and mode == kv.KV_HOST_STAGED, f"{c}: {ex}"
                both(kv.KV_HOST_DIRECT)
            assert_pool_equal(tB3, B3)
        finally:
            torch.cuda.synchronize()
            for hp in hps:
                kv.kv_host_free(hp)
        torch.cuda.synchronize()
    finally:
        torch.cuda.synchronize()
        ctx.close()


MEDIUM = [  # Ts, Td, H, order_s, order_d, layout, tokens: sizes at which AUTO's rules and the re-shaped ring engage
    (16, 16, 4, 0, 0, 0, 3000), (16, 16, 1, 0, 0, 0, 9000), (16, 16, 2, 0, 1, 0, 5000), (16, 64, 4, 0, 0, 0, 2048 * 3 - 37),
    (64, 16, 4, 0, 0, 1, 4000), (16, 24, 4, 0, 0, 0, 3100), (5, 7, 4, 0, 0, 0, 3001), (1, 1, 4, 0, 0, 0, 2500),
    (16, 16, 4, 1, 1, 0, 3000), (16, 64, 2, 1, 0, 0, 5000), (16, 16, 1, 0, 0, 1, 7000), (7, 5, 2, 0, 0, 0, 4100),
    (16, 16, 1, 0, 0, 0, 5000), (16, 16, 2, 1, 1, 0, 2400),  # < 40 MiB of narrow rows: the bulk ring, re-shaped
]


@pytest.mark.parametrize("Ts,Td,H,order_s,order_d,layout,ntok", MEDIUM)
def test_medium_sizes_with_default_options(kv, Ts, Td, H, order_s, order_d, layout, ntok):
    """Tens of MiB per call with nothing overridden: the sizes at which the automatic choices engage -- kv_move_shot
    (general form: gcd chunking, zero tails, tensor maps on HND pools) for segments of 4 KiB or more, the ring re-shaped
    for narrow rows with guided claiming for 2-4 KiB, kv_move_small for segments <= 1 KiB -- through pack -> re-paging
    unpack -> fused re-page, against the oracle."""
    L, C, D, e = 12, 2, 128, 2
    rng = np.random.default_rng(hash((Ts, Td, H, order_s, order_d, layout, ntok)) % 2**31)
    ctx = kv.Ctx(0)
    try:
        ns, nd = -(-ntok // Ts), -(-ntok // Td)
        A = host_pool(rng, L, C, ns + 7, Ts, H, D, e, order=order_s)
        B = host_pool(rng, L, C, nd + 9, Td, H, D, e, order=order_d)
        B2 = ko.HostPool([s.copy() for s in B.slabs], L, C, nd + 9, Td, H, D, e, B.page_stride_bytes, order_d)
        tA, dA = to_device(A, kv, torch)
        tB, dB = to_device(B, kv, torch)
        tB2, dB2 = to_device(B2, kv, torch)
        sids = rng.permutation(ns + 7)[:ns].astype(np.int32)
        dids = rng.permutation(nd + 9)[:nd].astype(np.int32)
        buf = torch.zeros(ns * dA.page_bytes(), dtype=torch.uint8, device="cuda")
        kv.kv_pack(ctx, dA, L, sids, buf, layout=layout)
        want = ko.pack(A, sids, layout=layout, threads=8)
        assert np.array_equal(buf.cpu().numpy(), want), "pack"
        kv.kv_unpack(ctx, buf, dids, dB, L, Ts, Td, ntok, layout=layout, flags=kv.KV_FLAG_VALIDATE)
        ko.unpack(want, dids, B, Ts=Ts, n_tokens=ntok, layout=layout, threads=8)
        assert_pool_equal(tB, B)
        kv.kv_repage(ctx, dA, sids, dB2, dids, L, ntok)
        ko.repage(A, sids, B2, dids, n_tokens=ntok, threads=8)
        assert_pool_equal(tB2, B2)
        assert_pool_equal(tA, A)
    finally:
        torch.cuda.synchronize()
        ctx.close()
