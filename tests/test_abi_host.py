"""CPU-only checks of the C ABI: the library loads, exports every symbol include/kvtier.h
declares, and its host logic (validation order, planning) is right -- through a planning-only
context (device = -1) that touches no CUDA API.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

from paper_2606_31093_b200 import kvtier as kv  # noqa: E402
from paper_2606_31093_b200 import workloads as W  # noqa: E402


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "kvtier.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(kv_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(kv.LIB_PATH)
    names = declared_symbols()
    assert len(names) >= 20 and "kv_pack" in names and "kv_reload_batched" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/kvtier.h but not exported"


def test_binding_has_the_same_names():
    skip = {"kv_ctx_set_option", "kv_ctx_get_stat", "kv_last_cuda_error", "kv_device_status"}  # Ctx methods
    for n in declared_symbols():
        if n not in skip:
            assert hasattr(kv, n), f"binding lacks {n}"


def test_version_and_strerror():
    assert kv.kv_version() == 0x00010000
    seen = set()
    for code in range(0, -11, -1):
        msg = kv.kv_strerror(code)
        assert msg and msg not in seen
        seen.add(msg)
    assert "unknown" in kv.kv_strerror(-99)


def fake_pool(shape, stride=None, base0=0x7000_0000_0000, align=0):
    slab = shape.P * (stride or shape.row_bytes)
    bases = [base0 + align + i * ((slab + 4095) // 4096 * 4096) for i in range(shape.L * shape.C)]
    return kv.PoolDesc(bases, shape.L, shape.C, shape.P, shape.T, shape.H, shape.D, shape.e, stride)


BUF = 0x7100_0000_0000


def status_of(fn):
    with pytest.raises(kv.KvError) as ei:
        fn()
    return ei.value.status


@pytest.fixture()
def ctx():
    c = kv.Ctx(-1)
    yield c
    c.close()


def test_planning_ctx_never_launches(ctx):
    s = W.QWEN3_OMNI
    d = fake_pool(s)
    case = W.prefix_case(0)
    n = len(case.src_ids)
    assert n == 512
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, case.src_ids, BUF, dst_bytes=n * s.page_bytes)) == kv.KV_ERR_NO_DEVICE
    # 512 pages x 48 layers x 2 = 49,152 segments of one 16 KiB row
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 49152
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 768 << 20
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT  # AUTO: one 16 KiB segment per single-warp CTA
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == 0 and ctx.stat(kv.KV_STAT_MEMCPYS) == 0


def test_plan_repage_16_to_64(ctx):
    """BASELINE.json:configs[4]: 2,048 tokens -> 32 pages of 64; segment = min(Ts,Td) tokens."""
    c5 = W.crossrole_case(0)
    d = fake_pool(c5.dst_shape)
    s = c5.dst_shape
    srcs = [BUF + r * (1 << 32) for r in range(32)]
    assert status_of(lambda: kv.kv_unpack_batched(ctx, srcs, c5.dst_ids, c5.dst_offsets, c5.n_tokens, d, s.L, 16, 64)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 32 * 32 * 4 * 96
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 32 * 32 * s.page_bytes == 6 << 30
    # neither page size divides the other: segment = gcd(16, 24) = 8 tokens = 8 KiB
    d24 = fake_pool(s.with_(T=24))
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, np.arange(2), d24, s.L, 16, 24, 48, src_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 8 * 1024
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 2 * 3 * 96


def test_plan_splits_rows_longer_than_a_stage(ctx):
    s = W.QWEN3_OMNI.with_(T=64)
    d = fake_pool(s)
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [1, 2, 3], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384  # 64 KiB row cut into 4 stage-sized pieces
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 3 * 96 * 4
    ctx.set_option(kv.KV_OPT_STAGE_BYTES, 32768)
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [1, 2, 3], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 3 * 96 * 2


def test_misalignment_selects_elem_kernel_never_rejects(ctx):
    s = W.TINY
    for d, buf in [(fake_pool(s, align=2), BUF), (fake_pool(s), BUF + 6), (fake_pool(s, stride=s.row_bytes + 2), BUF)]:
        assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0], buf, dst_bytes=1 << 30)) == kv.KV_ERR_NO_DEVICE
        assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_ELEM
    # but elem_bytes alignment is required (SURVEY.md 8(b) KV_ERR_ALIGN)
    assert status_of(lambda: kv.kv_pack(ctx, fake_pool(s), s.L, [0], BUF + 1, dst_bytes=1 << 30)) == kv.KV_ERR_ALIGN
    assert status_of(lambda: kv.kv_pack(ctx, fake_pool(s, align=1), s.L, [0], BUF, dst_bytes=1 << 30)) == kv.KV_ERR_ALIGN


def test_validation_errors(ctx):
    s = W.TINY
    d = fake_pool(s)
    pg = s.page_bytes
    E = kv
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0, 256], BUF, dst_bytes=2 * pg)) == E.KV_ERR_PAGE_RANGE
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0, -1], BUF, dst_bytes=2 * pg)) == E.KV_ERR_PAGE_RANGE
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0, 1], BUF, dst_bytes=2 * pg - 1)) == E.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0, 1], None, dst_bytes=2 * pg)) == E.KV_ERR_NULL
    assert status_of(lambda: kv.kv_pack(ctx, d, 0, [0], BUF, dst_bytes=pg)) == E.KV_ERR_DESC
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L + 1, [0], BUF, dst_bytes=pg)) == E.KV_ERR_DESC
    assert status_of(lambda: kv.kv_pack(ctx, d, s.L, [0], BUF, dst_bytes=pg, layout=2)) == E.KV_ERR_LAYOUT
    # unpack: page count must be ceil(n_tokens / Td); Td must be the pool's page size
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [0, 1], d, s.L, 16, 16, 33, src_bytes=1 << 30)) == E.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [0, 1], d, s.L, 16, 32, 64, src_bytes=1 << 30)) == E.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [0, 1], d, s.L, 16, 16, 32, src_bytes=2 * pg - 1)) == E.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [3, 3], d, s.L, 16, 16, 32, src_bytes=2 * pg, flags=kv.KV_FLAG_VALIDATE)) == E.KV_ERR_DUP_PAGE
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [3, 3], d, s.L, 16, 16, 32, src_bytes=2 * pg)) == E.KV_ERR_NO_DEVICE  # unchecked without the flag
    assert status_of(lambda: kv.kv_offload(ctx, d, s.L, [0], BUF, pg, mode=3)) == E.KV_ERR_LAYOUT
    # malformed descriptors
    bad = fake_pool(s)
    bad.desc.elem_bytes = 3
    assert status_of(lambda: kv.kv_pack(ctx, bad, s.L, [0], BUF, dst_bytes=1 << 30)) == E.KV_ERR_DESC
    bad = fake_pool(s)
    bad.desc.page_stride_bytes = s.row_bytes - 2
    assert status_of(lambda: kv.kv_pack(ctx, bad, s.L, [0], BUF, dst_bytes=1 << 30)) == E.KV_ERR_DESC
    # batched: offsets must be non-decreasing
    assert status_of(lambda: kv.kv_pack_batched(ctx, d, s.L, [0, 1, 2], [0, 2, 1], [BUF, BUF + (1 << 30)])) == E.KV_ERR_SIZE
    # options
    with pytest.raises(kv.KvError):
        ctx.set_option(kv.KV_OPT_STAGE_BYTES, 1000)
    with pytest.raises(kv.KvError):
        ctx.set_option(99, 0)


def test_empty_calls_are_ok_even_without_a_device(ctx):
    """n == 0 / n_req == 0 -> KV_OK, no launch."""
    s = W.TINY
    d = fake_pool(s)
    kv.kv_pack(ctx, d, s.L, [], BUF, dst_bytes=0)
    kv.kv_unpack(ctx, BUF, [], d, s.L, 16, 16, 0, src_bytes=0)
    kv.kv_pack_batched(ctx, d, s.L, [], [0], [])
    kv.kv_pack_batched(ctx, d, s.L, [], [0, 0, 0], [BUF, BUF])
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 0


def test_auto_host_mode_policy(ctx):
    s = W.QWEN3_OMNI
    d = fake_pool(s)
    for n, want in [(1, kv.KV_HOST_DIRECT), (2, kv.KV_HOST_DIRECT), (3, kv.KV_HOST_STAGED), (11, kv.KV_HOST_STAGED), (512, kv.KV_HOST_STAGED)]:
        assert status_of(lambda: kv.kv_offload(ctx, d, s.L, np.arange(n), BUF, n * s.page_bytes)) == kv.KV_ERR_NO_DEVICE
        assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == want, n
    # layer-first buffers stage too (chunks of whole layers: each (layer, K|V) run of pages is contiguous)
    assert status_of(lambda: kv.kv_offload(ctx, d, s.L, np.arange(512), BUF, 512 * s.page_bytes, mode=kv.KV_HOST_STAGED, layout=1)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_STAGED
    assert status_of(lambda: kv.kv_offload(ctx, d, s.L, np.arange(512), BUF, 512 * s.page_bytes, layout=1)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_HOST_MODE) == kv.KV_HOST_STAGED
    # layerwise reload: flag array checked before anything else
    flags8 = 0x9000
    f = lambda fl: kv.kv_reload_layerwise(ctx, BUF, 512 * s.page_bytes, np.arange(512), d, s.L, 16, 16, 512 * 16, fl, 1)
    assert status_of(lambda: f(flags8)) == kv.KV_ERR_NO_DEVICE
    assert status_of(lambda: f(None)) == kv.KV_ERR_NULL
    assert status_of(lambda: f(flags8 + 4)) == kv.KV_ERR_ALIGN


def test_plan_fused_repage_and_cow(ctx):
    """SURVEY.md 8(f) NEXT-2 / NEXT-1 planning: segment counts and payloads, validation before launch."""
    c5 = W.crossrole_case(0)
    src, dst = fake_pool(c5.src_shape), fake_pool(c5.dst_shape, base0=0x7800_0000_0000)
    L = c5.dst_shape.L
    f = lambda **kw: kv.kv_repage_batched(ctx, src, c5.src_ids, c5.src_offsets, dst, c5.dst_ids,
                                          c5.dst_offsets, c5.n_tokens, L, **kw)
    assert status_of(f) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 32 * 32 * 4 * 96  # 16 KiB segments, 4 per 64-token row
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 6 << 30
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    # device-resident id lists: nothing is validated on the host (the arrays are never dereferenced here)
    import torch
    fd = lambda: kv.kv_repage_batched(ctx, src, torch.from_numpy(c5.src_ids), c5.src_offsets, dst,
                                      torch.from_numpy(c5.dst_ids), c5.dst_offsets, c5.n_tokens, L,
                                      flags=kv.KV_FLAG_IDS_ON_DEVICE)
    assert status_of(fd) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 32 * 32 * 4 * 96
    bad = c5.dst_ids.copy(); bad[5] = bad[4]
    assert status_of(lambda: kv.kv_repage_batched(ctx, src, c5.src_ids, c5.src_offsets, dst, bad, c5.dst_offsets,
                                                  c5.n_tokens, L, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    nt = np.array(c5.n_tokens).copy(); nt[0] += 1
    assert status_of(lambda: kv.kv_repage_batched(ctx, src, c5.src_ids, c5.src_offsets, dst, c5.dst_ids,
                                                  c5.dst_offsets, nt, L)) == kv.KV_ERR_SIZE
    # copy-on-write append on the Qwen3-Omni shape: 5 old tokens + 7 new ones, 96 (layer,kv) rows
    s = W.QWEN3_OMNI
    d = fake_pool(s)
    assert status_of(lambda: kv.kv_cow_append(ctx, d, s.L, 7, 9, 5, BUF, 7)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 96 * 2
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 96 * 12 * 1024
    assert status_of(lambda: kv.kv_cow_append(ctx, d, s.L, 7, 9, 10, BUF, 7)) == kv.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_cow_append(ctx, d, s.L, 7, 7, 1, BUF, 1)) == kv.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_cow_append(ctx, d, s.L, 7, s.P, 1, BUF, 1)) == kv.KV_ERR_PAGE_RANGE
    kv.kv_cow_append(ctx, d, s.L, 7, 9, 0, None, 0)  # nothing to do: KV_OK, even without a device


def test_plan_submit_one_launch_for_a_turn(ctx):
    """kv_submit (SURVEY.md 8(a) a8 / PAPER.md:L238): a turn's scatter + copy-on-write append + gather planned as ONE
    launch whose pieces carry their own direction; validation of every operation precedes it."""
    s = W.QWEN3_OMNI
    d = fake_pool(s)
    rng = np.random.default_rng(5)
    perm = rng.permutation(s.P).astype(np.int32)
    dst, src, old, new = perm[:100], perm[100:160], int(perm[160]), int(perm[161])
    ops = [kv.op_unpack(BUF, dst, 100 * s.T, src_bytes=100 * s.page_bytes),
           kv.op_cow_append(old, new, 5, BUF + (1 << 36), 7),
           kv.op_pack(src, BUF + (1 << 37), dst_bytes=60 * s.page_bytes)]
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, ops, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 100 * 96 + 96 * 2 + 60 * 96
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 160 * s.page_bytes + 96 * 12 * 1024
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384 and ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    assert ctx.stat(kv.KV_STAT_LAUNCHES) == 0
    # a ragged unpack: n_pages must be ceil(n_tokens / T)
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_unpack(BUF, dst, 100 * s.T - 16, src_bytes=1 << 40)])) == kv.KV_ERR_SIZE
    kv_ok = [kv.op_unpack(BUF, dst, 100 * s.T - 15, src_bytes=1 << 40)]
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, kv_ok)) == kv.KV_ERR_NO_DEVICE
    # buffer too small, id out of range, bad kind, device ids
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_pack(src, BUF, dst_bytes=59 * s.page_bytes)])) == kv.KV_ERR_SIZE
    bad = src.copy(); bad[3] = s.P
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_pack(bad, BUF, dst_bytes=1 << 40)])) == kv.KV_ERR_PAGE_RANGE
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [(2, src, BUF, 1 << 40, 0, 0, 0)])) == kv.KV_ERR_LAYOUT
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, ops, flags=kv.KV_FLAG_IDS_ON_DEVICE)) == kv.KV_ERR_LAYOUT
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_cow_append(old, new, 10, BUF, 7)])) == kv.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_cow_append(old, old, 1, BUF, 1)])) == kv.KV_ERR_SIZE
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, [kv.op_cow_append(old, new, 1, None, 1)])) == kv.KV_ERR_NULL
    # under KV_FLAG_VALIDATE: two operations writing one page; an operation reading a page another one writes
    two = [kv.op_unpack(BUF, dst, 100 * s.T, src_bytes=1 << 40), kv.op_cow_append(old, int(dst[7]), 1, BUF, 1)]
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, two, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    rw = [kv.op_unpack(BUF, dst, 100 * s.T, src_bytes=1 << 40), kv.op_pack(dst[:3], BUF + (1 << 37), dst_bytes=1 << 40)]
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, rw, flags=kv.KV_FLAG_VALIDATE)) == kv.KV_ERR_DUP_PAGE
    assert status_of(lambda: kv.kv_submit(ctx, d, s.L, rw)) == kv.KV_ERR_NO_DEVICE  # unchecked without the flag
    kv.kv_submit(ctx, d, s.L, [])  # nothing to do: KV_OK
    kv.kv_submit(ctx, d, s.L, [kv.op_pack(np.zeros(0, np.int32), BUF, dst_bytes=0), kv.op_cow_append(old, new, 0, None, 0)])


def test_plan_hnd_pools(ctx):
    """SURVEY.md 8(f) NEXT-2, HND pools: kernel and segment chosen per direction;
    a malformed order is KV_ERR_DESC; degenerate HND (one head) plans as a plain copy."""
    s = W.QWEN3_OMNI

    def pool(order, shape=s, **kw):
        d = fake_pool(shape, **kw)
        d.desc.order = order
        return d

    hnd = pool(kv.KV_ORDER_HND)
    # pack out of an HND pool (no tensor maps on a planning ctx): strided source, whole 16 KiB rows per CTA (64 head_dim
    # rows each, gathered by cp.async)
    assert status_of(lambda: kv.kv_pack(ctx, hnd, s.L, [1, 2, 3], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 3 * 96
    assert ctx.stat(kv.KV_STAT_LAST_PAYLOAD) == 3 * s.page_bytes
    ctx.set_option(kv.KV_OPT_KERNEL, kv.KV_KERNEL_BULK)  # the ring's transposing geometry: 4 KiB stages (16 rows each)
    assert status_of(lambda: kv.kv_pack(ctx, hnd, s.L, [1, 2, 3], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_BULK and ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 4096
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 3 * 96 * 4
    ctx.set_option(kv.KV_OPT_KERNEL, kv.KV_KERNEL_AUTO)
    # unpack into an HND pool: strided destination, 16-byte stores from the stage
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, np.arange(10), hnd, s.L, 16, 16, 160, src_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 16384
    # pool -> pool: HND -> NHD is a strided source, NHD -> HND a strided destination
    nhd64 = pool(kv.KV_ORDER_NHD, s.with_(T=64, P=64), base0=0x7800_0000_0000)
    hnd64 = pool(kv.KV_ORDER_HND, s.with_(T=64, P=64), base0=0x7800_0000_0000)
    assert status_of(lambda: kv.kv_repage(ctx, hnd, np.arange(8), nhd64, [0, 1], s.L, 128)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    assert status_of(lambda: kv.kv_repage(ctx, pool(0), np.arange(8), hnd64, [0, 1], s.L, 128)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    # short segments keep the earlier choices: 2 KiB token rows of a one-token-per-chunk re-page (5 -> 7) go to the ring,
    # 1 KiB segments to kv_move_small (vec) once the call is large enough
    s2 = W.QWEN3_OMNI.with_(T=7, H=8, P=4096)
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, np.arange(100), fake_pool(s2), s2.L, 5, 7, 700, src_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 2048 and ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_BULK
    s1 = W.QWEN3_OMNI.with_(T=7, P=4096)
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, np.arange(100), fake_pool(s1), s1.L, 5, 7, 700, src_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 1024 and ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_VEC
    # head_dim rows that are not multiples of 16 bytes: element-wise kernel, never rejected
    odd = pool(kv.KV_ORDER_HND, s.with_(D=20))
    assert status_of(lambda: kv.kv_pack(ctx, odd, s.L, [1], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_ELEM
    # one head: [token][head] == [head][token]; planned as the contiguous copy it is
    one = pool(kv.KV_ORDER_HND, s.with_(H=1))
    assert status_of(lambda: kv.kv_unpack(ctx, BUF, [1], one, s.L, 16, 16, 16, src_bytes=1 << 40)) == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_KERNEL) == kv.KV_KERNEL_SHOT
    assert ctx.stat(kv.KV_STAT_LAST_SEGMENT) == 4096  # the whole 4 KiB row
    assert status_of(lambda: kv.kv_pack(ctx, pool(2), s.L, [1], BUF, dst_bytes=1 << 40)) == kv.KV_ERR_DESC


def test_peer_and_signal_argument_errors(ctx):
    """SURVEY.md 8(f) NEXT-3 entries on a planning-only ctx: argument errors come first, then
    KV_ERR_NO_DEVICE (nothing is launched, no CUDA call is made)."""
    with pytest.raises(kv.KvError) as ei:
        kv.kv_peer_enable(ctx, 1)
    assert ei.value.status == kv.KV_ERR_NO_DEVICE
    word = np.zeros(2, dtype=np.uint64)
    with pytest.raises(kv.KvError) as ei:
        kv.kv_signal(ctx, None, 1, stream=0)
    assert ei.value.status == kv.KV_ERR_NULL
    with pytest.raises(kv.KvError) as ei:
        kv.kv_signal(ctx, int(word.ctypes.data) + 4, 1, stream=0)
    assert ei.value.status == kv.KV_ERR_ALIGN
    with pytest.raises(kv.KvError) as ei:
        kv.kv_signal(ctx, word, 1, stream=0)
    assert ei.value.status == kv.KV_ERR_NO_DEVICE
    assert word[0] == 0


def test_chain_hash_planning_and_errors(ctx):
    """kv_chain_hash on a planning-only ctx: offsets are validated and page offsets written (H4: whole
    pages only), then KV_ERR_NO_DEVICE; nothing is dereferenced on the device side."""
    ident, out = 0x1000, 0x2000  # never touched without a device
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, ident, [0, 40, 40, 75], 16, out, out_capacity=4)
    assert ei.value.status == kv.KV_ERR_NO_DEVICE
    assert ctx.stat(kv.KV_STAT_LAST_ITEMS) == 4  # 2 + 0 + 2 whole pages
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, ident, [0, 40, 40, 75], 16, out, out_capacity=3)
    assert ei.value.status == kv.KV_ERR_SIZE
    for bad in ([0, 5, 3], [-1, 4]):
        with pytest.raises(kv.KvError) as ei:
            kv.kv_chain_hash(ctx, ident, bad, 1, out, out_capacity=100)
        assert ei.value.status == kv.KV_ERR_SIZE
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, ident, [0, 16], 0, out, out_capacity=1)
    assert ei.value.status == kv.KV_ERR_SIZE
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, ident + 4, [0, 16], 16, out, out_capacity=1)
    assert ei.value.status == kv.KV_ERR_ALIGN
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, None, [0, 16], 16, out, out_capacity=1)
    assert ei.value.status == kv.KV_ERR_NULL
    # nothing to hash: KV_OK even without a device
    assert kv.kv_chain_hash(ctx, None, [0, 15, 15], 16, None, out_capacity=0).tolist() == [0, 0, 0]
    assert kv.kv_chain_hash(ctx, None, [0], 16, None, out_capacity=0).tolist() == [0]


def test_header_is_c_and_links_from_c(tmp_path):
    """include/kvtier.h compiles as C99 with -Wall -Wextra -Werror -pedantic and a plain-C program drives the
    library through it (planning-only ctx: validation, planning and errors, no CUDA call)."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2606_31093_b200")
    exe = str(tmp_path / "abi_smoke")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(root, "include"),
                           os.path.join(root, "tests", "c", "abi_smoke.c"), "-o", exe, "-L", pkg, "-l:libkvtier.so",
                           "-Wl,-rpath," + pkg])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert "abi_smoke ok" in out.stdout
