"""kv_pack_static: the one entry point of libkvtier.so that allocates nothing.

Who needs it: callers that may not call cudaMalloc (directly, or through a library) at the moment they move KV pages --
a serving engine whose KV pools already own the GPU's memory (the allocation would fail), a step on the latency path
(cudaMalloc / cudaFree stall every stream of the device), a process tied to a fixed memory budget.  Every other entry
point takes a kv_ctx, which allocates when it is created and again when a call's page-id tables outgrow the kernel
parameters; kv_pack_static takes no ctx and keeps its tables in a fixed array built into the library
(include/kvtier.h, "kv_pack without any allocation").

What is checked here: its bytes equal those of the existing path (kv_pack through a ctx) -- bit for bit, the bar of
every transfer test in this suite -- on consecutive calls that share the array, including a shorter call after a longer
one (stale table contents behind the prefix in use) and a call big enough to need several fill launches and, on the
existing path, the allocated table arena; and that requests beyond the array's capacity are refused, not truncated.

This file is named to be collected LAST: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  The GPU tests call kv_pack_static BEFORE they create a ctx, so that a run of this file alone in a fresh
process exercises the first-call set-up on a device no ctx has touched; after the other tests the same code runs on a
device many ctxs have used.
"""
import numpy as np
import pytest

from paper_2606_31093_b200 import kvtier as kv
from tests.kvhelpers import host_pool, to_device

torch = pytest.importorskip("torch")


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _reference_pack(desc, L, ids):
    """The existing path: kv_pack through a ctx (which allocates), into a buffer of its own."""
    out = torch.full((len(ids) * desc.page_bytes(L),), 0xEE, dtype=torch.uint8, device="cuda")
    with kv.Ctx(0, staging_bytes=1 << 20) as ctx:
        kv.kv_pack(ctx, desc, L, ids, out)
        torch.cuda.synchronize()
    return out


# L, C, P, T, H, D, e, pad
SHAPES = [
    (4, 2, 256, 16, 2, 64, 2, 0),    # BASELINE.json:configs[0] Tiny: 4 KiB rows
    (3, 2, 64, 16, 4, 128, 2, 0),    # the paper's Qwen3-Omni row (16 KiB), few layers
    (2, 2, 40, 64, 4, 128, 2, 256),  # 64 KiB rows cut into four segments; padded page stride
    (2, 1, 33, 5, 3, 24, 2, 0),      # odd sizes: 720-byte rows, one slab per layer
]


@pytest.mark.gpu
@pytest.mark.parametrize("shape", SHAPES)
def test_two_calls_in_a_row_match_the_existing_path(shape):
    """Two kv_pack_static calls back to back on one stream, the second shorter than the first and over other pages:
    each must equal kv_pack's result for the same ids.  No sync between the two: stream order alone has to keep the
    second call's table fill behind the first call's copy."""
    _need_gpu()
    L, C, P, T, H, D, e, pad = shape
    rng = np.random.default_rng(20260611 + P)
    pool = host_pool(rng, L, C, P, T, H, D, e, pad)
    tens, desc = to_device(pool, kv, torch)
    n1 = min(37, P - 2)
    ids1 = rng.choice(P, n1, replace=False).astype(np.int32)
    ids2 = rng.permutation(P)[:n1 // 3].astype(np.int32)
    page = desc.page_bytes(L)
    tail = 256
    got1 = torch.full((n1 * page + tail,), 0xCD, dtype=torch.uint8, device="cuda")
    got2 = torch.full((len(ids2) * page + tail,), 0xCD, dtype=torch.uint8, device="cuda")
    before = [t.clone() for t in tens]
    kv.kv_pack_static(desc, L, ids1, got1, dst_bytes=n1 * page)
    kv.kv_pack_static(desc, L, ids2, got2, dst_bytes=len(ids2) * page)
    torch.cuda.synchronize()
    want1 = _reference_pack(desc, L, ids1)
    want2 = _reference_pack(desc, L, ids2)
    assert torch.equal(got1[:n1 * page], want1), "first call differs from kv_pack"
    assert torch.equal(got2[:len(ids2) * page], want2), "second call differs from kv_pack"
    assert bool((got1[n1 * page:] == 0xCD).all()) and bool((got2[len(ids2) * page:] == 0xCD).all()), \
        "wrote past the end of the buffer"
    assert all(torch.equal(a, b) for a, b in zip(tens, before)), "the source pool was written"


@pytest.mark.gpu
def test_large_then_small_then_large_and_no_device_memory_is_taken():
    """9,000 page ids (more than the kernel parameters hold: the existing path grows its allocated table arena for this,
    and kv_pack_static needs two fill launches), then 3 ids, then 9,000 others.  From the second call on, the device's
    free memory must not move: everything the path needs was in place after the first call."""
    _need_gpu()
    L, C, P, T, H, D, e = 2, 2, 1024, 16, 1, 64, 2  # 2 KiB rows: 8 KiB per page, 70 MiB per 9,000-page call
    rng = np.random.default_rng(31093)
    pool = host_pool(rng, L, C, P, T, H, D, e)
    tens, desc = to_device(pool, kv, torch)
    page = desc.page_bytes(L)
    big1 = rng.integers(0, P, 9000).astype(np.int32)   # pack only reads: duplicates are allowed
    small = np.array([5, 1023, 0], dtype=np.int32)
    big2 = rng.integers(0, P, 9000).astype(np.int32)
    outs = [torch.full((len(i) * page,), 0xCD, dtype=torch.uint8, device="cuda") for i in (big1, small, big2)]
    kv.kv_pack_static(desc, L, big1, outs[0])
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    kv.kv_pack_static(desc, L, small, outs[1])
    kv.kv_pack_static(desc, L, big2, outs[2])
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, f"device memory moved by {free_before - free_after} bytes across two calls"
    for ids, got in zip((big1, small, big2), outs):
        assert torch.equal(got, _reference_pack(desc, L, ids)), f"{len(ids)}-page call differs from kv_pack"


@pytest.mark.gpu
def test_on_a_side_stream_and_into_pinned_host_memory():
    """The stream is the caller's: two calls on a non-default stream, the second one writing to mapped pinned host
    memory (the offload direction), both equal to the existing path."""
    _need_gpu()
    L, C, P, T, H, D, e, pad = SHAPES[1]
    rng = np.random.default_rng(7)
    pool = host_pool(rng, L, C, P, T, H, D, e, pad)
    _, desc = to_device(pool, kv, torch)
    ids = rng.choice(P, 20, replace=False).astype(np.int32)
    nbytes = len(ids) * desc.page_bytes(L)
    dev = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    host = kv.kv_host_alloc(nbytes)
    try:
        view = kv.host_view(host, nbytes)
        view[:] = 0
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        kv.kv_pack_static(desc, L, ids, dev, stream=side)
        kv.kv_pack_static(desc, L, ids[::-1].copy(), host, dst_bytes=nbytes, stream=side)
        side.synchronize()
        assert torch.equal(dev, _reference_pack(desc, L, ids))
        assert np.array_equal(view, _reference_pack(desc, L, ids[::-1].copy()).cpu().numpy())
    finally:
        kv.kv_host_free(host)


@pytest.mark.gpu
def test_refusals_enqueue_nothing():
    """Beyond the array's capacity, an HND pool, a misaligned buffer, a bad page id: an error code, and not one byte of
    the destination changes."""
    _need_gpu()
    L, C, P, T, H, D, e, pad = SHAPES[0]
    rng = np.random.default_rng(3)
    pool = host_pool(rng, L, C, P, T, H, D, e, pad)
    _, desc = to_device(pool, kv, torch)
    page = desc.page_bytes(L)
    out = torch.full((8 * page + 64,), 0xCD, dtype=torch.uint8, device="cuda")

    def status(fn):
        with pytest.raises(kv.KvError) as ei:
            fn()
        return ei.value.status

    too_many = np.zeros(kv.KV_STATIC_MAX_PAGES + 1, dtype=np.int32)
    assert status(lambda: kv.kv_pack_static(desc, L, too_many, out, dst_bytes=1 << 62)) == kv.KV_ERR_STATIC_LIMIT
    assert status(lambda: kv.kv_pack_static(desc, L, [0, 1], out[8:], dst_bytes=2 * page)) == kv.KV_ERR_ALIGN
    assert status(lambda: kv.kv_pack_static(desc, L, [0, P], out)) == kv.KV_ERR_PAGE_RANGE
    assert status(lambda: kv.kv_pack_static(desc, L, [0, 1], out, dst_bytes=2 * page - 1)) == kv.KV_ERR_SIZE
    hnd = kv.PoolDesc(desc._tensors, L, C, P, T, H, D, e, order=kv.KV_ORDER_HND)
    assert status(lambda: kv.kv_pack_static(hnd, L, [0, 1], out)) == kv.KV_ERR_LAYOUT
    kv.kv_pack_static(desc, L, [], out)  # nothing to do: fine
    torch.cuda.synchronize()
    assert bool((out == 0xCD).all())


def test_capacity_limits_are_checked_before_any_cuda_call():
    """Runs without a GPU: the limits of include/kvtier.h are enforced ahead of the first CUDA call, with an error of
    their own and a message that names them."""
    assert kv.KV_STATIC_TABLE_BYTES == 270592
    P = 1 << 20
    bases = [0x7000_0000_0000 + i * (1 << 32) for i in range(4)]
    desc = kv.PoolDesc(bases, 2, 2, P, 16, 2, 64, 2)
    ids = np.zeros(kv.KV_STATIC_MAX_PAGES + 1, dtype=np.int32)
    with pytest.raises(kv.KvError) as ei:
        kv.kv_pack_static(desc, 2, ids, 0x7100_0000_0000, dst_bytes=1 << 62)
    assert ei.value.status == kv.KV_ERR_STATIC_LIMIT
    assert "65536" in str(ei.value) and "1024" in str(ei.value)
    wide = kv.PoolDesc([0x7000_0000_0000 + i * (1 << 24) for i in range(1026)], 513, 2, 16, 16, 2, 64, 2)
    with pytest.raises(kv.KvError) as ei:
        kv.kv_pack_static(wide, 513, [0], 0x7100_0000_0000, dst_bytes=1 << 62)
    assert ei.value.status == kv.KV_ERR_STATIC_LIMIT
    with pytest.raises(kv.KvError) as ei:
        kv.kv_pack_static(desc, 2, [0], 0x7100_0000_0000, dst_bytes=1 << 62, device=64)
    assert ei.value.status == kv.KV_ERR_SIZE
