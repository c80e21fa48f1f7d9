"""Test-side glue: host pools for the oracle <-> device pools for the CUDA path.
Holds no transfer arithmetic: it only allocates, fills with seeded random bytes and copies
whole slabs between host and device with torch."""
import numpy as np

from oracle import kv_oracle as ko


def host_pool(rng, L, C, P, T, H, D, e, pad=0):
    """Random-byte HostPool (random 8-bit patterns => random 16/32-bit patterns)."""
    row = T * H * D * e
    stride = row + pad
    slabs = [rng.integers(0, 256, size=P * stride, dtype=np.uint8) for _ in range(L * C)]
    return ko.HostPool(slabs, L, C, P, T, H, D, e, stride)


def to_device(pool, kvtier, torch, offset_bytes=0):
    """Upload a HostPool; returns (tensors, PoolDesc).  offset_bytes misaligns every slab base."""
    tens = []
    bases = []
    for s in pool.slabs:
        t = torch.empty(s.size + 64, dtype=torch.uint8, device="cuda")
        v = t[offset_bytes:offset_bytes + s.size]
        v.copy_(torch.from_numpy(s))
        tens.append(v)
        bases.append(v.data_ptr())
    desc = kvtier.PoolDesc(bases, pool.L, pool.C, pool.num_pages, pool.T, pool.H, pool.D, pool.e,
                           pool.page_stride_bytes)
    desc._tensors = tens
    return tens, desc


def assert_pool_equal(tens, pool):
    for i, (t, s) in enumerate(zip(tens, pool.slabs)):
        got = t.cpu().numpy()
        if not np.array_equal(got, s):
            bad = np.flatnonzero(got != s)
            raise AssertionError(f"slab {i}: {bad.size} bytes differ, first at {bad[0]} "
                                 f"(page {bad[0] // pool.page_stride_bytes})")
