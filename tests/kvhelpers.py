"""Test-side glue: host pools for the oracle <-> device pools for the CUDA path.
Holds no transfer arithmetic: it only allocates, fills with seeded random bytes and copies
whole slabs between host and device with torch."""
import numpy as np

from oracle import kv_oracle as ko


def host_pool(rng, L, C, P, T, H, D, e, pad=0, order=0):
    """Random-byte HostPool (random 8-bit patterns => random 16/32-bit patterns)."""
    row = T * H * D * e
    stride = row + pad
    slabs = [rng.integers(0, 256, size=P * stride, dtype=np.uint8) for _ in range(L * C)]
    return ko.HostPool(slabs, L, C, P, T, H, D, e, stride, order)


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
                           pool.page_stride_bytes, pool.order)
    desc._tensors = tens
    return tens, desc


def assert_pool_equal(tens, pool):
    for i, (t, s) in enumerate(zip(tens, pool.slabs)):
        got = t.cpu().numpy()
        if not np.array_equal(got, s):
            bad = np.flatnonzero(got != s)
            raise AssertionError(f"slab {i}: {bad.size} bytes differ, first at {bad[0]} "
                                 f"(page {bad[0] // pool.page_stride_bytes})")


# ---------------------------------------------------------------------------------------------
# full-scale helpers: pools that live only on the device (96 GiB >> what we want in host RAM)
# ---------------------------------------------------------------------------------------------
def device_pool(torch, kvtier, shape, seed, fill="randn"):
    """2*L slabs of [P][T][H][D] bf16 filled on the device with a seeded torch generator
    (BASELINE.json:configs[1]: normal(0,1) values).  Returns (slabs as uint8 views, PoolDesc)."""
    gen = torch.Generator(device="cuda").manual_seed(seed)
    slabs = []
    for _ in range(shape.L * shape.C):
        t = torch.empty(shape.P * shape.T * shape.H * shape.D, dtype=torch.bfloat16, device="cuda")
        if fill == "randn":
            t.normal_(generator=gen)
        else:
            t.view(torch.int16).random_(-32768, 32767, generator=gen)
        slabs.append(t.view(torch.uint8))
    desc = kvtier.PoolDesc(slabs, shape.L, shape.C, shape.P, shape.T, shape.H, shape.D, shape.e)
    return slabs, desc


def snapshot_pages(torch, slabs, ids, shape, layer_count=None):
    """Copy ONLY the pages `ids` of every slab to the host with torch indexing (shares nothing
    with the library) as a compact HostPool whose page k is device page ids[k]."""
    L = shape.L if layer_count is None else layer_count
    row = shape.row_bytes
    idx = torch.as_tensor(np.asarray(ids, dtype=np.int64), device="cuda")
    out = []
    for s in slabs[:L * shape.C]:
        out.append(s.view(shape.P, row).index_select(0, idx).cpu().numpy().reshape(-1))
    return ko.HostPool(out, L, shape.C, len(ids), shape.T, shape.H, shape.D, shape.e, row)


def page_checksums(torch, slabs, shape):
    """Per-page wrap-around 64-bit sums of every slab: [LC][P] int64 on the device."""
    return torch.stack([s.view(torch.int64).view(shape.P, -1).sum(dim=1) for s in slabs])
