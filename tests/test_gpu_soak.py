"""Concurrent soak: three lanes -- three CUDA streams sharing ONE ctx (its staging slots, its table ring, its
programmatic-dependent-launch chains) -- each issue a long random sequence of transfers with NO synchronisation in
between: pack, unpack (also ragged), fused re-page within the pool, batched copy-on-write appends, kv_submit turns,
offload and reload in every host mode.  A lane owns a disjoint third of the pool's pages, a device buffer and a
pinned host buffer, so the lanes are independent and the expected final state is each lane's operations applied in
order by the CPU oracle ("a page may simultaneously be used by inference or by loading, offloading,
and uploading operations"; SURVEY.md 8(c) reading 21: calls on different streams are independent when their
destination page sets are disjoint).  What this catches that the sequential fuzz cannot: a staging slot or a table
slot reused before its reader is done, a kernel started early (PDL) that reads what its predecessor has not
written yet, stream-order bugs in the fork / join of the staged pipeline."""
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


LANES = 3
PAGES_PER_LANE = 160
MAX_N = 60  # pages per transfer


class Lane:
    def __init__(self, kv, idx, page_bytes, rng):
        self.idx = idx
        self.pages = np.arange(idx * PAGES_PER_LANE, (idx + 1) * PAGES_PER_LANE, dtype=np.int32)
        self.stream = torch.cuda.Stream()
        nb = MAX_N * page_bytes
        self.dbuf = torch.empty(nb, dtype=torch.uint8, device="cuda")
        self.hp = kv.kv_host_alloc(nb)
        init = rng.integers(0, 256, size=nb, dtype=np.uint8)
        self.dbuf.copy_(torch.from_numpy(init))
        kv.host_view(self.hp, nb)[:] = init
        self.want_d = init.copy()  # the oracle's image of the device buffer
        self.want_h = init.copy()  # ... and of the pinned host buffer


@pytest.mark.parametrize("seed,order,kernel", [(0, 0, 0), (1, 0, 0), (2, 1, 0), (3, 0, 1), (4, 1, 4), (5, 0, 2)])
def test_three_streams_one_ctx_no_syncs(kv, seed, order, kernel):
    L, C, T, H, D, e = 4, 2, 16, 4, 128, 2  # 16 KiB rows, 128 KiB pages
    P = LANES * PAGES_PER_LANE
    rng = np.random.default_rng(9000 + seed)
    A = host_pool(rng, L, C, P, T, H, D, e, order=order)
    tA, dA = to_device(A, kv, torch)
    page = dA.page_bytes()
    tok = L * C * H * D * e
    ctx = kv.Ctx(0, staging_bytes=6 << 20)  # two slots of 3 MiB: transfers of up to 7.5 MiB pipeline through several chunks
    ctx.set_option(kv.KV_OPT_KERNEL, kernel)
    lanes = [Lane(kv, i, page, rng) for i in range(LANES)]
    torch.cuda.synchronize()
    modes = [kv.KV_HOST_AUTO, kv.KV_HOST_DIRECT, kv.KV_HOST_STAGED]
    try:
        # Phase 1: draw every operation, then issue them back to back (nothing but the C calls between two launches, so
        # the streams really run ahead of the host and against one another).  Phase 2: the oracle replays the same list.
        plan = []
        for step in range(70):
            for ln in lanes:  # round-robin over the lanes: their work interleaves on the device
                n = int(rng.integers(1, MAX_N + 1))
                op = int(rng.integers(0, 8))
                ids = rng.choice(ln.pages, n, replace=False).astype(np.int32)
                a = dict(ln=ln, op=op, n=n, ids=ids)
                if op == 1:
                    a["ntok"] = n * T - (int(rng.integers(0, T)) if rng.random() < 0.3 else 0)
                elif op in (2, 3):
                    a["mode"] = modes[int(rng.integers(0, 3))]
                elif op == 4:
                    k = max(1, n // 2)
                    a.update(k=k, src=ids[:k], dst=rng.choice(np.setdiff1d(ln.pages, ids[:k]), k, replace=False).astype(np.int32))
                elif op == 5:
                    k = max(1, n // 4)
                    n_old = rng.integers(0, T, size=k)
                    n_app = np.array([rng.integers(1, T - o + 1) for o in n_old])
                    apps_h = [rng.integers(0, 256, size=int(x) * tok, dtype=np.uint8) for x in n_app]
                    a.update(k=k, old=ids[:k], new=rng.choice(np.setdiff1d(ln.pages, ids[:k]), k, replace=False).astype(np.int32),
                             n_old=n_old, n_app=n_app, apps_h=apps_h, apps_d=[torch.from_numpy(x).cuda() for x in apps_h])
                elif op == 6:
                    k = max(1, n // 2)
                    a.update(k=k, dst=ids[:k],
                             src=rng.choice(np.setdiff1d(ln.pages, ids[:k]), min(k, MAX_N - k), replace=False).astype(np.int32))
                plan.append(a)
        torch.cuda.synchronize()  # the append blocks are uploaded
        for a in plan:
            ln, op, n, ids, s = a["ln"], a["op"], a["n"], a["ids"], a["ln"].stream
            if op == 0:  # pack -> device buffer
                kv.kv_pack(ctx, dA, L, ids, ln.dbuf, dst_bytes=n * page, stream=s)
            elif op == 1:  # unpack the device buffer's first n pages, now and then with a ragged tail
                kv.kv_unpack(ctx, ln.dbuf, ids, dA, L, T, T, a["ntok"], src_bytes=n * page, stream=s)
            elif op == 2:  # offload -> pinned host buffer
                kv.kv_offload(ctx, dA, L, ids, ln.hp, n * page, mode=a["mode"], stream=s)
            elif op == 3:  # reload from the pinned host buffer
                kv.kv_reload(ctx, ln.hp, n * page, ids, dA, L, T, T, n * T, mode=a["mode"], stream=s)
            elif op == 4:  # fused re-page inside the pool: k source pages -> k other pages of the lane
                kv.kv_repage(ctx, dA, a["src"], dA, a["dst"], L, a["k"] * T, stream=s)
            elif op == 5:  # batched copy-on-write append: k sessions
                kv.kv_cow_append_batched(ctx, dA, L, a["old"], a["new"], a["n_old"], a["n_app"], a["apps_d"], stream=s)
            elif op == 6:  # a turn in ONE launch: scatter the buffer's first k pages + gather other pages behind them
                k = a["k"]
                ops = [kv.op_unpack(ln.dbuf, a["dst"], k * T, src_bytes=k * page),
                       kv.op_pack(a["src"], ln.dbuf[k * page:], dst_bytes=len(a["src"]) * page)]
                kv.kv_submit(ctx, dA, L, ops, flags=kv.KV_FLAG_VALIDATE, stream=s)
            else:  # pack, then offload of the same pages
                kv.kv_pack(ctx, dA, L, ids, ln.dbuf, dst_bytes=n * page, stream=s)
                kv.kv_offload(ctx, dA, L, ids, ln.hp, n * page, stream=s)
        for a in plan:  # the oracle, in issue order (lanes are independent, so this is each lane's order)
            ln, op, n, ids = a["ln"], a["op"], a["n"], a["ids"]
            if op == 0:
                ln.want_d[:n * page] = ko.pack(A, ids)
            elif op == 1:
                ko.unpack(ln.want_d[:n * page], ids, A, Ts=T, n_tokens=a["ntok"])
            elif op == 2:
                ln.want_h[:n * page] = ko.pack(A, ids)
            elif op == 3:
                ko.unpack(ln.want_h[:n * page], ids, A, Ts=T, n_tokens=n * T)
            elif op == 4:
                ko.repage(A, a["src"], A, a["dst"], a["k"] * T)
            elif op == 5:
                ko.cow_append_batched(A, a["old"], a["new"], a["n_old"], a["n_app"], a["apps_h"])
            elif op == 6:
                k = a["k"]
                packed = ko.pack(A, a["src"])  # (reads pages the unpack of the same call does not write: unordered is fine)
                ko.unpack(ln.want_d[:k * page], a["dst"], A, Ts=T, n_tokens=k * T)
                ln.want_d[k * page:(k + len(a["src"])) * page] = packed
            else:
                ln.want_d[:n * page] = ko.pack(A, ids)
                ln.want_h[:n * page] = ln.want_d[:n * page]
        torch.cuda.synchronize()
        assert ctx.device_status() == 0
        assert_pool_equal(tA, A)
        for ln in lanes:
            assert np.array_equal(ln.dbuf.cpu().numpy(), ln.want_d), f"lane {ln.idx}: device buffer"
            assert np.array_equal(kv.host_view(ln.hp, ln.want_h.size), ln.want_h), f"lane {ln.idx}: pinned host buffer"
    finally:
        torch.cuda.synchronize()
        for ln in lanes:
            kv.kv_host_free(ln.hp)
        ctx.close()
