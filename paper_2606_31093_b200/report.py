"""Per-config measurement report (SURVEY.md 8(d) "Report schema"): every BASELINE.json config x
op x mode, device-timed with CUDA events on the launch stream, as GB/s and fraction of the
measured peaks.  Called by ``bench.py --report`` with the bench's 96 GiB pool; writes
``gpurun_out/report.json``.  Timing only -- parity is the business of tests/ (a torch gather check
guards each device-side result here so a wrong-but-fast run cannot be reported).

Conventions: device-side pack/unpack GB/s = (bytes read + bytes written) / time = 2*payload/time
(re-paging with padding: n_tokens*tok read + n_dst*page written); host tier GB/s = payload/time
against the pinned cudaMemcpy peak measured in the same run.
"""
from __future__ import annotations

import json
import os
import time

import numpy as np

from . import kvtier as kv
from . import workloads as W


# Isolated calls up to this payload run on a cold AND clean L2 (write 512 MiB, then read 512 MiB).
# asks for the flush below 256 MiB; up to 2 GiB the previous repetition's ~126 MB of dirty lines would otherwise be
# written back inside the timed call (~19 us: 20 % of a 256 MiB transfer), so the flush is kept on to 2 GiB.
FLUSH_UP_TO = 2 << 30
NOMINAL_HBM_GBPS = 7700.0  # HBM3e on B200 as the task statement quotes it (~7.7 TB/s); the measured copy peak is the bar


def _events(torch, fn, reps, warm, flush=None):
    """Median / best duration in us of `fn` between two CUDA events on the current stream.
    `flush` = (w, r): write 512 MiB then read another 512 MiB before every timed call, so the 126 MB
    L2 is cold AND clean -- a write-only flush leaves up to an L2's worth of dirty lines whose
    write-back (~20 us of DRAM time) would be billed to the timed call."""
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    stream.synchronize()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush[0].fill_(1)
            flush[1].view(torch.int64).sum()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fn()
        b.record(stream)
        stream.synchronize()
        ts.append(a.elapsed_time(b) * 1e3)  # us
    return float(np.median(ts)), float(np.min(ts))


def run(ctx, desc, shape, slabs, seed=0, out_dir="gpurun_out", hbm_peak=None):
    import torch

    rng = np.random.default_rng(seed + 77)
    recs = []
    flush = (torch.empty(512 << 20, dtype=torch.uint8, device="cuda"),
             torch.zeros(512 << 20, dtype=torch.uint8, device="cuda"))

    # ---- peaks measured in this run -----------------------------------------------------------
    N = 1 << 30
    a = torch.empty(N, dtype=torch.uint8, device="cuda")
    b = torch.empty(N, dtype=torch.uint8, device="cuda")
    h = torch.empty(N, dtype=torch.uint8, pin_memory=True)
    _, t = _events(torch, lambda: b.copy_(a), 10, 3)
    d2d = 2 * N / t / 1e3
    _, t = _events(torch, lambda: a.copy_(h, non_blocking=True), 10, 2)
    h2d = N / t / 1e3
    _, t = _events(torch, lambda: h.copy_(a, non_blocking=True), 10, 2)
    d2h = N / t / 1e3
    del a, b, h
    peaks = {"hbm_copy_GBps_this_run": d2d, "h2d_GBps": h2d, "d2h_GBps": d2h,
             "hbm_peak_GBps": hbm_peak or d2d}
    hbm = peaks["hbm_peak_GBps"]

    def rec(cfg, op, mode, payload, traffic, n_pages, fn, reps=7, warm=2, link=None, check=None):
        med, best = _events(torch, fn, reps, warm, flush if payload <= FLUSH_UP_TO else None)
        r = {"config": cfg, "op": op, "mode": mode, "payload_bytes": int(payload),
             "traffic_bytes": int(traffic), "n_pages": int(n_pages), "time_us_median": med,
             "time_us_best": best}
        if link is None:
            r["GBps"] = traffic / med / 1e3
            r["pct_of_measured_hbm_peak"] = 100 * r["GBps"] / hbm
            r["pct_of_nominal_hbm_peak"] = 100 * r["GBps"] / NOMINAL_HBM_GBPS
        else:
            r["GBps"] = payload / med / 1e3
            r["pct_of_link_peak"] = 100 * r["GBps"] / link
        if check is not None:
            r["verified"] = bool(check())
        recs.append(r)
        return r

    L, T = shape.L, shape.T
    LC, row, page = shape.L * shape.C, shape.row_bytes, shape.page_bytes

    def gather_ok(buf, ids, layers=L):
        idx = torch.as_tensor(np.asarray(ids, dtype=np.int64), device="cuda")
        v = buf[:len(ids) * layers * shape.C * row].view(len(ids), layers * shape.C, row)
        return all(torch.equal(v[:, lc], slabs[lc].view(shape.P, row).index_select(0, idx))
                   for lc in range(0, layers * shape.C, 11))

    def scatter_ok(buf, ids, layers=L):  # same-page-size unpack: page ids[p] == buffer page p
        return gather_ok(buf, ids, layers)

    # ---- config 1: Tiny (launch-bound; correctness config) --------------------------------------
    tc = W.tiny_case(seed)
    ts_ = tc.shape
    tslabs = [torch.randint(0, 256, (ts_.P * ts_.row_bytes,), dtype=torch.uint8, device="cuda") for _ in range(ts_.L * ts_.C)]
    tdesc = kv.PoolDesc(tslabs, ts_.L, ts_.C, ts_.P, ts_.T, ts_.H, ts_.D, ts_.e)
    tbuf = torch.empty(37 * ts_.page_bytes, dtype=torch.uint8, device="cuda")
    pl = 37 * ts_.page_bytes
    rec("1 tiny", "pack", "device", pl, 2 * pl, 37, lambda: kv.kv_pack(ctx, tdesc, ts_.L, tc.src_ids, tbuf), reps=20)
    rec("1 tiny", "unpack", "device", pl, 2 * pl, 37,
        lambda: kv.kv_unpack(ctx, tbuf, tc.dst_ids, tdesc, ts_.L, ts_.T, ts_.T, 37 * ts_.T), reps=20)

    # ---- config 2: single-request prefix ---------------------------------------------------------
    c2 = W.prefix_case(seed, shape=shape)
    n = len(c2.src_ids)
    pl = n * page
    buf = torch.empty(pl, dtype=torch.uint8, device="cuda")
    rec("2 prefix", "pack", "device", pl, 2 * pl, n, lambda: kv.kv_pack(ctx, desc, L, c2.src_ids, buf),
        reps=20, warm=3, check=lambda: gather_ok(buf, c2.src_ids))
    rec("2 prefix", "unpack", "device", pl, 2 * pl, n,
        lambda: kv.kv_unpack(ctx, buf, c2.dst_ids, desc, L, T, T, n * T), reps=20, warm=3,
        check=lambda: scatter_ok(buf, c2.dst_ids))
    # ---- fragmentation (SURVEY.md 8(d) "structure of the workloads" (i)): the same 512 pages in runs of r
    # consecutive ids (run starts drawn at random, runs disjoint); r = 1 is the aged pool of the configs,
    # r = n a fresh one.  Consecutive pages are adjacent within a slab but stay a page apart in the buffer,
    # so segments do not grow: only DRAM/TLB locality of the pool side changes.
    for r_len in (1, 4, 16, 64, n):
        starts = rng.choice(shape.P // r_len, n // r_len, replace=False) * r_len
        ids_r = (starts[:, None] + np.arange(r_len)[None, :]).reshape(-1).astype(np.int32)
        rec("2 prefix, ids in runs", f"pack, runs of {r_len}", "device", pl, 2 * pl, n,
            lambda: kv.kv_pack(ctx, desc, L, ids_r, buf), reps=20, warm=3)
        rec("2 prefix, ids in runs", f"unpack, runs of {r_len}", "device", pl, 2 * pl, n,
            lambda: kv.kv_unpack(ctx, buf, ids_r, desc, L, T, T, n * T), reps=20, warm=3)

    # ---- tensor-parallel head partitions ("head partitions"): the same slabs read as pools of 1 and 2
    # KV heads per rank -> 4 KiB / 8 KiB rows, 4x / 2x the pages for the same 768 MiB (timing only)
    for Hp in (1, 2):
        f = shape.H // Hp
        desc_p = kv.PoolDesc(slabs, L, shape.C, shape.P * f, T, Hp, shape.D, shape.e)
        ids_p = rng.choice(shape.P * f, n * f, replace=False).astype(np.int32)
        dst_p = rng.choice(shape.P * f, n * f, replace=False).astype(np.int32)
        rec(f"2 prefix, {Hp} KV head(s) per rank", f"pack ({4 * Hp} KiB rows)", "device", pl, 2 * pl, n * f,
            lambda: kv.kv_pack(ctx, desc_p, L, ids_p, buf), reps=20, warm=3)
        rec(f"2 prefix, {Hp} KV head(s) per rank", f"unpack ({4 * Hp} KiB rows)", "device", pl, 2 * pl, n * f,
            lambda: kv.kv_unpack(ctx, buf, dst_p, desc_p, L, T, T, n * f * T), reps=20, warm=3)

    # ---- NEXT-2: the same prefix on an HND pool ([head][token][dim] pages; the buffer stays NHD, so the
    # transfer transposes).  Same slabs, HND descriptor: timing only (parity: tests/test_gpu_hnd.py).
    desc_h = kv.PoolDesc(slabs, L, shape.C, shape.P, T, shape.H, shape.D, shape.e, order=kv.KV_ORDER_HND)
    for tm, label in ((1, "tensor maps (cp.async.bulk.tensor)"), (0, "lane paths (cp.async gather / STG.128)")):
        ctx.set_option(kv.KV_OPT_TENSOR_MAPS, tm)
        rec("2 prefix, HND pool", "pack", label, pl, 2 * pl, n,
            lambda: kv.kv_pack(ctx, desc_h, L, c2.src_ids, buf), reps=20, warm=3)
        rec("2 prefix, HND pool", "unpack", label, pl, 2 * pl, n,
            lambda: kv.kv_unpack(ctx, buf, c2.dst_ids, desc_h, L, T, T, n * T), reps=20, warm=3)
        rec("2 prefix, HND pool", "repage HND->HND pool", label, pl, 2 * pl, n,
            lambda: kv.kv_repage(ctx, desc_h, c2.src_ids, desc_h, c2.dst_ids, L, n * T), reps=20, warm=3)
    ctx.set_option(kv.KV_OPT_TENSOR_MAPS, 1)
    host_total = 0
    hp = None
    try:
        # one pinned allocation serves configs 2-5 (26.5 GiB for config 4)
        b4 = W.batch_case(seed, shape=shape)
        host_total = int(b4.req_offsets[-1]) * page
        t0 = time.perf_counter()
        hp = kv.kv_host_alloc(host_total)
        peaks["pinned_alloc_GiB"] = host_total / 2**30
        peaks["pinned_alloc_seconds"] = time.perf_counter() - t0
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged"), (kv.KV_HOST_AUTO, "auto")):
            rec("2 prefix", "offload", name, pl, pl, n,
                lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, mode=mode), reps=7, link=d2h)
            rec("2 prefix", "reload", name, pl, pl, n,
                lambda: kv.kv_reload(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, mode=mode), reps=7, link=h2d)
        torch.cuda.synchronize()
        recs[-1]["verified"] = bool(scatter_ok(buf, c2.dst_ids))

        # layer-first host buffer (NEXT-2): staged in chunks of whole layers; layer-by-layer reload with flags
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            rec("2 prefix, layer-first buffer", "offload", name, pl, pl, n,
                lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, mode=mode, layout=kv.KV_LAYOUT_LAYER_FIRST),
                reps=7, link=d2h)
            rec("2 prefix, layer-first buffer", "reload", name, pl, pl, n,
                lambda: kv.kv_reload(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, mode=mode,
                                     layout=kv.KV_LAYOUT_LAYER_FIRST), reps=7, link=h2d)
        flp = kv.kv_host_alloc(L * 8)
        fh = kv.host_view(flp, L * 8).view(np.uint64)
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            first, last = [], []
            for it in range(5):
                fh[:] = 0
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                kv.kv_reload_layerwise(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, flp, 1, mode=mode)
                while fh[0] != 1:
                    pass
                t1 = time.perf_counter()
                while fh[L - 1] != 1:
                    pass
                t2 = time.perf_counter()
                first.append((t1 - t0) * 1e6)
                last.append((t2 - t0) * 1e6)
            recs.append({"config": "2 prefix, layer-first buffer", "op": "reload_layerwise", "mode": name,
                         "payload_bytes": int(pl), "first_layer_us": float(np.median(first)),
                         "last_layer_us": float(np.median(last)), "GBps": pl / float(np.median(last)) / 1e3,
                         "timing": "host wall clock from the call to the flag seen in mapped pinned memory"})
        kv.kv_host_free(flp)

        # both directions of the link at once: offload on one stream (ctx), reload of ANOTHER buffer on a
        # second stream (ctx2) -- eviction of one session while another is restored.  Peak = two plain
        # cudaMemcpyAsync of the same sizes on the same two streams.
        ctx2 = kv.Ctx(torch.cuda.current_device())
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        dev2 = torch.empty(pl, dtype=torch.uint8, device="cuda")
        hA = torch.from_numpy(kv.host_view(hp, 2 * pl))

        def both(f, g):
            sa.wait_stream(torch.cuda.current_stream())
            sb.wait_stream(torch.cuda.current_stream())
            f()
            g()
            torch.cuda.current_stream().wait_stream(sa)
            torch.cuda.current_stream().wait_stream(sb)

        def mc_a():
            with torch.cuda.stream(sa):
                hA[:pl].copy_(buf, non_blocking=True)

        def mc_b():
            with torch.cuda.stream(sb):
                dev2.copy_(hA[pl:], non_blocking=True)

        _, t = _events(torch, lambda: both(mc_a, mc_b), 7, 2)
        peaks["duplex_memcpy_GBps"] = duplex = 2 * pl / t / 1e3
        rec("2 prefix", "offload and reload at once (two ctxs, two streams)", "auto", 2 * pl, 2 * pl, 2 * n,
            lambda: both(lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, stream=sa),
                         lambda: kv.kv_reload(ctx2, hp + pl, pl, c2.dst_ids, desc, L, T, T, n * T, stream=sb)),
            reps=7, link=duplex)
        torch.cuda.synchronize()
        ctx2.close()
        del dev2, hA

        # ---- config 3: 50-turn session ------------------------------------------------------------
        turns = W.session_turns(seed, T=T)
        fl = W.FreeList(shape.P, np.random.default_rng(seed))
        stream = torch.cuda.current_stream()
        in_host, moved, per_turn = 0, 0, []
        t_reload = t_offload = 0.0
        for tn in turns:
            ids = fl.pop(in_host)
            n_new = tn.cum_tokens // T - in_host
            new_ids = fl.pop(n_new)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record(stream)
            kv.kv_reload(ctx, hp, in_host * page, ids, desc, L, T, T, in_host * T)
            e[1].record(stream)
            kv.kv_offload(ctx, desc, L, new_ids, hp + in_host * page, n_new * page)
            e[2].record(stream)
            stream.synchronize()
            r_us, o_us = e[0].elapsed_time(e[1]) * 1e3, e[1].elapsed_time(e[2]) * 1e3
            per_turn.append({"turn": tn.k, "reload_pages": in_host, "reload_us": r_us,
                             "offload_pages": n_new, "offload_us": o_us})
            t_reload += r_us
            t_offload += o_us
            moved += (in_host + n_new) * page
            in_host += n_new
            fl.give_back(ids)
            fl.give_back(new_ids)
        n50 = per_turn[-1]["reload_pages"]
        recs.append({"config": "3 session", "op": "50 turns: reload matched prefix + offload new pages", "mode": "auto",
                     "payload_bytes": int(moved), "n_pages": int(moved // page),
                     "time_us_total": t_reload + t_offload,
                     "reload_GBps": sum(p["reload_pages"] for p in per_turn) * page / t_reload / 1e3,
                     "offload_GBps": sum(p["offload_pages"] for p in per_turn) * page / t_offload / 1e3,
                     "pct_of_link_peak_reload": 100 * sum(p["reload_pages"] for p in per_turn) * page / t_reload / 1e3 / h2d,
                     "turn50_reload_pages": n50, "turn50_reload_us": per_turn[-1]["reload_us"],
                     "turn50_reload_GBps": n50 * page / per_turn[-1]["reload_us"] / 1e3,
                     "per_turn": per_turn})
        buf50 = torch.empty(n50 * page, dtype=torch.uint8, device="cuda")
        ids50 = fl.pop(n50)
        rec("3 session", "turn-50 unpack from a device copy of the buffer", "device", n50 * page, 2 * n50 * page, n50,
            lambda: kv.kv_unpack(ctx, buf50, ids50, desc, L, T, T, n50 * T), reps=10,
            check=lambda: scatter_ok(buf50, ids50))
        fl.give_back(ids50)
        del buf50

        # ---- config 4: concurrent batch -------------------------------------------------------------
        R = len(b4.lens)
        counts = np.diff(b4.req_offsets)
        big = torch.empty(host_total, dtype=torch.uint8, device="cuda")
        bufs = [big[int(b4.req_offsets[r]) * page:int(b4.req_offsets[r + 1]) * page] for r in range(R)]
        hps = [hp + int(b4.req_offsets[r]) * page for r in range(R)]
        sizes = [int(c) * page for c in counts]
        pl4 = host_total
        rec("4 batch", "pack_batched", "device", pl4, 2 * pl4, pl4 // page,
            lambda: kv.kv_pack_batched(ctx, desc, L, b4.src_ids, b4.req_offsets, bufs), reps=7,
            check=lambda: gather_ok(big, b4.src_ids))
        rec("4 batch", "unpack_batched", "device", pl4, 2 * pl4, pl4 // page,
            lambda: kv.kv_unpack_batched(ctx, bufs, b4.dst_ids, b4.req_offsets, counts * T, desc, L, T, T), reps=7,
            check=lambda: scatter_ok(big, b4.dst_ids))
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            rec("4 batch", "offload_batched", name, pl4, pl4, pl4 // page,
                lambda: kv.kv_offload_batched(ctx, desc, L, b4.src_ids, b4.req_offsets, hps, host_bytes=sizes, mode=mode),
                reps=3, warm=1, link=d2h)
            rec("4 batch", "reload_batched", name, pl4, pl4, pl4 // page,
                lambda: kv.kv_reload_batched(ctx, hps, b4.dst_ids, b4.req_offsets, counts * T, desc, L, T, T,
                                             host_bytes=sizes, mode=mode), reps=3, warm=1, link=h2d)
        del big, bufs

        # ---- config 5: cross-role re-paging 16 -> 64 -------------------------------------------------
        half = (shape.P // 2) * row
        s_src = shape.with_(P=shape.P // 2)
        s_dst = shape.with_(T=64, P=shape.P // 8)
        d_src = kv.PoolDesc([s[:half] for s in slabs], L, shape.C, s_src.P, 16, shape.H, shape.D, shape.e)
        d_dst = kv.PoolDesc([s[half:] for s in slabs], L, shape.C, s_dst.P, 64, shape.H, shape.D, shape.e)
        for ragged in (False, True):
            c5 = W.crossrole_case(seed, ragged=ragged, src_shape=s_src, dst_shape=s_dst)
            R5 = len(c5.n_tokens)
            big5 = torch.empty(int(c5.src_offsets[-1]) * page, dtype=torch.uint8, device="cuda")
            bufs5 = [big5[int(c5.src_offsets[r]) * page:int(c5.src_offsets[r + 1]) * page] for r in range(R5)]
            pl5 = int(c5.src_offsets[-1]) * page
            name = "5 cross-role ragged" if ragged else "5 cross-role"
            rec(name, "pack_batched (T=16)", "device", pl5, 2 * pl5, pl5 // page,
                lambda: kv.kv_pack_batched(ctx, d_src, L, c5.src_ids, c5.src_offsets, bufs5), reps=10)
            wr = int(c5.dst_offsets[-1]) * s_dst.page_bytes
            rd = int(c5.n_tokens.sum()) * shape.tok_bytes
            rec(name, "unpack_batched re-page 16->64", "device", wr, rd + wr, int(c5.dst_offsets[-1]),
                lambda: kv.kv_unpack_batched(ctx, bufs5, c5.dst_ids, c5.dst_offsets, c5.n_tokens, d_dst, L, 16, 64),
                reps=10)
            rec(name, "repage_batched fused pool->pool 16->64", "device", wr, rd + wr, int(c5.dst_offsets[-1]),
                lambda: kv.kv_repage_batched(ctx, d_src, c5.src_ids, c5.src_offsets, d_dst, c5.dst_ids,
                                             c5.dst_offsets, c5.n_tokens, L), reps=10)
            del big5, bufs5

        # ---- NEXT-1: copy-on-write tail-page append, 64 sessions in one launch -------
        S = 64
        perm = rng.permutation(shape.P).astype(np.int32)
        n_old = rng.integers(0, T, size=S)
        n_app = np.array([rng.integers(1, T - o + 1) for o in n_old])
        apps = [torch.empty(int(a) * shape.tok_bytes, dtype=torch.uint8, device="cuda") for a in n_app]
        plc = int((n_old + n_app).sum()) * shape.tok_bytes
        rec("3 session", "cow_append_batched (64 sessions' tail pages)", "device", plc, 2 * plc, S,
            lambda: kv.kv_cow_append_batched(ctx, desc, L, perm[:S], perm[S:2 * S], n_old, n_app, apps), reps=20)
        del apps

        # ---- NEXT-4: chained paged hashing: ids of whole sessions / batches ----------
        def chain_rec(name, wb):
            d_ident = torch.from_numpy(wb.ident.view(np.int64)).cuda()
            lens = np.diff(wb.tok_offsets)
            npg = int((lens // T).sum())
            outc = torch.empty(max(npg, 1), dtype=torch.int64, device="cuda")
            med, best = _events(torch, lambda: kv.kv_chain_hash(ctx, d_ident, wb.tok_offsets, T, outc), 20, 3)
            longest = int((lens // T).max())
            recs.append({"config": "NEXT-4 chain hash", "op": name, "sessions": int(lens.size), "tokens": int(lens.sum()),
                         "pages": npg, "longest_chain_pages": longest, "chain_us_median": med, "chain_us_best": best,
                         "Mpages_per_s": npg / med, "ns_per_link_longest_chain": 1e3 * med / max(longest, 1)})
        turns = W.session_turns(seed)
        chain_rec("config 3: one 50-turn session history (a single chain)", W.identity_batch(seed + 3, lens=[turns[-1].cum_tokens]))
        chain_rec("config 4: 64 requests, log-uniform 512-16,384 tokens", W.identity_batch(seed + 4, lens=W.batch_case(seed).lens))
        chain_rec("4,096 sessions, log-uniform 512-16,384 tokens", W.identity_batch(seed + 5, n_sessions=4096))

        # ---- transfer-size sweep 1 MiB .. 8 GiB (layer_count = 32 => 1 MiB pages) --------------------
        Ls = 32
        pg = Ls * shape.C * row
        sweep = []
        bufS = torch.empty(8 << 30, dtype=torch.uint8, device="cuda")
        for npg in W.sweep_sizes_pages():
            ids = rng.choice(shape.P, npg, replace=False).astype(np.int32)
            dst = rng.choice(shape.P, npg, replace=False).astype(np.int32)
            ids_s = rng.choice(s_src.P, npg, replace=False).astype(np.int32)
            nd = -(-npg * 16 // 64)
            dst64 = rng.choice(s_dst.P, nd, replace=False).astype(np.int32)
            pls = npg * pg
            reps = 20 if pls <= (256 << 20) else 7
            row_ = {"MiB": pls >> 20, "n_pages": npg}
            fl_ = flush if pls <= FLUSH_UP_TO else None
            m, bst = _events(torch, lambda: kv.kv_pack(ctx, desc, Ls, ids, bufS), reps, 2, fl_)
            row_["pack_GBps"], row_["pack_us"], row_["pack_us_best"] = 2 * pls / m / 1e3, m, bst
            m, bst = _events(torch, lambda: kv.kv_unpack(ctx, bufS, dst, desc, Ls, T, T, npg * T), reps, 2, fl_)
            row_["unpack_GBps"], row_["unpack_us"] = 2 * pls / m / 1e3, m
            m, bst = _events(torch, lambda: kv.kv_unpack(ctx, bufS, dst64, d_dst, Ls, 16, 64, npg * 16), reps, 2, fl_)
            row_["repage_GBps"], row_["repage_us"] = (pls + nd * Ls * shape.C * 4 * row) / m / 1e3, m
            m, bst = _events(torch, lambda: kv.kv_repage(ctx, d_src, ids_s, d_dst, dst64, Ls, npg * 16), reps, 2, fl_)
            row_["repage_fused_GBps"], row_["repage_fused_us"] = (pls + nd * Ls * shape.C * 4 * row) / m / 1e3, m
            reps_h = 7 if pls <= (1 << 30) else 3
            m, bst = _events(torch, lambda: kv.kv_offload(ctx, desc, Ls, ids, hp, pls), reps_h, 1)
            row_["offload_GBps"], row_["offload_us"], row_["offload_mode"] = pls / m / 1e3, m, ctx.stat(kv.KV_STAT_LAST_HOST_MODE)
            m, bst = _events(torch, lambda: kv.kv_reload(ctx, hp, pls, dst, desc, Ls, T, T, npg * T), reps_h, 1)
            row_["reload_GBps"], row_["reload_us"] = pls / m / 1e3, m
            row_["pack_pct_hbm_peak"] = 100 * row_["pack_GBps"] / hbm
            row_["offload_pct_link_peak"] = 100 * row_["offload_GBps"] / d2h
            row_["reload_pct_link_peak"] = 100 * row_["reload_GBps"] / h2d
            sweep.append(row_)
        del bufS
        first80 = next((r["MiB"] for r in sweep if r["pack_pct_hbm_peak"] >= 80), None)
        recs.append({"config": "5 sweep", "op": "1 MiB - 8 GiB, layer_count 32", "rows": sweep,
                     "smallest_MiB_reaching_80pct_hbm_pack": first80})
    finally:
        torch.cuda.synchronize()
        if hp is not None:
            kv.kv_host_free(hp)

    try:
        import pynvml
        pynvml.nvmlInit()
        driver = pynvml.nvmlSystemGetDriverVersion()
        driver = driver.decode() if isinstance(driver, bytes) else driver
    except Exception:
        driver = None
    peaks["peak_source"] = "MEASURED_PEAKS.json hbm_gbs (torch copy_, read+write)" if hbm_peak else "D2D copy measured in this run"
    peaks["nominal_hbm_GBps"] = NOMINAL_HBM_GBPS
    out = {"peaks": peaks, "records": recs, "gpu": torch.cuda.get_device_name(0), "driver": driver,
           "cuda": torch.version.cuda, "cores": len(os.sched_getaffinity(0))}
    os.makedirs(out_dir, exist_ok=True)
    with open(os.path.join(out_dir, "report.json"), "w") as f:
        json.dump(out, f, indent=1)
    # compact summary for the bench line
    return {"peaks": peaks,
            "summary": [{k: r[k] for k in ("config", "op", "mode", "GBps", "pct_of_measured_hbm_peak", "pct_of_link_peak", "verified") if k in r}
                        for r in recs if "GBps" in r],
            "file": os.path.join(out_dir, "report.json")}


def markdown(rep: dict) -> str:
    """Summary tables of a report.json (what profiles/*_report_summary.md holds)."""
    pk = rep["peaks"]
    out = [f"Peaks measured in the same run: D2D copy {pk['hbm_copy_GBps_this_run']:.0f} GB/s (read+write), pinned H2D "
           f"{pk['h2d_GBps']:.1f} GB/s, D2H {pk['d2h_GBps']:.1f} GB/s, both at once {pk.get('duplex_memcpy_GBps', 0):.1f} GB/s; denominator for HBM fractions: "
           f"{pk['hbm_peak_GBps']:.1f} GB/s (MEASURED_PEAKS.json). GPU: {rep.get('gpu')}; host cores: {rep.get('cores')}.", "",
           "| config | op | mode | payload MiB | median us | GB/s | % of peak | verified |",
           "|---|---|---|---:|---:|---:|---:|---|"]
    for r in rep["records"]:
        if "time_us_median" in r:
            pct = (f"{r['pct_of_measured_hbm_peak']:.1f} (HBM)" if "pct_of_measured_hbm_peak" in r
                   else f"{r['pct_of_link_peak']:.1f} (link)")
            out.append(f"| {r['config']} | {r['op']} | {r['mode']} | {r['payload_bytes'] / 2**20:.1f} | "
                       f"{r['time_us_median']:.1f} | {r['GBps']:.1f} | {pct} | {r.get('verified', '')} |")
        elif "time_us_total" in r:
            out.append(f"| {r['config']} | {r['op']} | {r['mode']} | {r['payload_bytes'] / 2**20:.0f} | "
                       f"{r['time_us_total']:.0f} (total) | reload {r['reload_GBps']:.1f} / offload {r['offload_GBps']:.1f} | "
                       f"{r['pct_of_link_peak_reload']:.1f} (link, reload) | turn 50: {r['turn50_reload_pages']} pages in "
                       f"{r['turn50_reload_us'] / 1e3:.1f} ms |")
    lw = [r for r in rep["records"] if "first_layer_us" in r]
    if lw:
        out += ["", "Layer-by-layer reload of a layer-first host buffer (kv_reload_layerwise, 768 MiB, 48 layers; host wall clock from the "
                    "call to the flag seen in mapped pinned memory):", "",
                "| mode | first layer usable after us | last layer after us | GB/s |", "|---|---:|---:|---:|"]
        for r in lw:
            out.append(f"| {r['mode']} | {r['first_layer_us']:.0f} | {r['last_layer_us']:.0f} | {r['GBps']:.1f} |")
    ch = [r for r in rep["records"] if "chain_us_median" in r]
    if ch:
        out += ["", "Chained paged hashing (kv_chain_hash: digest launch + link launch, events around the call; the chain is serial, "
                    "so the floor of a call is its LONGEST chain x 16 dependent xor/multiply steps):", "",
                "| input | sessions | tokens | ids | longest chain | median us | M ids/s | ns per link of the longest chain |"
                + (" oracle 1 thread us | oracle all cores us |" if "chain_oracle" in rep else ""),
                "|---|---:|---:|---:|---:|---:|---:|---:|" + ("---:|---:|" if "chain_oracle" in rep else "")]
        for r in ch:
            o = rep.get("chain_oracle", {}).get(r["op"])
            out.append(f"| {r['op']} | {r['sessions']} | {r['tokens']} | {r['pages']} | {r['longest_chain_pages']} | "
                       f"{r['chain_us_median']:.1f} | {r['Mpages_per_s']:.1f} | {r['ns_per_link_longest_chain']:.1f} |"
                       + (f" {o['us_1thread']:.0f} | {o['us_all_cores']:.0f} ({o['cores']}) |" if o else ""))
    for r in rep["records"]:
        if "rows" not in r:
            continue
        out += ["", f"{r['config']}: {r['op']} (isolated calls; L2 flushed clean up to 2 GiB):", "",
                "| MiB | pack us | pack GB/s | % HBM | unpack GB/s | re-page 16->64 GB/s | fused re-page GB/s | offload GB/s (mode) | % link | reload GB/s | % link |",
                "|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|"]
        for w in r["rows"]:
            mode = {1: "direct", 2: "staged"}.get(w.get("offload_mode"), "?")
            out.append(f"| {w['MiB']} | {w['pack_us']:.1f} | {w['pack_GBps']:.0f} | {w['pack_pct_hbm_peak']:.1f} | "
                       f"{w['unpack_GBps']:.0f} | {w['repage_GBps']:.0f} | {w.get('repage_fused_GBps', 0):.0f} | "
                       f"{w['offload_GBps']:.1f} ({mode}) | {w['offload_pct_link_peak']:.1f} | {w['reload_GBps']:.1f} | "
                       f"{w['reload_pct_link_peak']:.1f} |")
        out += ["", f"Smallest size reaching 80 % of the HBM peak (pack, isolated call): "
                    f"{r.get('smallest_MiB_reaching_80pct_hbm_pack')} MiB."]
    return "\n".join(out) + "\n"


if __name__ == "__main__":  # python -m paper_2606_31093_b200.report gpurun_out/report.json
    import sys

    with open(sys.argv[1]) as f:
        sys.stdout.write(markdown(json.load(f)))
