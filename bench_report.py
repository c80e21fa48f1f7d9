"""bench_report.py -- measurement harness beside bench.py (SURVEY.md 8(d) "Report schema"; not part of the library).

Two entry points, both called by bench.py with the bench's own 96 GiB pool:

  compact(...)  what the DEFAULT `python bench.py` line carries besides the configs[1] headline: pinned cudaMemcpyAsync
                peaks of the host link measured in the same run (`roofline_host`), and `per_config` -- device-timed
                GB/s and fraction of the HBM peak for BASELINE.json configs[2] (turn 50), configs[3] (26.5 GiB batched),
                configs[4] (exact and ragged: pack, re-paging unpack, fused re-page) and six points of the 1 MiB-8 GiB
                sweep, every record with a `bit_exact` flag.
  run(...)      `python bench.py --report`: every config x op x mode -> gpurun_out/report.json; markdown() prints the
                tables kept under profiles/.

Every record carries `verified` / `bit_exact`: True or False, never blank.  The checks here are written with plain
torch indexing (index_select / reshape / permute on the pool's slabs): they share nothing with the library and do not
touch oracle/ (parity against the oracle is the business of tests/; bench.py may run the oracle only in its
cpu_baseline leg).  Destinations are poisoned before the timed calls, so a transfer that delivers nothing fails.

Conventions: device-side GB/s = (bytes read + bytes written) / time = 2*payload/time (re-paging with padding:
n_tokens*tok read + n_dst*page written); host tier GB/s = payload/time against the pinned cudaMemcpyAsync peak measured
in the same run.
"""
from __future__ import annotations

import json
import os
import time

import numpy as np

from paper_2606_31093_b200 import kvtier as kv
from paper_2606_31093_b200 import workloads as W

# Isolated calls up to this payload run on a cold AND clean L2 (write 512 MiB, then read 512 MiB).
# asks for the flush below 256 MiB; up to 2 GiB the previous repetition's ~126 MB of dirty lines would otherwise be
# written back inside the timed call (~19 us: 20 % of a 256 MiB transfer), so the flush is kept on to 2 GiB.
FLUSH_UP_TO = 2 << 30
NOMINAL_HBM_GBPS = 7700.0  # HBM3e on B200 as the task statement quotes it (~7.7 TB/s); the measured copy peak is the bar
GATE_CYCLES = 400_000      # ~200 us of torch.cuda._sleep: long enough for the host to queue the call behind it
LC_STEP = 11               # checks compare ALL pages of every 11th (layer, K|V) slab (9 of the 96)


def _events(torch, fn, reps, warm, flush=None, gate=False):
    """Median / best duration in us of `fn` between two CUDA events on the current stream.
    `flush` = (w, r): write 512 MiB then read another 512 MiB before every timed call, so the 126 MB
    L2 is cold AND clean -- a write-only flush leaves up to an L2's worth of dirty lines whose
    write-back (~20 us of DRAM time) would be billed to the timed call.
    `gate`: a ~200 us spin kernel is enqueued before the first event, so the host has already queued the call and
    the closing event when the GPU gets there: the interval is then what the DEVICE needs for an isolated call
    (event -> launch from the queue -> kernel -> event), with the host's cost of issuing the call taken out."""
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    stream.synchronize()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush[0].fill_(1)
            flush[1].view(torch.int64).sum()
        if gate:
            torch.cuda._sleep(GATE_CYCLES)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fn()
        b.record(stream)
        stream.synchronize()
        ts.append(a.elapsed_time(b) * 1e3)  # us
    return float(np.median(ts)), float(np.min(ts))


def _back_to_back(torch, fn, reps, warm):
    """us per call of `reps` calls issued back to back between two events (the bench's headline convention)."""
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    stream.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(reps):
        fn()
    b.record(stream)
    stream.synchronize()
    return a.elapsed_time(b) * 1e3 / reps


# ------------------------------------------------------------------------------------------------
# torch-only checks (no library code, no oracle)
# ------------------------------------------------------------------------------------------------
class Checker:
    def __init__(self, torch, slabs, shape, lc_step=LC_STEP):
        self.t, self.slabs, self.shape, self.step = torch, slabs, shape, lc_step

    def idx(self, ids):
        return self.t.as_tensor(np.asarray(ids, dtype=np.int64), device="cuda")

    def lcs(self, layers=None):
        return range(0, (layers or self.shape.L) * self.shape.C, self.step)

    def rows(self, lc, ids, P=None, row=None, hnd=None, slabs=None):
        """Pages `ids` of slab lc as [n][row] bytes in NHD-linear order.  hnd = (H, T, drow): the pool's pages are
        [head][token][dim] and are permuted to [token][head][dim] here."""
        P, row = P or self.shape.P, row or self.shape.row_bytes
        s = (slabs or self.slabs)[lc][:P * row]
        if hnd is None:
            return s.view(P, row).index_select(0, self.idx(ids))
        H, T, drow = hnd
        return s.view(P, H, T, drow).index_select(0, self.idx(ids)).permute(0, 2, 1, 3).reshape(len(ids), row)

    def pack_ok(self, buf, ids, layers=None, P=None, row=None, hnd=None, layer_first=False, slabs=None):
        """buffer == gather of the pool's pages (page-first [page][lc][row] or layer-first [lc][page][row])."""
        row_b = row or self.shape.row_bytes
        LC = (layers or self.shape.L) * self.shape.C
        n = len(ids)
        if n == 0:
            return True
        v = buf[:n * LC * row_b]
        v = v.view(LC, n, row_b) if layer_first else v.view(n, LC, row_b)
        for lc in self.lcs(layers):
            got = v[lc] if layer_first else v[:, lc]
            if not self.t.equal(got, self.rows(lc, ids, P, row, hnd, slabs)):
                return False
        return True

    unpack_ok = pack_ok  # same page size: pool page ids[p] == buffer page p

    def poison(self, ids, P=None, row=None, layers=None, slabs=None):
        """Overwrite pages `ids` of the checked slabs, so that a scatter that writes nothing cannot pass."""
        P, row = P or self.shape.P, row or self.shape.row_bytes
        for lc in self.lcs(layers):
            (slabs or self.slabs)[lc][:P * row].view(P, row).index_fill_(0, self.idx(ids), 0xEE)

    def repage_ok(self, src_rows, n_tokens, Ts, dst_slabs, dst_P, Td, dst_ids, lc):
        """Token stream of `src_rows` ([n_src][Ts*tokrow], NHD) re-paged to pages of Td tokens, zero-padded tail,
        == pages dst_ids of dst_slabs[lc]."""
        tokrow = self.shape.tokrow_bytes
        n_dst = -(-int(n_tokens) // Td)
        exp = self.t.zeros(n_dst * Td, tokrow, dtype=self.t.uint8, device="cuda")
        exp[:n_tokens] = src_rows.reshape(-1, tokrow)[:n_tokens]
        got = dst_slabs[lc][:dst_P * Td * tokrow].view(dst_P, Td * tokrow).index_select(0, self.idx(dst_ids))
        return bool(self.t.equal(got, exp.view(n_dst, Td * tokrow)))

    def host_equals_device(self, hp, dev, n_pages, layers=None, row=None):
        """Pinned host buffer (page-first) == device buffer, compared on the checked slabs (strided numpy views of
        the host buffer: 9/96 of the bytes cross the link again)."""
        row_b = row or self.shape.row_bytes
        LC = (layers or self.shape.L) * self.shape.C
        if n_pages == 0:
            return True
        hv = kv.host_view(hp, n_pages * LC * row_b).reshape(n_pages, LC, row_b)
        dv = dev[:n_pages * LC * row_b].view(n_pages, LC, row_b)
        for lc in self.lcs(layers):
            if not self.t.equal(self.t.from_numpy(np.ascontiguousarray(hv[:, lc])).cuda(), dv[:, lc]):
                return False
        return True


def link_peaks(torch, nbytes=1 << 30, reps=20):
    """Pinned cudaMemcpyAsync peaks of the host link, measured here and now (>= 1 GiB, best of 20, each
    direction) + both directions at once on two streams."""
    a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    h = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    h2 = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    h.zero_()
    h2.zero_()  # touch the pages from the CPU once (first DMA passes over untouched pinned pages are slow)
    m_h2d, t = _events(torch, lambda: a.copy_(h, non_blocking=True), reps, 2)
    h2d = nbytes / t / 1e3
    m_d2h, t = _events(torch, lambda: h.copy_(a, non_blocking=True), reps, 2)
    d2h = nbytes / t / 1e3
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()

    def both():
        cur = torch.cuda.current_stream()
        sa.wait_stream(cur)
        sb.wait_stream(cur)
        with torch.cuda.stream(sa):
            h.copy_(a, non_blocking=True)
        with torch.cuda.stream(sb):
            b.copy_(h2, non_blocking=True)
        cur.wait_stream(sa)
        cur.wait_stream(sb)

    m_dup, t = _events(torch, both, reps, 2)
    duplex = 2 * nbytes / t / 1e3
    # the same bytes as TWO back-to-back copies per direction (the chunking of a staged 768 MiB transfer): with both
    # directions busy every copy boundary costs the link ~0.25 ms on this platform, for plain cudaMemcpyAsync too
    K = 2
    c = nbytes // K // 4096 * 4096

    def both3():
        cur = torch.cuda.current_stream()
        sa.wait_stream(cur)
        sb.wait_stream(cur)
        with torch.cuda.stream(sa):
            for i in range(K):
                h[i * c:(i + 1) * c].copy_(a[i * c:(i + 1) * c], non_blocking=True)
        with torch.cuda.stream(sb):
            for i in range(K):
                b[i * c:(i + 1) * c].copy_(h2[i * c:(i + 1) * c], non_blocking=True)
        cur.wait_stream(sa)
        cur.wait_stream(sb)

    _, t = _events(torch, both3, reps, 2)
    duplex3 = 2 * K * c / t / 1e3
    del a, b, h, h2
    return {"h2d_GBps": h2d, "d2h_GBps": d2h, "duplex_GBps": duplex, "duplex_chunked_GBps": duplex3, "duplex_chunked_copies_each_way": K,
            "bytes": nbytes, "reps": reps,
            "median": {"h2d_GBps": nbytes / m_h2d / 1e3, "d2h_GBps": nbytes / m_d2h / 1e3, "duplex_GBps": 2 * nbytes / m_dup / 1e3,
                       "what": "the same passes, median instead of best (how far the link itself varies from pass to pass)"},
            "how": "pinned cudaMemcpyAsync (torch copy_ non_blocking), best of reps, CUDA events; duplex = D2H and H2D "
                   "of the same size on two streams, 2*bytes / time; duplex_chunked = the same bytes issued as "
                   "two back-to-back copies per direction (what chunking alone costs plain copies when both directions are busy)"}


def empty_launch_us(torch, reps=30):
    """What a launch that moves nothing costs between two events on this box: a one-element torch fill_ (a store-only
    kernel of one thread), after the same L2 flush as the sweep's calls.  With the flush kernels queued ahead the host
    has issued everything before the GPU gets there, so this is device time: event -> launch -> event."""
    flag = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = (torch.empty(64 << 20, dtype=torch.uint8, device="cuda"), torch.zeros(64 << 20, dtype=torch.uint8, device="cuda"))
    med, _ = _events(torch, lambda: flag.fill_(1), reps, 3, flush)
    return med


def sweep_row(torch, ctx, desc, shape, chk, buf, src, flush, npg, rng, hbm, t_launch, layers=32, reps=None):
    """One point of the transfer-size sweep (pack of npg pages of `layers` layers = npg MiB): isolated call on a cold,
    clean L2 (the flush kernels are queued ahead of it, so the host's cost of issuing the call is hidden: device time),
    against (a) the floor empty launch + 2*payload/peak and (b) a plain contiguous copy of the same bytes (torch copy_
    = cudaMemcpyAsync device to device, `src` -> `buf`) timed the same way: what the hardware gives a transfer of that
    size when nothing has to be gathered."""
    pg = layers * shape.C * shape.row_bytes
    pls = npg * pg
    ids = rng.choice(shape.P, npg, replace=False).astype(np.int32)
    reps = reps or (20 if pls <= (256 << 20) else 7)
    fl_ = flush if pls <= FLUSH_UP_TO else None
    cm, _ = _events(torch, lambda: buf[:pls].copy_(src[:pls]), reps, 2, fl_)
    buf[:pls].fill_(0xEE)
    m, bst = _events(torch, lambda: kv.kv_pack(ctx, desc, layers, ids, buf), reps, 2, fl_)
    floor = t_launch + 2 * pls / hbm / 1e3
    return {"MiB": pls >> 20, "n_pages": int(npg), "pack_us": m, "pack_us_best": bst,
            "pack_GBps": 2 * pls / m / 1e3, "pack_frac_hbm": 2 * pls / m / 1e3 / hbm,
            "floor_us": floor, "vs_floor": m / floor,
            "plain_copy_us": cm, "plain_copy_frac_hbm": 2 * pls / cm / 1e3 / hbm, "vs_plain_copy": m / cm,
            "kernel": {1: "bulk", 2: "vec", 3: "elem", 4: "shot"}.get(ctx.stat(kv.KV_STAT_LAST_KERNEL), "?"),
            "bit_exact": bool(chk.pack_ok(buf, ids, layers=layers)), "_ids": ids}


# ------------------------------------------------------------------------------------------------
# the compact per-config block of the default bench line
# ------------------------------------------------------------------------------------------------
def compact(ctx, desc, shape, slabs, seed, hbm_peak):
    import torch

    L, T, page, row = shape.L, shape.T, shape.page_bytes, shape.row_bytes
    chk = Checker(torch, slabs, shape)
    rng = np.random.default_rng(seed + 177)
    out = []

    def rec(config, op, payload, traffic, us, ok, **kw):
        r = {"config": config, "op": op, "payload_MiB": payload / 2**20, "us": us, "GBps": traffic / us / 1e3,
             "frac_hbm": traffic / us / 1e3 / hbm_peak, "bit_exact": bool(ok)}
        r.update(kw)
        out.append(r)

    # ---- configs[3]: 64 requests, 18,091 pages, 26.5 GiB, one batched launch each way ------------------------
    b4 = W.batch_case(seed, shape=shape)
    counts = np.diff(b4.req_offsets)
    total = int(b4.req_offsets[-1]) * page
    big = torch.empty(total, dtype=torch.uint8, device="cuda")
    bufs = [big[int(b4.req_offsets[r]) * page:int(b4.req_offsets[r + 1]) * page] for r in range(len(counts))]
    big[::4096].fill_(0xEE)
    l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
    us = _back_to_back(torch, lambda: kv.kv_pack_batched(ctx, desc, L, b4.src_ids, b4.req_offsets, bufs), 3, 1)
    rec("configs[3] concurrent batch (64 requests, 18,091 pages)", "kv_pack_batched", total, 2 * total, us,
        chk.pack_ok(big, b4.src_ids), launches_per_call=(ctx.stat(kv.KV_STAT_LAUNCHES) - l0) // 4)
    chk.poison(b4.dst_ids)
    l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
    us = _back_to_back(torch, lambda: kv.kv_unpack_batched(ctx, bufs, b4.dst_ids, b4.req_offsets, counts * T, desc, L, T, T), 3, 1)
    rec("configs[3] concurrent batch (64 requests, 18,091 pages)", "kv_unpack_batched", total, 2 * total, us,
        chk.unpack_ok(big, b4.dst_ids), launches_per_call=(ctx.stat(kv.KV_STAT_LAUNCHES) - l0) // 4)

    # ---- configs[2], turn 50: the matched prefix of the 50-turn session, device side --------------------------
    turns = W.session_turns(seed, T=T)
    n50 = turns[-1].n_matched_pages
    ids50 = rng.choice(shape.P, n50, replace=False).astype(np.int32)
    buf50 = big[:n50 * page]  # holds packed pages of configs[3]: any bytes will do for a scatter
    chk.poison(ids50)
    us = _back_to_back(torch, lambda: kv.kv_unpack(ctx, buf50, ids50, desc, L, T, T, n50 * T), 5, 2)
    rec(f"configs[2] 50-turn session, turn 50 ({n50} pages)", "kv_unpack (device copy of the host buffer)", n50 * page,
        2 * n50 * page, us, chk.unpack_ok(buf50, ids50))

    # ---- configs[4]: cross-role 16 -> 64 re-paging, exact and ragged ---------------------------------------------
    half = (shape.P // 2) * row
    s_src, s_dst = shape.with_(P=shape.P // 2), shape.with_(T=64, P=shape.P // 8)
    src_slabs, dst_slabs = [s[:half] for s in slabs], [s[half:] for s in slabs]
    d_src = kv.PoolDesc(src_slabs, L, shape.C, s_src.P, 16, shape.H, shape.D, shape.e)
    d_dst = kv.PoolDesc(dst_slabs, L, shape.C, s_dst.P, 64, shape.H, shape.D, shape.e)
    for ragged in (False, True):
        c5 = W.crossrole_case(seed, ragged=ragged, src_shape=s_src, dst_shape=s_dst)
        R5 = len(c5.n_tokens)
        pl5 = int(c5.src_offsets[-1]) * page
        bufs5 = [big[int(c5.src_offsets[r]) * page:int(c5.src_offsets[r + 1]) * page] for r in range(R5)]
        name = "configs[4] cross-role 16->64, 32 requests" + (" (ragged tails)" if ragged else " (2,048 tokens each)")
        big[:pl5:4096].fill_(0xEE)
        us = _back_to_back(torch, lambda: kv.kv_pack_batched(ctx, d_src, L, c5.src_ids, c5.src_offsets, bufs5), 5, 2)
        rec(name, "kv_pack_batched (T=16)", pl5, 2 * pl5, us, chk.pack_ok(big, c5.src_ids, P=s_src.P, slabs=src_slabs))
        wr = int(c5.dst_offsets[-1]) * s_dst.page_bytes
        rd = int(c5.n_tokens.sum()) * shape.tok_bytes

        def repage_all_ok(from_buffer):
            for lc in chk.lcs():
                for r in range(R5):
                    so, se = int(c5.src_offsets[r]), int(c5.src_offsets[r + 1])
                    if from_buffer:
                        rows = bufs5[r].view(se - so, L * shape.C, row)[:, lc]
                    else:
                        rows = chk.rows(lc, c5.src_ids[so:se], P=s_src.P, slabs=src_slabs)
                    if not chk.repage_ok(rows, int(c5.n_tokens[r]), 16, dst_slabs, s_dst.P, 64,
                                         c5.dst_ids[c5.dst_offsets[r]:c5.dst_offsets[r + 1]], lc):
                        return False
            return True

        chk.poison(c5.dst_ids, P=s_dst.P, row=s_dst.row_bytes, slabs=dst_slabs)
        us = _back_to_back(torch, lambda: kv.kv_unpack_batched(ctx, bufs5, c5.dst_ids, c5.dst_offsets, c5.n_tokens,
                                                               d_dst, L, 16, 64), 5, 2)
        rec(name, "kv_unpack_batched re-paging 16->64", wr, rd + wr, us, repage_all_ok(True))
        chk.poison(c5.dst_ids, P=s_dst.P, row=s_dst.row_bytes, slabs=dst_slabs)
        us = _back_to_back(torch, lambda: kv.kv_repage_batched(ctx, d_src, c5.src_ids, c5.src_offsets, d_dst, c5.dst_ids,
                                                               c5.dst_offsets, c5.n_tokens, L), 5, 2)
        rec(name, "kv_repage_batched fused pool->pool 16->64", wr, rd + wr, us, repage_all_ok(False))

    # ---- a config-3 turn on the device as ONE launch (kv_submit): scatter the matched prefix, extend the retained
    # partial page copy-on-write, gather the pages that became full ------------------------------------------------
    tk = turns[9]  # turn 10: ~600 matched pages
    n_m, n_new = tk.n_matched_pages, tk.cum_tokens // T - tk.n_matched_pages
    perm = rng.permutation(shape.P).astype(np.int32)
    ids_m, ids_new, old_id, new_id = perm[:n_m], perm[n_m:n_m + n_new], int(perm[n_m + n_new]), int(perm[n_m + n_new + 1])
    n_old, n_app = 5, 9
    app = torch.randint(0, 256, (L * shape.C * n_app * shape.tokrow_bytes,), dtype=torch.uint8, device="cuda")
    src_t, dst_t = big[:n_m * page], big[(n_m + 8) * page:(n_m + 8 + n_new) * page]
    ops = [kv.op_unpack(src_t, ids_m, n_m * T), kv.op_cow_append(old_id, new_id, n_old, app, n_app),
           kv.op_pack(ids_new, dst_t)]
    pl_t = (n_m + n_new) * page + L * shape.C * (n_old + n_app) * shape.tokrow_bytes

    def three():
        kv.kv_unpack(ctx, src_t, ids_m, desc, L, T, T, n_m * T)
        kv.kv_cow_append(ctx, desc, L, old_id, new_id, n_old, app, n_app)
        kv.kv_pack(ctx, desc, L, ids_new, dst_t)

    flush = (torch.empty(512 << 20, dtype=torch.uint8, device="cuda"), torch.zeros(512 << 20, dtype=torch.uint8, device="cuda"))
    l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
    us3, _ = _events(torch, three, 7, 2, flush)
    l1 = ctx.stat(kv.KV_STAT_LAUNCHES)
    chk.poison(ids_m)
    dst_t.fill_(0xEE)
    us1, _ = _events(torch, lambda: kv.kv_submit(ctx, desc, L, ops), 7, 2, flush)
    l2 = ctx.stat(kv.KV_STAT_LAUNCHES)
    ok = chk.unpack_ok(src_t, ids_m) and chk.pack_ok(dst_t, ids_new)
    for lc in chk.lcs():  # the copy-on-write page: n_old tokens of the old page, then the append block's rows
        newp, oldp = chk.rows(lc, [new_id]).view(T, -1), chk.rows(lc, [old_id]).view(T, -1)
        ok = ok and bool(torch.equal(newp[:n_old], oldp[:n_old])) and \
            bool(torch.equal(newp[n_old:n_old + n_app], app.view(L * shape.C, n_app, -1)[lc]))
    rec(f"configs[2] turn 10 on the device: unpack {n_m} pages + CoW append + pack {n_new} pages", "kv_submit (ONE launch)",
        pl_t, 2 * pl_t, us1, ok, launches_per_call=(l2 - l1) // 9, isolated=True,
        three_calls_us=us3, three_calls_launches=(l1 - l0) // 9)

    # ---- six points of the 1 MiB - 8 GiB sweep (layer_count 32 => 1 MiB pages), isolated calls -------------------
    t_launch = empty_launch_us(torch)
    sweep = []
    for npg in (1, 16, 64, 256, 1024, 8192):
        r = sweep_row(torch, ctx, desc, shape, chk, big, big[13 << 30:], flush, npg, rng, hbm_peak, t_launch)
        r.pop("_ids")
        sweep.append(r)
    del big, bufs, flush
    return {"records": out, "sweep": sweep, "empty_launch_us": t_launch,
            "check": f"bit_exact: torch index_select / reshape compare of ALL pages on every {LC_STEP}th (layer,K|V) slab, "
                     "destinations poisoned before the timed calls",
            "timing": "records: calls issued back to back between two CUDA events (us per call); sweep and the kv_submit "
                      "turn: isolated calls on a cold, clean L2 (the flush kernels are queued ahead of the call, so the host's cost "
                      "of issuing it is hidden: device time); floor = empty launch (one-element fill_) + 2*payload/peak; "
                      "plain_copy = torch copy_ (cudaMemcpyAsync D2D) of the same bytes, contiguous, timed the same way"}


# ------------------------------------------------------------------------------------------------
# the full report
# ------------------------------------------------------------------------------------------------
def run(ctx, desc, shape, slabs, seed=0, out_dir="gpurun_out", hbm_peak=None):
    import torch

    rng = np.random.default_rng(seed + 77)
    recs = []
    flush = (torch.empty(512 << 20, dtype=torch.uint8, device="cuda"),
             torch.zeros(512 << 20, dtype=torch.uint8, device="cuda"))
    chk = Checker(torch, slabs, shape)

    # ---- peaks measured in this run -----------------------------------------------------------
    N = 1 << 30
    a = torch.empty(N, dtype=torch.uint8, device="cuda")
    b = torch.empty(N, dtype=torch.uint8, device="cuda")
    _, t = _events(torch, lambda: b.copy_(a), 10, 3)
    d2d = 2 * N / t / 1e3
    del a, b
    lp = link_peaks(torch)
    h2d, d2h = lp["h2d_GBps"], lp["d2h_GBps"]
    peaks = {"hbm_copy_GBps_this_run": d2d, "h2d_GBps": h2d, "d2h_GBps": d2h, "duplex_memcpy_GBps": lp["duplex_GBps"],
             "hbm_peak_GBps": hbm_peak or d2d}
    hbm = peaks["hbm_peak_GBps"]
    duplex = lp["duplex_GBps"]

    def rec(cfg, op, mode, payload, traffic, n_pages, fn, reps=7, warm=2, link=None, check=None, before=None):
        if before is not None:
            before()  # poison the destination: the check below then proves that the timed calls delivered
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
        torch.cuda.synchronize()
        r["verified"] = bool(check())  # every record is checked: True or False, never blank
        recs.append(r)
        return r

    L, T = shape.L, shape.T
    LC, row, page = shape.L * shape.C, shape.row_bytes, shape.page_bytes

    # ---- config 1: Tiny (launch-bound; correctness config) --------------------------------------
    tc = W.tiny_case(seed)
    ts_ = tc.shape
    tslabs = [torch.randint(0, 256, (ts_.P * ts_.row_bytes,), dtype=torch.uint8, device="cuda") for _ in range(ts_.L * ts_.C)]
    tdesc = kv.PoolDesc(tslabs, ts_.L, ts_.C, ts_.P, ts_.T, ts_.H, ts_.D, ts_.e)
    tchk = Checker(torch, tslabs, ts_, lc_step=1)
    tbuf = torch.empty(37 * ts_.page_bytes, dtype=torch.uint8, device="cuda")
    pl = 37 * ts_.page_bytes
    rec("1 tiny", "pack", "device", pl, 2 * pl, 37, lambda: kv.kv_pack(ctx, tdesc, ts_.L, tc.src_ids, tbuf), reps=20,
        before=lambda: tbuf.fill_(0xEE), check=lambda: tchk.pack_ok(tbuf, tc.src_ids))
    rec("1 tiny", "unpack", "device", pl, 2 * pl, 37,
        lambda: kv.kv_unpack(ctx, tbuf, tc.dst_ids, tdesc, ts_.L, ts_.T, ts_.T, 37 * ts_.T), reps=20,
        before=lambda: tchk.poison(tc.dst_ids), check=lambda: tchk.unpack_ok(tbuf, tc.dst_ids))

    # ---- config 2: single-request prefix ---------------------------------------------------------
    c2 = W.prefix_case(seed, shape=shape)
    n = len(c2.src_ids)
    pl = n * page
    buf = torch.empty(pl, dtype=torch.uint8, device="cuda")
    poison_buf = lambda: buf.fill_(0xEE)
    rec("2 prefix", "pack", "device", pl, 2 * pl, n, lambda: kv.kv_pack(ctx, desc, L, c2.src_ids, buf),
        reps=20, warm=3, before=poison_buf, check=lambda: chk.pack_ok(buf, c2.src_ids))
    rec("2 prefix", "unpack", "device", pl, 2 * pl, n,
        lambda: kv.kv_unpack(ctx, buf, c2.dst_ids, desc, L, T, T, n * T), reps=20, warm=3,
        before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids))
    # What the paper's "PyTorch fallback for unsupported layouts" would pay for the same two transfers on
    # this GPU: plain torch indexing, one gather / scatter per (layer, K|V) slab (96 launches each) -- context beside the
    # kernel's figure, not a baseline the library uses (it has no PyTorch path).
    idx_src = torch.as_tensor(c2.src_ids.astype(np.int64), device="cuda")
    idx_dst = torch.as_tensor(c2.dst_ids.astype(np.int64), device="cuda")
    slab_rows = [s_.view(shape.P, row) for s_ in slabs]
    buf3 = buf.view(n, LC, row)
    tbuf = {}

    def torch_pack():
        tbuf["x"] = torch.stack([sr.index_select(0, idx_src) for sr in slab_rows], dim=1)  # [page][layer*kv][row]: page-first

    def torch_unpack():
        for lc_, sr in enumerate(slab_rows):
            sr.index_copy_(0, idx_dst, buf3[:, lc_])

    rec("2 prefix", "pack by torch index_select + stack (the paper's PyTorch-fallback shape)", "torch, 97 launches", pl, 2 * pl, n,
        torch_pack, reps=7, warm=2, check=lambda: bool(torch.equal(tbuf["x"].view(-1), buf)))
    tbuf.clear()
    rec("2 prefix", "unpack by torch index_copy_ per slab (the paper's PyTorch-fallback shape)", "torch, 96 launches", pl, 2 * pl, n,
        torch_unpack, reps=7, warm=2, before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids))
    # ---- fragmentation (SURVEY.md 8(d) "structure of the workloads" (i)): the same 512 pages in runs of r
    # consecutive ids (run starts drawn at random, runs disjoint); r = 1 is the aged pool of the configs,
    # r = n a fresh one.  Consecutive pages are adjacent within a slab but stay a page apart in the buffer,
    # so segments do not grow: only DRAM/TLB locality of the pool side changes.
    for r_len in (1, 4, 16, 64, n):
        starts = rng.choice(shape.P // r_len, n // r_len, replace=False) * r_len
        ids_r = (starts[:, None] + np.arange(r_len)[None, :]).reshape(-1).astype(np.int32)
        rec("2 prefix, ids in runs", f"pack, runs of {r_len}", "device", pl, 2 * pl, n,
            lambda: kv.kv_pack(ctx, desc, L, ids_r, buf), reps=20, warm=3, before=poison_buf,
            check=lambda: chk.pack_ok(buf, ids_r))
        rec("2 prefix, ids in runs", f"unpack, runs of {r_len}", "device", pl, 2 * pl, n,
            lambda: kv.kv_unpack(ctx, buf, ids_r, desc, L, T, T, n * T), reps=20, warm=3,
            before=lambda: chk.poison(ids_r), check=lambda: chk.unpack_ok(buf, ids_r))

    # ---- tensor-parallel head partitions ("head partitions"): the same slabs read as pools of 1 and 2
    # KV heads per rank -> 4 KiB / 8 KiB rows, 4x / 2x the pages for the same 768 MiB
    for Hp in (1, 2):
        f = shape.H // Hp
        desc_p = kv.PoolDesc(slabs, L, shape.C, shape.P * f, T, Hp, shape.D, shape.e)
        ids_p = rng.choice(shape.P * f, n * f, replace=False).astype(np.int32)
        dst_p = rng.choice(shape.P * f, n * f, replace=False).astype(np.int32)
        rec(f"2 prefix, {Hp} KV head(s) per rank", f"pack ({4 * Hp} KiB rows)", "device", pl, 2 * pl, n * f,
            lambda: kv.kv_pack(ctx, desc_p, L, ids_p, buf), reps=20, warm=3, before=poison_buf,
            check=lambda: chk.pack_ok(buf, ids_p, P=shape.P * f, row=row // f))
        rec(f"2 prefix, {Hp} KV head(s) per rank", f"unpack ({4 * Hp} KiB rows)", "device", pl, 2 * pl, n * f,
            lambda: kv.kv_unpack(ctx, buf, dst_p, desc_p, L, T, T, n * f * T), reps=20, warm=3,
            before=lambda: chk.poison(dst_p, P=shape.P * f, row=row // f),
            check=lambda: chk.unpack_ok(buf, dst_p, P=shape.P * f, row=row // f))

    # ---- NEXT-2: the same prefix on an HND pool ([head][token][dim] pages; the buffer stays NHD, so the
    # transfer transposes).  Same slabs, HND descriptor; the check permutes the pool's pages with torch.
    desc_h = kv.PoolDesc(slabs, L, shape.C, shape.P, T, shape.H, shape.D, shape.e, order=kv.KV_ORDER_HND)
    hnd = (shape.H, T, shape.D * shape.e)
    for tm, label in ((1, "tensor maps (cp.async.bulk.tensor)"), (0, "lane paths (cp.async gather / STG.128)")):
        ctx.set_option(kv.KV_OPT_TENSOR_MAPS, tm)
        rec("2 prefix, HND pool", "pack", label, pl, 2 * pl, n,
            lambda: kv.kv_pack(ctx, desc_h, L, c2.src_ids, buf), reps=20, warm=3, before=poison_buf,
            check=lambda: chk.pack_ok(buf, c2.src_ids, hnd=hnd))
        rec("2 prefix, HND pool", "unpack", label, pl, 2 * pl, n,
            lambda: kv.kv_unpack(ctx, buf, c2.dst_ids, desc_h, L, T, T, n * T), reps=20, warm=3,
            before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids, hnd=hnd))
        rec("2 prefix, HND pool", "repage HND->HND pool", label, pl, 2 * pl, n,
            lambda: kv.kv_repage(ctx, desc_h, c2.src_ids, desc_h, c2.dst_ids, L, n * T), reps=20, warm=3,
            before=lambda: chk.poison(c2.dst_ids),
            check=lambda: all(torch.equal(chk.rows(lc, c2.src_ids), chk.rows(lc, c2.dst_ids)) for lc in chk.lcs()))
    ctx.set_option(kv.KV_OPT_TENSOR_MAPS, 1)
    kv.kv_pack(ctx, desc, L, c2.src_ids, buf)  # buf = the NHD pack of the prefix again (the host-tier checks compare with it)
    torch.cuda.synchronize()
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
        kv.host_view(hp, host_total)[::4096] = 0  # touch every page once from the CPU
        poison_host = lambda: kv.host_view(hp, pl).__setitem__(slice(0, None, 512), 0xEE)
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged"), (kv.KV_HOST_AUTO, "auto")):
            rec("2 prefix", "offload", name, pl, pl, n,
                lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, mode=mode), reps=7, link=d2h,
                before=poison_host, check=lambda: chk.host_equals_device(hp, buf, n))
            rec("2 prefix", "reload", name, pl, pl, n,
                lambda: kv.kv_reload(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, mode=mode), reps=7, link=h2d,
                before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids))

        # layer-first host buffer (NEXT-2): staged in chunks of whole layers; layer-by-layer reload with flags
        buf_lf = torch.empty(pl, dtype=torch.uint8, device="cuda")
        kv.kv_pack(ctx, desc, L, c2.src_ids, buf_lf, layout=kv.KV_LAYOUT_LAYER_FIRST)
        torch.cuda.synchronize()
        lf_ok = chk.pack_ok(buf_lf, c2.src_ids, layer_first=True)

        def host_lf_ok():  # the layer-first host buffer == the (checked) layer-first device pack, on the checked slabs
            hv = kv.host_view(hp, pl).reshape(LC, n, row)
            dv = buf_lf.view(LC, n, row)
            return lf_ok and all(torch.equal(torch.from_numpy(hv[lc]).cuda(), dv[lc]) for lc in chk.lcs())

        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            rec("2 prefix, layer-first buffer", "offload", name, pl, pl, n,
                lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, mode=mode, layout=kv.KV_LAYOUT_LAYER_FIRST),
                reps=7, link=d2h, before=poison_host, check=host_lf_ok)
            rec("2 prefix, layer-first buffer", "reload", name, pl, pl, n,
                lambda: kv.kv_reload(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, mode=mode,
                                     layout=kv.KV_LAYOUT_LAYER_FIRST), reps=7, link=h2d,
                before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids))
        flp = kv.kv_host_alloc(L * 8)
        fh = kv.host_view(flp, L * 8).view(np.uint64)
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            first, last = [], []
            chk.poison(c2.dst_ids)
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
            torch.cuda.synchronize()
            recs.append({"config": "2 prefix, layer-first buffer", "op": "reload_layerwise", "mode": name,
                         "payload_bytes": int(pl), "first_layer_us": float(np.median(first)),
                         "last_layer_us": float(np.median(last)), "GBps": pl / float(np.median(last)) / 1e3,
                         "timing": "host wall clock from the call to the flag seen in mapped pinned memory",
                         "verified": bool(chk.unpack_ok(buf, c2.dst_ids))})
        kv.kv_host_free(flp)
        del buf_lf

        # a captured STAGED offload / reload replayed from a CUDA graph (copy nodes + one kernel node per chunk)
        ctx.set_option(kv.KV_OPT_RESERVE_STAGING, 0)
        cap_stream = torch.cuda.Stream()
        g_off, g_rel = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
        with torch.cuda.graph(g_off, stream=cap_stream):
            kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, stream=cap_stream)
        cap_mode = {1: "direct", 2: "staged"}.get(ctx.stat(kv.KV_STAT_LAST_HOST_MODE), "?")
        with torch.cuda.graph(g_rel, stream=cap_stream):
            kv.kv_reload(ctx, hp, pl, c2.dst_ids, desc, L, T, T, n * T, stream=cap_stream)
        rec("2 prefix", "offload, CUDA-graph replay", f"auto = {cap_mode} (captured)", pl, pl, n, g_off.replay, reps=7,
            link=d2h, before=poison_host, check=lambda: chk.host_equals_device(hp, buf, n))
        rec("2 prefix", "reload, CUDA-graph replay", f"auto = {cap_mode} (captured)", pl, pl, n, g_rel.replay, reps=7,
            link=h2d, before=lambda: chk.poison(c2.dst_ids), check=lambda: chk.unpack_ok(buf, c2.dst_ids))
        del g_off, g_rel

        # both directions of the link at once: offload on one stream (ctx), reload of ANOTHER buffer on a
        # second stream (ctx2) -- eviction of one session while another is restored.  Peak = two plain
        # cudaMemcpyAsync of the same sizes on the same two streams (link_peaks).
        ctx2 = kv.Ctx(torch.cuda.current_device())
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        kv.kv_offload(ctx, desc, L, c2.src_ids, hp + pl, pl)  # the buffer the reload leg reads
        torch.cuda.synchronize()

        def both(f, g):
            sa.wait_stream(torch.cuda.current_stream())
            sb.wait_stream(torch.cuda.current_stream())
            f()
            g()
            torch.cuda.current_stream().wait_stream(sa)
            torch.cuda.current_stream().wait_stream(sb)

        rec("2 prefix", "offload and reload at once (two ctxs, two streams)", "auto", 2 * pl, 2 * pl, 2 * n,
            lambda: both(lambda: kv.kv_offload(ctx, desc, L, c2.src_ids, hp, pl, stream=sa),
                         lambda: kv.kv_reload(ctx2, hp + pl, pl, c2.dst_ids, desc, L, T, T, n * T, stream=sb)),
            reps=15, link=duplex, before=lambda: (poison_host(), chk.poison(c2.dst_ids)),  # the shared link varies by +-5 % from pass to pass
            check=lambda: chk.host_equals_device(hp, buf, n) and chk.unpack_ok(buf, c2.dst_ids))
        torch.cuda.synchronize()
        ctx2.close()

        # ---- config 3: 50-turn session ------------------------------------------------------------
        turns = W.session_turns(seed, T=T)
        fl = W.FreeList(shape.P, np.random.default_rng(seed))
        stream = torch.cuda.current_stream()
        in_host, moved, per_turn = 0, 0, []
        t_reload = t_offload = 0.0
        session_ok = True
        hv_all = kv.host_view(hp, host_total)
        for tn in turns:
            ids = fl.pop(in_host)
            n_new = tn.cum_tokens // T - in_host
            new_ids = fl.pop(n_new)
            chk.poison(ids)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record(stream)
            kv.kv_reload(ctx, hp, in_host * page, ids, desc, L, T, T, in_host * T)
            e[1].record(stream)
            kv.kv_offload(ctx, desc, L, new_ids, hp + in_host * page, n_new * page)
            e[2].record(stream)
            stream.synchronize()
            r_us, o_us = e[0].elapsed_time(e[1]) * 1e3, e[1].elapsed_time(e[2]) * 1e3
            # every turn checked on the sampled slabs: reloaded pages == the host buffer's prefix, appended host pages
            # == the pool's new pages
            hv3 = hv_all[:(in_host + n_new) * page].reshape(in_host + n_new, LC, row)
            for lc in chk.lcs():
                col = torch.from_numpy(np.ascontiguousarray(hv3[:, lc])).cuda()
                session_ok = session_ok and bool(torch.equal(col[:in_host], chk.rows(lc, ids))) and \
                    bool(torch.equal(col[in_host:], chk.rows(lc, new_ids)))
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
                     "per_turn": per_turn, "verified": bool(session_ok)})
        buf50 = torch.empty(n50 * page, dtype=torch.uint8, device="cuda")
        buf50.random_(0, 256)
        ids50 = fl.pop(n50)
        rec("3 session", "turn-50 unpack from a device copy of the buffer", "device", n50 * page, 2 * n50 * page, n50,
            lambda: kv.kv_unpack(ctx, buf50, ids50, desc, L, T, T, n50 * T), reps=10,
            before=lambda: chk.poison(ids50), check=lambda: chk.unpack_ok(buf50, ids50))
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
        n4 = pl4 // page
        rec("4 batch", "pack_batched", "device", pl4, 2 * pl4, n4,
            lambda: kv.kv_pack_batched(ctx, desc, L, b4.src_ids, b4.req_offsets, bufs), reps=7,
            before=lambda: big[::4096].fill_(0xEE), check=lambda: chk.pack_ok(big, b4.src_ids))
        rec("4 batch", "unpack_batched", "device", pl4, 2 * pl4, n4,
            lambda: kv.kv_unpack_batched(ctx, bufs, b4.dst_ids, b4.req_offsets, counts * T, desc, L, T, T), reps=7,
            before=lambda: chk.poison(b4.dst_ids), check=lambda: chk.unpack_ok(big, b4.dst_ids))
        poison_host4 = lambda: hv_all.__setitem__(slice(0, None, 4096), 0xEE)
        for mode, name in ((kv.KV_HOST_DIRECT, "direct"), (kv.KV_HOST_STAGED, "staged")):
            rec("4 batch", "offload_batched (64 pinned per-request buffers)", name, pl4, pl4, n4,
                lambda: kv.kv_offload_batched(ctx, desc, L, b4.src_ids, b4.req_offsets, hps, host_bytes=sizes, mode=mode),
                reps=3, warm=1, link=d2h, before=poison_host4, check=lambda: chk.host_equals_device(hp, big, n4))
            rec("4 batch", "reload_batched (64 pinned per-request buffers)", name, pl4, pl4, n4,
                lambda: kv.kv_reload_batched(ctx, hps, b4.dst_ids, b4.req_offsets, counts * T, desc, L, T, T,
                                             host_bytes=sizes, mode=mode), reps=3, warm=1, link=h2d,
                before=lambda: chk.poison(b4.dst_ids), check=lambda: chk.unpack_ok(big, b4.dst_ids))

        # ---- config 5: cross-role re-paging 16 -> 64 -------------------------------------------------
        half = (shape.P // 2) * row
        s_src = shape.with_(P=shape.P // 2)
        s_dst = shape.with_(T=64, P=shape.P // 8)
        src_slabs, dst_slabs = [s[:half] for s in slabs], [s[half:] for s in slabs]
        d_src = kv.PoolDesc(src_slabs, L, shape.C, s_src.P, 16, shape.H, shape.D, shape.e)
        d_dst = kv.PoolDesc(dst_slabs, L, shape.C, s_dst.P, 64, shape.H, shape.D, shape.e)
        poison_dst64 = lambda ids: chk.poison(ids, P=s_dst.P, row=s_dst.row_bytes, slabs=dst_slabs)
        for ragged in (False, True):
            c5 = W.crossrole_case(seed, ragged=ragged, src_shape=s_src, dst_shape=s_dst)
            R5 = len(c5.n_tokens)
            pl5 = int(c5.src_offsets[-1]) * page
            bufs5 = [big[int(c5.src_offsets[r]) * page:int(c5.src_offsets[r + 1]) * page] for r in range(R5)]
            name = "5 cross-role ragged" if ragged else "5 cross-role"

            def repage_all_ok(from_buffer, c5=c5, bufs5=bufs5, R5=R5):
                for lc in chk.lcs():
                    for r in range(R5):
                        so, se = int(c5.src_offsets[r]), int(c5.src_offsets[r + 1])
                        rows = bufs5[r].view(se - so, LC, row)[:, lc] if from_buffer else \
                            chk.rows(lc, c5.src_ids[so:se], P=s_src.P, slabs=src_slabs)
                        if not chk.repage_ok(rows, int(c5.n_tokens[r]), 16, dst_slabs, s_dst.P, 64,
                                             c5.dst_ids[c5.dst_offsets[r]:c5.dst_offsets[r + 1]], lc):
                            return False
                return True

            rec(name, "pack_batched (T=16)", "device", pl5, 2 * pl5, pl5 // page,
                lambda: kv.kv_pack_batched(ctx, d_src, L, c5.src_ids, c5.src_offsets, bufs5), reps=10,
                before=lambda: big[:pl5:4096].fill_(0xEE),
                check=lambda: chk.pack_ok(big, c5.src_ids, P=s_src.P, slabs=src_slabs))
            wr = int(c5.dst_offsets[-1]) * s_dst.page_bytes
            rd = int(c5.n_tokens.sum()) * shape.tok_bytes
            rec(name, "unpack_batched re-page 16->64", "device", wr, rd + wr, int(c5.dst_offsets[-1]),
                lambda: kv.kv_unpack_batched(ctx, bufs5, c5.dst_ids, c5.dst_offsets, c5.n_tokens, d_dst, L, 16, 64),
                reps=10, before=lambda: poison_dst64(c5.dst_ids), check=lambda: repage_all_ok(True))
            rec(name, "repage_batched fused pool->pool 16->64", "device", wr, rd + wr, int(c5.dst_offsets[-1]),
                lambda: kv.kv_repage_batched(ctx, d_src, c5.src_ids, c5.src_offsets, d_dst, c5.dst_ids,
                                             c5.dst_offsets, c5.n_tokens, L), reps=10,
                before=lambda: poison_dst64(c5.dst_ids), check=lambda: repage_all_ok(False))
        del bufs, bufs5

        # ---- NEXT-1: copy-on-write tail-page append, 64 sessions in one launch -------
        S = 64
        perm = rng.permutation(shape.P).astype(np.int32)
        n_old = rng.integers(0, T, size=S)
        n_app = np.array([rng.integers(1, T - o + 1) for o in n_old])
        apps = [torch.randint(0, 256, (int(a) * shape.tok_bytes,), dtype=torch.uint8, device="cuda") for a in n_app]
        plc = int((n_old + n_app).sum()) * shape.tok_bytes
        old_c, new_c = perm[:S], perm[S:2 * S]

        def cow_ok():
            tokrow = shape.tokrow_bytes
            for lc in chk.lcs():
                newp, oldp = chk.rows(lc, new_c).view(S, T, tokrow), chk.rows(lc, old_c).view(S, T, tokrow)
                for s_ in range(S):
                    o, a_ = int(n_old[s_]), int(n_app[s_])
                    if not torch.equal(newp[s_, :o], oldp[s_, :o]):
                        return False
                    if not torch.equal(newp[s_, o:o + a_], apps[s_].view(LC, a_, tokrow)[lc]):
                        return False
                    if not bool((newp[s_, o + a_:] == 0xEE).all()):  # slots beyond are left as they were (poisoned)
                        return False
            return True

        rec("3 session", "cow_append_batched (64 sessions' tail pages)", "device", plc, 2 * plc, S,
            lambda: kv.kv_cow_append_batched(ctx, desc, L, old_c, new_c, n_old, n_app, apps), reps=20,
            before=lambda: chk.poison(new_c), check=cow_ok)

        # ---- a config-3 turn on the device as ONE launch (kv_submit) vs the three single calls -------------------
        for k in (5, 10, 25, 50):
            tk = turns[k - 1]
            n_m, n_new = tk.n_matched_pages, tk.cum_tokens // T - tk.n_matched_pages
            pm = rng.permutation(shape.P).astype(np.int32)
            ids_m, ids_new = pm[:n_m], pm[n_m:n_m + n_new]
            o_id, n_id = int(pm[n_m + n_new]), int(pm[n_m + n_new + 1])
            no_, na_ = 5, 9
            app = torch.randint(0, 256, (na_ * shape.tok_bytes,), dtype=torch.uint8, device="cuda")
            src_t, dst_t = big[:n_m * page], big[(n_m + 8) * page:(n_m + 8 + n_new) * page]
            ops = [kv.op_unpack(src_t, ids_m, n_m * T), kv.op_cow_append(o_id, n_id, no_, app, na_), kv.op_pack(ids_new, dst_t)]
            pl_t = (n_m + n_new) * page + (no_ + na_) * shape.tok_bytes

            def three():
                kv.kv_unpack(ctx, src_t, ids_m, desc, L, T, T, n_m * T)
                kv.kv_cow_append(ctx, desc, L, o_id, n_id, no_, app, na_)
                kv.kv_pack(ctx, desc, L, ids_new, dst_t)

            def turn_ok():
                ok = chk.unpack_ok(src_t, ids_m) and chk.pack_ok(dst_t, ids_new)
                for lc in chk.lcs():
                    newp, oldp = chk.rows(lc, [n_id]).view(T, -1), chk.rows(lc, [o_id]).view(T, -1)
                    ok = ok and bool(torch.equal(newp[:no_], oldp[:no_])) and \
                        bool(torch.equal(newp[no_:no_ + na_], app.view(LC, na_, -1)[lc]))
                return ok

            poison_turn = lambda: (chk.poison(ids_m), chk.poison([n_id]), dst_t.fill_(0xEE))
            l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
            r3 = rec("3 session", f"turn {k} on the device: unpack {n_m} + CoW append + pack {n_new} pages", "three calls",
                     pl_t, 2 * pl_t, n_m + n_new, three, reps=7, before=poison_turn, check=turn_ok)
            l1 = ctx.stat(kv.KV_STAT_LAUNCHES)
            r1 = rec("3 session", f"turn {k} on the device: unpack {n_m} + CoW append + pack {n_new} pages", "kv_submit",
                     pl_t, 2 * pl_t, n_m + n_new, lambda: kv.kv_submit(ctx, desc, L, ops), reps=7, before=poison_turn,
                     check=turn_ok)
            l2 = ctx.stat(kv.KV_STAT_LAUNCHES)
            r3["launches_per_turn"], r1["launches_per_turn"] = (l1 - l0) // 9, (l2 - l1) // 9
        del big

        # ---- NEXT-4: chained paged hashing: ids of whole sessions / batches ----------
        def chain_rec(name, wb):
            d_ident = torch.from_numpy(wb.ident.view(np.int64)).cuda()
            lens = np.diff(wb.tok_offsets)
            npg = int((lens // T).sum())
            outc = torch.empty(max(npg, 1), dtype=torch.int64, device="cuda")
            l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
            med, best = _events(torch, lambda: kv.kv_chain_hash(ctx, d_ident, wb.tok_offsets, T, outc), 20, 3)
            launches = (ctx.stat(kv.KV_STAT_LAUNCHES) - l0) // 23
            longest = int((lens // T).max())
            # `_ids`: the GPU's ids, compared with the oracle's in bench.py's cpu_baseline leg (the one place that may run
            # oracle/); until then the record says so
            recs.append({"config": "NEXT-4 chain hash", "op": name, "sessions": int(lens.size), "tokens": int(lens.sum()),
                         "pages": npg, "longest_chain_pages": longest, "chain_us_median": med, "chain_us_best": best,
                         "launches_per_call": int(launches), "Mpages_per_s": npg / med,
                         "ns_per_link_longest_chain": 1e3 * med / max(longest, 1), "verified": False,
                         "_ids": outc.cpu().numpy().view(np.uint64)[:npg].copy()})
        chain_rec("config 3: one 50-turn session history (a single chain)", W.identity_batch(seed + 3, lens=[turns[-1].cum_tokens]))
        chain_rec("config 3: one turn's increment (60 pages, a single chain)", W.identity_batch(seed + 6, lens=[60 * T]))
        chain_rec("config 4: 64 requests, log-uniform 512-16,384 tokens", W.identity_batch(seed + 4, lens=W.batch_case(seed).lens))
        chain_rec("4,096 sessions, log-uniform 512-16,384 tokens", W.identity_batch(seed + 5, n_sessions=4096))

        # ---- transfer-size sweep 1 MiB .. 8 GiB (layer_count = 32 => 1 MiB pages) --------------------
        Ls = 32
        pg = Ls * shape.C * row
        sweep = []
        bufS = torch.empty(8 << 30, dtype=torch.uint8, device="cuda")
        srcS = torch.empty(8 << 30, dtype=torch.uint8, device="cuda")
        t_launch = empty_launch_us(torch)
        peaks["empty_launch_us"] = t_launch
        for npg in W.sweep_sizes_pages():
            row_ = sweep_row(torch, ctx, desc, shape, chk, bufS, srcS, flush, npg, rng, hbm, t_launch, layers=Ls)
            ids = row_.pop("_ids")
            ok = row_.pop("bit_exact")
            dst = rng.choice(shape.P, npg, replace=False).astype(np.int32)
            ids_s = rng.choice(s_src.P, npg, replace=False).astype(np.int32)
            nd = -(-npg * 16 // 64)
            dst64 = rng.choice(s_dst.P, nd, replace=False).astype(np.int32)
            pls = npg * pg
            reps = 20 if pls <= (256 << 20) else 7
            fl_ = flush if pls <= FLUSH_UP_TO else None
            chk.poison(dst, layers=Ls)
            m, bst = _events(torch, lambda: kv.kv_unpack(ctx, bufS, dst, desc, Ls, T, T, npg * T), reps, 2, fl_)
            row_["unpack_GBps"], row_["unpack_us"] = 2 * pls / m / 1e3, m
            ok = ok and chk.unpack_ok(bufS, dst, layers=Ls)

            def rep_ok(from_buffer):
                return all(chk.repage_ok(bufS[:pls].view(npg, Ls * shape.C, row)[:, lc] if from_buffer else
                                         chk.rows(lc, ids_s, P=s_src.P, slabs=src_slabs),
                                         npg * 16, 16, dst_slabs, s_dst.P, 64, dst64, lc) for lc in chk.lcs(Ls))

            poison_dst64(dst64)
            m, bst = _events(torch, lambda: kv.kv_unpack(ctx, bufS, dst64, d_dst, Ls, 16, 64, npg * 16), reps, 2, fl_)
            row_["repage_GBps"], row_["repage_us"] = (pls + nd * Ls * shape.C * 4 * row) / m / 1e3, m
            ok = ok and rep_ok(True)
            poison_dst64(dst64)
            m, bst = _events(torch, lambda: kv.kv_repage(ctx, d_src, ids_s, d_dst, dst64, Ls, npg * 16), reps, 2, fl_)
            row_["repage_fused_GBps"], row_["repage_fused_us"] = (pls + nd * Ls * shape.C * 4 * row) / m / 1e3, m
            ok = ok and rep_ok(False)
            reps_h = 7 if pls <= (1 << 30) else 5  # D2H over this pool's VMs is noisy (+-2 % between passes): medians of >= 5
            kv.kv_pack(ctx, desc, Ls, ids, bufS)  # the device-side expectation of the offload
            hv_all[:pls:512] = 0xEE
            m, bst = _events(torch, lambda: kv.kv_offload(ctx, desc, Ls, ids, hp, pls), reps_h, 2)
            row_["offload_GBps"], row_["offload_us"], row_["offload_mode"] = pls / m / 1e3, m, ctx.stat(kv.KV_STAT_LAST_HOST_MODE)
            ok = ok and chk.host_equals_device(hp, bufS, npg, layers=Ls)
            chk.poison(dst, layers=Ls)
            m, bst = _events(torch, lambda: kv.kv_reload(ctx, hp, pls, dst, desc, Ls, T, T, npg * T), reps_h, 1)
            row_["reload_GBps"], row_["reload_us"] = pls / m / 1e3, m
            ok = ok and chk.unpack_ok(bufS, dst, layers=Ls)
            row_["pack_pct_hbm_peak"] = 100 * row_["pack_GBps"] / hbm
            row_["offload_pct_link_peak"] = 100 * row_["offload_GBps"] / d2h
            row_["reload_pct_link_peak"] = 100 * row_["reload_GBps"] / h2d
            row_["verified"] = bool(ok)
            sweep.append(row_)
        del bufS, srcS
        first80 = next((r["MiB"] for r in sweep if r["pack_pct_hbm_peak"] >= 80), None)
        recs.append({"config": "5 sweep", "op": "1 MiB - 8 GiB, layer_count 32", "rows": sweep,
                     "smallest_MiB_reaching_80pct_hbm_pack": first80,
                     "verified": bool(all(r["verified"] for r in sweep))})
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
    return {"peaks": peaks, "records": recs, "gpu": torch.cuda.get_device_name(0), "driver": driver,
            "cuda": torch.version.cuda, "cores": len(os.sched_getaffinity(0)),
            "check": f"verified: torch index_select / reshape / permute compare of ALL pages on every {LC_STEP}th "
                     "(layer,K|V) slab, destinations poisoned before the timed calls; chain ids against the oracle "
                     "(bench.py cpu_baseline leg)"}


def write(rep: dict, out_dir="gpurun_out") -> dict:
    """Drop the private keys, write report.json, return the compact summary for the bench line."""
    for r in rep["records"]:
        r.pop("_ids", None)
    os.makedirs(out_dir, exist_ok=True)
    with open(os.path.join(out_dir, "report.json"), "w") as f:
        json.dump(rep, f, indent=1)
    recs = rep["records"]
    return {"peaks": rep["peaks"],
            "summary": [{k: r[k] for k in ("config", "op", "mode", "GBps", "pct_of_measured_hbm_peak", "pct_of_link_peak", "verified") if k in r}
                        for r in recs if "GBps" in r],
            "all_verified": bool(all(r.get("verified") is True for r in recs)),
            "file": os.path.join(out_dir, "report.json")}


def markdown(rep: dict) -> str:
    """Summary tables of a report.json (what profiles/*_report_summary.md holds)."""
    pk = rep["peaks"]
    out = [f"Peaks measured in the same run: D2D copy {pk['hbm_copy_GBps_this_run']:.0f} GB/s (read+write), pinned H2D "
           f"{pk['h2d_GBps']:.1f} GB/s, D2H {pk['d2h_GBps']:.1f} GB/s, both at once {pk.get('duplex_memcpy_GBps', 0):.1f} GB/s; denominator for HBM fractions: "
           f"{pk['hbm_peak_GBps']:.1f} GB/s (MEASURED_PEAKS.json). GPU: {rep.get('gpu')}; host cores: {rep.get('cores')}. "
           f"Empty launch (one-element fill_) between two events, device time: {pk.get('empty_launch_us', 0):.1f} us.", "",
           f"Checks ({rep.get('check', '')}).", "",
           "| config | op | mode | payload MiB | median us | GB/s | % of peak | verified |",
           "|---|---|---|---:|---:|---:|---:|---|"]
    for r in rep["records"]:
        if "time_us_median" in r:
            pct = (f"{r['pct_of_measured_hbm_peak']:.1f} (HBM)" if "pct_of_measured_hbm_peak" in r
                   else f"{r['pct_of_link_peak']:.1f} (link)")
            extra = f" [{r['launches_per_turn']} launch(es)]" if "launches_per_turn" in r else ""
            out.append(f"| {r['config']} | {r['op']}{extra} | {r['mode']} | {r['payload_bytes'] / 2**20:.1f} | "
                       f"{r['time_us_median']:.1f} | {r['GBps']:.1f} | {pct} | {r['verified']} |")
        elif "time_us_total" in r:
            out.append(f"| {r['config']} | {r['op']} | {r['mode']} | {r['payload_bytes'] / 2**20:.0f} | "
                       f"{r['time_us_total']:.0f} (total) | reload {r['reload_GBps']:.1f} / offload {r['offload_GBps']:.1f} | "
                       f"{r['pct_of_link_peak_reload']:.1f} (link, reload) | {r['verified']} (every turn; turn 50: "
                       f"{r['turn50_reload_pages']} pages in {r['turn50_reload_us'] / 1e3:.1f} ms) |")
    lw = [r for r in rep["records"] if "first_layer_us" in r]
    if lw:
        out += ["", "Layer-by-layer reload of a layer-first host buffer (kv_reload_layerwise, 768 MiB, 48 layers; host wall clock from the "
                    "call to the flag seen in mapped pinned memory):", "",
                "| mode | first layer usable after us | last layer after us | GB/s | verified |", "|---|---:|---:|---:|---|"]
        for r in lw:
            out.append(f"| {r['mode']} | {r['first_layer_us']:.0f} | {r['last_layer_us']:.0f} | {r['GBps']:.1f} | {r['verified']} |")
    ch = [r for r in rep["records"] if "chain_us_median" in r]
    if ch:
        out += ["", "Chained paged hashing (kv_chain_hash, events around the call; the chain is serial, "
                    "so the floor of a call is its LONGEST chain x 16 dependent xor/multiply steps):", "",
                "| input | sessions | tokens | ids | longest chain | launches | median us | M ids/s | ns per link of the longest chain |"
                + (" oracle 1 thread us | oracle all cores us |" if "chain_oracle" in rep else "") + " verified (== oracle) |",
                "|---|---:|---:|---:|---:|---:|---:|---:|---:|" + ("---:|---:|" if "chain_oracle" in rep else "") + "---|"]
        for r in ch:
            o = rep.get("chain_oracle", {}).get(r["op"])
            out.append(f"| {r['op']} | {r['sessions']} | {r['tokens']} | {r['pages']} | {r['longest_chain_pages']} | "
                       f"{r.get('launches_per_call', '')} | {r['chain_us_median']:.1f} | {r['Mpages_per_s']:.1f} | {r['ns_per_link_longest_chain']:.1f} |"
                       + (f" {o['us_1thread']:.0f} | {o['us_all_cores']:.0f} ({o['cores']}) |" if o else "") + f" {r['verified']} |")
    for r in rep["records"]:
        if "rows" not in r:
            continue
        out += ["", f"{r['config']}: {r['op']} (isolated calls; L2 flushed clean up to 2 GiB -- the flush kernels are queued ahead of the "
                    "call, so the host's cost of issuing it is hidden and the interval is device time; floor = empty launch + 2*payload/peak; "
                    "plain copy = torch copy_ (cudaMemcpyAsync device to device) of the same bytes, contiguous, timed the same way):", "",
                "| MiB | kernel | pack us | % HBM | floor us | x floor | plain copy us | its % HBM | pack / plain copy | unpack GB/s | re-page 16->64 GB/s | fused re-page GB/s | offload GB/s (mode) | % link | reload GB/s | % link | verified |",
                "|---:|---|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---|"]
        for w in r["rows"]:
            mode = {1: "direct", 2: "staged"}.get(w.get("offload_mode"), "?")
            out.append(f"| {w['MiB']} | {w.get('kernel', '')} | {w['pack_us']:.1f} | {w['pack_pct_hbm_peak']:.1f} | {w['floor_us']:.1f} | {w['vs_floor']:.2f} | "
                       f"{w['plain_copy_us']:.1f} | {100 * w['plain_copy_frac_hbm']:.1f} | {w['vs_plain_copy']:.2f} | "
                       f"{w['unpack_GBps']:.0f} | {w['repage_GBps']:.0f} | {w.get('repage_fused_GBps', 0):.0f} | "
                       f"{w['offload_GBps']:.1f} ({mode}) | {w['offload_pct_link_peak']:.1f} | {w['reload_GBps']:.1f} | "
                       f"{w['reload_pct_link_peak']:.1f} | {w['verified']} |")
        out += ["", f"Smallest size reaching 80 % of the HBM peak (pack, isolated call, host cost inside): "
                    f"{r.get('smallest_MiB_reaching_80pct_hbm_pack')} MiB."]
    bad = [r for r in rep["records"] if r.get("verified") is not True]
    out += ["", f"Records: {len(rep['records'])}; not verified: {len(bad)}."]
    return "\n".join(out) + "\n"


if __name__ == "__main__":  # python bench_report.py gpurun_out/report.json
    import sys

    with open(sys.argv[1]) as f:
        sys.stdout.write(markdown(json.load(f)))
