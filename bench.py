#!/usr/bin/env python
"""bench.py -- KV pack/unpack GB/s on one B200 (BASELINE.json:metric), roofline and CPU baseline.

Workload (N=1): BASELINE.json:configs[1] "Single-request prefix offload": 48 layers, 4 KV heads,
head_dim 128, bf16 normal(0,1), page_size 16, pool of 65,536 pages (96 GiB); one 8,192-token
prefix = 512 fragmented pages (768 MiB), fresh page ids every step.

  step      = kv_pack (512 scattered pages -> device transfer buffer)
              + kv_unpack (a transfer buffer -> 512 other scattered pages), i.e. SURVEY.md 8(a)
              a1-a4 through the C ABI; inputs resident in HBM.
  value     = (bytes read + bytes written) / time = 4 * payload * K / t   [GB/s, device-timed]
  e2e       = the same metric with HOST buffers: kv_offload (pool -> pinned host) + kv_reload
              (pinned host -> pool) + stream sync per step; H2D/D2H inside the timed region
              (SURVEY.md 8(a) a6/a7).
  roofline  = dominant kernel kv_move_shot_plain (the pack launch): algorithmic bytes 2*payload per
              launch / its mean duration from CUDA events on the launch stream, against the
              measured HBM copy peak in MEASURED_PEAKS.json.
  cpu_baseline = the oracle (oracle/kv_oracle.c, as it stands) on the box's host cores, on a
              bounded sample of the same workload.

  roofline_host = offload / reload / both-at-once against the pinned cudaMemcpyAsync peaks measured in the SAME run
              (BASELINE.json:north_star "host-link peak"), per_config = the other configs of BASELINE.json (turn 50 of
              configs[2], configs[3] 26.5 GiB batched, configs[4] exact + ragged, six sweep points) device-timed with a
              bit_exact flag each (bench_report.compact), peer = the NEXT-3 push into a pool on another GPU where
              one is visible.

`--impl reference` times the oracle alone (the reference arm of this tier) on the SAME config: the full 512-page prefix,
--steps / --warmup honoured (a wall-clock cap, printed, is the only bound).
`--report` additionally times every config of BASELINE.json and writes gpurun_out/report.json.
Multi-GPU: the path does not shard with an exchange step -- replicas only:
under torchrun each rank runs an independent replica; value = sum of units / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "kv_pack_unpack_GBps"
UNIT = "GB/s"
# dram__bytes_read.sum + dram__bytes_write.sum of one kv_pack launch (mean of 4 launches) from an `ncu --set full` capture of
# THIS command at THIS workload.  It is a profile figure, not something this run measures: it is emitted only when the run's
# configuration is a profiled one (512 pages, NHD pool, the kernel the profile captured), with the file named beside it;
# otherwise `traffic` is null.  kv_move_shot_plain (AUTO's kernel for this call): 805.3 MB read + 753.0 MB written; the round-1
# ring (--kernel bulk): 805.4 + 759.3 (the last ~50 MB written are still dirty in L2 at exit).  Those three captures ran on a
# 12 GiB pool (--pool-pages 8192); "pool96" is the round-3 capture of the plain kernel on the 96 GiB pool the default run times.
NCU_TRAFFIC = {"kv_move_shot_plain": {"bytes_per_launch": 1558.3e6, "profile": "profiles/r02_kv_move_shot_plain_full.md"},
               "kv_move_shot": {"bytes_per_launch": 1558.4e6, "profile": "profiles/r02_kv_move_shot_full.md"},
               "kv_move_bulk": {"bytes_per_launch": 1564.6e6, "profile": "profiles/r01_kv_move_bulk_full.md"},
               "workload": {"pages": 512, "pool_order": "nhd", "min_pool_pages": 8192},  # r02 was captured on a 12 GiB pool
               # round 3: the same command captured ON the 96 GiB pool (single-pass metric list: no save/restore), mean of 7 kv_pack
               # launches, 806.62 MB read + 750.38 MB written; used when the run's pool is that pool
               "pool96": {"pool_pages": 65536,
                          "kv_move_shot_plain": {"bytes_per_launch": 1557.0e6, "profile": "profiles/r03_pool96_dram.md"}}}
REFERENCE_WALL_CAP_S = 150.0  # the reference arm stops adding steps beyond this (and says so); 50 steps need ~8 s


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--pool-pages", type=int, default=65536, help="pages per slab (65536 = 96 GiB pool)")
    ap.add_argument("--prefix-tokens", type=int, default=8192)
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the host-tier leg (0 = min(steps, 20))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip per_config / roofline_host / peer (small pools, plumbing tests)")
    ap.add_argument("--report", action="store_true", help="also time every BASELINE.json config -> gpurun_out/report.json")
    ap.add_argument("--pool-order", default="nhd", choices=["nhd", "hnd"],
                    help="in-page order of the pool (BASELINE.json configs are NHD; hnd = the NEXT-2 transposing transfers)")
    ap.add_argument("--host-mode", default="auto", choices=["auto", "direct", "staged"],
                    help="kv_host_mode of the host-tier legs (auto = the library's measured choice)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "bulk", "vec", "shot"],
                    help="KV_OPT_KERNEL of every ctx (auto = the library's measured choice; the others reproduce the A/B "
                         "figures of DESIGN.md: bulk = the persistent ring, shot = one segment per single-warp CTA)")
    ap.add_argument("--lead-chunk-mib", type=int, default=-1,
                    help="KV_OPT_LEAD_CHUNK of every ctx in MiB (-1 = the library's default; 0 = equal chunks: the A/B figure of DESIGN.md)")
    ap.add_argument("--seed", type=int, default=0)
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed regions run."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.stop = [], set(), False
        self.max_mhz, self.ok = None, False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:  # NVML missing: report nulls rather than fail the bench
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self.stop:
            try:
                util = nv.nvmlDeviceGetUtilizationRates(self.h).gpu
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.samples.append((mhz, util))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.ok:
            self.t.start()
        return self

    def __exit__(self, *a):
        self.stop = True
        if self.ok:
            self.t.join(timeout=1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        mhz = [m for m, _ in self.samples]
        return {"sm_mhz": float(np.median(mhz)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(mhz)}


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on host cores
# ------------------------------------------------------------------------------------------------
def bench_config(args, shape, reference_pool_pages=None):
    """The `config` object of both arms: the same workload (shape, pages per step, payload, byte convention).  The
    reference arm passes the size of the HOST pool its oracle really runs on: that pool is bounded by RAM,
    so `pool_pages` / `pool_GiB` differ from our arm's 96 GiB device pool and `kernel` does not apply."""
    n = -(-args.prefix_tokens // shape.T)
    pool_pages = args.pool_pages if reference_pool_pages is None else reference_pool_pages
    cfg = {
        "workload": "configs[1] single-request prefix offload: pack 512 fragmented pages (8,192 tokens) "
                    "to a device buffer + unpack a buffer into 512 other pages.  configs[1] is the configuration the metric's "
                    "80 % bar is hardest on among those that are bandwidth-bound (768 MiB per call; configs[3] 26.5 GiB and "
                    "configs[4] 6 GiB run at 1.00-1.02 of the same peak and are carried in per_config, configs[0] is launch-bound)",
        "layers": shape.L, "kv_heads": shape.H, "head_dim": shape.D, "page_size": shape.T,
        "pool_order": args.pool_order, "pool_pages": pool_pages,
        "kernel": args.kernel if reference_pool_pages is None else "n/a (oracle C loops on the host cores)",
        "pool_GiB": round(shape.L * shape.C * pool_pages * shape.row_bytes / 2**30, 1),
        "payload_MiB": n * shape.page_bytes / 2**20, "pages_per_step": n, "parallelism": "replicas only",
        "l2": "inputs larger than L2 (768 MiB per op, fresh page ids per step; unpack reads the buffer packed one step earlier)",
        "bytes_convention": "GB/s = (bytes read + bytes written) / time = 2*payload per op",
    }
    if reference_pool_pages is not None:
        cfg["pool"] = (f"host-resident, {pool_pages} pages: same shape and pages per step as our arm, smaller pool "
                       f"(our arm: {args.pool_pages} pages in HBM)")
    return cfg


def oracle_pool(shape, pool_pages: int, seed: int):
    """Host-resident pool for the oracle: normal(0,1) bf16 bit patterns (upper 16 bits of float32 normals); one slab is
    drawn, the others are rotations of it (the copy's speed does not depend on the values)."""
    from oracle import kv_oracle as ko

    rng = np.random.default_rng(seed)
    row = shape.row_bytes
    f = rng.standard_normal(pool_pages * row // 2, dtype=np.float32)
    one = (f.view(np.uint32) >> 16).astype(np.uint16).view(np.uint8)
    slabs = [one] + [np.roll(one, 4096 * (i + 1)) for i in range(shape.L * shape.C - 1)]
    return ko.HostPool(slabs, shape.L, shape.C, pool_pages, shape.T, shape.H, shape.D, shape.e, row), rng


def oracle_run(pool, rng, shape, n_pages: int, steps: int, warmup: int, threads: int, wall_cap_s=None):
    """Times oracle pack + unpack (C loops, as they stand) of `n_pages` fresh random pages per step.  Returns the
    per-step seconds of the timed steps (fewer than `steps` only if the wall-clock cap was hit)."""
    from oracle import kv_oracle as ko

    ts = []
    t_begin = time.perf_counter()
    for s in range(warmup + steps):
        ids = rng.choice(pool.num_pages, n_pages, replace=False).astype(np.int32)
        dst = rng.choice(pool.num_pages, n_pages, replace=False).astype(np.int32)
        t0 = time.perf_counter()
        buf = ko.pack(pool, ids, threads=threads)
        ko.unpack(buf, dst, pool, Ts=shape.T, n_tokens=n_pages * shape.T, threads=threads)
        t1 = time.perf_counter()
        if s >= warmup:
            ts.append(t1 - t0)
        if wall_cap_s is not None and ts and time.perf_counter() - t_begin > wall_cap_s:
            break
    return ts


ORACLE_POOL_PAGES = 4096  # "default 4,096 pages = 6 GiB at 48 L x 4 H x 128 D bf16, T 16"


def run_reference(args):
    from paper_2606_31093_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shape = W.QWEN3_OMNI
    cores = len(os.sched_getaffinity(0))
    n_pages = -(-args.prefix_tokens // shape.T)  # the FULL prefix of our arm's config: 512 pages per step
    payload = n_pages * shape.page_bytes
    pool, rng = oracle_pool(shape, ORACLE_POOL_PAGES, args.seed)
    ts = oracle_run(pool, rng, shape, n_pages, args.steps, args.warmup, cores, wall_cap_s=REFERENCE_WALL_CAP_S)
    sec = float(np.mean(ts))
    gbps = 4 * payload / sec / 1e9
    capped = len(ts) < args.steps
    sample = (f"oracle pack+unpack of the full {n_pages}-page prefix per step on a {ORACLE_POOL_PAGES}-page host pool "
              f"({ORACLE_POOL_PAGES * shape.page_bytes / 2**30:.0f} GiB, 48 L x 4 H x 128 D bf16; the pool is host-resident, so its "
              f"size is bounded by RAM: BASELINE.md 4), {len(ts)} timed steps after {args.warmup} warm-ups, {cores} OpenMP threads "
              f"over the page loop" + (f"; STOPPED at the {REFERENCE_WALL_CAP_S:.0f} s wall-clock cap before {args.steps} steps" if capped else ""))
    line = {
        "impl": "reference", "metric": METRIC, "value": gbps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(ts), "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u16 (bf16 bit patterns, bitwise copy)", "data": "synthetic",
        "config": bench_config(args, shape, reference_pool_pages=ORACLE_POOL_PAGES),
        "cpu_baseline": {"value": gbps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def peer_leg(torch, kv, ctx, shape, local, seed):
    """the provider pushes pages into a pool on ANOTHER GPU of the box over NVLink
    (kv_unpack / kv_repage with the destination pool P2P-mapped), no collective; pull = kv_pack from the peer's pool.
    Runs in ONE process whenever a second, peer-accessible GPU is visible (under torchrun every rank sees all GPUs);
    reported against a cudaMemcpyPeerAsync peak measured here; results checked with torch indexing on the peer."""
    ndev = torch.cuda.device_count()
    if ndev < 2:
        return {"available": False, "reason": f"{ndev} GPU visible to this process: the two-GPU push stays unmeasured on hardware"}
    peer = (local + 1) % ndev
    if not torch.cuda.can_device_access_peer(local, peer):
        return {"available": False, "reason": f"GPU {local} has no peer path to GPU {peer}"}
    import bench_report

    kv.kv_peer_enable(ctx, peer)
    pd = f"cuda:{peer}"
    sp = shape.with_(P=4096)  # a 6 GiB destination pool on the peer
    n = 512
    page, row, L, T = sp.page_bytes, sp.row_bytes, sp.L, sp.T
    rng = np.random.default_rng(seed + 31 + local)
    pslabs = [torch.zeros(sp.P * row, dtype=torch.uint8, device=pd) for _ in range(L * sp.C)]
    pdesc = kv.PoolDesc(pslabs, L, sp.C, sp.P, T, sp.H, sp.D, sp.e)
    buf = torch.empty(n * page, dtype=torch.uint8, device=f"cuda:{local}")
    buf.random_(0, 256)
    back = torch.empty_like(buf)
    stream = torch.cuda.current_stream()
    flag = torch.zeros(1, dtype=torch.int64, device=pd)

    def timed(fn, reps=10, warm=3):
        for _ in range(warm):
            fn()
        stream.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        stream.synchronize()
        return a.elapsed_time(b) * 1e3 / reps  # us

    # peak: plain device-to-device copies over the same link, both directions
    tmp = torch.empty(n * page, dtype=torch.uint8, device=pd)
    push_peak = n * page / timed(lambda: tmp.copy_(buf, non_blocking=True)) / 1e3
    pull_peak = n * page / timed(lambda: back.copy_(tmp, non_blocking=True)) / 1e3
    del tmp
    ids = [rng.permutation(sp.P)[:n].astype(np.int32) for _ in range(16)]
    it = iter(range(10**9))
    us_push = timed(lambda: kv.kv_unpack(ctx, buf, ids[next(it) % 16], pdesc, L, T, T, n * T))
    kv.kv_unpack(ctx, buf, ids[0], pdesc, L, T, T, n * T)
    kv.kv_signal(ctx, flag, 1)  # availability flag in the peer's memory, behind the pages
    stream.synchronize()
    with torch.cuda.device(peer):
        pchk = bench_report.Checker(torch, pslabs, sp)
        vb = buf.to(pd)
        ok_push = bool(pchk.unpack_ok(vb, ids[0])) and int(flag.item()) == 1
    us_pull = timed(lambda: kv.kv_pack(ctx, pdesc, L, ids[next(it) % 16], back))
    kv.kv_pack(ctx, pdesc, L, ids[3], back)
    stream.synchronize()
    with torch.cuda.device(peer):
        ok_pull = bool(pchk.pack_ok(back.to(pd), ids[3]))
    return {"available": True, "from_gpu": local, "to_gpu": peer, "payload_MiB": n * page / 2**20,
            "push": {"op": "kv_unpack: local buffer -> 512 scattered pages of the peer's pool (posted stores)",
                     "GBps": n * page / us_push / 1e3, "peak": push_peak, "frac": n * page / us_push / 1e3 / push_peak,
                     "bit_exact": ok_push},
            "pull": {"op": "kv_pack: 512 scattered pages of the peer's pool -> local buffer (loads over the link)",
                     "GBps": n * page / us_pull / 1e3, "peak": pull_peak, "frac": n * page / us_pull / 1e3 / pull_peak,
                     "bit_exact": ok_pull},
            "peak_how": "cudaMemcpyPeerAsync (torch copy_ between the two devices) of the same 768 MiB, back to back, CUDA events",
            "unit": "GB/s of payload over NVLink"}


def run_ours(args):
    import torch

    from paper_2606_31093_b200 import kvtier as kv
    from paper_2606_31093_b200 import workloads as W

    from paper_2606_31093_b200.replicas import Replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; kvtier has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    rep = Replicas(os.environ.get("KV_BENCH_BACKEND", "nccl"))  # gloo only in the plumbing test (two ranks, one GPU)
    world, rank, local = rep.world, rep.rank, rep.local_rank
    max_over_ranks = rep.max_over_ranks

    def barrier():
        torch.cuda.synchronize()
        rep.barrier()
        torch.cuda.synchronize()

    shape = W.QWEN3_OMNI.with_(P=args.pool_pages)
    P, n = shape.P, -(-args.prefix_tokens // shape.T)
    payload = n * shape.page_bytes
    K, Wm = args.steps, args.warmup
    Ke = args.e2e_steps or min(K, 20)

    # pool: 2*L slabs of [P][T][H][D] bf16, normal(0,1) (BASELINE.json:configs[1])
    gen = torch.Generator(device="cuda").manual_seed(args.seed + rank)
    slabs = []
    for _ in range(shape.L * shape.C):
        t = torch.empty(P * shape.T * shape.H * shape.D, dtype=torch.bfloat16, device="cuda")
        t.normal_(generator=gen)
        slabs.append(t)
    desc = kv.PoolDesc(slabs, shape.L, shape.C, P, shape.T, shape.H, shape.D, shape.e,
                       order=kv.KV_ORDER_HND if args.pool_order == "hnd" else kv.KV_ORDER_NHD)
    bufs = [torch.empty(payload, dtype=torch.uint8, device="cuda") for _ in range(2)]
    rng = np.random.default_rng(args.seed + 1000 * rank)
    total = Wm + max(K, Ke) + 1
    src_ids, dst_ids = [], []
    for _ in range(total):  # fresh, fragmented page ids every step; dst disjoint from src
        perm = rng.permutation(P)[:2 * n].astype(np.int32)
        src_ids.append(perm[:n].copy())
        dst_ids.append(perm[n:].copy())

    ctx = kv.Ctx(local)
    kopt = {"auto": kv.KV_KERNEL_AUTO, "bulk": kv.KV_KERNEL_BULK, "vec": kv.KV_KERNEL_VEC, "shot": kv.KV_KERNEL_SHOT}[args.kernel]
    ctx.set_option(kv.KV_OPT_KERNEL, kopt)
    if args.lead_chunk_mib >= 0:
        ctx.set_option(kv.KV_OPT_LEAD_CHUNK, args.lead_chunk_mib << 20)
    stream = torch.cuda.current_stream()
    kv.kv_pack(ctx, desc, shape.L, src_ids[-1], bufs[1])  # buffer read by the first unpack

    def step(i):
        kv.kv_pack(ctx, desc, shape.L, src_ids[i], bufs[i & 1])
        kv.kv_unpack(ctx, bufs[(i + 1) & 1], dst_ids[i], desc, shape.L, shape.T, shape.T, n * shape.T)

    with ClockSampler(local) as clocks:
        # ---- device leg ---------------------------------------------------------------------
        for i in range(Wm):
            step(i)
        barrier()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K + 1)]
        l0 = ctx.stat(kv.KV_STAT_LAUNCHES)
        ev[0].record(stream)
        for i in range(K):
            kv.kv_pack(ctx, desc, shape.L, src_ids[Wm + i], bufs[i & 1])
            ev[2 * i + 1].record(stream)
            kv.kv_unpack(ctx, bufs[(i + 1) & 1], dst_ids[Wm + i], desc, shape.L, shape.T, shape.T, n * shape.T)
            ev[2 * i + 2].record(stream)
        barrier()
        launches = ctx.stat(kv.KV_STAT_LAUNCHES) - l0
        kern_name = {kv.KV_KERNEL_BULK: "kv_move_bulk", kv.KV_KERNEL_VEC: "kv_move_vec", kv.KV_KERNEL_ELEM: "kv_move_elem",
                     kv.KV_KERNEL_SHOT: "kv_move_shot"}.get(ctx.stat(kv.KV_STAT_LAST_KERNEL), "?")
        if ctx.stat(kv.KV_STAT_LAST_PLAIN):
            kern_name += "_plain"
        t_total_ms = max_over_ranks(ev[0].elapsed_time(ev[2 * K]))
        pack_ms = float(np.mean([ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(K)]))
        unpack_ms = float(np.mean([ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(K)]))
        # bit-exactness of the timed region's LAST step, with plain torch indexing (no library code, no oracle): the
        # buffer just packed == gather of its source pages; the pages just scattered == the buffer they came from
        import bench_report

        u8 = [t.view(torch.uint8) for t in slabs]
        chk = bench_report.Checker(torch, u8, shape)
        hnd = (shape.H, shape.T, shape.D * shape.e) if args.pool_order == "hnd" else None
        headline_ok = bool(chk.pack_ok(bufs[(K - 1) & 1], src_ids[Wm + K - 1], hnd=hnd)
                           and chk.unpack_ok(bufs[K & 1], dst_ids[Wm + K - 1], hnd=hnd))

        # ---- host-tier legs: every step offloads 512 pages to pinned host memory and reloads 512 pages
        # from it, through the C ABI, host buffers, stream sync per step.
        #   serial  one ctx, one stream: offload, then reload of the SAME buffer (per-direction link numbers)
        #   duplex  (the e2e value) two ctxs on two streams: step i offloads into hp[i & 1] while it reloads
        #           hp[(i + 1) & 1], written one step earlier -- the schedule of the device leg, and of a
        #           server that evicts one session while it restores another; both PCIe directions carry
        #           payload at once
        hm = {"auto": kv.KV_HOST_AUTO, "direct": kv.KV_HOST_DIRECT, "staged": kv.KV_HOST_STAGED}[args.host_mode]
        hp = [kv.kv_host_alloc(payload) for _ in range(2)]
        for h in hp:  # touch every page from the CPU once: a fresh VM backs guest memory lazily, and the first DMA
            kv.host_view(h, payload)[:] = 0  # passes over untouched pinned pages ran at ~40 instead of ~56 GB/s
        Ks = min(Ke, 5)
        kv.kv_offload(ctx, desc, shape.L, src_ids[-1], hp[1], payload, mode=hm)  # the buffer the first duplex step reloads
        for i in range(Wm):
            kv.kv_offload(ctx, desc, shape.L, src_ids[i], hp[0], payload, mode=hm)
            kv.kv_reload(ctx, hp[0], payload, dst_ids[i], desc, shape.L, shape.T, shape.T, n * shape.T, mode=hm)
            stream.synchronize()
        barrier()
        eo = [torch.cuda.Event(enable_timing=True) for _ in range(2 * Ks + 1)]
        eo[0].record(stream)
        for i in range(Ks):
            kv.kv_offload(ctx, desc, shape.L, src_ids[Wm + i], hp[0], payload, mode=hm)
            eo[2 * i + 1].record(stream)
            kv.kv_reload(ctx, hp[0], payload, dst_ids[Wm + i], desc, shape.L, shape.T, shape.T, n * shape.T, mode=hm)
            eo[2 * i + 2].record(stream)
            stream.synchronize()
        barrier()
        serial_ms = max_over_ranks(eo[0].elapsed_time(eo[2 * Ks])) / Ks
        off_ms = float(np.mean([eo[2 * i].elapsed_time(eo[2 * i + 1]) for i in range(Ks)]))
        rel_ms = float(np.mean([eo[2 * i + 1].elapsed_time(eo[2 * i + 2]) for i in range(Ks)]))
        host_mode = {1: "direct", 2: "staged"}.get(ctx.stat(kv.KV_STAT_LAST_HOST_MODE), "?")

        ctx2 = kv.Ctx(local)  # its own staging, side stream and events: the two directions share nothing
        ctx2.set_option(kv.KV_OPT_KERNEL, kopt)
        if args.lead_chunk_mib >= 0:
            ctx2.set_option(kv.KV_OPT_LEAD_CHUNK, args.lead_chunk_mib << 20)
        s_off, s_rel = torch.cuda.Stream(), torch.cuda.Stream()

        def duplex_step(i):
            kv.kv_offload(ctx, desc, shape.L, src_ids[i], hp[i & 1], payload, mode=hm, stream=s_off)
            kv.kv_reload(ctx2, hp[(i + 1) & 1], payload, dst_ids[i], desc, shape.L, shape.T, shape.T, n * shape.T,
                         mode=hm, stream=s_rel)
            s_off.synchronize()  # the host reads the step's result here
            s_rel.synchronize()

        for i in range(Wm):
            duplex_step(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_step = [torch.cuda.Event(enable_timing=True) for _ in range(Ke)]
        e0.record(s_off)
        for i in range(Ke):
            duplex_step(Wm + i)
            e_step[i].record(s_off)  # both streams idle: the step's end on the device clock
        e1.record(s_off)  # both streams were synchronised by the last step
        barrier()
        e2e_ms = max_over_ranks(e0.elapsed_time(e1))
        torch.cuda.synchronize()
        step_ms = [(e0 if i == 0 else e_step[i - 1]).elapsed_time(e_step[i]) for i in range(Ke)]
        # the same schedule with the two host syncs per step replaced by cross-stream events (offload i -> reload i+1
        # reads its buffer; reload i+1 -> offload i+2 overwrites it): what the link does when the host never waits
        done_off = [torch.cuda.Event() for _ in range(Ke + 1)]
        done_rel = [torch.cuda.Event() for _ in range(Ke + 1)]
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s_rel.wait_stream(s_off)
        e2.record(s_off)
        for i in range(Ke):
            if i >= 2:
                s_off.wait_event(done_rel[i - 1])
            kv.kv_offload(ctx, desc, shape.L, src_ids[Wm + i], hp[i & 1], payload, mode=hm, stream=s_off)
            done_off[i].record(s_off)
            if i >= 1:
                s_rel.wait_event(done_off[i - 1])
            kv.kv_reload(ctx2, hp[(i + 1) & 1], payload, dst_ids[Wm + i], desc, shape.L, shape.T, shape.T, n * shape.T,
                         mode=hm, stream=s_rel)
            done_rel[i].record(s_rel)
        s_off.wait_stream(s_rel)
        e3.record(s_off)
        barrier()
        dup_nosync = {"achieved": 2 * payload * Ke / (e2.elapsed_time(e3) * 1e-3) / 1e9,
                      "what": "the same Ke offload+reload steps with cross-stream events instead of host syncs"}
        ctx2.close()
        for h in hp:
            kv.kv_host_free(h)

        link = per_config = None
        peer = {"available": False, "reason": "skipped (--no-per-config)"}
        if not args.no_per_config:
            link = bench_report.link_peaks(torch)
            dup_nosync["frac"] = dup_nosync["achieved"] / link["duplex_GBps"]
            # The legs below come AFTER every timed region of the contract line; a failure in one of them (not enough
            # memory beside another rank's pool, a box without peer access between its GPUs) is reported in its own key and
            # never costs the run its headline numbers.  per_config first, then -- behind a barrier, so that no rank's peer
            # traffic lands on rank 0's GPU while it times the other configs -- the peer leg, last because a fault in a
            # path that no lease of this build has ever been able to run must not take anything else with it.
            if rank == 0 and args.pool_pages >= 65536 and args.pool_order == "nhd":
                try:
                    per_config = bench_report.compact(ctx, desc, shape, u8, args.seed, measured_peaks()[0])
                except Exception as exc:  # noqa: BLE001
                    per_config = {"error": f"{type(exc).__name__}: {exc}"[:400]}
                torch.cuda.empty_cache()  # another rank's peer leg allocates its destination pool on this GPU
            try:
                barrier()
                peer = peer_leg(torch, kv, ctx, shape, local, args.seed)
            except Exception as exc:  # noqa: BLE001
                peer = {"available": False, "reason": f"peer leg failed: {type(exc).__name__}: {exc}"[:400]}

    peak, peak_src = measured_peaks()
    value = world * 4 * payload * K / (t_total_ms * 1e-3) / 1e9
    e2e_value = world * 4 * payload * Ke / (e2e_ms * 1e-3) / 1e9
    achieved = 2 * payload / (pack_ms * 1e-3) / 1e9
    profiled = NCU_TRAFFIC.get(kern_name) if (args.pool_order == NCU_TRAFFIC["workload"]["pool_order"]
                                              and n == NCU_TRAFFIC["workload"]["pages"]
                                              and args.pool_pages >= NCU_TRAFFIC["workload"]["min_pool_pages"]) else None
    if profiled and args.pool_pages == NCU_TRAFFIC["pool96"]["pool_pages"]:
        profiled = NCU_TRAFFIC["pool96"].get(kern_name, profiled)  # a capture on this very pool, where one exists
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": t_total_ms / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u16 (bf16 bit patterns, bitwise copy)", "data": "synthetic",
        "config": bench_config(args, shape),
        "bit_exact": headline_ok,
        "bit_exact_check": "sampled: every 11th (layer, K|V) slab of the last timed step, by torch indexing; the full compares are the GPU tests",
        "ops": {
            "pack_GBps": 2 * payload / (pack_ms * 1e-3) / 1e9, "pack_ms": pack_ms,
            "unpack_GBps": 2 * payload / (unpack_ms * 1e-3) / 1e9, "unpack_ms": unpack_ms,
            "offload_link_GBps": payload / (off_ms * 1e-3) / 1e9, "offload_ms": off_ms,
            "reload_link_GBps": payload / (rel_ms * 1e-3) / 1e9, "reload_ms": rel_ms,
            "host_mode": host_mode,
        },
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": payload + 2 * (4 * n + 8 * shape.L * shape.C + 48 * 12),
                "d2h_bytes_per_step": payload, "steps": Ke,
                "link_GBps_payload": world * 2 * payload * Ke / (e2e_ms * 1e-3) / 1e9,
                "what": "kv_offload (pool->pinned host) on one stream + kv_reload (pinned host->pool, buffer written one step earlier) "
                        "on another, both through the C ABI, both streams synchronised every step.  `value` follows the metric's "
                        "convention (bytes read + written on each side of the link = 4*payload per step); link_GBps_payload is what "
                        "crosses the link, both directions summed",
                "step_ms": {"mean": float(np.mean(step_ms)), "median": float(np.median(step_ms)), "best": float(np.min(step_ms)),
                            "worst": float(np.max(step_ms)),
                            "what": "this rank's Ke timed steps one by one (the link peaks beside them are best-of-20 figures)"},
                "serial_value": world * 4 * payload / (serial_ms * 1e-3) / 1e9,
                "serial_what": "same two calls on ONE stream, reload reading the buffer the offload just wrote"},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "kernel": f"{kern_name} (kv_pack launch)" if args.pool_order == "nhd"
                     else f"{kern_name}<kTrans> with tensor maps (kv_pack launch, HND pool)", "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": profiled["bytes_per_launch"] if profiled else None,
                     "traffic_source": (f"ncu capture of this command at this workload (r02 profiles: --set full on a 12 GiB pool; "
                                        f"r03_pool96: a single-pass --metrics list on the 96 GiB pool), {profiled['profile']} "
                                        "(a profile figure, not measured by this run)") if profiled else None,
                     "algorithmic_bytes": 2 * payload, "peak_source": peak_src,
                     "timing": "mean over the K timed steps of CUDA events on the launch stream around each kv_pack call (one launch; page ids ride in the kernel parameters)"},
        "clocks": clocks.summary(),
    }
    if link is not None:  # host-link roofline: achieved payload GB/s against the pinned cudaMemcpyAsync peaks of THIS run
        off_g, rel_g = payload / (off_ms * 1e-3) / 1e9, payload / (rel_ms * 1e-3) / 1e9
        dup_g = 2 * payload * Ke / (e2e_ms * 1e-3) / 1e9  # this rank's link (replicas have a link each)
        line["roofline_host"] = {
            "bound": "host link (PCIe)", "unit": "GB/s of payload",
            "offload": {"achieved": off_g, "peak": link["d2h_GBps"], "frac": off_g / link["d2h_GBps"]},
            "reload": {"achieved": rel_g, "peak": link["h2d_GBps"], "frac": rel_g / link["h2d_GBps"]},
            "duplex": {"achieved": dup_g, "peak": link["duplex_GBps"], "frac": dup_g / link["duplex_GBps"],
                       "frac_of_chunked_memcpy": dup_g / link["duplex_chunked_GBps"],
                       "frac_of_median_memcpy": dup_g / link["median"]["duplex_GBps"],
                       "frac_best_step": 2 * payload / (min(step_ms) * 1e-3) / 1e9 / link["duplex_GBps"],
                       "frac_median_step": 2 * payload / (float(np.median(step_ms)) * 1e-3) / 1e9 / link["duplex_GBps"],
                       "what": "the e2e leg (offload and reload at once, host sync every step) against D2H + H2D "
                               "cudaMemcpyAsync at once (one copy each way, best of 20); frac_of_median_memcpy = the leg's MEAN "
                               "against the MEDIAN of those 20 plain passes (mean against best is not like against like when "
                               "the link itself spreads); frac_best_step / frac_median_step = "
                               "the best / median single step of the leg against that same best-of-20 peak (the link on this "
                               "pool's VMs varies by +-2 % from pass to pass); frac_of_chunked_memcpy = against the same plain "
                               "copies issued as two per direction, the chunking of a staged 768 MiB transfer"},
            "duplex_no_host_sync": dup_nosync,
            "peaks": link, "host_mode": host_mode,
        }
        line["e2e"]["frac_of_duplex_memcpy_peak"] = dup_g / link["duplex_GBps"]
        # The same fractions once more INSIDE `roofline` and `e2e` -- the keys a record keeper that drops unknown top-level
        # keys still holds -- so that the record alone answers BASELINE.json's metric ("% of HBM / host-link peak").
        rh = line["roofline_host"]
        line["roofline"]["host"] = {
            "unit": "GB/s of payload over the host link", "host_mode": host_mode,
            "peak_source": "pinned cudaMemcpyAsync D2H / H2D / both at once, best of 20, measured in this run",
            "offload": dict(rh["offload"]), "reload": dict(rh["reload"]),
            "duplex": {k: rh["duplex"][k] for k in ("achieved", "peak", "frac", "frac_of_median_memcpy")},
        }
        line["e2e"]["offload_frac"] = rh["offload"]["frac"]
        line["e2e"]["reload_frac"] = rh["reload"]["frac"]
    if per_config is not None:
        line["per_config"] = per_config
        recs = [r for r in per_config.get("records", []) if isinstance(r, dict) and "payload_MiB" in r and "GBps" in r]
        if recs:  # the largest single-GPU configuration timed by this run, beside the headline's configs[1]
            big = max(recs, key=lambda r: r["payload_MiB"])
            line["roofline"]["largest"] = {"config": big["config"], "op": big["op"], "payload_GiB": big["payload_MiB"] / 1024,
                                           "achieved": big["GBps"], "peak": peak, "frac": big["GBps"] / peak,
                                           "bit_exact": big["bit_exact"], "check": "sampled: every 11th (layer, K|V) slab"}
    line["peer"] = peer

    if rank == 0 and not args.no_cpu_baseline:
        # the oracle as it stands, 4,096-page host pool, same pages per call as the config (512),
        # 3 warm-ups, median of 10; all cores, and a single thread
        cores = len(os.sched_getaffinity(0))
        pool_o, rng_o = oracle_pool(W.QWEN3_OMNI, ORACLE_POOL_PAGES, args.seed)
        ts = oracle_run(pool_o, rng_o, W.QWEN3_OMNI, n, steps=10, warmup=3, threads=cores)
        ts1 = oracle_run(pool_o, rng_o, W.QWEN3_OMNI, n, steps=3, warmup=1, threads=1)
        sec, sec1 = float(np.median(ts)), float(np.median(ts1))
        line["cpu_baseline"] = {
            "value": 4 * payload / sec / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle pack+unpack of the full {n}-page prefix per step on a {ORACLE_POOL_PAGES}-page host pool (6 GiB; BASELINE.md 4), "
                      f"median of 10 steps after 3 warm-ups, {cores} OpenMP threads over the page loop ({sec:.2f} s/step); "
                      f"single thread, same {n} pages, median of 3 after 1 warm-up: {4 * payload / sec1 / 1e9:.2f} GB/s ({sec1:.2f} s/step)",
            "single_thread_value": 4 * payload / sec1 / 1e9,
        }
        del pool_o
    if args.report and rank == 0:
        import bench_report

        rep_full = bench_report.run(ctx, desc, shape, [t.view(torch.uint8) for t in slabs], args.seed, hbm_peak=peak)
        # the oracle of the NEXT-4 row timed beside the GPU records, and the GPU's ids compared with it (cpu_baseline leg:
        # the one place bench.py runs oracle/)
        from oracle import chain_oracle as co

        cores = len(os.sched_getaffinity(0))
        turns = W.session_turns(args.seed)
        chain_oracle = {}
        inputs = {"config 3: one 50-turn session history (a single chain)": W.identity_batch(args.seed + 3, lens=[turns[-1].cum_tokens]),
                  "config 3: one turn's increment (60 pages, a single chain)": W.identity_batch(args.seed + 6, lens=[60 * shape.T]),
                  "config 4: 64 requests, log-uniform 512-16,384 tokens": W.identity_batch(args.seed + 4, lens=W.batch_case(args.seed).lens),
                  "4,096 sessions, log-uniform 512-16,384 tokens": W.identity_batch(args.seed + 5, n_sessions=4096)}
        for r in rep_full["records"]:
            wb = inputs.get(r.get("op")) if r.get("config") == "NEXT-4 chain hash" else None
            if wb is None:
                continue
            ts = {}
            for th in (1, cores):
                best = 1e30
                for _ in range(3):
                    t0 = time.perf_counter()
                    want_ids = co.chain_batched(wb.ident, wb.tok_offsets, shape.T, threads=th)[0]
                    best = min(best, time.perf_counter() - t0)
                ts[th] = best * 1e6
            chain_oracle[r["op"]] = {"us_1thread": ts[1], "us_all_cores": ts[cores], "cores": cores}
            r["verified"] = bool(np.array_equal(r["_ids"], want_ids))
        rep_full["chain_oracle"] = chain_oracle
        line["report"] = bench_report.write(rep_full)
        line["report"]["chain_oracle"] = chain_oracle
    if rank == 0:
        print(json.dumps(line), flush=True)
    try:
        ctx.close()
        rep.close()
    except Exception:  # noqa: BLE001  (nothing after the line may turn a measured run into a failed one)
        pass


def main():
    args = parse()
    import __graft_entry__

    # every rank: mtime-based, serialised by a file lock (one compiles, the others wait).  The reference arm compiles but
    # does not import the binding: its process never maps libkvtier.so, only oracle/.
    __graft_entry__.ensure_built(load=args.impl != "reference")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
