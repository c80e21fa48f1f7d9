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
  roofline  = dominant kernel kv_move_bulk (the pack launch): algorithmic bytes 2*payload per
              launch / its mean duration from CUDA events on the launch stream, against the
              measured HBM copy peak in MEASURED_PEAKS.json.
  cpu_baseline = the oracle (oracle/kv_oracle.c, as it stands) on the box's host cores, on a
              bounded sample of the same workload.

`--impl reference` times the oracle alone (the reference arm of this tier).
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
# dram__bytes_read.sum + dram__bytes_write.sum of one kv_move_bulk launch at this workload (mean of 4
# launches), from the `ncu --set full` capture summarised in profiles/r01_kv_move_bulk_full.md:
# 805.4 MB read + 759.3 MB written (the last ~46 MB of the destination is still dirty in L2 at exit).
NCU_TRAFFIC_BYTES_PER_LAUNCH = 1564.6e6


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
    ap.add_argument("--report", action="store_true", help="also time every BASELINE.json config -> gpurun_out/report.json")
    ap.add_argument("--pool-order", default="nhd", choices=["nhd", "hnd"],
                    help="in-page order of the pool (BASELINE.json configs are NHD; hnd = the NEXT-2 transposing transfers)")
    ap.add_argument("--host-mode", default="auto", choices=["auto", "direct", "staged"],
                    help="kv_host_mode of the host-tier legs (auto = the library's measured choice)")
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
def oracle_run(shape, pool_pages: int, n_pages: int, steps: int, warmup: int, threads: int, seed: int):
    """Times oracle pack + unpack (C loops, as they stand) on a host pool.  Returns
    (GB/s in the (read+written)/time convention, seconds per step)."""
    from oracle import kv_oracle as ko

    rng = np.random.default_rng(seed)
    row = shape.row_bytes
    # normal(0,1) bf16 bit patterns = upper 16 bits of float32 normals
    def slab():
        f = rng.standard_normal(pool_pages * row // 2, dtype=np.float32)
        return (f.view(np.uint32) >> 16).astype(np.uint16).view(np.uint8)

    one = slab()
    slabs = [one] + [np.roll(one, 4096 * (i + 1)) for i in range(shape.L * shape.C - 1)]
    pool = ko.HostPool(slabs, shape.L, shape.C, pool_pages, shape.T, shape.H, shape.D, shape.e, row)
    payload = n_pages * shape.page_bytes
    ts = []
    for s in range(warmup + steps):
        ids = rng.choice(pool_pages, n_pages, replace=False).astype(np.int32)
        dst = rng.choice(pool_pages, n_pages, replace=False).astype(np.int32)
        t0 = time.perf_counter()
        buf = ko.pack(pool, ids, threads=threads)
        ko.unpack(buf, dst, pool, Ts=shape.T, n_tokens=n_pages * shape.T, threads=threads)
        t1 = time.perf_counter()
        if s >= warmup:
            ts.append(t1 - t0)
    sec = float(np.mean(ts))
    return 4 * payload / sec / 1e9, sec


def run_reference(args):
    from paper_2606_31093_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shape = W.QWEN3_OMNI
    cores = len(os.sched_getaffinity(0))
    n_pages = 64  # bounded sample of the 512-page prefix
    steps, warmup = max(1, min(args.steps, 10)), max(1, min(args.warmup, 2))
    gbps, sec = oracle_run(shape, 256, n_pages, steps, warmup, cores, args.seed)
    sample = (f"oracle pack+unpack of {n_pages} of the 512 pages per step on a 256-page host pool "
              f"(48 L x 4 H x 128 D bf16), {steps} steps, {cores} OpenMP threads over the page loop")
    line = {
        "impl": "reference", "metric": METRIC, "value": gbps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
        "config": {"workload": "configs[1] single-request prefix offload (bounded sample)",
                   "layers": shape.L, "kv_heads": shape.H, "head_dim": shape.D, "page_size": shape.T,
                   "pages_per_step": n_pages},
        "cpu_baseline": {"value": gbps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
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
        kern_name = {kv.KV_KERNEL_BULK: "kv_move_bulk", kv.KV_KERNEL_VEC: "kv_move_vec",
                     kv.KV_KERNEL_ELEM: "kv_move_elem"}.get(ctx.stat(kv.KV_STAT_LAST_KERNEL), "?")
        t_total_ms = max_over_ranks(ev[0].elapsed_time(ev[2 * K]))
        pack_ms = float(np.mean([ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(K)]))
        unpack_ms = float(np.mean([ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(K)]))

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
        e0.record(s_off)
        for i in range(Ke):
            duplex_step(Wm + i)
        e1.record(s_off)  # both streams were synchronised by the last step
        barrier()
        e2e_ms = max_over_ranks(e0.elapsed_time(e1))
        ctx2.close()
        for h in hp:
            kv.kv_host_free(h)

    peak, peak_src = measured_peaks()
    value = world * 4 * payload * K / (t_total_ms * 1e-3) / 1e9
    e2e_value = world * 4 * payload * Ke / (e2e_ms * 1e-3) / 1e9
    achieved = 2 * payload / (pack_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": t_total_ms / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u16 (bf16 bit patterns, bitwise copy)", "data": "synthetic",
        "config": {
            "workload": "configs[1] single-request prefix offload: pack 512 fragmented pages (8,192 tokens) "
                        "to a device buffer + unpack a buffer into 512 other pages",
            "layers": shape.L, "kv_heads": shape.H, "head_dim": shape.D, "page_size": shape.T,
            "pool_order": args.pool_order, "pool_pages": P, "pool_GiB": round(shape.L * shape.C * P * shape.row_bytes / 2**30, 1),
            "payload_MiB": payload / 2**20, "pages_per_step": n, "parallelism": "replicas only",
            "l2": "inputs larger than L2 (768 MiB per op, fresh page ids per step; unpack reads the buffer packed one step earlier)",
            "bytes_convention": "GB/s = (bytes read + bytes written) / time = 2*payload per op",
        },
        "ops": {
            "pack_GBps": 2 * payload / (pack_ms * 1e-3) / 1e9, "pack_ms": pack_ms,
            "unpack_GBps": 2 * payload / (unpack_ms * 1e-3) / 1e9, "unpack_ms": unpack_ms,
            "offload_link_GBps": payload / (off_ms * 1e-3) / 1e9, "offload_ms": off_ms,
            "reload_link_GBps": payload / (rel_ms * 1e-3) / 1e9, "reload_ms": rel_ms,
            "host_mode": host_mode,
        },
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": payload + 2 * (4 * n + 8 * shape.L * shape.C + 40 * 12),
                "d2h_bytes_per_step": payload, "steps": Ke,
                "what": "kv_offload (pool->pinned host) on one stream + kv_reload (pinned host->pool, buffer written one step earlier) "
                        "on another, both through the C ABI, both streams synchronised every step",
                "serial_value": world * 4 * payload / (serial_ms * 1e-3) / 1e9,
                "serial_what": "same two calls on ONE stream, reload reading the buffer the offload just wrote",
                "link_GBps_payload": world * 2 * payload * Ke / (e2e_ms * 1e-3) / 1e9},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "kernel": f"{kern_name} (kv_pack launch)" if args.pool_order == "nhd"
                     else f"{kern_name}<kTrans> with tensor maps (kv_pack launch, HND pool)", "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH if args.pool_order == "nhd" and n == 512 else None, "algorithmic_bytes": 2 * payload,
                     "peak_source": peak_src,
                     "timing": "mean over the K timed steps of CUDA events on the launch stream around each kv_pack call (one launch; page ids ride in the kernel parameters)"},
        "clocks": clocks.summary(),
    }

    if rank == 0 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        gbps, sec = oracle_run(W.QWEN3_OMNI, 1024, n, steps=6, warmup=1, threads=cores, seed=args.seed)
        gbps1, _ = oracle_run(W.QWEN3_OMNI, 256, 64, steps=1, warmup=1, threads=1, seed=args.seed)
        line["cpu_baseline"] = {
            "value": gbps, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle pack+unpack of the full {n}-page prefix on a 1,024-page host pool, 6 steps after 1 warm-up, "
                      f"{cores} OpenMP threads over the page loop ({sec:.2f} s/step); single thread on a 64-page sample: {gbps1:.2f} GB/s",
            "single_thread_value": gbps1,
        }
    if args.report and rank == 0:
        from paper_2606_31093_b200 import report

        line["report"] = report.run(ctx, desc, shape, [t.view(torch.uint8) for t in slabs], args.seed, hbm_peak=peak)
        # the oracle of the NEXT-4 row timed beside the GPU records (cpu_baseline leg: the one place bench.py runs oracle/)
        from oracle import chain_oracle as co

        cores = len(os.sched_getaffinity(0))
        turns = W.session_turns(args.seed)
        chain_oracle = {}
        for name, wb in (("config 3: one 50-turn session history (a single chain)", W.identity_batch(args.seed + 3, lens=[turns[-1].cum_tokens])),
                         ("config 4: 64 requests, log-uniform 512-16,384 tokens", W.identity_batch(args.seed + 4, lens=W.batch_case(args.seed).lens)),
                         ("4,096 sessions, log-uniform 512-16,384 tokens", W.identity_batch(args.seed + 5, n_sessions=4096))):
            ts = {}
            for th in (1, cores):
                best = 1e30
                for _ in range(3):
                    t0 = time.perf_counter()
                    co.chain_batched(wb.ident, wb.tok_offsets, shape.T, threads=th)
                    best = min(best, time.perf_counter() - t0)
                ts[th] = best * 1e6
            chain_oracle[name] = {"us_1thread": ts[1], "us_all_cores": ts[cores], "cores": cores}
        rp = os.path.join(ROOT, "gpurun_out", "report.json")
        with open(rp) as f:
            full = json.load(f)
        full["chain_oracle"] = chain_oracle
        with open(rp, "w") as f:
            json.dump(full, f, indent=1)
        line["report"]["chain_oracle"] = chain_oracle
    if rank == 0:
        print(json.dumps(line))
    ctx.close()
    rep.close()


def main():
    args = parse()
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:  # fresh checkout: build what is missing (one rank per node)
        import __graft_entry__

        __graft_entry__.ensure_built()
    else:  # the other ranks of the node wait for rank 0's build instead of racing it
        lib = os.path.join(ROOT, "paper_2606_31093_b200", "libkvtier.so")
        t0 = time.time()
        while args.impl == "ours" and not os.path.exists(lib) and time.time() - t0 < 300:
            time.sleep(1.0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
