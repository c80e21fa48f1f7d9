// kv_run.inl -- execution: one launch (device / DIRECT host), or the STAGED chunk pipeline between the kernels and the copy engines
// Part of the host side of libkvtier.so; included by kvtier.cu only (one translation unit).
// Shares nothing with oracle/.
#pragma once

namespace {

// one launch over all requests (device buffers, or mapped pinned host buffers = DIRECT mode)
int run_single_launch(kv_ctx *ctx, const kv_pool_desc *pools, const Call &c, const int32_t *ids,
                      uint32_t flags, uint32_t cta_cap, cudaStream_t s) {
  std::vector<Piece> pieces;
  pieces.reserve(c.reqs.size());
  uint64_t acc = 0;
  for (const Req &q : c.reqs) {
    Piece pc{};
    pc.item_begin = acc; pc.buf = q.buf; pc.n_tokens = q.n_tokens; pc.id_begin = q.id_begin;
    pc.n_buf_pages = q.n_buf_pages; pc.dir = q.dir;
    pieces.push_back(pc);
    acc += q.items;
  }
  const bool dev_ids = flags & KV_FLAG_IDS_ON_DEVICE;
  HostBlob hb;
  build_blob(pools, c.geom, pieces.data(), pieces.size(), ids, c.n_ids, dev_ids, &hb);
  int rcm = append_maps(ctx, c.geom, &hb);
  if (rcm) return rcm;
  Blob b;
  if (ctx->inline_tables && c.geom.kernel != KERNEL_ELEM && hb.bytes.size() <= (size_t)kInlineLarge) {
    b.inl = &hb;  // tables travel inside the kernel parameters: one launch, no copy
    b.d_ids = dev_ids ? ids : nullptr;
    b.caller_ids = dev_ids;
    return launch(ctx, c.geom, b, 0, (uint32_t)pieces.size(), acc, cta_cap, s);
  }
  if (ctx->cur_capturing) return KV_ERR_CAPTURE;
  int rc = upload_blob(ctx, hb, ids, dev_ids, s, &b);
  if (rc) return rc;
  BlobGuard guard(ctx, &b, s);  // records the slot's event behind the launch, on every way out
  return launch(ctx, c.geom, b, 0, (uint32_t)pieces.size(), acc, cta_cap, s);
}

int ensure_staging(kv_ctx *ctx) {
  if (ctx->staging) return KV_OK;
  if (ctx->cur_capturing) return KV_ERR_CAPTURE;  // an allocation would invalidate the capture: reserve the staging first
  // 1 GiB = two 512 MiB slots (0.6 % of the 180 GB): with both link directions busy every chunk boundary costs ~0.25 ms,
  // for plain cudaMemcpyAsync too (768 MiB each way as 1 / 2 / 3 / 6 copies: 99.2 / 96.1 / 96.5 / 93.7 GB/s summed), so
  // chunks are as large as the pipeline allows
  if (!ctx->staging_bytes) ctx->staging_bytes = (size_t)1024 << 20;
  const cudaError_t e = cudaMalloc(&ctx->staging, ctx->staging_bytes);
  if (e != cudaSuccess) {
    ctx->staging = nullptr;
    ctx->staging_denied = true;  // KV_HOST_AUTO stops asking (run_host)
    ctx->last_cuda_error = (int)e;
    (void)cudaGetLastError();
    return KV_ERR_CUDA;
  }
  ctx->staging_denied = false;
  return KV_OK;
}

// KV_HOST_STAGED: the flattened page sequence of all requests is cut into chunks that fit one
// staging slot; per chunk: kernel <-> slot on `s`, copy engine slot <-> pinned host on the side
// stream, double (or deeper) buffered with events.  Page-first: a chunk is a run of whole pages,
// contiguous in the host buffer (one copy).  Layer-first: a chunk is a range of whole layers of one or more page
// ranges; its (layer, K|V) runs are a layer apart in the host buffer and move as ONE 2-D copy.
// Layer flags of kv_reload_layerwise: after the pages of layers [l0, l0 + n) have landed in the pool,
// flags[l] = value is stored (release, system scope) in stream order.
struct LayerFlags { uint64_t *flags = nullptr; uint64_t value = 0; };

int run_staged(kv_ctx *ctx, const kv_pool_desc *pools, const Call &c, const int32_t *ids,
               uint32_t flags, cudaStream_t s, LayerFlags lf = LayerFlags()) {
  int rc = ensure_staging(ctx);
  if (rc) return rc;
  const Geom &g = c.geom;
  const uint32_t n_slots = ctx->staging_slots;
  const bool cap = ctx->cur_capturing;
  const bool dev_ids = flags & KV_FLAG_IDS_ON_DEVICE;
  // unit of chunking: tokens that are whole pages on both sides
  const uint64_t unit_tokens = (uint64_t)g.Tpool / g.g * g.Tbuf;  // lcm(Tpool, Tbuf)
  const bool layer_first = g.layout == KV_LAYOUT_LAYER_FIRST;
  const uint64_t unit_bytes = unit_tokens * g.tokrow * (layer_first ? g.C : g.LC);
  // slot i = staging + i * slot_pitch for EVERY call of this ctx; slot_bytes (what a chunk of THIS call may fill) is a
  // prefix of it.  The per-slot events thus guard the same bytes whatever the chunk size of the call that recorded them
  // and whatever stream it ran on (two staged calls of one ctx on two streams share the slots safely).
  const size_t slot_pitch = ctx->staging_bytes / n_slots / 256 * 256;
  size_t slot_bytes = slot_pitch;
  uint64_t lead_bytes = 0;
  if (ctx->chunk_bytes) slot_bytes = std::min(slot_bytes, ctx->chunk_bytes / 256 * 256);
  // Equal chunks: at least two per transfer where that leaves >= 64 MiB each (the first chunk's kernel of an offload, or
  // the last one's of a reload, is not hidden behind a copy: 0.8 % of a two-chunk transfer; a third chunk would halve
  // that and cost more than it saves once the other link direction is busy too), as many as the slot size demands, and
  // the payload divided evenly among them in whole chunking units (no two-page leftover chunk at the end).
  // From 128 MiB a SHORT chunk (32 MiB) leads an offload, or ends a reload, when KV_OPT_LEAD_CHUNK allows it: the one
  // kernel that no copy hides -- the first of an offload, the last of a reload -- is then a 32 MiB kernel (~12 us)
  // instead of one over half the payload (~120 us of a 14.3 ms transfer at 768 MiB), and the short copy beside it is
  // still long enough (0.57 ms) to hide the neighbouring large chunk's kernel.
  else {
    const uint64_t cap = slot_bytes / unit_bytes * unit_bytes, min_chunk = (uint64_t)64 << 20;
    if (cap < unit_bytes) return KV_ERR_SIZE;  // one chunking unit does not fit a staging slot
    if (ctx->lead_chunk && !lf.flags && !layer_first && c.payload >= 2 * min_chunk) {
      lead_bytes = std::max<uint64_t>(unit_bytes, ((uint64_t)ctx->lead_chunk + unit_bytes - 1) / unit_bytes * unit_bytes);
      if (lead_bytes > cap || lead_bytes * 2 > c.payload) lead_bytes = 0;
    }
    const uint64_t rest = c.payload - lead_bytes;
    uint64_t n = lead_bytes ? 1 : std::max<uint64_t>(1, std::min<uint64_t>(2, c.payload / min_chunk));
    uint64_t per = cap;
    for (;; ++n) {
      per = ((rest + n - 1) / n + unit_bytes - 1) / unit_bytes * unit_bytes;
      if (per <= cap) break;
    }
    slot_bytes = (size_t)std::max<uint64_t>(per, unit_bytes);
  }
  // layer-by-layer reload: the first flag should come early, so chunks stay small (a 64 MiB chunk of the
  // Qwen3-Omni prefix is 4 layers: first layer usable after 1.3 ms; 256 MiB chunks would make it 5 ms)
  if (lf.flags) slot_bytes = std::min<size_t>(slot_bytes, (size_t)64 << 20);
  if (slot_bytes < unit_bytes) return KV_ERR_SIZE;
  const uint64_t chunk_tokens = slot_bytes / unit_bytes * unit_tokens;
  // an offload's FIRST chunk is the short one; a reload's short chunk is the remainder its equal chunks leave at the end
  const uint64_t lead_tokens = g.dir == 0 ? lead_bytes / unit_bytes * unit_tokens : 0;

  // A chunk = what one staging slot holds: pieces for the kernel, copies for the copy engine.  Page-first:
  // a run of whole pages, all layers (contiguous in the host buffer).  Layer-first: a range of layers
  // [l0, l0 + nl) of one or more page ranges; every (layer, K|V) of a page range is one contiguous host run.
  struct Chunk { uint32_t piece_first, n_pieces; uint64_t items; uint32_t l0, nl, sig_n; uint64_t id_lo = ~0ull, id_hi = 0; };
  // rows > 1: a strided copy of `rows` runs of `bytes` each, host_pitch apart in the host buffer and dense in the
  // slot (the (layer, K|V) runs of a layer-first page range): ONE 2-D copy-engine transfer instead of `rows`
  struct Copy { uint64_t host, dev_off, bytes; uint64_t rows = 1, host_pitch = 0; };
  std::vector<Piece> pieces;
  std::vector<Chunk> chunks;
  std::vector<std::vector<Copy>> copies;
  if (layer_first) {
    const uint64_t row = g.buf_row;  // bytes of one buffer page of one (layer, K|V)
    uint64_t widest = 1;
    for (const Req &q : c.reqs) widest = std::max<uint64_t>(widest, q.n_buf_pages);
    // as many layers per chunk as the widest request allows; a request wider than a slot is cut by page ranges
    const uint32_t kl = (uint32_t)std::min<uint64_t>(g.L, std::max<uint64_t>(1, slot_bytes / (widest * g.C * row)));
    const uint64_t unit_pool_pages = unit_tokens / g.Tpool;
    for (uint32_t l0 = 0; l0 < g.L; l0 += kl) {
      const uint32_t nl = std::min(kl, g.L - l0);
      const uint64_t per_buf_page = (uint64_t)nl * g.C * row;  // slot bytes one buffer page costs in this layer range
      const uint64_t max_pool_pages = slot_bytes / per_buf_page * g.Tbuf / g.Tpool / unit_pool_pages * unit_pool_pages;
      if (!max_pool_pages) return KV_ERR_SIZE;
      Chunk cur{(uint32_t)pieces.size(), 0, 0, l0, nl, 0};
      std::vector<Copy> cur_copies;
      uint64_t fill = 0;
      auto close = [&]() {
        if (cur.n_pieces) { chunks.push_back(cur); copies.push_back(cur_copies); }
        cur = Chunk{(uint32_t)pieces.size(), 0, 0, l0, nl, 0};
        cur_copies.clear();
        fill = 0;
      };
      for (const Req &q : c.reqs) {
        for (uint64_t q0 = 0; q0 < q.n_ids; q0 += max_pool_pages) {
          const uint64_t q1 = std::min(q.n_ids, q0 + max_pool_pages);
          const uint64_t t0 = q0 * g.Tpool, t1 = q1 * g.Tpool;
          const uint64_t b0 = std::min(t0 / g.Tbuf, q.n_buf_pages);
          const uint64_t b1 = std::min((t1 + g.Tbuf - 1) / g.Tbuf, q.n_buf_pages);
          const uint64_t nb = b1 - b0, region = nb * per_buf_page;
          if (fill + region > slot_bytes) close();
          Piece pc{};
          pc.item_begin = cur.items;
          pc.buf = fill;  // offset within the slot; the slot base is added below
          pc.n_tokens = q.n_tokens > t0 ? std::min(q.n_tokens - t0, t1 - t0) : 0;
          pc.id_begin = q.id_begin + q0;
          pc.n_buf_pages = nb;
          pieces.push_back(pc);
          cur.n_pieces++;
          cur.id_lo = std::min(cur.id_lo, pc.id_begin); cur.id_hi = std::max(cur.id_hi, pc.id_begin + (q1 - q0));
          cur.items += (q1 - q0) * (g.Tpool / g.g) * nl * g.C * g.subs;
          if (nb) {
            const uint64_t pitch = q.n_buf_pages * row;  // host bytes between consecutive (layer, K|V) runs
            if (pitch <= (1ull << 30)) {
              cur_copies.push_back(Copy{q.buf + ((uint64_t)l0 * g.C * q.n_buf_pages + b0) * row, fill, nb * row,
                                        (uint64_t)nl * g.C, pitch});
            } else {  // beyond the 2-D copy's pitch limit: one copy per run
              for (uint32_t l = 0; l < nl; ++l)
                for (uint32_t kc = 0; kc < g.C; ++kc)
                  cur_copies.push_back(Copy{q.buf + (((uint64_t)(l0 + l) * g.C + kc) * q.n_buf_pages + b0) * row,
                                            fill + ((uint64_t)l * g.C + kc) * nb * row, nb * row});
            }
          }
          fill += (region + 255) / 256 * 256;
        }
      }
      close();
      if (!chunks.empty()) chunks.back().sig_n = nl;  // layers [l0, l0 + nl) are complete after this chunk
    }
  } else {
    uint64_t fill_tokens = 0;  // tokens (in buffer-page units) already placed in the open chunk
    Chunk cur{0, 0, 0, 0, g.L, 0};
    std::vector<Copy> cur_copies;
    auto close = [&]() {
      if (cur.n_pieces) { chunks.push_back(cur); copies.push_back(cur_copies); }
      cur = Chunk{(uint32_t)pieces.size(), 0, 0, 0, g.L, 0};
      cur_copies.clear();
      fill_tokens = 0;
    };
    for (const Req &q : c.reqs) {
      // the request covers n_ids pool pages = n_ids*Tpool token slots; its buffer holds
      // n_buf_pages*Tbuf token slots.  Walk it in token ranges [t0, t1) of whole units.
      const uint64_t slots_pool = q.n_ids * g.Tpool;
      uint64_t t0 = 0;
      while (t0 < slots_pool) {
        const uint64_t cap_tokens = (lead_tokens && chunks.empty()) ? lead_tokens : chunk_tokens;
        if (fill_tokens == cap_tokens) close();
        const uint64_t cap_now = (lead_tokens && chunks.empty()) ? lead_tokens : chunk_tokens;  // (close() may have opened chunk 1)
        const uint64_t t1 = std::min(slots_pool, t0 + (cap_now - fill_tokens));
        const uint64_t span = t1 - t0;  // multiple of Tpool; multiple of unit except at the request's end
        const uint64_t buf_pages = (std::min(t1, q.n_buf_pages * g.Tbuf) - std::min(t0, q.n_buf_pages * g.Tbuf) + g.Tbuf - 1) / g.Tbuf;
        const uint64_t dev_off = fill_tokens * g.tokrow * g.LC;
        Piece pc{};
        pc.item_begin = cur.items;
        pc.buf = dev_off;  // offset within the slot; the slot base is added below
        pc.n_tokens = q.n_tokens > t0 ? std::min(q.n_tokens - t0, span) : 0;
        pc.id_begin = q.id_begin + t0 / g.Tpool;
        pc.n_buf_pages = buf_pages;
        pieces.push_back(pc);
        cur.n_pieces++;
        cur.id_lo = std::min(cur.id_lo, pc.id_begin); cur.id_hi = std::max(cur.id_hi, pc.id_begin + span / g.Tpool);
        cur.items += items_of(g, span / g.Tpool);
        if (buf_pages)
          cur_copies.push_back(Copy{q.buf + t0 / g.Tbuf * g.buf_page, dev_off, buf_pages * g.buf_page});
        // buffer-page units consumed in the slot (a ragged tail still occupies whole units)
        fill_tokens += (span + unit_tokens - 1) / unit_tokens * unit_tokens;
        t0 = t1;
      }
    }
    close();
  }
  // patch slot bases
  for (size_t ci = 0; ci < chunks.size(); ++ci) {
    const uint64_t base = (uint64_t)(uintptr_t)ctx->staging + (ci % n_slots) * slot_pitch;
    for (uint32_t k = 0; k < chunks[ci].n_pieces; ++k) pieces[chunks[ci].piece_first + k].buf += base;
  }
  // Tables.  A chunk's launch needs its slab bases, its pieces and ITS page ids (a contiguous range of the call's id
  // array): a few hundred bytes at the paper's shapes (a 256 MiB chunk of the Qwen3-Omni pool is 170 pages), so each
  // chunk launch carries them inside its kernel parameters -- no table copy, no pinned ring, and therefore nothing
  // that a CUDA graph could not replay.  Only calls with a chunk whose tables exceed the parameter space (tens of
  // thousands of tiny pages per chunk) stage ONE blob for all chunks through the pinned ring; those cannot be captured.
  const bool layer_range = layer_first;  // layer-first chunks launch over a slab range [l0*C, (l0+nl)*C)
  bool inline_ok = ctx->inline_tables && g.kernel != KERNEL_ELEM;
  for (const Chunk &ch : chunks) {
    const size_t n_lc = layer_range ? ch.nl * g.C : g.LC;
    const size_t need = n_lc * 8 + (size_t)ch.n_pieces * sizeof(Piece) + (dev_ids ? 0 : (size_t)(ch.id_hi - ch.id_lo) * 4) +
                        (g.tma_inline ? 64 + n_lc * sizeof(CUtensorMap) : 0);
    if (need > (size_t)kInlineLarge) inline_ok = false;
  }
  if (cap && !inline_ok) return KV_ERR_CAPTURE;
  // An eager transfer of several chunks forks to the ctx's side stream.  While a staged transfer of this ctx is being
  // captured on another stream -- between its cudaStreamBeginCapture and cudaStreamEndCapture -- the side stream is part
  // of that capture: work enqueued onto it now would end up inside the foreign graph or invalidate it.  Refuse before
  // anything is enqueued (KV_HOST_AUTO then runs DIRECT, run_host).
  if (!cap && chunks.size() > 1 && capturing(ctx->side)) return KV_ERR_CAPTURE;
  Blob shared;  // the one staged blob of the fallback
  HostBlob hb_all;
  if (!inline_ok) {
    build_blob(pools, g, pieces.data(), pieces.size(), ids, c.n_ids, dev_ids, &hb_all);
    rc = upload_blob(ctx, hb_all, ids, dev_ids, s, &shared);
    if (rc) return rc;
  }
  BlobGuard guard(ctx, &shared, s);  // no-op for inline tables
  HostBlob hb_chunk;
  std::vector<Piece> chunk_pieces;
  auto launch_chunk = [&](const Chunk &ch) -> int {
    if (!inline_ok)
      return launch(ctx, g, shared, ch.piece_first, ch.n_pieces, ch.items, 0, s, ch.l0 * g.C, ch.nl * g.C);
    chunk_pieces.assign(pieces.begin() + ch.piece_first, pieces.begin() + ch.piece_first + ch.n_pieces);
    if (!dev_ids)
      for (Piece &pc : chunk_pieces) pc.id_begin -= ch.id_lo;  // ids of the chunk start at 0 in its own table
    build_blob(pools, g, chunk_pieces.data(), chunk_pieces.size(), dev_ids ? nullptr : ids + ch.id_lo,
               dev_ids ? 0 : ch.id_hi - ch.id_lo, dev_ids, &hb_chunk, layer_range ? ch.l0 * g.C : 0,
               layer_range ? ch.nl * g.C : 0);
    int rcm = append_maps(ctx, g, &hb_chunk, layer_range ? ch.l0 * g.C : 0, layer_range ? ch.nl * g.C : 0);
    if (rcm) return rcm;
    Blob b;
    b.inl = &hb_chunk;
    b.d_ids = dev_ids ? ids : nullptr;
    b.caller_ids = dev_ids;
    return launch(ctx, g, b, 0, ch.n_pieces, ch.items, 0, s, ch.l0 * g.C, ch.nl * g.C);
  };
  // Events.  Eager calls order slot reuse across calls with the ctx's per-slot events.  Inside a capture the same
  // fork / join pattern is recorded with events of its own (a captured record is an edge of the graph, not a real
  // record), and there is no earlier call to wait for: a replayed graph is ordered against other work of the ctx by
  // the stream it is launched on (kvtier.h "CUDA graphs").
  cudaEvent_t ev_entry = cap ? ctx->cap_entry : ctx->ev_entry;
  cudaEvent_t *ev_full = cap ? ctx->cap_full : ctx->ev_full;
  cudaEvent_t *ev_free = cap ? ctx->cap_free : ctx->ev_free;
  std::vector<uint8_t> cap_used(kMaxStagingSlots, 0);  // capture: slots this call has already been through
  // A transfer of ONE chunk has nothing to overlap: its kernel and its copy run back to back on the caller's stream, with
  // no fork to the side stream and no cross-stream events (each costs a few microseconds: 8 MiB offload 168 -> 16x us
  // against 155 us for the bare cudaMemcpyAsync).  The slot is still guarded by its event for whoever uses it next.
  const bool single = chunks.size() == 1;
  cudaStream_t cs = single ? s : ctx->side;
  if (!single) {
    KV_CUDA(ctx, cudaEventRecord(ev_entry, s));
    KV_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ev_entry, 0));
  }
  for (size_t ci = 0; ci < chunks.size(); ++ci) {
    const uint32_t slot = (uint32_t)(ci % n_slots);
    uint8_t *slot_base = (uint8_t *)ctx->staging + (size_t)slot * slot_pitch;
    const bool wait_free = cap ? cap_used[slot] != 0 : ctx->free_valid[slot];
    if (g.dir == 0) {  // offload: kernel fills the slot on s, copy engine drains it on side
      if (wait_free) KV_CUDA(ctx, cudaStreamWaitEvent(s, ev_free[slot], 0));
      rc = launch_chunk(chunks[ci]);
      if (rc) return rc;
      if (!single) {
        KV_CUDA(ctx, cudaEventRecord(ev_full[slot], s));
        KV_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ev_full[slot], 0));
      }
      for (const Copy &cp : copies[ci]) {
        if (cp.rows > 1)
          KV_CUDA(ctx, cudaMemcpy2DAsync((void *)(uintptr_t)cp.host, cp.host_pitch, slot_base + cp.dev_off, cp.bytes,
                                         cp.bytes, cp.rows, cudaMemcpyDeviceToHost, cs));
        else
          KV_CUDA(ctx, cudaMemcpyAsync((void *)(uintptr_t)cp.host, slot_base + cp.dev_off, cp.bytes,
                                       cudaMemcpyDeviceToHost, cs));
        ctx->memcpys++;
      }
      KV_CUDA(ctx, cudaEventRecord(ev_free[slot], cs));
    } else {  // reload: copy engine fills the slot on side, kernel drains it on s
      if (wait_free) KV_CUDA(ctx, cudaStreamWaitEvent(cs, ev_free[slot], 0));
      for (const Copy &cp : copies[ci]) {
        if (cp.rows > 1)
          KV_CUDA(ctx, cudaMemcpy2DAsync(slot_base + cp.dev_off, cp.bytes, (const void *)(uintptr_t)cp.host,
                                         cp.host_pitch, cp.bytes, cp.rows, cudaMemcpyHostToDevice, cs));
        else
          KV_CUDA(ctx, cudaMemcpyAsync(slot_base + cp.dev_off, (const void *)(uintptr_t)cp.host,
                                       cp.bytes, cudaMemcpyHostToDevice, cs));
        ctx->memcpys++;
      }
      if (!single) {
        KV_CUDA(ctx, cudaEventRecord(ev_full[slot], ctx->side));
        KV_CUDA(ctx, cudaStreamWaitEvent(s, ev_full[slot], 0));
      }
      rc = launch_chunk(chunks[ci]);
      if (rc) return rc;
      if (lf.flags && chunks[ci].sig_n) {  // these layers' pages are in the pool: publish
        kvt::kv_signal_range<<<1, 32, 0, s>>>(lf.flags + chunks[ci].l0, chunks[ci].sig_n, lf.value);  // strides over > 32
        KV_CUDA(ctx, cudaGetLastError());
        ctx->launches++;
      }
      KV_CUDA(ctx, cudaEventRecord(ev_free[slot], s));
    }
    if (cap) cap_used[slot] = 1; else ctx->free_valid[slot] = true;
  }
  if (g.dir == 0 && !single) {  // join the copy engine's tail back into s
    const size_t first = chunks.size() > n_slots ? chunks.size() - n_slots : 0;
    for (size_t ci = first; ci < chunks.size(); ++ci)
      KV_CUDA(ctx, cudaStreamWaitEvent(s, ev_free[ci % n_slots], 0));
  }
  return KV_OK;
}

// Is `p` pinned host memory?  Returns its device alias (UVA: normally the same address).
int host_alias(kv_ctx *ctx, const void *p, uint64_t *alias) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) { (void)cudaGetLastError(); return KV_ERR_HOST_MEM; }
  if (a.type != cudaMemoryTypeHost || !a.devicePointer) return KV_ERR_HOST_MEM;
  (void)ctx;
  *alias = (uint64_t)(uintptr_t)a.devicePointer;
  return KV_OK;
}

int resolve_mode(const kv_ctx *ctx, int mode, const Call &c, int *out) {
  if (mode != KV_HOST_AUTO && mode != KV_HOST_DIRECT && mode != KV_HOST_STAGED) return KV_ERR_LAYOUT;
  int m = mode;
  // Measured on B200 / PCIe Gen5 x16: the copy engines reach 98-99 % of the
  // cudaMemcpy peak, SM-issued stores/loads over the link 92 % (128-byte TLP payloads).  A one-chunk staged
  // transfer is a kernel and a copy back to back on the caller's stream; it is ahead of DIRECT from 4 MiB
  // (92 vs 98 us; 8 MiB 167 vs 178; 16 MiB 314 vs 336), level at 2 MiB, behind at 1 MiB (reload 41 vs 38 us),
  // where DIRECT is one launch with no staging traffic.
  if (m == KV_HOST_AUTO) m = c.payload >= kAutoStagedMinBytes ? KV_HOST_STAGED : KV_HOST_DIRECT;
  (void)ctx;
  *out = m;
  return KV_OK;
}

// Device alias of a flag word (device memory, or mapped pinned host memory).
int flag_alias(const void *p, uint64_t **out) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return KV_ERR_HOST_MEM; }
  if (a.type == cudaMemoryTypeUnregistered) return KV_ERR_HOST_MEM;
  if (a.type == cudaMemoryTypeHost) {
    if (!a.devicePointer) return KV_ERR_HOST_MEM;
    *out = (uint64_t *)a.devicePointer;
  } else {
    *out = (uint64_t *)p;
  }
  return KV_OK;
}

int run_host(kv_ctx *ctx, const kv_pool_desc *pools, Call &c, const int32_t *ids, int mode,
             uint32_t flags, cudaStream_t s, LayerFlags lf = LayerFlags()) {
  int m = 0;
  int rc = resolve_mode(ctx, mode, c, &m);
  if (rc) return rc;
  note_plan(ctx, c);
  ctx->last_mode = (uint64_t)m;
  if (c.reqs.empty()) return KV_OK;  // n == 0: nothing to do, no launch
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  DeviceGuard guard(ctx);
  std::vector<uint64_t> alias(c.reqs.size());
  for (size_t i = 0; i < c.reqs.size(); ++i) {
    rc = host_alias(ctx, (const void *)(uintptr_t)c.reqs[i].buf, &alias[i]);
    if (rc) return rc;
  }
  if (lf.flags) {
    rc = flag_alias(lf.flags, &lf.flags);
    if (rc) return rc;
  }
  if (m == KV_HOST_STAGED && mode == KV_HOST_AUTO && !ctx->staging) {
    // AUTO prefers the staged pipeline but the ctx has no staging yet: this call would allocate it.  No staging to be
    // had -- the stream is being captured, or the allocation fails or has failed before (HBM is full of KV pools: the
    // normal state of a serving engine) -- is no reason to fail a transfer that DIRECT can do without any staging.
    // Nothing has been enqueued at this point.
    if (ctx->staging_denied) m = KV_HOST_DIRECT;
    else {
      rc = ensure_staging(ctx);
      if (rc == KV_ERR_CUDA || rc == KV_ERR_CAPTURE) m = KV_HOST_DIRECT;
      else if (rc) return rc;
    }
    ctx->last_mode = (uint64_t)m;
  }
  if (m == KV_HOST_STAGED) {
    // The chunk pipeline is copies, events and kernels with their tables in the kernel parameters: all of it can be
    // captured into a CUDA graph.  What cannot: allocating the staging during the capture (reserve it first:
    // KV_OPT_RESERVE_STAGING, or any earlier staged call) and tables too large for the parameters.  Then an explicit
    // KV_HOST_STAGED is KV_ERR_CAPTURE and KV_HOST_AUTO takes DIRECT, as it did before staged transfers were capturable.
    rc = run_staged(ctx, pools, c, ids, flags, s, lf);
    if (!(rc == KV_ERR_CAPTURE && mode == KV_HOST_AUTO)) return rc;
    m = KV_HOST_DIRECT;
    ctx->last_mode = (uint64_t)m;
  }
  // DIRECT: one launch moves every layer (the flags follow it together)
  for (size_t i = 0; i < c.reqs.size(); ++i) c.reqs[i].buf = alias[i];
  // Small DIRECT transfers (the only ones AUTO still sends this way) finish sooner with few CTAs: the link saturates with
  // far fewer of them than HBM (1 MiB: 39 us with 256 CTAs, 34 with 64; 2 MiB 58 -> 54).  Large ones keep the device
  // grid: with the general kernel (batches, layer-first buffers) 64 CTAs cost 2-3 % of the link (26.5 GiB batched
  // 52.7 -> 50.8 GB/s).
  const uint32_t cta_cap = ctx->host_max_ctas ? ctx->host_max_ctas : (c.payload <= ((uint64_t)16 << 20) ? 64u : 0u);
  rc = run_single_launch(ctx, pools, c, ids, flags, cta_cap, s);
  if (rc || !lf.flags) return rc;
  for (uint32_t l0 = 0; l0 < c.geom.L; l0 += 32) {
    kvt::kv_signal_range<<<1, 32, 0, s>>>(lf.flags + l0, std::min(32u, c.geom.L - l0), lf.value);
    KV_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
  }
  return KV_OK;
}

int run_device(kv_ctx *ctx, const kv_pool_desc *pools, const Call &c, const int32_t *ids,
               uint32_t flags, cudaStream_t s) {
  note_plan(ctx, c);
  if (c.reqs.empty()) return KV_OK;  // n == 0: nothing to do, no launch
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  DeviceGuard guard(ctx);
  return run_single_launch(ctx, pools, c, ids, flags, 0, s);
}

}  // namespace
