// kv_launch.inl -- lookup tables of a launch (inline in the kernel parameters, or staged through the pinned ring) and the launches themselves
// Part of the host side of libkvtier.so; included by kvtier.cu only (one translation unit).
// Shares nothing with oracle/.
#pragma once

namespace {

// ---------------------------------------------------------------------------------------------
// blob = [bases: LC x u64][pieces: n x Piece][ids: n_ids x i32], staged through a pinned ring
// ---------------------------------------------------------------------------------------------
struct HostBlob {
  std::vector<uint8_t> bytes;
  size_t off_pieces = 0, off_ids = 0;
  size_t off_maps_pool = 0, off_maps_src = 0;  // tensor maps carried in the blob (0 = none); 64-byte aligned
};

// `pieces` / `n_pieces`: the pieces of the launch(es) the blob serves.  lc0 / lc_n: only the slab bases
// [lc0, lc0 + lc_n) go in (a layer-range chunk of the staged pipeline with tables of its own); lc_n == 0: all.
void build_blob(const kv_pool_desc *p, const Geom &g, const Piece *pieces, size_t n_pieces,
                const int32_t *ids, uint64_t n_ids, bool ids_on_device, HostBlob *hb,
                uint32_t lc0 = 0, uint32_t lc_n = 0) {
  if (!lc_n) lc_n = g.LC;
  hb->off_pieces = (size_t)lc_n * 8 * (g.src_pool ? 2 : 1);
  hb->off_ids = hb->off_pieces + n_pieces * sizeof(Piece);
  hb->bytes.resize(hb->off_ids + (ids_on_device ? 0 : (size_t)n_ids * 4));
  uint8_t *h = hb->bytes.data();
  for (uint32_t i = 0; i < lc_n; ++i) ((uint64_t *)h)[i] = (uint64_t)(uintptr_t)p->base[lc0 + i];
  if (g.src_pool)
    for (uint32_t i = 0; i < lc_n; ++i) ((uint64_t *)h)[lc_n + i] = (uint64_t)(uintptr_t)g.src_pool->base[lc0 + i];
  if (n_pieces) std::memcpy(h + hb->off_pieces, pieces, n_pieces * sizeof(Piece));
  if (!ids_on_device && n_ids) std::memcpy(h + hb->off_ids, ids, (size_t)n_ids * 4);
}

// A captured HND call whose pool has no maps in device memory yet (Geom::tma_inline): the maps of slabs
// [lc0, lc0 + lc_n) are encoded on the host and appended to the blob, 64-byte aligned (the blob itself is 64-byte
// aligned inside the kernel parameters).
int append_maps(kv_ctx *ctx, const Geom &g, HostBlob *hb, uint32_t lc0 = 0, uint32_t lc_n = 0) {
  hb->off_maps_pool = hb->off_maps_src = 0;
  if (!g.tma_inline) return KV_OK;
  if (!lc_n) lc_n = g.LC;
  auto add = [&](const kv_pool_desc *p, size_t *off) -> int {
    const size_t at = (hb->bytes.size() + 63) / 64 * 64;
    hb->bytes.resize(at + (size_t)lc_n * sizeof(CUtensorMap));
    *off = at;
    std::vector<CUtensorMap> maps(lc_n);  // (the vector's storage satisfies the encoder's alignment; the blob's may not)
    int rc = encode_maps(ctx, p, lc0, lc_n, g.tb, g.tma_es, maps.data());
    if (rc) return rc;
    std::memcpy(hb->bytes.data() + at, maps.data(), (size_t)lc_n * sizeof(CUtensorMap));
    return KV_OK;
  };
  if (g.pool_hnd) { int rc = add(g.dst_pool, &hb->off_maps_pool); if (rc) return rc; }
  if (g.src_hnd) { int rc = add(g.src_pool, &hb->off_maps_src); if (rc) return rc; }
  return KV_OK;
}

// Tables of a launch: either resident in device memory (slot of the pinned ring) or carried
// inside the kernel parameters (inline; no copy, no slot).
struct Blob {
  BlobSlot *slot = nullptr;
  const uint64_t *d_bases = nullptr;
  const Piece *d_pieces = nullptr;
  const int32_t *d_ids = nullptr;  // also set for caller-supplied device ids in inline mode
  const HostBlob *inl = nullptr;   // non-null: inline tables
  bool caller_ids = false;          // the page ids are the caller's device array (KV_FLAG_IDS_ON_DEVICE): unvalidated
  const Piece *h_pieces = nullptr; // host copy of the blob's pieces (a single-piece launch carries its piece in the Job header)
};

int upload_blob(kv_ctx *ctx, const HostBlob &hb, const int32_t *ids, bool ids_on_device,
                cudaStream_t s, Blob *out) {
  const size_t bytes = hb.bytes.size();
  BlobSlot &slot = ctx->blobs[ctx->next_blob++ % kBlobSlots];
  if (slot.used) KV_CUDA(ctx, cudaEventSynchronize(slot.ev));  // last reader of this slot is done
  if (slot.cap < bytes) {
    // The 16 slots are views into ONE pinned + ONE device arena, (re)allocated together: a slot that grew on its own
    // cost a cudaFree (a device-wide sync) and a millisecond of cudaMallocHost per slot, i.e. 16 hiccups in a row.
    for (BlobSlot &o : ctx->blobs)
      if (o.used) KV_CUDA(ctx, cudaEventSynchronize(o.ev));
    if (ctx->blob_arena_h) cudaFreeHost(ctx->blob_arena_h);
    if (ctx->blob_arena_d) cudaFree(ctx->blob_arena_d);
    ctx->blob_arena_h = ctx->blob_arena_d = nullptr;
    for (BlobSlot &o : ctx->blobs) { o.h = o.d = nullptr; o.cap = 0; o.used = false; }
    const size_t cap = (std::max<size_t>((size_t)256 << 10, bytes + bytes / 2) + 255) / 256 * 256;
    KV_CUDA(ctx, cudaMallocHost(&ctx->blob_arena_h, cap * kBlobSlots));
    KV_CUDA(ctx, cudaMalloc(&ctx->blob_arena_d, cap * kBlobSlots));
    for (int i = 0; i < kBlobSlots; ++i) {
      ctx->blobs[i].h = (uint8_t *)ctx->blob_arena_h + (size_t)i * cap;
      ctx->blobs[i].d = (uint8_t *)ctx->blob_arena_d + (size_t)i * cap;
      ctx->blobs[i].cap = cap;
    }
  }
  std::memcpy(slot.h, hb.bytes.data(), bytes);
  KV_CUDA(ctx, cudaMemcpyAsync(slot.d, slot.h, bytes, cudaMemcpyHostToDevice, s));
  ctx->memcpys++;
  // From here on the slot is in flight.  Its event must be recorded behind the last reader on EVERY way out of the
  // caller, failures included: BlobGuard (below) does that.
  slot.used = true;
  out->slot = &slot;
  out->d_bases = (const uint64_t *)slot.d;
  out->d_pieces = (const Piece *)((uint8_t *)slot.d + hb.off_pieces);
  out->h_pieces = (const Piece *)(hb.bytes.data() + hb.off_pieces);  // the caller's HostBlob outlives its launches
  out->d_ids = ids_on_device ? ids : (const int32_t *)((uint8_t *)slot.d + hb.off_ids);
  out->caller_ids = ids_on_device;
  return KV_OK;
}

// Records the slot's event on `s` when the caller's scope ends -- after the launches on the way out of a successful
// call, and equally after a launch / tensor-map failure in between, so that the slot is never reused on the strength
// of a stale or never-recorded event while its table copy or a kernel reading it may still be pending.
struct BlobGuard {
  kv_ctx *ctx; const Blob *b; cudaStream_t s;
  BlobGuard(kv_ctx *c, const Blob *bl, cudaStream_t st) : ctx(c), b(bl), s(st) {}
  ~BlobGuard() {
    if (!b->slot) return;
    if (cudaEventRecord(b->slot->ev, s) != cudaSuccess) {  // cannot order the slot's reuse behind its readers: drain them
      (void)cudaGetLastError();
      cudaStreamSynchronize(s);
      (void)cudaGetLastError();
      b->slot->used = false;
    }
  }
};


template <int N>
void launch_bulk(const Job &j, const HostBlob *hb, bool trans, uint32_t grid, uint32_t block, size_t smem,
                 cudaStream_t s, bool pdl) {
  static thread_local kvt::JobT<N> p;
  p.j = j;
  if constexpr (N > 0) std::memcpy(p.blob, hb->bytes.data(), hb->bytes.size());
  // Programmatic dependent launch: this grid may become resident while the previous kernel of the stream
  // is still draining (its CTAs leave half of each SM's shared memory free); it runs its prologue and then
  // blocks in griddepcontrol.wait until that kernel has completed and flushed.
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  if (trans) (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_bulk<N, true>, p);
  else (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_bulk<N, false>, p);
}
template <int N>
void launch_shot(const Job &j, const HostBlob *hb, bool trans, uint32_t grid, size_t smem, cudaStream_t s, bool pdl) {
  static thread_local kvt::JobT<N> p;
  p.j = j;
  if constexpr (N > 0) std::memcpy(p.blob, hb->bytes.data(), hb->bytes.size());
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  if (j.lean && !j.l2_hint) {  // the plain case (for an HND pool: whole boxes by tensor copies)
    if (trans) (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_shot_plain<N, true>, p);
    else (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_shot_plain<N, false>, p);
  } else if (trans) (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_shot<N, true>, p);
  else (void)cudaLaunchKernelEx(&cfg, kvt::kv_move_shot<N, false>, p);
}
template <int N>
void launch_vec(const Job &j, const HostBlob *hb, bool trans, uint32_t grid, cudaStream_t s) {
  static thread_local kvt::JobT<N> p;
  p.j = j;
  if constexpr (N > 0) std::memcpy(p.blob, hb->bytes.data(), hb->bytes.size());
  if (trans) kvt::kv_move_vec<8, N, true><<<grid, 256, 0, s>>>(p);
  else kvt::kv_move_vec<8, N, false><<<grid, 256, 0, s>>>(p);
}
template <int N>
void launch_small(const Job &j, const HostBlob *hb, uint32_t grid, cudaStream_t s) {
  static thread_local kvt::JobT<N> p;
  p.j = j;
  if constexpr (N > 0) std::memcpy(p.blob, hb->bytes.data(), hb->bytes.size());
  kvt::kv_move_small<N><<<grid, 256, 0, s>>>(p);
}
template <typename U>
void launch_elem(const kvt::JobT<0> &p, bool trans, uint32_t grid, cudaStream_t s) {
  if (trans) kvt::kv_move_elem<U, true><<<grid, 256, 0, s>>>(p);
  else kvt::kv_move_elem<U, false><<<grid, 256, 0, s>>>(p);
}

// lc0 / lc_count: the launch covers slabs [lc0, lc0 + lc_count) of the call only (layer-range chunks of the
// layer-first staged pipeline; tables in device memory); lc_count == 0: all of them.
int launch(kv_ctx *ctx, const Geom &g, const Blob &b, uint32_t piece_first, uint32_t n_pieces,
           uint64_t total_items, uint32_t cta_cap, cudaStream_t s, uint32_t lc0 = 0, uint32_t lc_count = 0) {
  if (!total_items) return KV_OK;
  Job j{};
  j.bases = b.d_bases ? b.d_bases + lc0 : nullptr; j.ids = b.d_ids;
  j.pieces = b.d_pieces ? b.d_pieces + piece_first : nullptr;
  if (b.inl) { j.off_pieces = (uint32_t)b.inl->off_pieces; j.off_ids = (uint32_t)b.inl->off_ids; }
  j.status = ctx->d_status;
  j.total_items = total_items;
  j.page_stride = g.page_stride; j.buf_row_bytes = g.buf_row; j.buf_page_bytes = g.buf_page;
  j.n_pieces = n_pieces; j.LC = lc_count ? lc_count : g.LC; j.dir = (uint32_t)g.dir; j.layout = (uint32_t)g.layout;
  j.g = g.g; j.cpp_pool = g.Tpool / g.g; j.cpp_buf = g.Tbuf / g.g;
  j.tokrow = g.tokrow; j.chunk_bytes = g.chunk_bytes; j.sub_bytes = g.sub_bytes; j.subs = g.subs;
  j.num_pages = g.num_pages;
  if (n_pieces == 1) {
    const Piece *hp = b.inl ? (const Piece *)(b.inl->bytes.data() + b.inl->off_pieces) : b.h_pieces;
    if (!hp) return KV_ERR_NULL;  // every Blob is built by build_blob / upload_blob, which keep the host copy
    j.one = hp[piece_first];
  }
  // the short decode path (kv_kernels.cuh Job::lean): host ids only (validated before any launch), nothing to zero-fill
  j.lean = 0;
  if ((g.dir == 0 || g.dir == 1) && g.layout == KV_LAYOUT_PAGE_FIRST && g.Tpool == g.Tbuf && !b.caller_ids &&
      (!g.trans || (g.tma && g.pool_hnd && g.kernel == KERNEL_SHOT && g.chunk_bytes % g.sub_bytes == 0)) &&
      total_items <= 0xffffffffull) {
    const Piece *hp = b.inl ? (const Piece *)(b.inl->bytes.data() + b.inl->off_pieces) : b.h_pieces;
    bool full = hp != nullptr && hp[piece_first].item_begin == 0;
    for (uint32_t k = 0; full && k < n_pieces; ++k)  // nothing to zero-fill in any request
      full = hp[piece_first + k].n_buf_pages * (uint64_t)g.Tbuf <= hp[piece_first + k].n_tokens;
    if (full) j.lean = n_pieces == 1 ? 1 : 2;
  }
  auto magic = [](uint32_t d) -> uint64_t { return d <= 1 ? 0ull : ~0ull / d + 1; };  // floor(2^64 / d) + 1 unless d | 2^64
  j.m_subs = magic(j.subs); j.m_LC = magic(j.LC); j.m_cpp_pool = magic(j.cpp_pool); j.m_cpp_buf = magic(j.cpp_buf);
  if (g.src_pool) { j.src_num_pages = g.src_pool->num_pages; j.src_page_stride = g.src_pool->page_stride_bytes; }
  j.src_ids = g.dev_src_ids;
  j.drow = g.drow; j.H = g.H;
  if (g.trans) {
    // the pool of this geometry is the destination pool of dir 2 and "the" pool otherwise; g.Tpool is its page size
    j.pool_hnd = g.pool_hnd; j.src_hnd = g.src_hnd;
    j.p_ts = g.drow; j.p_hs = (uint64_t)g.Tpool * g.drow;
    j.q_ts = g.drow; j.q_hs = (uint64_t)g.Tbuf * g.drow;  // dir 2: Tbuf is the source pool's page size
  }
  ctx->last_tma = 0;
  if (g.tma && is_async_kernel(g.kernel) && g.tma_inline) {
    if (!b.inl || (g.pool_hnd && !b.inl->off_maps_pool) || (g.src_hnd && !b.inl->off_maps_src)) return KV_ERR_CAPTURE;
    j.tb = g.tb;
    j.off_maps_pool = (uint32_t)b.inl->off_maps_pool;
    j.off_maps_src = (uint32_t)b.inl->off_maps_src;
    ctx->last_tma = 1;
  } else if (g.tma && is_async_kernel(g.kernel)) {
    j.tb = g.tb;
    if (g.pool_hnd) {
      int rc = get_maps(ctx, g.dst_pool, g.L, g.tb, g.tma_es, &j.maps_pool);
      if (rc) return rc;
    }
    if (g.src_hnd) {
      int rc = get_maps(ctx, g.src_pool, g.L, g.tb, g.tma_es, &j.maps_src);
      if (rc) return rc;
    }
    if (j.maps_pool) j.maps_pool += (size_t)lc0 * sizeof(CUtensorMap);
    ctx->last_tma = 1;
  }
  uint32_t cap = cta_cap ? cta_cap : ctx->max_ctas;
  uint32_t grid = 0;
  if (g.kernel == KERNEL_SHOT) {
    // one segment per single-warp CTA; the grid is the item list (capped only on request: a CTA then walks its items)
    j.stage_bytes = (g.sub_bytes + 127) / 128 * 128;
    j.l2_hint = ctx->l2_hint;
    grid = (uint32_t)std::min<uint64_t>(total_items, cap ? cap : 0x7fffffffu);
    const bool pdl = ctx->pdl && !ctx->cur_capturing;
    if (!b.inl) launch_shot<0>(j, nullptr, g.trans, grid, j.stage_bytes, s, pdl);
    else if (b.inl->bytes.size() <= kInlineSmall) launch_shot<kInlineSmall>(j, b.inl, g.trans, grid, j.stage_bytes, s, pdl);
    else launch_shot<kInlineLarge>(j, b.inl, g.trans, grid, j.stage_bytes, s, pdl);
  } else if (g.kernel == KERNEL_BULK) {
    const bool lane_geom = g.trans && !g.tma;  // row gathers by all lanes want more, shallower warps
    j.stage_bytes = (g.sub_bytes + 127) / 128 * 128;
    j.stages = lane_geom ? ctx->t_stages : ctx->stages; j.lag = std::min(ctx->lag, j.stages - 1);
    j.zero_bytes = std::min<uint32_t>(4096, j.stage_bytes);
    j.l2_hint = ctx->l2_hint;
    uint32_t warps = lane_geom ? ctx->t_warps : ctx->warps;
    if (!lane_geom && ctx->auto_geom && j.stage_bytes < 16384) {
      // Narrow rows (a tensor-parallel head partition: 1 KV head = 4 KiB rows, 2 heads = 8 KiB): what saturates HBM is
      // the BYTES in flight per SM (~128 KiB of stages), so smaller stages need more of them.  Measured on B200,
      // 768 MiB back to back: 4 KiB rows 3.46 TB/s with the 2 x 4 ring, 6.2 with 8 x 4; 8 KiB rows 5.09 -> 6.24 with
      // 4 x 4.  Launch-sized calls keep the 2-warp ring (more CTAs, each with little to do).
      const uint32_t total = 131072u / j.stage_bytes;          // stages per SM
      const uint32_t w = std::min<uint32_t>(kvt::kMaxWarps, std::max<uint32_t>(2, total / 4));
      if (total_items >= 4ull * ctx->sm_count * w) {
        warps = w;
        j.stages = std::min<uint32_t>(kvt::kMaxStages, std::max<uint32_t>(4, total / w));
        j.lag = std::min(ctx->lag, j.stages - 1);
      }
    }
    size_t smem = (size_t)j.zero_bytes + (size_t)warps * j.stages * j.stage_bytes;
    while (smem > (size_t)ctx->max_smem - kStaticSmemReserve && j.stages > 2) {  // static smem holds barriers + meta
      --j.stages; j.lag = std::min(j.lag, j.stages - 1);
      smem = (size_t)j.zero_bytes + (size_t)warps * j.stages * j.stage_bytes;
    }
    while (smem > (size_t)ctx->max_smem - kStaticSmemReserve && warps > 1) {
      --warps;
      smem = (size_t)j.zero_bytes + (size_t)warps * j.stages * j.stage_bytes;
    }
    const uint64_t want = (total_items + warps - 1) / warps;
    grid = (uint32_t)std::min<uint64_t>(want, cap ? cap : (uint32_t)ctx->sm_count);
    const uint64_t G = (uint64_t)grid * warps;
    if (ctx->dynamic && total_items >= 8 * G && !ctx->cur_capturing) {  // enough work for claiming to pay
      uint8_t *slot = (uint8_t *)ctx->d_status + 256 + (size_t)(ctx->next_sched++ % kSchedSlots) * 16;
      j.sched = (unsigned long long *)slot;
      j.sched_done = (uint32_t *)(slot + 8);
      j.first_batch = (uint32_t)std::min<uint64_t>(32, total_items / (4 * G));
    }
    const bool pdl = ctx->pdl && !ctx->cur_capturing;
    if (!b.inl) launch_bulk<0>(j, nullptr, g.trans, grid, warps * 32, smem, s, pdl);
    else if (b.inl->bytes.size() <= kInlineSmall) launch_bulk<kInlineSmall>(j, b.inl, g.trans, grid, warps * 32, smem, s, pdl);
    else launch_bulk<kInlineLarge>(j, b.inl, g.trans, grid, warps * 32, smem, s, pdl);
  } else {
    const uint32_t wpb = 8;  // warps per 256-thread CTA
    const uint64_t want = (total_items + wpb - 1) / wpb;
    grid = (uint32_t)std::min<uint64_t>(want, cap ? cap : (uint32_t)ctx->sm_count * 8);
    kvt::JobT<0> p0;
    p0.j = j;
    if (g.kernel == KERNEL_VEC && !g.trans && g.dir != 3 && g.sub_bytes <= 1024) {
      // segments of <= 1 KiB: 32 of them per warp and pass (kv_move_small)
      grid = (uint32_t)std::min<uint64_t>((total_items + wpb * 32 - 1) / (wpb * 32), cap ? cap : (uint32_t)ctx->sm_count * 8);
      if (!b.inl) launch_small<0>(j, nullptr, grid, s);
      else if (b.inl->bytes.size() <= kInlineSmall) launch_small<kInlineSmall>(j, b.inl, grid, s);
      else launch_small<kInlineLarge>(j, b.inl, grid, s);
    } else if (g.kernel == KERNEL_VEC) {
      if (!b.inl) launch_vec<0>(j, nullptr, g.trans, grid, s);
      else if (b.inl->bytes.size() <= kInlineSmall) launch_vec<kInlineSmall>(j, b.inl, g.trans, grid, s);
      else launch_vec<kInlineLarge>(j, b.inl, g.trans, grid, s);
    }
    else if (g.unit >= 8) launch_elem<uint64_t>(p0, g.trans, grid, s);
    else if (g.unit == 4) launch_elem<uint32_t>(p0, g.trans, grid, s);
    else if (g.unit == 2) launch_elem<uint16_t>(p0, g.trans, grid, s);
    else launch_elem<uint8_t>(p0, g.trans, grid, s);
  }
  KV_CUDA(ctx, cudaGetLastError());
  ctx->launches++;
  ctx->last_grid = grid;
  ctx->last_plain = g.kernel == KERNEL_SHOT && j.lean && !j.l2_hint;
  return KV_OK;
}

}  // namespace
