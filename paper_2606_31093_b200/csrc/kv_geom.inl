// kv_geom.inl -- descriptor checks, tensor maps of HND pools, and the geometry of a call (what a segment is, which kernel moves it)
// Part of the host side of libkvtier.so; included by kvtier.cu only (one translation unit).
// Shares nothing with oracle/.
#pragma once

namespace {

// Geometry of one call: everything derived from the descriptor, the buffer page size and the
// kernel options; no pointers to transfer data.
struct Geom {
  uint32_t L = 0, C = 0, LC = 0;
  uint32_t Tpool = 0, Tbuf = 0, g = 0;
  uint32_t tokrow = 0, chunk_bytes = 0, sub_bytes = 0, subs = 0;
  uint64_t pool_row = 0, buf_row = 0, buf_page = 0;
  uint64_t page_stride = 0;
  uint32_t num_pages = 0, elem = 0;
  int dir = 0, layout = 0;
  int kernel = KERNEL_BULK;
  uint32_t unit = 16;  // widest power of two dividing every address/length (elem kernel)
  // dir 2 (pool -> pool): the source pool; its bases follow the destination's in the tables
  const kv_pool_desc *src_pool = nullptr;
  const kv_pool_desc *dst_pool = nullptr;  // the pool of the call (destination pool of dir 2)
  const int32_t *dev_src_ids = nullptr;    // dir 2 with device-resident ids: the source list
  // an HND pool on either side makes the transfer a [token] x [head] transposition (kTrans kernels)
  bool trans = false;
  uint32_t drow = 0, H = 0, pool_hnd = 0, src_hnd = 0;
  // HND sides served by tensor copies: box of `tb` whole tokens, element width `tma_es` bytes
  bool tma = false;
  uint32_t tb = 0, tma_es = 0;
  // the maps travel inside the kernel parameters (a captured call whose pool has no maps in device memory yet)
  bool tma_inline = false;
};

struct Req {          // one request as the caller states it
  uint64_t buf = 0;   // transfer buffer (device-accessible address)
  uint64_t n_tokens = 0;
  uint64_t id_begin = 0, n_ids = 0;  // its page ids in the call's id array
  uint64_t n_buf_pages = 0;
  uint64_t items = 0;  // work items of this request (filled by the planners)
  uint32_t dir = 0;    // kv_submit only: this request's direction (0 pack, 1 unpack, 3 copy-on-write append)
};

int check_desc(const kv_pool_desc *p, uint32_t layer_count) {
  if (!p || !p->base) return KV_ERR_NULL;
  if (!p->layer_count || !p->kv_count || !p->num_pages || !p->page_size || !p->num_heads ||
      !p->head_dim || p->order > KV_ORDER_HND)
    return KV_ERR_DESC;
  if (p->elem_bytes != 1 && p->elem_bytes != 2 && p->elem_bytes != 4 && p->elem_bytes != 8)
    return KV_ERR_DESC;
  if (!layer_count || layer_count > p->layer_count) return KV_ERR_DESC;
  if ((uint64_t)p->layer_count * p->kv_count > kMaxLayersKv) return KV_ERR_DESC;
  const uint64_t row = (uint64_t)p->page_size * p->num_heads * p->head_dim * p->elem_bytes;
  if (row > 0xFFFFFFFFull) return KV_ERR_DESC;
  if (p->page_stride_bytes < row) return KV_ERR_DESC;
  if (p->page_stride_bytes % p->elem_bytes) return KV_ERR_ALIGN;
  for (uint64_t i = 0; i < (uint64_t)layer_count * p->kv_count; ++i) {
    if (!p->base[i]) return KV_ERR_NULL;
    if ((uint64_t)(uintptr_t)p->base[i] % p->elem_bytes) return KV_ERR_ALIGN;
  }
  return KV_OK;
}

// Is `s` being captured into a CUDA graph?  Captured launches must be self-contained: tables inline
// in the kernel parameters (a staged table copy would read the ctx's pinned ring at REPLAY time),
// static work distribution (a baked claim-counter slot could be shared with a live launch).
bool capturing(cudaStream_t s) {
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(s, &st) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return st != cudaStreamCaptureStatusNone;
}
// Every entry point that may launch calls this first: one capture query per call, not one per launch.
void enter(kv_ctx *ctx, kv_stream_t stream) {
  if (!ctx) return;
  ctx->cur_stream = (cudaStream_t)stream;
  ctx->cur_capturing = !ctx->host_only && capturing(ctx->cur_stream);
}

uint32_t gcd32(uint32_t a, uint32_t b) {
  while (b) { uint32_t t = a % b; a = b; b = t; }
  return a;
}

uint32_t low_pow2(uint64_t v) {  // largest power of two (<= 16) dividing v; 16 for v == 0
  uint32_t u = 16;
  while (u > 1 && (v % u)) u >>= 1;
  return u;
}

// ---- tensor maps of HND pools ----------------------------------------------------------------
void map_key(const kv_pool_desc *p, uint32_t layer_count, uint32_t tb, uint32_t es, std::vector<uint64_t> *k) {
  const uint32_t LC = layer_count * p->kv_count;
  k->clear();
  k->reserve(LC + 8);
  const uint64_t f[8] = {LC, p->num_pages, p->page_size, p->num_heads, (uint64_t)p->head_dim * p->elem_bytes,
                         p->page_stride_bytes, tb, es};
  k->insert(k->end(), f, f + 8);
  for (uint32_t i = 0; i < LC; ++i) k->push_back((uint64_t)(uintptr_t)p->base[i]);
}

const MapSet *find_maps(const kv_ctx *ctx, const std::vector<uint64_t> &key) {
  for (const MapSet &m : ctx->map_sets)
    if (m.key == key) return &m;
  return nullptr;
}

// Smallest element width that keeps the innermost box dimension within the 256-element limit.
uint32_t tma_elem_bytes(uint32_t drow) {
  for (uint32_t es : {1u, 2u, 4u, 8u})
    if (drow % es == 0 && drow / es <= 256) return es;
  return 0;
}

// Tensor maps of slabs [lc0, lc0 + lc_n) of pool `p` (slab = tensor (dim, head, token, page), box (drow, H, tb, 1)),
// written to `maps`.  Pure host work: no CUDA call, so it is legal while a stream is being captured.
int encode_maps(kv_ctx *ctx, const kv_pool_desc *p, uint32_t lc0, uint32_t lc_n, uint32_t tb, uint32_t es, CUtensorMap *maps) {
  const uint32_t drow = p->head_dim * p->elem_bytes;
  static const CUtensorMapDataType kTypes[9] = {CU_TENSOR_MAP_DATA_TYPE_UINT8, CU_TENSOR_MAP_DATA_TYPE_UINT8,
      CU_TENSOR_MAP_DATA_TYPE_UINT16, CU_TENSOR_MAP_DATA_TYPE_UINT16, CU_TENSOR_MAP_DATA_TYPE_UINT32,
      CU_TENSOR_MAP_DATA_TYPE_UINT32, CU_TENSOR_MAP_DATA_TYPE_UINT32, CU_TENSOR_MAP_DATA_TYPE_UINT32,
      CU_TENSOR_MAP_DATA_TYPE_UINT64};
  const cuuint64_t dims[4] = {drow / es, p->num_heads, p->page_size, p->num_pages};
  const cuuint64_t strides[3] = {(cuuint64_t)p->page_size * drow, drow, p->page_stride_bytes};
  const cuuint32_t box[4] = {drow / es, p->num_heads, tb, 1};
  const cuuint32_t ones[4] = {1, 1, 1, 1};
  for (uint32_t i = 0; i < lc_n; ++i) {
    CUresult r = ctx->encode_tiled(&maps[i], kTypes[es], 4, p->base[lc0 + i], dims, strides, box, ones,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { ctx->last_cuda_error = (int)r; return KV_ERR_CUDA; }
  }
  return KV_OK;
}

// Device array of LC tensor maps for pool `p`, cached in the ctx per (pool, box).  Built on first use: LC encoder calls +
// one blocking copy; never during stream capture (a captured call carries its maps in its parameters instead).
int get_maps(kv_ctx *ctx, const kv_pool_desc *p, uint32_t layer_count, uint32_t tb, uint32_t es, const uint8_t **out) {
  std::vector<uint64_t> key;
  map_key(p, layer_count, tb, es, &key);
  if (const MapSet *m = find_maps(ctx, key)) { *out = (const uint8_t *)m->d; return KV_OK; }
  const uint32_t LC = layer_count * p->kv_count;
  std::vector<CUtensorMap> maps(LC);
  int rc = encode_maps(ctx, p, 0, LC, tb, es, maps.data());
  if (rc) return rc;
  if (ctx->map_sets.size() >= kMaxMapSets) {  // rare: drop everything once nothing can still be reading it
    KV_CUDA(ctx, cudaDeviceSynchronize());
    for (MapSet &m : ctx->map_sets) cudaFree(m.d);
    ctx->map_sets.clear();
  }
  MapSet ms;
  ms.key = key;
  KV_CUDA(ctx, cudaMalloc(&ms.d, (size_t)LC * sizeof(CUtensorMap)));
  cudaError_t e = cudaMemcpy(ms.d, maps.data(), (size_t)LC * sizeof(CUtensorMap), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(ms.d); ctx->last_cuda_error = (int)e; (void)cudaGetLastError(); return KV_ERR_CUDA; }
  ctx->map_sets.push_back(ms);
  *out = (const uint8_t *)ms.d;
  return KV_OK;
}

// Can the HND side(s) of this geometry move by tensor copies?  (Planning only: no CUDA calls except
// the capture query.)  While `cur_stream` is being captured, only maps already in the cache may be used.
bool tma_eligible(const kv_ctx *ctx, const kv_pool_desc *p, const kv_pool_desc *src_pool, uint32_t layer_count,
                  uint32_t gtok, uint64_t tokrow, uint32_t drow, uint32_t cap, uint32_t *tb_out, uint32_t *es_out) {
  if (!ctx->tensor_maps || !ctx->encode_tiled) return false;
  const uint32_t es = tma_elem_bytes(drow);
  if (!es || (drow % 16) || p->num_heads > 256 || tokrow > cap) return false;
  uint32_t tb = (uint32_t)std::min<uint64_t>(std::min<uint64_t>(gtok, 256), cap / tokrow);
  while (tb > 1 && gtok % tb) --tb;  // boxes tile the chunk exactly
  auto side_ok = [&](const kv_pool_desc *q) {
    return q->page_stride_bytes % 16 == 0 && q->page_stride_bytes < (1ull << 40) &&
           (uint64_t)q->page_size * drow < (1ull << 40);
  };
  if (!side_ok(p) || (src_pool && !side_ok(src_pool))) return false;
  *tb_out = tb; *es_out = es;
  return true;
}

int make_geom(const kv_ctx *ctx, const kv_pool_desc *p, uint32_t layer_count, uint32_t Tbuf,
              int dir, int layout, const std::vector<Req> &reqs, Geom *out,
              const kv_pool_desc *src_pool = nullptr) {
  if (layout != KV_LAYOUT_PAGE_FIRST && layout != KV_LAYOUT_LAYER_FIRST) return KV_ERR_LAYOUT;
  Geom g;
  g.L = layer_count; g.C = p->kv_count; g.LC = g.L * g.C;
  g.dst_pool = p;
  g.Tpool = p->page_size; g.Tbuf = Tbuf;
  g.g = gcd32(g.Tpool, g.Tbuf);
  g.elem = p->elem_bytes;
  const uint64_t tokrow = (uint64_t)p->num_heads * p->head_dim * p->elem_bytes;
  g.tokrow = (uint32_t)tokrow;
  g.pool_row = tokrow * g.Tpool;
  g.buf_row = tokrow * g.Tbuf;
  if (g.buf_row > 0xFFFFFFFFull) return KV_ERR_SIZE;
  g.buf_page = g.buf_row * g.LC;
  g.chunk_bytes = (uint32_t)(tokrow * g.g);
  g.page_stride = p->page_stride_bytes;
  g.num_pages = p->num_pages;
  g.dir = dir; g.layout = layout;
  // widest unit every address and length of this call is a multiple of
  uint32_t unit = 16;
  unit = std::min(unit, low_pow2(tokrow));
  unit = std::min(unit, low_pow2(g.page_stride));
  for (uint32_t i = 0; i < g.LC; ++i) unit = std::min(unit, low_pow2((uint64_t)(uintptr_t)p->base[i]));
  if (dir != 2)  // dir 2 keeps an id index in Req::buf, not an address
    for (const Req &r : reqs) {
      if (r.buf % g.elem) return KV_ERR_ALIGN;
      unit = std::min(unit, low_pow2(r.buf));
    }
  if (src_pool) {
    g.src_pool = src_pool;
    unit = std::min(unit, low_pow2(src_pool->page_stride_bytes));
    for (uint32_t i = 0; i < g.LC; ++i) unit = std::min(unit, low_pow2((uint64_t)(uintptr_t)src_pool->base[i]));
  }
  g.H = p->num_heads;
  g.drow = p->head_dim * p->elem_bytes;
  // With one head, or one token per page, [token][head] and [head][token] are the same bytes.
  auto is_hnd = [](const kv_pool_desc *q) { return q->order == KV_ORDER_HND && q->num_heads > 1 && q->page_size > 1; };
  g.pool_hnd = is_hnd(p); g.src_hnd = src_pool && is_hnd(src_pool);
  g.trans = g.pool_hnd || g.src_hnd;
  if (g.trans) unit = std::min(unit, low_pow2(g.drow));  // rows are moved one by one
  g.unit = unit;
  int kernel = ctx->kernel;
  if (unit < 16) kernel = KERNEL_ELEM;  // 16-byte paths need 16-byte alignment everywhere
  if (g.trans && dir != 3 && kernel != KERNEL_ELEM && kernel != KERNEL_VEC) {
    // HND sides by tensor copies: the bulk ring with its contiguous-path geometry, one box per item
    uint32_t tb = 0, es = 0;
    const uint32_t cap16 = std::max(16u, ctx->stage_bytes / 16 * 16);
    if (tma_eligible(ctx, p, g.src_hnd ? src_pool : nullptr, layer_count, g.g, tokrow, g.drow, cap16, &tb, &es)) {
      bool cached_or_free = true;
      if (!ctx->host_only && ctx->cur_capturing) {
        std::vector<uint64_t> key;
        if (g.pool_hnd) { map_key(p, layer_count, tb, es, &key); cached_or_free = find_maps(ctx, key) != nullptr; }
        if (cached_or_free && g.src_hnd) { map_key(src_pool, layer_count, tb, es, &key); cached_or_free = find_maps(ctx, key) != nullptr; }
      }
      if (cached_or_free) {
        g.tma = true; g.tb = tb; g.tma_es = es;
      } else if (ctx->inline_tables) {
        // Capturing, and (one of) the pool(s) has no maps in device memory yet: encode them on the host and let them
        // ride in the kernel parameters beside the tables, if everything fits there (one-request device transfers and
        // DIRECT host transfers always do at the paper's shapes: 96 slabs x 128 B = 12 KiB).  Otherwise: lane paths.
        uint64_t n_ids = 0;
        for (const Req &r : reqs) n_ids += r.n_ids + (dir == 2 ? r.n_buf_pages : 0);
        const uint64_t tables = (uint64_t)g.LC * 8 * (src_pool ? 2 : 1) + reqs.size() * sizeof(Piece) + n_ids * 4;
        const uint64_t maps = (uint64_t)g.LC * sizeof(CUtensorMap) * ((g.pool_hnd ? 1 : 0) + (g.src_hnd ? 1 : 0));
        if (tables + 128 + maps <= (uint64_t)kInlineLarge) { g.tma = true; g.tma_inline = true; g.tb = tb; g.tma_es = es; }
      }
    }
  }
  if (kernel == KERNEL_AUTO) {
    // One segment per single-warp CTA (kv_move_shot) wherever a segment is at least 4 KiB: measured on B200 against the
    // persistent ring and the 16-byte LDG/STG kernel (round 2) it is ahead on every such shape --
    // 768 MiB back to back 6.64 vs 6.38 / 6.01 TB/s at 16 KiB rows, 6.63 vs 6.19 / 5.95 at 4 KiB rows, HND pools with
    // tensor maps 6.62 vs 6.33, HND lane paths 6.58 / 6.48 vs 6.13 / 4.25, copy-on-write batches 5.6 vs 3.3 / 5.2 -- and
    // on every size from 1 MiB (7.2 vs 9.2 us isolated) to 1 GiB (320 vs 331 us).  Below 4 KiB the rate at which an SM
    // retires bulk copies takes over (about 11 M a second): 2 KiB segments 3.9 TB/s against the ring's 6.2 (more,
    // shallower stages per SM), 1 KiB 2.0 against kv_move_small's 6.0.
    const uint32_t cap16 = std::max(16u, ctx->stage_bytes / 16 * 16);
    uint32_t seg = std::min(g.chunk_bytes, cap16);
    if (g.tma) seg = g.tb * g.tokrow;
    else if (g.trans) seg = std::min(g.chunk_bytes, std::max(g.drow, cap16 / g.drow * g.drow));
    if (dir == 3) seg = (uint32_t)std::min<uint64_t>(g.pool_row / 2, cap16);  // ragged pieces: half a page row on average
    const bool shot = seg >= kShotMinSegment && (!g.trans || g.drow <= cap16);
    if (shot) {
      kernel = KERNEL_SHOT;
    } else {
      // Short segments.  Paths without tensor maps on an HND pool: a strided DESTINATION is fastest with 16-byte STG from
      // many warps (vec); a strided source alone gathered by cp.async into the bulk ring; everything contiguous: the ring,
      // re-shaped for narrow rows (kv_launch.inl).
      const bool dst_strided = g.pool_hnd && dir != 0;
      kernel = (dst_strided && !g.tma) ? KERNEL_VEC : KERNEL_BULK;  // small tensor boxes: the ring, as before
      if (!g.trans && dir != 3) {
        uint64_t bytes = 0;
        for (const Req &r : reqs) bytes += r.n_ids * g.pool_row * g.LC;
        // Segments of 1 KiB or less (one-token pages; re-paging between page sizes with no common divisor): an SM
        // retires small bulk copies too slowly (3.4 TB/s at 1 KiB); kv_move_small (32 segments decoded per warp at once,
        // copied eight at a time) does 6.05-6.15 TB/s.  From 2 KiB the re-shaped ring is back at 6.2 TB/s.
        if (g.chunk_bytes <= 1024 && bytes >= (8ull << 20)) kernel = KERNEL_VEC;
      } else if (!g.trans) {
        // copy-on-write appends on narrow token rows: many short, ragged pieces; one warp per piece with 16-byte loads
        // beats one bulk copy per piece from ~16 MiB
        uint64_t bytes = 0;
        for (const Req &r : reqs) bytes += ((r.n_tokens & 0xffffffffull) + (r.n_tokens >> 32)) * tokrow * g.LC;
        if (bytes >= (16ull << 20)) kernel = KERNEL_VEC;
      }
    }
  }
  if (!is_async_kernel(kernel)) g.tma = false;  // tensor copies exist in the shared-memory kernels only
  uint32_t cap = kernel == KERNEL_BULK ? (g.trans && !g.tma ? ctx->t_stage_bytes : ctx->stage_bytes)
                 : (kernel == KERNEL_SHOT ? ctx->stage_bytes : 16384u);
  cap = std::max(16u, cap / 16 * 16);
  if (g.trans && is_async_kernel(kernel) && g.drow > cap) kernel = KERNEL_VEC;  // a row must fit one stage
  g.kernel = kernel;
  g.sub_bytes = std::min(g.chunk_bytes, cap);
  if (!g.trans && g.chunk_bytes > cap && g.chunk_bytes % 16 == 0) {
    // A row a little longer than a stage (say 17,280 B) would be cut into one full stage and a 896-byte crumb, and
    // crumbs are copied at the small-copy rate.  Cut it into equal pieces instead (two of 8,704 / 8,576 B):
    // measured on a 5-token x 3-head x 576-dim pool: 4.96 -> 6.05 TB/s; 20 KiB rows: 5.4 -> 6.2.
    const uint32_t n = (g.chunk_bytes + cap - 1) / cap;
    const uint32_t even = ((g.chunk_bytes + n - 1) / n + 127) / 128 * 128;
    if (even <= cap) g.sub_bytes = even;
  }
  if (g.trans) g.sub_bytes = std::min(g.chunk_bytes, std::max(g.drow, cap / g.drow * g.drow));  // whole rows
  if (g.tma) g.sub_bytes = g.tb * g.tokrow;  // whole tokens: one box
  if (is_async_kernel(kernel) && dir != 3) {
    // Launch-bound calls: with fewer segments than issuing warps most SMs would idle while a few
    // move 16 KiB each; cutting segments down to >= 4 KiB spreads a small transfer over the chip
    // (measured on B200, 1 MiB pack back to back: 6.1 -> 5.0 us per call).
    uint64_t chunks = 0;
    for (const Req &r : reqs) chunks += r.n_ids * (g.Tpool / g.g) * g.LC;
    const uint64_t lanes = (uint64_t)ctx->sm_count * (kernel == KERNEL_SHOT ? 2 : (g.trans && !g.tma ? ctx->t_warps : ctx->warps));
    while (g.sub_bytes >= 8192 && g.sub_bytes % 32 == 0 && (!g.trans || (g.sub_bytes / 2) % g.drow == 0) &&
           (!g.tma || g.tb % 2 == 0) &&
           chunks * ((g.chunk_bytes + g.sub_bytes - 1) / g.sub_bytes) * 2 <= lanes) {
      g.sub_bytes /= 2;
      if (g.tma) g.tb /= 2;
    }
  }
  g.subs = (g.chunk_bytes + g.sub_bytes - 1) / g.sub_bytes;
  *out = g;
  return KV_OK;
}

uint64_t items_of(const Geom &g, uint64_t n_pool_pages) {
  return n_pool_pages * (g.Tpool / g.g) * g.LC * g.subs;
}

int check_ids(const int32_t *ids, uint64_t n, uint32_t num_pages) {
  for (uint64_t i = 0; i < n; ++i)
    if (ids[i] < 0 || (uint32_t)ids[i] >= num_pages) return KV_ERR_PAGE_RANGE;
  return KV_OK;
}

int check_dups(const int32_t *ids, uint64_t n, uint32_t num_pages) {
  std::vector<uint8_t> seen((size_t)(num_pages + 7) / 8, 0);
  for (uint64_t i = 0; i < n; ++i) {
    const uint32_t g = (uint32_t)ids[i];
    if (seen[g >> 3] & (1u << (g & 7))) return KV_ERR_DUP_PAGE;
    seen[g >> 3] |= (uint8_t)(1u << (g & 7));
  }
  return KV_OK;
}

}  // namespace
