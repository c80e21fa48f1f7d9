// kvtier.cu -- C ABI (include/kvtier.h) of the paged-KV tier transfer: host validation, page-id
// staging, planning of the flat segment list (a2) and launches (a3-a8).
// Every byte of the path is moved by the kernels in kv_kernels.cuh or, in KV_HOST_STAGED mode,
// by the copy engines between the ctx's device staging and pinned host memory.
// There is no CPU fallback: without a CUDA device transfer calls fail (KV_ERR_CUDA / NO_DEVICE).
#include "../../include/kvtier.h"

#include <cuda.h>  // CUtensorMap types only; the encoder is fetched through cudaGetDriverEntryPoint
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <new>
#include <numeric>
#include <vector>

#include "kv_chain.cuh"
#include "kv_kernels.cuh"

namespace {

using kvt::Job;
using kvt::Piece;

constexpr int kBlobSlots = 16;
constexpr int kMaxStagingSlots = 4;
constexpr uint32_t kMaxLayersKv = 4096;  // layer_count * kv_count
constexpr uint64_t kAutoStagedMinBytes = 16ull << 20;
constexpr uint64_t kAutoVecMinBytes = 40ull << 20, kAutoVecMaxBytes = 384ull << 20;  // AUTO: vec kernel in between
constexpr uint32_t kSchedSlots = 256;  // claim counters, handed out round-robin per launch
constexpr int kStaticSmemReserve = 8192;  // static shared memory of kv_move_bulk (barriers + stage metadata, 6 KiB) rounded up

enum KernelKind { KERNEL_AUTO = 0, KERNEL_BULK = 1, KERNEL_VEC = 2, KERNEL_ELEM = 3 };

// Tensor maps of one HND pool for one box size (kv_kernels.cuh "TMA tensor maps"): built once per
// (pool, box) and kept in device memory for the life of the ctx.
struct MapSet {
  std::vector<uint64_t> key;  // slab bases + every descriptor field the maps depend on + box tokens
  void *d = nullptr;          // device array of LC CUtensorMap
};
constexpr size_t kMaxMapSets = 64;
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct BlobSlot {
  void *h = nullptr;  // pinned host
  void *d = nullptr;  // device
  size_t cap = 0;
  cudaEvent_t ev = nullptr;  // recorded after the last kernel that reads `d`
  bool used = false;
};

}  // namespace

struct kv_ctx {
  int device = -1;
  bool host_only = false;
  int sm_count = 148;
  int max_smem = 0;
  cudaStream_t side = nullptr;
  cudaEvent_t ev_entry = nullptr;
  BlobSlot blobs[kBlobSlots];
  uint32_t next_blob = 0;
  uint32_t *d_status = nullptr;
  // staging for KV_HOST_STAGED
  void *staging = nullptr;
  size_t staging_bytes = 0;
  cudaEvent_t ev_full[kMaxStagingSlots] = {};  // producer into the slot finished
  cudaEvent_t ev_free[kMaxStagingSlots] = {};  // consumer of the slot finished
  bool free_valid[kMaxStagingSlots] = {};
  int last_cuda_error = 0;
  // options
  int kernel = KERNEL_AUTO;
  uint32_t stage_bytes = 16384, stages = 4, warps = 2, lag = 2, max_ctas = 0, host_max_ctas = 0;
  // bulk geometry of transposing transfers (an HND pool): rows are gathered with 16-byte cp.async by all
  // lanes, which wants more, shallower issuing warps (measured: 8 x 4 x 4 KiB)
  uint32_t t_stage_bytes = 4096, t_stages = 4, t_warps = 8;
  uint32_t staging_slots = 2, l2_hint = 0, inline_tables = 1, dynamic = 1, tensor_maps = 1, pdl = 1;
  uint32_t next_sched = 0;
  EncodeTiledFn encode_tiled = nullptr;  // cuTensorMapEncodeTiled, nullptr if the driver has none
  std::vector<MapSet> map_sets;
  cudaStream_t cur_stream = nullptr;     // stream of the entry point being served (capture check while planning)
  uint64_t last_tma = 0;
  size_t chunk_bytes = 0;
  // stats
  uint64_t launches = 0, memcpys = 0, last_items = 0, last_payload = 0, last_kernel = 0,
           last_mode = 0, last_grid = 0, last_segment = 0;
};

namespace {

#define KV_CUDA(ctx, expr)                         \
  do {                                             \
    cudaError_t e__ = (expr);                      \
    if (e__ != cudaSuccess) {                      \
      (ctx)->last_cuda_error = (int)e__;           \
      (void)cudaGetLastError();                    \
      return KV_ERR_CUDA;                          \
    }                                              \
  } while (0)

struct DeviceGuard {
  int prev = -1;
  bool active = false;
  explicit DeviceGuard(const kv_ctx *ctx) {
    if (ctx->host_only) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) {
      cudaSetDevice(ctx->device);
      active = true;
    }
  }
  ~DeviceGuard() {
    if (active) cudaSetDevice(prev);
  }
};

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
};

struct Req {          // one request as the caller states it
  uint64_t buf = 0;   // transfer buffer (device-accessible address)
  uint64_t n_tokens = 0;
  uint64_t id_begin = 0, n_ids = 0;  // its page ids in the call's id array
  uint64_t n_buf_pages = 0;
  uint64_t items = 0;  // work items of this request (filled by the planners)
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

// Device array of LC tensor maps for pool `p` (slab = tensor (dim, head, token, page), box (drow, H, tb, 1)).
// Built on first use: LC encoder calls + one blocking copy; never during stream capture (the caller checks).
int get_maps(kv_ctx *ctx, const kv_pool_desc *p, uint32_t layer_count, uint32_t tb, uint32_t es, const uint8_t **out) {
  std::vector<uint64_t> key;
  map_key(p, layer_count, tb, es, &key);
  if (const MapSet *m = find_maps(ctx, key)) { *out = (const uint8_t *)m->d; return KV_OK; }
  const uint32_t LC = layer_count * p->kv_count;
  const uint32_t drow = p->head_dim * p->elem_bytes;
  static const CUtensorMapDataType kTypes[9] = {CU_TENSOR_MAP_DATA_TYPE_UINT8, CU_TENSOR_MAP_DATA_TYPE_UINT8,
      CU_TENSOR_MAP_DATA_TYPE_UINT16, CU_TENSOR_MAP_DATA_TYPE_UINT16, CU_TENSOR_MAP_DATA_TYPE_UINT32,
      CU_TENSOR_MAP_DATA_TYPE_UINT32, CU_TENSOR_MAP_DATA_TYPE_UINT32, CU_TENSOR_MAP_DATA_TYPE_UINT32,
      CU_TENSOR_MAP_DATA_TYPE_UINT64};
  std::vector<CUtensorMap> maps(LC);
  const cuuint64_t dims[4] = {drow / es, p->num_heads, p->page_size, p->num_pages};
  const cuuint64_t strides[3] = {(cuuint64_t)p->page_size * drow, drow, p->page_stride_bytes};
  const cuuint32_t box[4] = {drow / es, p->num_heads, tb, 1};
  const cuuint32_t ones[4] = {1, 1, 1, 1};
  for (uint32_t i = 0; i < LC; ++i) {
    CUresult r = ctx->encode_tiled(&maps[i], kTypes[es], 4, p->base[i], dims, strides, box, ones,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { ctx->last_cuda_error = (int)r; return KV_ERR_CUDA; }
  }
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
      if (!ctx->host_only && capturing(ctx->cur_stream)) {
        std::vector<uint64_t> key;
        if (g.pool_hnd) { map_key(p, layer_count, tb, es, &key); cached_or_free = find_maps(ctx, key) != nullptr; }
        if (cached_or_free && g.src_hnd) { map_key(src_pool, layer_count, tb, es, &key); cached_or_free = find_maps(ctx, key) != nullptr; }
      }
      if (cached_or_free) { g.tma = true; g.tb = tb; g.tma_es = es; kernel = KERNEL_BULK; }
    }
  }
  if (kernel == KERNEL_AUTO) {
    // Measured on B200 for the paths without tensor maps: a strided DESTINATION is
    // fastest with 16-byte STG from many warps (vec, 5.5 TB/s); a strided source alone is fastest gathered by
    // cp.async into the bulk ring and stored with one bulk copy (5.8 TB/s); everything contiguous is the
    // bulk path (6.3 TB/s).
    const bool dst_strided = g.pool_hnd && dir != 0;
    kernel = dst_strided ? KERNEL_VEC : KERNEL_BULK;
    // Mid-sized contiguous transfers are latency-bound: 14 MB in flight through 296 issuing warps ramps slower
    // than 16-byte loads from 1,184 CTAs' worth of warps.  Measured on B200, isolated calls on a cold L2
    // (DESIGN.md "Kernels"): 48 MiB 23.6 -> 18.5 us, 64 MiB 27.7 -> 23.6, 192 MiB 68.6 -> 64.6; equal at
    // <= 32 MiB (launch-bound) and 128 MiB; bulk ahead again from 512 MiB (171 vs 177 us).
    if (!g.trans && dir != 3) {
      uint64_t bytes = 0;
      for (const Req &r : reqs) bytes += r.n_ids * g.pool_row * g.LC;
      if (bytes >= kAutoVecMinBytes && bytes < kAutoVecMaxBytes) kernel = KERNEL_VEC;
    } else if (!g.trans) {
      // copy-on-write appends are many short, ragged pieces (about 6 KiB each): one warp per piece with 16-byte
      // loads beats one bulk copy per piece at every size where they differ (64 sessions: 44 -> 30 us,
      // 512 sessions: 279 -> 225 us; equal below ~16 MiB)
      uint64_t bytes = 0;
      for (const Req &r : reqs) bytes += ((r.n_tokens & 0xffffffffull) + (r.n_tokens >> 32)) * tokrow * g.LC;
      if (bytes >= (16ull << 20)) kernel = KERNEL_VEC;
    }
  }
  uint32_t cap = kernel == KERNEL_BULK ? (g.trans && !g.tma ? ctx->t_stage_bytes : ctx->stage_bytes) : 16384u;
  cap = std::max(16u, cap / 16 * 16);
  if (g.trans && kernel == KERNEL_BULK && g.drow > cap) kernel = KERNEL_VEC;  // a row must fit one stage
  g.kernel = kernel;
  g.sub_bytes = std::min(g.chunk_bytes, cap);
  if (g.trans) g.sub_bytes = std::min(g.chunk_bytes, std::max(g.drow, cap / g.drow * g.drow));  // whole rows
  if (g.tma) g.sub_bytes = g.tb * g.tokrow;  // whole tokens: one box
  if (kernel == KERNEL_BULK && dir != 3) {
    // Launch-bound calls: with fewer segments than issuing warps most SMs would idle while a few
    // move 16 KiB each; cutting segments down to >= 4 KiB spreads a small transfer over the chip
    // (measured on B200, 1 MiB pack back to back: 6.1 -> 5.0 us per call).
    uint64_t chunks = 0;
    for (const Req &r : reqs) chunks += r.n_ids * (g.Tpool / g.g) * g.LC;
    const uint64_t lanes = (uint64_t)ctx->sm_count * (g.trans && !g.tma ? ctx->t_warps : ctx->warps);
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

// ---------------------------------------------------------------------------------------------
// blob = [bases: LC x u64][pieces: n x Piece][ids: n_ids x i32], staged through a pinned ring
// ---------------------------------------------------------------------------------------------
struct HostBlob {
  std::vector<uint8_t> bytes;
  size_t off_pieces = 0, off_ids = 0;
};

void build_blob(const kv_pool_desc *p, const Geom &g, const std::vector<Piece> &pieces,
                const int32_t *ids, uint64_t n_ids, bool ids_on_device, HostBlob *hb) {
  hb->off_pieces = (size_t)g.LC * 8 * (g.src_pool ? 2 : 1);
  hb->off_ids = hb->off_pieces + pieces.size() * sizeof(Piece);
  hb->bytes.resize(hb->off_ids + (ids_on_device ? 0 : (size_t)n_ids * 4));
  uint8_t *h = hb->bytes.data();
  for (uint32_t i = 0; i < g.LC; ++i) ((uint64_t *)h)[i] = (uint64_t)(uintptr_t)p->base[i];
  if (g.src_pool)
    for (uint32_t i = 0; i < g.LC; ++i) ((uint64_t *)h)[g.LC + i] = (uint64_t)(uintptr_t)g.src_pool->base[i];
  std::memcpy(h + hb->off_pieces, pieces.data(), pieces.size() * sizeof(Piece));
  if (!ids_on_device && n_ids) std::memcpy(h + hb->off_ids, ids, (size_t)n_ids * 4);
}

// Tables of a launch: either resident in device memory (slot of the pinned ring) or carried
// inside the kernel parameters (inline; no copy, no slot).
struct Blob {
  BlobSlot *slot = nullptr;
  const uint64_t *d_bases = nullptr;
  const Piece *d_pieces = nullptr;
  const int32_t *d_ids = nullptr;  // also set for caller-supplied device ids in inline mode
  const HostBlob *inl = nullptr;   // non-null: inline tables
};

int upload_blob(kv_ctx *ctx, const HostBlob &hb, const int32_t *ids, bool ids_on_device,
                cudaStream_t s, Blob *out) {
  const size_t bytes = hb.bytes.size();
  BlobSlot &slot = ctx->blobs[ctx->next_blob++ % kBlobSlots];
  if (slot.used) KV_CUDA(ctx, cudaEventSynchronize(slot.ev));  // last reader of this slot is done
  if (slot.cap < bytes) {
    if (slot.h) cudaFreeHost(slot.h);
    if (slot.d) cudaFree(slot.d);
    slot.h = slot.d = nullptr; slot.cap = 0;
    size_t cap = std::max<size_t>(65536, bytes + bytes / 2);
    KV_CUDA(ctx, cudaMallocHost(&slot.h, cap));
    KV_CUDA(ctx, cudaMalloc(&slot.d, cap));
    slot.cap = cap;
  }
  std::memcpy(slot.h, hb.bytes.data(), bytes);
  KV_CUDA(ctx, cudaMemcpyAsync(slot.d, slot.h, bytes, cudaMemcpyHostToDevice, s));
  ctx->memcpys++;
  slot.used = true;
  out->slot = &slot;
  out->d_bases = (const uint64_t *)slot.d;
  out->d_pieces = (const Piece *)((uint8_t *)slot.d + hb.off_pieces);
  out->d_ids = ids_on_device ? ids : (const int32_t *)((uint8_t *)slot.d + hb.off_ids);
  return KV_OK;
}

constexpr int kInlineSmall = 3840;   // whole parameter block stays under the classic 4 KiB
constexpr int kInlineLarge = 31744;  // CUDA 12.1+ large kernel parameters (<= 32,764 B)

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
void launch_vec(const Job &j, const HostBlob *hb, bool trans, uint32_t grid, cudaStream_t s) {
  static thread_local kvt::JobT<N> p;
  p.j = j;
  if constexpr (N > 0) std::memcpy(p.blob, hb->bytes.data(), hb->bytes.size());
  if (trans) kvt::kv_move_vec<8, N, true><<<grid, 256, 0, s>>>(p);
  else kvt::kv_move_vec<8, N, false><<<grid, 256, 0, s>>>(p);
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
  if (g.tma && g.kernel == KERNEL_BULK) {
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
  if (g.kernel == KERNEL_BULK) {
    const bool lane_geom = g.trans && !g.tma;  // row gathers by all lanes want more, shallower warps
    j.stage_bytes = (g.sub_bytes + 127) / 128 * 128;
    j.stages = lane_geom ? ctx->t_stages : ctx->stages; j.lag = std::min(ctx->lag, j.stages - 1);
    j.zero_bytes = std::min<uint32_t>(4096, j.stage_bytes);
    j.l2_hint = ctx->l2_hint;
    uint32_t warps = lane_geom ? ctx->t_warps : ctx->warps;
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
    if (ctx->dynamic && total_items >= 8 * G && !capturing(s)) {  // enough work for claiming to pay
      uint8_t *slot = (uint8_t *)ctx->d_status + 256 + (size_t)(ctx->next_sched++ % kSchedSlots) * 16;
      j.sched = (unsigned long long *)slot;
      j.sched_done = (uint32_t *)(slot + 8);
      j.first_batch = (uint32_t)std::min<uint64_t>(32, total_items / (4 * G));
    }
    const bool pdl = ctx->pdl && !capturing(s);
    if (!b.inl) launch_bulk<0>(j, nullptr, g.trans, grid, warps * 32, smem, s, pdl);
    else if (b.inl->bytes.size() <= kInlineSmall) launch_bulk<kInlineSmall>(j, b.inl, g.trans, grid, warps * 32, smem, s, pdl);
    else launch_bulk<kInlineLarge>(j, b.inl, g.trans, grid, warps * 32, smem, s, pdl);
  } else {
    const uint32_t wpb = 8;  // warps per 256-thread CTA
    const uint64_t want = (total_items + wpb - 1) / wpb;
    grid = (uint32_t)std::min<uint64_t>(want, cap ? cap : (uint32_t)ctx->sm_count * 8);
    kvt::JobT<0> p0;
    p0.j = j;
    if (g.kernel == KERNEL_VEC) {
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
  return KV_OK;
}

// Validation shared by every entry point.  Fills reqs/geom; returns before any CUDA call.
struct Call {
  Geom geom;
  std::vector<Req> reqs;
  uint64_t n_ids = 0;
  uint64_t total_items = 0;
  uint64_t payload = 0;
};

int plan_pack(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *ids,
              const int64_t *off, uint32_t n_req, int layout, void *const *dsts,
              const uint64_t *dst_bytes, uint32_t flags, Call *c) {
  if (!ctx) return KV_ERR_NULL;
  int rc = check_desc(pools, layer_count);
  if (rc) return rc;
  if (n_req && (!off || !dsts)) return KV_ERR_NULL;
  const uint64_t page = (uint64_t)layer_count * pools->kv_count * pools->page_size *
                        pools->num_heads * pools->head_dim * pools->elem_bytes;
  c->reqs.clear();
  for (uint32_t r = 0; r < n_req; ++r) {
    if (off[r + 1] < off[r] || off[r] < 0) return KV_ERR_SIZE;
    const uint64_t n = (uint64_t)(off[r + 1] - off[r]);
    if (!n) continue;
    if (!dsts[r]) return KV_ERR_NULL;
    if (dst_bytes && dst_bytes[r] < n * page) return KV_ERR_SIZE;
    Req q;
    q.buf = (uint64_t)(uintptr_t)dsts[r];
    q.n_tokens = n * pools->page_size;
    q.id_begin = (uint64_t)off[r]; q.n_ids = n; q.n_buf_pages = n;
    c->reqs.push_back(q);
  }
  c->n_ids = n_req ? (uint64_t)off[n_req] : 0;
  if (c->n_ids && !ids) return KV_ERR_NULL;
  rc = make_geom(ctx, pools, layer_count, pools->page_size, /*dir=*/0, layout, c->reqs, &c->geom);
  if (rc) return rc;
  if (!(flags & KV_FLAG_IDS_ON_DEVICE)) {
    rc = check_ids(ids, c->n_ids, pools->num_pages);
    if (rc) return rc;
  }
  c->total_items = 0; c->payload = 0;
  for (Req &q : c->reqs) {
    q.items = items_of(c->geom, q.n_ids);
    if (q.items > 0xFFFFFFFFull) return KV_ERR_SIZE;
    c->total_items += q.items;
    c->payload += q.n_ids * page;
  }
  return KV_OK;
}

int plan_unpack(kv_ctx *ctx, const void *const *srcs, const uint64_t *src_bytes,
                const int32_t *ids, const int64_t *off, const uint64_t *n_tokens, uint32_t n_req,
                const kv_pool_desc *pools, uint32_t layer_count, uint32_t Ts, uint32_t Td,
                int layout, uint32_t flags, Call *c) {
  if (!ctx) return KV_ERR_NULL;
  int rc = check_desc(pools, layer_count);
  if (rc) return rc;
  if (!Ts || !Td || Td != pools->page_size) return KV_ERR_SIZE;
  if (n_req && (!off || !srcs || !n_tokens)) return KV_ERR_NULL;
  const uint64_t tokrow = (uint64_t)pools->num_heads * pools->head_dim * pools->elem_bytes;
  const uint64_t lc = (uint64_t)layer_count * pools->kv_count;
  c->reqs.clear();
  for (uint32_t r = 0; r < n_req; ++r) {
    if (off[r + 1] < off[r] || off[r] < 0) return KV_ERR_SIZE;
    const uint64_t n = (uint64_t)(off[r + 1] - off[r]);
    if (n != (n_tokens[r] + Td - 1) / Td) return KV_ERR_SIZE;
    if (!n) continue;
    if (!srcs[r]) return KV_ERR_NULL;
    const uint64_t n_src = (n_tokens[r] + Ts - 1) / Ts;
    if (src_bytes && src_bytes[r] < n_src * lc * Ts * tokrow) return KV_ERR_SIZE;
    Req q;
    q.buf = (uint64_t)(uintptr_t)srcs[r];
    q.n_tokens = n_tokens[r];
    q.id_begin = (uint64_t)off[r]; q.n_ids = n; q.n_buf_pages = n_src;
    c->reqs.push_back(q);
  }
  c->n_ids = n_req ? (uint64_t)off[n_req] : 0;
  if (c->n_ids && !ids) return KV_ERR_NULL;
  rc = make_geom(ctx, pools, layer_count, Ts, /*dir=*/1, layout, c->reqs, &c->geom);
  if (rc) return rc;
  if (!(flags & KV_FLAG_IDS_ON_DEVICE)) {
    rc = check_ids(ids, c->n_ids, pools->num_pages);
    if (rc) return rc;
    if (flags & KV_FLAG_VALIDATE) {
      rc = check_dups(ids, c->n_ids, pools->num_pages);
      if (rc) return rc;
    }
  }
  c->total_items = 0; c->payload = 0;
  for (Req &q : c->reqs) {
    q.items = items_of(c->geom, q.n_ids);
    if (q.items > 0xFFFFFFFFull) return KV_ERR_SIZE;
    c->total_items += q.items;
    c->payload += q.n_ids * lc * Td * tokrow;
  }
  return KV_OK;
}

// kv_repage[_batched]: destination pool `dp` (page size Td), source pool `sp` (page size Ts);
// the combined id array is [all destination ids][all source ids] and Req::buf indexes into it.
int plan_repage(kv_ctx *ctx, const kv_pool_desc *sp, const int32_t *src_ids, const int64_t *src_off,
                const kv_pool_desc *dp, const int32_t *dst_ids, const int64_t *dst_off,
                const uint64_t *n_tokens, uint32_t n_req, uint32_t layer_count, uint32_t flags,
                Call *c, std::vector<int32_t> *all_ids) {
  if (!ctx) return KV_ERR_NULL;
  int rc = check_desc(dp, layer_count);
  if (rc) return rc;
  rc = check_desc(sp, layer_count);
  if (rc) return rc;
  const bool dev_ids = flags & KV_FLAG_IDS_ON_DEVICE;
  if (sp->kv_count != dp->kv_count || sp->num_heads != dp->num_heads || sp->head_dim != dp->head_dim ||
      sp->elem_bytes != dp->elem_bytes)
    return KV_ERR_DESC;
  if (n_req && (!src_off || !dst_off || !n_tokens)) return KV_ERR_NULL;
  const uint32_t Ts = sp->page_size, Td = dp->page_size;
  const uint64_t tokrow = (uint64_t)dp->num_heads * dp->head_dim * dp->elem_bytes;
  const uint64_t lc = (uint64_t)layer_count * dp->kv_count;
  const uint64_t n_dst_total = n_req ? (uint64_t)dst_off[n_req] : 0;
  c->reqs.clear();
  for (uint32_t r = 0; r < n_req; ++r) {
    if (dst_off[r + 1] < dst_off[r] || dst_off[r] < 0 || src_off[r + 1] < src_off[r] || src_off[r] < 0)
      return KV_ERR_SIZE;
    const uint64_t nd = (uint64_t)(dst_off[r + 1] - dst_off[r]), ns = (uint64_t)(src_off[r + 1] - src_off[r]);
    if (nd != (n_tokens[r] + Td - 1) / Td || ns != (n_tokens[r] + Ts - 1) / Ts) return KV_ERR_SIZE;
    if (!nd) continue;
    Req q;
    // index of its first source id: in the combined host array, or in the caller's device array
    q.buf = (dev_ids ? 0 : n_dst_total) + (uint64_t)src_off[r];
    q.n_tokens = n_tokens[r];
    q.id_begin = (uint64_t)dst_off[r]; q.n_ids = nd; q.n_buf_pages = ns;
    c->reqs.push_back(q);
  }
  const uint64_t n_src_total = n_req ? (uint64_t)src_off[n_req] : 0;
  c->n_ids = n_dst_total + n_src_total;
  if ((n_dst_total && !dst_ids) || (n_src_total && !src_ids)) return KV_ERR_NULL;
  rc = make_geom(ctx, dp, layer_count, Ts, /*dir=*/2, KV_LAYOUT_PAGE_FIRST, c->reqs, &c->geom, sp);
  if (rc) return rc;
  if (dev_ids) {  // nothing to validate on the host: out-of-range ids skip their page and set the status word
    c->geom.dev_src_ids = src_ids;
  } else {
    rc = check_ids(dst_ids, n_dst_total, dp->num_pages);
    if (rc) return rc;
    rc = check_ids(src_ids, n_src_total, sp->num_pages);
    if (rc) return rc;
    if (flags & KV_FLAG_VALIDATE) {
      rc = check_dups(dst_ids, n_dst_total, dp->num_pages);
      if (rc) return rc;
    }
    all_ids->resize((size_t)c->n_ids);
    if (n_dst_total) std::memcpy(all_ids->data(), dst_ids, (size_t)n_dst_total * 4);
    if (n_src_total) std::memcpy(all_ids->data() + n_dst_total, src_ids, (size_t)n_src_total * 4);
  }
  c->total_items = 0; c->payload = 0;
  for (Req &q : c->reqs) {
    q.items = items_of(c->geom, q.n_ids);
    if (q.items > 0xFFFFFFFFull) return KV_ERR_SIZE;
    c->total_items += q.items;
    c->payload += q.n_ids * lc * Td * tokrow;
  }
  return KV_OK;
}

// kv_cow_append[_batched]: one Req per session with something to move.
int plan_cow(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *old_ids,
             const int32_t *new_ids, const uint32_t *n_old, const uint32_t *n_app,
             const void *const *apps, uint32_t n_sessions, uint32_t flags, Call *c) {
  if (!ctx) return KV_ERR_NULL;
  int rc = check_desc(pools, layer_count);
  if (rc) return rc;
  if (flags & KV_FLAG_IDS_ON_DEVICE) return KV_ERR_LAYOUT;
  if (n_sessions && (!old_ids || !new_ids || !n_old || !n_app || !apps)) return KV_ERR_NULL;
  const uint64_t tokrow = (uint64_t)pools->num_heads * pools->head_dim * pools->elem_bytes;
  const uint64_t lc = (uint64_t)layer_count * pools->kv_count;
  c->reqs.clear();
  for (uint32_t s = 0; s < n_sessions; ++s) {
    if ((uint64_t)n_old[s] + n_app[s] > pools->page_size || old_ids[s] == new_ids[s]) return KV_ERR_SIZE;
    if (old_ids[s] < 0 || new_ids[s] < 0 || (uint32_t)old_ids[s] >= pools->num_pages ||
        (uint32_t)new_ids[s] >= pools->num_pages)
      return KV_ERR_PAGE_RANGE;
    if (n_app[s] && !apps[s]) return KV_ERR_NULL;
    if (!n_old[s] && !n_app[s]) continue;
    Req q;
    q.buf = (uint64_t)(uintptr_t)apps[s];
    q.n_tokens = (uint64_t)n_old[s] | ((uint64_t)n_app[s] << 32);
    q.id_begin = (uint64_t)(uint32_t)old_ids[s] | ((uint64_t)(uint32_t)new_ids[s] << 32);
    c->reqs.push_back(q);
  }
  if (flags & KV_FLAG_VALIDATE) {  // new pages distinct, and none of them is some session's old page
    std::vector<uint8_t> is_new((size_t)(pools->num_pages + 7) / 8, 0);
    for (uint32_t s = 0; s < n_sessions; ++s) {
      const uint32_t g = (uint32_t)new_ids[s];
      if (is_new[g >> 3] & (1u << (g & 7))) return KV_ERR_DUP_PAGE;
      is_new[g >> 3] |= (uint8_t)(1u << (g & 7));
    }
    for (uint32_t s = 0; s < n_sessions; ++s) {
      const uint32_t g = (uint32_t)old_ids[s];
      if (is_new[g >> 3] & (1u << (g & 7))) return KV_ERR_DUP_PAGE;
    }
  }
  c->n_ids = 0;
  rc = make_geom(ctx, pools, layer_count, pools->page_size, /*dir=*/3, KV_LAYOUT_PAGE_FIRST, c->reqs, &c->geom);
  if (rc) return rc;
  c->total_items = 0; c->payload = 0;
  const uint64_t sub = c->geom.sub_bytes;
  for (Req &q : c->reqs) {
    const uint64_t b_old = (q.n_tokens & 0xffffffffull) * tokrow, b_app = (q.n_tokens >> 32) * tokrow;
    q.items = lc * ((b_old + sub - 1) / sub + (b_app + sub - 1) / sub);
    c->total_items += q.items;
    c->payload += lc * (b_old + b_app);
  }
  return KV_OK;
}

void note_plan(kv_ctx *ctx, const Call &c) {
  ctx->last_items = c.total_items;
  ctx->last_payload = c.payload;
  ctx->last_kernel = (uint64_t)c.geom.kernel;
  ctx->last_segment = c.geom.sub_bytes;
}

// one launch over all requests (device buffers, or mapped pinned host buffers = DIRECT mode)
int run_single_launch(kv_ctx *ctx, const kv_pool_desc *pools, const Call &c, const int32_t *ids,
                      uint32_t flags, uint32_t cta_cap, cudaStream_t s) {
  std::vector<Piece> pieces;
  pieces.reserve(c.reqs.size());
  uint64_t acc = 0;
  for (const Req &q : c.reqs) {
    Piece pc;
    pc.item_begin = acc; pc.buf = q.buf; pc.n_tokens = q.n_tokens; pc.id_begin = q.id_begin;
    pc.n_buf_pages = q.n_buf_pages;
    pieces.push_back(pc);
    acc += q.items;
  }
  const bool dev_ids = flags & KV_FLAG_IDS_ON_DEVICE;
  HostBlob hb;
  build_blob(pools, c.geom, pieces, ids, c.n_ids, dev_ids, &hb);
  Blob b;
  if (ctx->inline_tables && c.geom.kernel != KERNEL_ELEM && hb.bytes.size() <= (size_t)kInlineLarge) {
    b.inl = &hb;  // tables travel inside the kernel parameters: one launch, no copy
    b.d_ids = dev_ids ? ids : nullptr;
    return launch(ctx, c.geom, b, 0, (uint32_t)pieces.size(), acc, cta_cap, s);
  }
  if (capturing(s)) return KV_ERR_CAPTURE;
  int rc = upload_blob(ctx, hb, ids, dev_ids, s, &b);
  if (rc) return rc;
  rc = launch(ctx, c.geom, b, 0, (uint32_t)pieces.size(), acc, cta_cap, s);
  if (rc) return rc;
  KV_CUDA(ctx, cudaEventRecord(b.slot->ev, s));
  return KV_OK;
}

int ensure_staging(kv_ctx *ctx) {
  if (ctx->staging) return KV_OK;
  if (!ctx->staging_bytes) ctx->staging_bytes = (size_t)128 << 20;
  KV_CUDA(ctx, cudaMalloc(&ctx->staging, ctx->staging_bytes));
  return KV_OK;
}

// KV_HOST_STAGED: the flattened page sequence of all requests is cut into chunks that fit one
// staging slot; per chunk: kernel <-> slot on `s`, copy engine slot <-> pinned host on the side
// stream, double (or deeper) buffered with events.  Page-first only (a chunk of pages is then
// contiguous in the host buffer); layer-first falls back to DIRECT.
// Layer flags of kv_reload_layerwise: after the pages of layers [l0, l0 + n) have landed in the pool,
// flags[l] = value is stored (release, system scope) in stream order.
struct LayerFlags { uint64_t *flags = nullptr; uint64_t value = 0; };

int run_staged(kv_ctx *ctx, const kv_pool_desc *pools, const Call &c, const int32_t *ids,
               uint32_t flags, cudaStream_t s, LayerFlags lf = LayerFlags()) {
  int rc = ensure_staging(ctx);
  if (rc) return rc;
  const Geom &g = c.geom;
  const uint32_t n_slots = ctx->staging_slots;
  // unit of chunking: tokens that are whole pages on both sides
  const uint64_t unit_tokens = (uint64_t)g.Tpool / g.g * g.Tbuf;  // lcm(Tpool, Tbuf)
  const bool layer_first = g.layout == KV_LAYOUT_LAYER_FIRST;
  const uint64_t unit_bytes = unit_tokens * g.tokrow * (layer_first ? g.C : g.LC);
  size_t slot_bytes = ctx->staging_bytes / n_slots / 256 * 256;
  if (ctx->chunk_bytes) slot_bytes = std::min(slot_bytes, ctx->chunk_bytes / 256 * 256);
  if (slot_bytes < unit_bytes) return KV_ERR_SIZE;
  const uint64_t chunk_tokens = slot_bytes / unit_bytes * unit_tokens;

  // A chunk = what one staging slot holds: pieces for the kernel, copies for the copy engine.  Page-first:
  // a run of whole pages, all layers (contiguous in the host buffer).  Layer-first: a range of layers
  // [l0, l0 + nl) of one or more page ranges; every (layer, K|V) of a page range is one contiguous host run.
  struct Chunk { uint32_t piece_first, n_pieces; uint64_t items; uint32_t l0, nl, sig_n; };
  struct Copy { uint64_t host, dev_off, bytes; };
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
          Piece pc;
          pc.item_begin = cur.items;
          pc.buf = fill;  // offset within the slot; the slot base is added below
          pc.n_tokens = q.n_tokens > t0 ? std::min(q.n_tokens - t0, t1 - t0) : 0;
          pc.id_begin = q.id_begin + q0;
          pc.n_buf_pages = nb;
          pieces.push_back(pc);
          cur.n_pieces++;
          cur.items += (q1 - q0) * (g.Tpool / g.g) * nl * g.C * g.subs;
          if (nb)
            for (uint32_t l = 0; l < nl; ++l)
              for (uint32_t kc = 0; kc < g.C; ++kc)
                cur_copies.push_back(Copy{q.buf + (((uint64_t)(l0 + l) * g.C + kc) * q.n_buf_pages + b0) * row,
                                          fill + ((uint64_t)l * g.C + kc) * nb * row, nb * row});
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
        if (fill_tokens == chunk_tokens) close();
        const uint64_t t1 = std::min(slots_pool, t0 + (chunk_tokens - fill_tokens));
        const uint64_t span = t1 - t0;  // multiple of Tpool; multiple of unit except at the request's end
        const uint64_t buf_pages = (std::min(t1, q.n_buf_pages * g.Tbuf) - std::min(t0, q.n_buf_pages * g.Tbuf) + g.Tbuf - 1) / g.Tbuf;
        const uint64_t dev_off = fill_tokens * g.tokrow * g.LC;
        Piece pc;
        pc.item_begin = cur.items;
        pc.buf = (uint64_t)(uintptr_t)ctx->staging;  // + slot base, patched per chunk below
        pc.buf = dev_off;                              // offset within the slot for now
        pc.n_tokens = q.n_tokens > t0 ? std::min(q.n_tokens - t0, span) : 0;
        pc.id_begin = q.id_begin + t0 / g.Tpool;
        pc.n_buf_pages = buf_pages;
        pieces.push_back(pc);
        cur.n_pieces++;
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
    const uint64_t base = (uint64_t)(uintptr_t)ctx->staging + (ci % n_slots) * slot_bytes;
    for (uint32_t k = 0; k < chunks[ci].n_pieces; ++k) pieces[chunks[ci].piece_first + k].buf += base;
  }
  HostBlob hb;
  build_blob(pools, g, pieces, ids, c.n_ids, flags & KV_FLAG_IDS_ON_DEVICE, &hb);
  Blob b;
  rc = upload_blob(ctx, hb, ids, flags & KV_FLAG_IDS_ON_DEVICE, s, &b);
  if (rc) return rc;
  KV_CUDA(ctx, cudaEventRecord(ctx->ev_entry, s));
  KV_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_entry, 0));
  for (size_t ci = 0; ci < chunks.size(); ++ci) {
    const uint32_t slot = (uint32_t)(ci % n_slots);
    uint8_t *slot_base = (uint8_t *)ctx->staging + (size_t)slot * slot_bytes;
    if (g.dir == 0) {  // offload: kernel fills the slot on s, copy engine drains it on side
      if (ctx->free_valid[slot]) KV_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_free[slot], 0));
      rc = launch(ctx, g, b, chunks[ci].piece_first, chunks[ci].n_pieces, chunks[ci].items, 0, s,
                  chunks[ci].l0 * g.C, chunks[ci].nl * g.C);
      if (rc) return rc;
      KV_CUDA(ctx, cudaEventRecord(ctx->ev_full[slot], s));
      KV_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_full[slot], 0));
      for (const Copy &cp : copies[ci]) {
        KV_CUDA(ctx, cudaMemcpyAsync((void *)(uintptr_t)cp.host, slot_base + cp.dev_off, cp.bytes,
                                     cudaMemcpyDeviceToHost, ctx->side));
        ctx->memcpys++;
      }
      KV_CUDA(ctx, cudaEventRecord(ctx->ev_free[slot], ctx->side));
      ctx->free_valid[slot] = true;
    } else {  // reload: copy engine fills the slot on side, kernel drains it on s
      if (ctx->free_valid[slot]) KV_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_free[slot], 0));
      for (const Copy &cp : copies[ci]) {
        KV_CUDA(ctx, cudaMemcpyAsync(slot_base + cp.dev_off, (const void *)(uintptr_t)cp.host,
                                     cp.bytes, cudaMemcpyHostToDevice, ctx->side));
        ctx->memcpys++;
      }
      KV_CUDA(ctx, cudaEventRecord(ctx->ev_full[slot], ctx->side));
      KV_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_full[slot], 0));
      rc = launch(ctx, g, b, chunks[ci].piece_first, chunks[ci].n_pieces, chunks[ci].items, 0, s,
                  chunks[ci].l0 * g.C, chunks[ci].nl * g.C);
      if (rc) return rc;
      if (lf.flags && chunks[ci].sig_n) {  // these layers' pages are in the pool: publish
        kvt::kv_signal_range<<<1, 32, 0, s>>>(lf.flags + chunks[ci].l0, chunks[ci].sig_n, lf.value);  // strides over > 32
        KV_CUDA(ctx, cudaGetLastError());
        ctx->launches++;
      }
      KV_CUDA(ctx, cudaEventRecord(ctx->ev_free[slot], s));
      ctx->free_valid[slot] = true;
    }
  }
  if (g.dir == 0) {  // join the copy engine's tail back into s
    const size_t first = chunks.size() > n_slots ? chunks.size() - n_slots : 0;
    for (size_t ci = first; ci < chunks.size(); ++ci)
      KV_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_free[ci % n_slots], 0));
  }
  KV_CUDA(ctx, cudaEventRecord(b.slot->ev, s));
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
  // cudaMemcpy peak, SM-issued stores/loads over the link 92 % (128-byte TLP payloads); below
  // ~16 MiB both are latency-bound and equal, and DIRECT is one launch with no staging traffic.
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
  if (capturing(s)) {  // the chunk pipeline (side stream, staging slots, table upload) is not replayable
    if (mode == KV_HOST_STAGED) return KV_ERR_CAPTURE;
    m = KV_HOST_DIRECT;
    ctx->last_mode = (uint64_t)m;
  }
  for (Req &q : c.reqs) {
    uint64_t alias = 0;
    rc = host_alias(ctx, (const void *)(uintptr_t)q.buf, &alias);
    if (rc) return rc;
    if (m == KV_HOST_DIRECT) q.buf = alias;
  }
  if (lf.flags) {
    rc = flag_alias(lf.flags, &lf.flags);
    if (rc) return rc;
  }
  if (m == KV_HOST_DIRECT) {  // one launch moves every layer: the flags follow it together
    rc = run_single_launch(ctx, pools, c, ids, flags, ctx->host_max_ctas, s);
    if (rc || !lf.flags) return rc;
    for (uint32_t l0 = 0; l0 < c.geom.L; l0 += 32) {
      kvt::kv_signal_range<<<1, 32, 0, s>>>(lf.flags + l0, std::min(32u, c.geom.L - l0), lf.value);
      KV_CUDA(ctx, cudaGetLastError());
      ctx->launches++;
    }
    return KV_OK;
  }
  return run_staged(ctx, pools, c, ids, flags, s, lf);
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

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

uint32_t kv_version(void) { return KVTIER_VERSION; }

const char *kv_strerror(int status) {
  switch (status) {
    case KV_OK: return "ok";
    case KV_ERR_NULL: return "required pointer is NULL";
    case KV_ERR_SIZE: return "size mismatch (buffer too small, inconsistent page sizes/counts, or too many items)";
    case KV_ERR_PAGE_RANGE: return "page id out of range";
    case KV_ERR_DUP_PAGE: return "duplicate destination page id";
    case KV_ERR_LAYOUT: return "unknown layout, host mode or option";
    case KV_ERR_ALIGN: return "pointer or stride not aligned to elem_bytes";
    case KV_ERR_CUDA: return "CUDA error (see kv_last_cuda_error)";
    case KV_ERR_HOST_MEM: return "host buffer is not pinned memory";
    case KV_ERR_DESC: return "malformed kv_pool_desc";
    case KV_ERR_NO_DEVICE: return "planning-only context: nothing launched";
    case KV_ERR_CAPTURE: return "call cannot be captured into a CUDA graph (tables exceed the kernel parameters, or staged host mode)";
    default: return "unknown kvtier status";
  }
}

int kv_ctx_create(kv_ctx **out, int device, size_t staging_bytes) {
  if (!out) return KV_ERR_NULL;
  *out = nullptr;
  kv_ctx *ctx = new (std::nothrow) kv_ctx();
  if (!ctx) return KV_ERR_SIZE;
  ctx->staging_bytes = staging_bytes;
  if (device < 0) {
    ctx->host_only = true;
    ctx->max_smem = 232448;
    *out = ctx;
    return KV_OK;
  }
  ctx->device = device;
  auto fail = [&](cudaError_t e) {
    (void)e;
    (void)cudaGetLastError();
    delete ctx;
    return KV_ERR_CUDA;
  };
  cudaError_t e;
  int prev = -1;
  if ((e = cudaGetDevice(&prev)) != cudaSuccess) return fail(e);
  if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(e);
  if ((e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return fail(e);
  if ((e = cudaDeviceGetAttribute(&ctx->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device)) != cudaSuccess) return fail(e);
  const void *bulk_kernels[] = {(const void *)kvt::kv_move_bulk<0, false>, (const void *)kvt::kv_move_bulk<kInlineSmall, false>,
                                (const void *)kvt::kv_move_bulk<kInlineLarge, false>, (const void *)kvt::kv_move_bulk<0, true>,
                                (const void *)kvt::kv_move_bulk<kInlineSmall, true>, (const void *)kvt::kv_move_bulk<kInlineLarge, true>};
  for (const void *k : bulk_kernels)
    if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->max_smem - kStaticSmemReserve)) != cudaSuccess) return fail(e);
  {  // cuTensorMapEncodeTiled without linking libcuda; absent -> HND pools keep to the lane paths
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess &&
        qr == cudaDriverEntryPointSuccess)
      ctx->encode_tiled = (EncodeTiledFn)fn;
    else
      (void)cudaGetLastError();
  }
  if ((e = cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking)) != cudaSuccess) return fail(e);
  if ((e = cudaEventCreateWithFlags(&ctx->ev_entry, cudaEventDisableTiming)) != cudaSuccess) return fail(e);
  for (int i = 0; i < kBlobSlots; ++i)
    if ((e = cudaEventCreateWithFlags(&ctx->blobs[i].ev, cudaEventDisableTiming)) != cudaSuccess) return fail(e);
  for (int i = 0; i < kMaxStagingSlots; ++i) {
    if ((e = cudaEventCreateWithFlags(&ctx->ev_full[i], cudaEventDisableTiming)) != cudaSuccess) return fail(e);
    if ((e = cudaEventCreateWithFlags(&ctx->ev_free[i], cudaEventDisableTiming)) != cudaSuccess) return fail(e);
  }
  if ((e = cudaMalloc((void **)&ctx->d_status, 256 + kSchedSlots * 16)) != cudaSuccess) return fail(e);
  if ((e = cudaMemset(ctx->d_status, 0, 256 + kSchedSlots * 16)) != cudaSuccess) return fail(e);
  if (prev >= 0 && prev != device) cudaSetDevice(prev);
  *out = ctx;
  return KV_OK;
}

int kv_ctx_destroy(kv_ctx *ctx) {
  if (!ctx) return KV_ERR_NULL;
  if (!ctx->host_only) {
    DeviceGuard guard(ctx);
    cudaStreamSynchronize(ctx->side);
    for (auto &b : ctx->blobs) {
      if (b.used) cudaEventSynchronize(b.ev);
      if (b.h) cudaFreeHost(b.h);
      if (b.d) cudaFree(b.d);
      if (b.ev) cudaEventDestroy(b.ev);
    }
    for (int i = 0; i < kMaxStagingSlots; ++i) {
      if (ctx->ev_full[i]) cudaEventDestroy(ctx->ev_full[i]);
      if (ctx->ev_free[i]) { cudaEventSynchronize(ctx->ev_free[i]); cudaEventDestroy(ctx->ev_free[i]); }
    }
    if (ctx->staging) cudaFree(ctx->staging);
    for (MapSet &m : ctx->map_sets) cudaFree(m.d);
    if (ctx->d_status) cudaFree(ctx->d_status);
    if (ctx->ev_entry) cudaEventDestroy(ctx->ev_entry);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    (void)cudaGetLastError();
  }
  delete ctx;
  return KV_OK;
}

int kv_ctx_set_option(kv_ctx *ctx, int option, int64_t v) {
  if (!ctx) return KV_ERR_NULL;
  switch (option) {
    case KV_OPT_KERNEL: if (v < 0 || v > 3) return KV_ERR_SIZE; ctx->kernel = (int)v; break;
    case KV_OPT_STAGE_BYTES: if (v < 1024 || v > 65536 || v % 16) return KV_ERR_SIZE; ctx->stage_bytes = ctx->t_stage_bytes = (uint32_t)v; break;
    case KV_OPT_STAGES_PER_WARP: if (v < 2 || v > kvt::kMaxStages) return KV_ERR_SIZE; ctx->stages = ctx->t_stages = (uint32_t)v; break;
    case KV_OPT_WARPS: if (v < 1 || v > kvt::kMaxWarps) return KV_ERR_SIZE; ctx->warps = ctx->t_warps = (uint32_t)v; break;
    case KV_OPT_STORE_LAG: if (v < 1 || v > 3) return KV_ERR_SIZE; ctx->lag = (uint32_t)v; break;
    case KV_OPT_MAX_CTAS: if (v < 0 || v > 65535) return KV_ERR_SIZE; ctx->max_ctas = (uint32_t)v; break;
    case KV_OPT_CHUNK_BYTES: if (v < 0) return KV_ERR_SIZE; ctx->chunk_bytes = (size_t)v; break;
    case KV_OPT_HOST_MAX_CTAS: if (v < 0 || v > 65535) return KV_ERR_SIZE; ctx->host_max_ctas = (uint32_t)v; break;
    case KV_OPT_STAGING_SLOTS: if (v < 2 || v > kMaxStagingSlots) return KV_ERR_SIZE; ctx->staging_slots = (uint32_t)v; break;
    case KV_OPT_L2_HINT: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->l2_hint = (uint32_t)v; break;
    case KV_OPT_INLINE_TABLES: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->inline_tables = (uint32_t)v; break;
    case KV_OPT_DYNAMIC: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->dynamic = (uint32_t)v; break;
    case KV_OPT_TENSOR_MAPS: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->tensor_maps = (uint32_t)v; break;
    case KV_OPT_PDL: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->pdl = (uint32_t)v; break;
    default: return KV_ERR_LAYOUT;
  }
  return KV_OK;
}

int kv_ctx_get_stat(kv_ctx *ctx, int stat, uint64_t *out) {
  if (!ctx || !out) return KV_ERR_NULL;
  switch (stat) {
    case KV_STAT_LAUNCHES: *out = ctx->launches; break;
    case KV_STAT_MEMCPYS: *out = ctx->memcpys; break;
    case KV_STAT_LAST_ITEMS: *out = ctx->last_items; break;
    case KV_STAT_LAST_PAYLOAD: *out = ctx->last_payload; break;
    case KV_STAT_LAST_KERNEL: *out = ctx->last_kernel; break;
    case KV_STAT_LAST_HOST_MODE: *out = ctx->last_mode; break;
    case KV_STAT_LAST_GRID: *out = ctx->last_grid; break;
    case KV_STAT_LAST_SEGMENT: *out = ctx->last_segment; break;
    case KV_STAT_LAST_TENSOR_MAPS: *out = ctx->last_tma; break;
    default: return KV_ERR_LAYOUT;
  }
  return KV_OK;
}

int kv_last_cuda_error(kv_ctx *ctx) { return ctx ? ctx->last_cuda_error : 0; }

int kv_device_status(kv_ctx *ctx, uint32_t *out) {
  if (!ctx || !out) return KV_ERR_NULL;
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  DeviceGuard guard(ctx);
  KV_CUDA(ctx, cudaDeviceSynchronize());
  KV_CUDA(ctx, cudaMemcpy(out, ctx->d_status, 4, cudaMemcpyDeviceToHost));
  KV_CUDA(ctx, cudaMemset(ctx->d_status, 0, 4));
  return KV_OK;
}

int kv_peer_enable(kv_ctx *ctx, int peer_device) {
  if (!ctx) return KV_ERR_NULL;
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  if (peer_device < 0 || peer_device == ctx->device) return KV_ERR_SIZE;
  DeviceGuard guard(ctx);
  int can = 0;
  KV_CUDA(ctx, cudaDeviceCanAccessPeer(&can, ctx->device, peer_device));
  if (!can) { ctx->last_cuda_error = (int)cudaErrorPeerAccessUnsupported; return KV_ERR_CUDA; }
  cudaError_t e = cudaDeviceEnablePeerAccess(peer_device, 0);
  if (e == cudaErrorPeerAccessAlreadyEnabled) { (void)cudaGetLastError(); e = cudaSuccess; }
  KV_CUDA(ctx, e);
  return KV_OK;
}

int kv_signal(kv_ctx *ctx, uint64_t *flag, uint64_t value, kv_stream_t stream) {
  if (!ctx || !flag) return KV_ERR_NULL;
  if ((uint64_t)(uintptr_t)flag % 8) return KV_ERR_ALIGN;
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  DeviceGuard guard(ctx);
  uint64_t *dev = flag;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, flag) != cudaSuccess) { (void)cudaGetLastError(); return KV_ERR_HOST_MEM; }
  if (a.type == cudaMemoryTypeUnregistered) return KV_ERR_HOST_MEM;  // pageable host memory
  if (a.type == cudaMemoryTypeHost) {
    if (!a.devicePointer) return KV_ERR_HOST_MEM;
    dev = (uint64_t *)a.devicePointer;
  }
  kvt::kv_signal_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(dev, value);
  KV_CUDA(ctx, cudaGetLastError());
  ctx->launches++;
  return KV_OK;
}

int kv_chain_hash(kv_ctx *ctx, const uint64_t *ident, const int64_t *tok_offsets, uint32_t n_sessions,
                  uint32_t page_size, const uint64_t *roots, uint64_t *out, size_t out_capacity,
                  int64_t *page_offsets, kv_stream_t stream) {
  if (!ctx) return KV_ERR_NULL;
  if (!page_size) return KV_ERR_SIZE;
  if (n_sessions && !tok_offsets) return KV_ERR_NULL;
  std::vector<int64_t> poff((size_t)n_sessions + 1, 0);
  for (uint32_t s = 0; s < n_sessions; ++s) {
    if (tok_offsets[s] < 0 || tok_offsets[s + 1] < tok_offsets[s]) return KV_ERR_SIZE;
    poff[s + 1] = poff[s] + (tok_offsets[s + 1] - tok_offsets[s]) / (int64_t)page_size;
  }
  const uint64_t total = (uint64_t)poff[n_sessions];
  if (total > out_capacity) return KV_ERR_SIZE;
  if (page_offsets) std::memcpy(page_offsets, poff.data(), poff.size() * sizeof(int64_t));
  ctx->last_items = total;
  if (!total) return KV_OK;
  if (!ident || !out) return KV_ERR_NULL;
  if (((uint64_t)(uintptr_t)ident | (uint64_t)(uintptr_t)out) % 8) return KV_ERR_ALIGN;
  if (ctx->host_only) return KV_ERR_NO_DEVICE;
  cudaStream_t s = (cudaStream_t)stream;
  DeviceGuard guard(ctx);
  if (capturing(s)) return KV_ERR_CAPTURE;
  // tables: [tok_off: S+1][page_off: S+1][roots: S], staged through the pinned ring
  HostBlob hb;
  const size_t n1 = (size_t)n_sessions + 1;
  hb.bytes.resize((2 * n1 + (roots ? n_sessions : 0)) * 8);
  std::memcpy(hb.bytes.data(), tok_offsets, n1 * 8);
  std::memcpy(hb.bytes.data() + n1 * 8, poff.data(), n1 * 8);
  if (roots) std::memcpy(hb.bytes.data() + 2 * n1 * 8, roots, (size_t)n_sessions * 8);
  Blob b;
  int rc = upload_blob(ctx, hb, nullptr, true, s, &b);
  if (rc) return rc;
  kvt::ChainJob j{};
  j.ident = ident; j.out = out;
  j.tok_off = (const int64_t *)b.slot->d;
  j.page_off = j.tok_off + n1;
  j.roots = roots ? (const uint64_t *)(j.page_off + n1) : nullptr;
  j.default_root = KV_CHAIN_ROOT;
  j.total_pages = total; j.n_sessions = n_sessions; j.T = page_size;
  const uint64_t blocks = (total + 127) / 128;
  if (blocks > 0x7fffffffull) return KV_ERR_SIZE;
  kvt::kv_chain_digest<<<(uint32_t)blocks, 128, 0, s>>>(j);
  KV_CUDA(ctx, cudaGetLastError());
  kvt::kv_chain_link<<<n_sessions, 32, 0, s>>>(j);
  KV_CUDA(ctx, cudaGetLastError());
  ctx->launches += 2;
  KV_CUDA(ctx, cudaEventRecord(b.slot->ev, s));
  return KV_OK;
}

int kv_host_alloc(void **p, size_t bytes) {
  if (!p) return KV_ERR_NULL;
  *p = nullptr;
  if (!bytes) return KV_ERR_SIZE;
  cudaError_t e = cudaHostAlloc(p, bytes, cudaHostAllocMapped | cudaHostAllocPortable);
  if (e != cudaSuccess) { (void)cudaGetLastError(); *p = nullptr; return KV_ERR_CUDA; }
  return KV_OK;
}

int kv_host_free(void *p) {
  if (!p) return KV_ERR_NULL;
  if (cudaFreeHost(p) != cudaSuccess) { (void)cudaGetLastError(); return KV_ERR_CUDA; }
  return KV_OK;
}

int kv_host_register(void *p, size_t bytes) {
  if (!p) return KV_ERR_NULL;
  if (!bytes) return KV_ERR_SIZE;
  if (cudaHostRegister(p, bytes, cudaHostRegisterMapped | cudaHostRegisterPortable) != cudaSuccess) {
    (void)cudaGetLastError();
    return KV_ERR_CUDA;
  }
  return KV_OK;
}

int kv_host_unregister(void *p) {
  if (!p) return KV_ERR_NULL;
  if (cudaHostUnregister(p) != cudaSuccess) { (void)cudaGetLastError(); return KV_ERR_CUDA; }
  return KV_OK;
}

int kv_pack(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *page_ids,
            uint32_t n, int layout, void *dst, size_t dst_bytes, uint32_t flags, kv_stream_t stream) {
  const int64_t off[2] = {0, (int64_t)n};
  void *const dsts[1] = {dst};
  const uint64_t nb[1] = {(uint64_t)dst_bytes};
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_pack(ctx, pools, layer_count, page_ids, off, 1, layout, dsts, nb, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, page_ids, flags, (cudaStream_t)stream);
}

int kv_unpack(kv_ctx *ctx, const void *src, size_t src_bytes, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
              uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens, int layout,
              uint32_t flags, kv_stream_t stream) {
  const int64_t off[2] = {0, (int64_t)n_dst_pages};
  const void *const srcs[1] = {src};
  const uint64_t nb[1] = {(uint64_t)src_bytes};
  const uint64_t nt[1] = {n_tokens};
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_unpack(ctx, srcs, nb, dst_page_ids, off, nt, 1, pools, layer_count, src_page_size,
                       dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, dst_page_ids, flags, (cudaStream_t)stream);
}

int kv_pack_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                    const int32_t *page_ids, const int64_t *req_offsets, uint32_t n_req, int layout,
                    void *const *dsts, const uint64_t *dst_bytes, uint32_t flags, kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_pack(ctx, pools, layer_count, page_ids, req_offsets, n_req, layout, dsts, dst_bytes, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, page_ids, flags, (cudaStream_t)stream);
}

int kv_unpack_batched(kv_ctx *ctx, const void *const *srcs, const uint64_t *src_bytes,
                      const int32_t *dst_page_ids, const int64_t *req_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                      uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                      int layout, uint32_t flags, kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_unpack(ctx, srcs, src_bytes, dst_page_ids, req_offsets, n_tokens, n_req, pools,
                       layer_count, src_page_size, dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, dst_page_ids, flags, (cudaStream_t)stream);
}

int kv_repage_batched(kv_ctx *ctx, const kv_pool_desc *src_pools, const int32_t *src_page_ids,
                      const int64_t *src_offsets, const kv_pool_desc *dst_pools,
                      const int32_t *dst_page_ids, const int64_t *dst_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, uint32_t layer_count, uint32_t flags,
                      kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  std::vector<int32_t> ids;
  int rc = plan_repage(ctx, src_pools, src_page_ids, src_offsets, dst_pools, dst_page_ids,
                       dst_offsets, n_tokens, n_req, layer_count, flags, &c, &ids);
  if (rc) return rc;
  return run_device(ctx, dst_pools, c, (flags & KV_FLAG_IDS_ON_DEVICE) ? dst_page_ids : ids.data(), flags,
                    (cudaStream_t)stream);
}

int kv_repage(kv_ctx *ctx, const kv_pool_desc *src_pools, const int32_t *src_page_ids,
              uint32_t n_src_pages, const kv_pool_desc *dst_pools, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, uint32_t layer_count, uint64_t n_tokens, uint32_t flags,
              kv_stream_t stream) {
  const int64_t soff[2] = {0, (int64_t)n_src_pages}, doff[2] = {0, (int64_t)n_dst_pages};
  const uint64_t nt[1] = {n_tokens};
  return kv_repage_batched(ctx, src_pools, src_page_ids, soff, dst_pools, dst_page_ids, doff, nt, 1,
                           layer_count, flags, stream);
}

int kv_cow_append_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                          const int32_t *old_ids, const int32_t *new_ids, const uint32_t *n_old,
                          const uint32_t *n_app, const void *const *apps, uint32_t n_sessions,
                          uint32_t flags, kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_cow(ctx, pools, layer_count, old_ids, new_ids, n_old, n_app, apps, n_sessions, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, nullptr, flags, (cudaStream_t)stream);
}

int kv_cow_append(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, int32_t old_id,
                  int32_t new_id, uint32_t n_old, const void *app, uint32_t n_app, uint32_t flags,
                  kv_stream_t stream) {
  const int32_t o[1] = {old_id}, n[1] = {new_id};
  const uint32_t no[1] = {n_old}, na[1] = {n_app};
  const void *const ap[1] = {app};
  return kv_cow_append_batched(ctx, pools, layer_count, o, n, no, na, ap, 1, flags, stream);
}

int kv_offload(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
               const int32_t *page_ids, uint32_t n, int layout, void *host_dst, size_t host_bytes,
               int mode, uint32_t flags, kv_stream_t stream) {
  const int64_t off[2] = {0, (int64_t)n};
  void *const dsts[1] = {host_dst};
  const uint64_t nb[1] = {(uint64_t)host_bytes};
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_pack(ctx, pools, layer_count, page_ids, off, 1, layout, dsts, nb, flags, &c);
  if (rc) return rc;
  return run_host(ctx, pools, c, page_ids, mode, flags, (cudaStream_t)stream);
}

int kv_reload(kv_ctx *ctx, const void *host_src, size_t host_bytes, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
              uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens, int layout,
              int mode, uint32_t flags, kv_stream_t stream) {
  const int64_t off[2] = {0, (int64_t)n_dst_pages};
  const void *const srcs[1] = {host_src};
  const uint64_t nb[1] = {(uint64_t)host_bytes};
  const uint64_t nt[1] = {n_tokens};
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_unpack(ctx, srcs, nb, dst_page_ids, off, nt, 1, pools, layer_count, src_page_size,
                       dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_host(ctx, pools, c, dst_page_ids, mode, flags, (cudaStream_t)stream);
}

int kv_reload_layerwise_batched(kv_ctx *ctx, const void *const *host_srcs, const uint64_t *host_bytes,
                                const int32_t *dst_page_ids, const int64_t *req_offsets,
                                const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                                uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                                uint64_t *layer_flags, uint64_t flag_value, int mode, uint32_t flags,
                                kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  if (!layer_flags) return KV_ERR_NULL;
  if ((uint64_t)(uintptr_t)layer_flags % 8) return KV_ERR_ALIGN;
  Call c;
  int rc = plan_unpack(ctx, host_srcs, host_bytes, dst_page_ids, req_offsets, n_tokens, n_req, pools,
                       layer_count, src_page_size, dst_page_size, KV_LAYOUT_LAYER_FIRST, flags, &c);
  if (rc) return rc;
  LayerFlags lf;
  lf.flags = layer_flags; lf.value = flag_value;
  if (c.reqs.empty() && !ctx->host_only) {  // nothing to move: every layer is trivially complete
    int m = 0;
    rc = resolve_mode(ctx, mode, c, &m);
    if (rc) return rc;
    DeviceGuard guard(ctx);
    rc = flag_alias(lf.flags, &lf.flags);
    if (rc) return rc;
    kvt::kv_signal_range<<<1, 32, 0, (cudaStream_t)stream>>>(lf.flags, layer_count, flag_value);
    KV_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return KV_OK;
  }
  return run_host(ctx, pools, c, dst_page_ids, mode, flags, (cudaStream_t)stream, lf);
}

int kv_reload_layerwise(kv_ctx *ctx, const void *host_src, size_t host_bytes, const int32_t *dst_page_ids,
                        uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
                        uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens,
                        uint64_t *layer_flags, uint64_t flag_value, int mode, uint32_t flags,
                        kv_stream_t stream) {
  const int64_t off[2] = {0, (int64_t)n_dst_pages};
  const void *const srcs[1] = {host_src};
  const uint64_t nb[1] = {(uint64_t)host_bytes};
  const uint64_t nt[1] = {n_tokens};
  return kv_reload_layerwise_batched(ctx, srcs, nb, dst_page_ids, off, nt, 1, pools, layer_count, src_page_size,
                                     dst_page_size, layer_flags, flag_value, mode, flags, stream);
}

int kv_offload_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                       const int32_t *page_ids, const int64_t *req_offsets, uint32_t n_req,
                       int layout, void *const *host_dsts, const uint64_t *host_bytes, int mode,
                       uint32_t flags, kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_pack(ctx, pools, layer_count, page_ids, req_offsets, n_req, layout, host_dsts, host_bytes, flags, &c);
  if (rc) return rc;
  return run_host(ctx, pools, c, page_ids, mode, flags, (cudaStream_t)stream);
}

int kv_reload_batched(kv_ctx *ctx, const void *const *host_srcs, const uint64_t *host_bytes,
                      const int32_t *dst_page_ids, const int64_t *req_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                      uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                      int layout, int mode, uint32_t flags, kv_stream_t stream) {
  if (ctx) ctx->cur_stream = (cudaStream_t)stream;
  Call c;
  int rc = plan_unpack(ctx, host_srcs, host_bytes, dst_page_ids, req_offsets, n_tokens, n_req,
                       pools, layer_count, src_page_size, dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_host(ctx, pools, c, dst_page_ids, mode, flags, (cudaStream_t)stream);
}

}  // extern "C"
