// kvtier.cu -- C ABI (include/kvtier.h) of the paged-KV tier transfer: host validation, page-id
// staging, planning of the flat segment list (a2) and launches (a3-a8).
// Every byte of the path is moved by the kernels in kv_kernels.cuh or, in KV_HOST_STAGED mode,
// by the copy engines between the ctx's device staging and pinned host memory.
// There is no CPU fallback: without a CUDA device transfer calls fail (KV_ERR_CUDA / NO_DEVICE).
#include "../../include/kvtier.h"

#include <cuda.h>  // CUtensorMap types only; the encoder is fetched through cudaGetDriverEntryPoint
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstddef>
#include <cstring>
#include <new>
#include <numeric>
#include <vector>

#include "kv_chain.cuh"
#include "kv_kernels.cuh"

#include "kv_host_state.h"
#include "kv_geom.inl"
#include "kv_launch.inl"
#include "kv_plan.inl"
#include "kv_run.inl"


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
    case KV_ERR_STATIC_LIMIT:
      return "request exceeds the fixed table array of kv_pack_static (at most 65536 page ids and 1024 layer x K/V slabs per call): split it";
    default: return "unknown kvtier status";
  }
}

}  // extern "C"

namespace {
// Frees everything a ctx owns on its device; null-safe member by member, so it also serves a ctx whose creation
// stopped half way.  The caller has made the ctx's device current.
void ctx_release(kv_ctx *ctx) {
  if (ctx->side) cudaStreamSynchronize(ctx->side);
  for (auto &b : ctx->blobs) {
    if (b.used && b.ev) cudaEventSynchronize(b.ev);
    if (b.ev) cudaEventDestroy(b.ev);
  }
  for (int i = 0; i < kMaxStagingSlots; ++i) {
    if (ctx->ev_full[i]) cudaEventDestroy(ctx->ev_full[i]);
    if (ctx->ev_free[i]) { if (ctx->free_valid[i]) cudaEventSynchronize(ctx->ev_free[i]); cudaEventDestroy(ctx->ev_free[i]); }
    if (ctx->cap_full[i]) cudaEventDestroy(ctx->cap_full[i]);
    if (ctx->cap_free[i]) cudaEventDestroy(ctx->cap_free[i]);
  }
  if (ctx->blob_arena_h) cudaFreeHost(ctx->blob_arena_h);
  if (ctx->blob_arena_d) cudaFree(ctx->blob_arena_d);
  if (ctx->staging) cudaFree(ctx->staging);
  for (MapSet &m : ctx->map_sets) cudaFree(m.d);
  if (ctx->d_status) cudaFree(ctx->d_status);
  if (ctx->ev_entry) cudaEventDestroy(ctx->ev_entry);
  if (ctx->cap_entry) cudaEventDestroy(ctx->cap_entry);
  if (ctx->side) cudaStreamDestroy(ctx->side);
  (void)cudaGetLastError();
}

cudaError_t ctx_init_device(kv_ctx *ctx, int device) {
  cudaError_t e;
  if ((e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&ctx->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device)) != cudaSuccess) return e;
  const void *bulk_kernels[] = {(const void *)kvt::kv_move_bulk<0, false>, (const void *)kvt::kv_move_bulk<kInlineSmall, false>,
                                (const void *)kvt::kv_move_bulk<kInlineLarge, false>, (const void *)kvt::kv_move_bulk<0, true>,
                                (const void *)kvt::kv_move_bulk<kInlineSmall, true>, (const void *)kvt::kv_move_bulk<kInlineLarge, true>};
  for (const void *k : bulk_kernels)
    if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->max_smem - kStaticSmemReserve)) != cudaSuccess) return e;
  const void *shot_kernels[] = {(const void *)kvt::kv_move_shot<0, false>, (const void *)kvt::kv_move_shot<kInlineSmall, false>,
                                (const void *)kvt::kv_move_shot<kInlineLarge, false>, (const void *)kvt::kv_move_shot<0, true>,
                                (const void *)kvt::kv_move_shot<kInlineSmall, true>, (const void *)kvt::kv_move_shot<kInlineLarge, true>,
                                (const void *)kvt::kv_move_shot_plain<0, false>, (const void *)kvt::kv_move_shot_plain<kInlineSmall, false>,
                                (const void *)kvt::kv_move_shot_plain<kInlineLarge, false>, (const void *)kvt::kv_move_shot_plain<0, true>,
                                (const void *)kvt::kv_move_shot_plain<kInlineSmall, true>,
                                (const void *)kvt::kv_move_shot_plain<kInlineLarge, true>};
  for (const void *k : shot_kernels) {  // stages up to 64 KiB (KV_OPT_STAGE_BYTES); as many CTAs per SM as shared memory holds
    if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return e;
  }
  {  // cuTensorMapEncodeTiled without linking libcuda; absent -> HND pools keep to the lane paths
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess &&
        qr == cudaDriverEntryPointSuccess)
      ctx->encode_tiled = (EncodeTiledFn)fn;
    else
      (void)cudaGetLastError();
  }
  if ((e = cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking)) != cudaSuccess) return e;
  if ((e = cudaEventCreateWithFlags(&ctx->ev_entry, cudaEventDisableTiming)) != cudaSuccess) return e;
  if ((e = cudaEventCreateWithFlags(&ctx->cap_entry, cudaEventDisableTiming)) != cudaSuccess) return e;
  for (int i = 0; i < kBlobSlots; ++i)
    if ((e = cudaEventCreateWithFlags(&ctx->blobs[i].ev, cudaEventDisableTiming)) != cudaSuccess) return e;
  for (int i = 0; i < kMaxStagingSlots; ++i) {
    if ((e = cudaEventCreateWithFlags(&ctx->ev_full[i], cudaEventDisableTiming)) != cudaSuccess) return e;
    if ((e = cudaEventCreateWithFlags(&ctx->ev_free[i], cudaEventDisableTiming)) != cudaSuccess) return e;
    if ((e = cudaEventCreateWithFlags(&ctx->cap_full[i], cudaEventDisableTiming)) != cudaSuccess) return e;
    if ((e = cudaEventCreateWithFlags(&ctx->cap_free[i], cudaEventDisableTiming)) != cudaSuccess) return e;
  }
  if ((e = cudaMalloc((void **)&ctx->d_status, 256 + kSchedSlots * 16)) != cudaSuccess) return e;
  if ((e = cudaMemset(ctx->d_status, 0, 256 + kSchedSlots * 16)) != cudaSuccess) return e;
  return cudaSuccess;
}
}  // namespace

extern "C" {

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
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e == cudaSuccess) e = cudaSetDevice(device);
  if (e == cudaSuccess) {
    e = ctx_init_device(ctx, device);
    if (e != cudaSuccess) ctx_release(ctx);  // same teardown as kv_ctx_destroy: nothing created so far leaks
  }
  if (prev >= 0 && prev != device) cudaSetDevice(prev);  // the caller's current device is restored on EVERY way out
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    delete ctx;
    return KV_ERR_CUDA;
  }
  *out = ctx;
  return KV_OK;
}

int kv_ctx_destroy(kv_ctx *ctx) {
  if (!ctx) return KV_ERR_NULL;
  if (!ctx->host_only) {
    DeviceGuard guard(ctx);
    ctx_release(ctx);
  }
  delete ctx;
  return KV_OK;
}

int kv_ctx_set_option(kv_ctx *ctx, int option, int64_t v) {
  if (!ctx) return KV_ERR_NULL;
  switch (option) {
    case KV_OPT_KERNEL: if (v < 0 || v > 4) return KV_ERR_SIZE; ctx->kernel = (int)v; break;
    case KV_OPT_STAGE_BYTES: if (v < 1024 || v > 65536 || v % 16) return KV_ERR_SIZE; ctx->stage_bytes = ctx->t_stage_bytes = (uint32_t)v; ctx->auto_geom = false; break;
    case KV_OPT_STAGES_PER_WARP: if (v < 2 || v > kvt::kMaxStages) return KV_ERR_SIZE; ctx->stages = ctx->t_stages = (uint32_t)v; ctx->auto_geom = false; break;
    case KV_OPT_WARPS: if (v < 1 || v > kvt::kMaxWarps) return KV_ERR_SIZE; ctx->warps = ctx->t_warps = (uint32_t)v; ctx->auto_geom = false; break;
    case KV_OPT_STORE_LAG: if (v < 1 || v > 3) return KV_ERR_SIZE; ctx->lag = (uint32_t)v; break;
    case KV_OPT_MAX_CTAS: if (v < 0 || v > 65535) return KV_ERR_SIZE; ctx->max_ctas = (uint32_t)v; break;
    case KV_OPT_CHUNK_BYTES: if (v < 0) return KV_ERR_SIZE; ctx->chunk_bytes = (size_t)v; break;
    case KV_OPT_HOST_MAX_CTAS: if (v < 0 || v > 65535) return KV_ERR_SIZE; ctx->host_max_ctas = (uint32_t)v; break;
    case KV_OPT_STAGING_SLOTS:
      if (v < 2 || v > kMaxStagingSlots) return KV_ERR_SIZE;
      if ((uint32_t)v != ctx->staging_slots && !ctx->host_only) {
        // the slots move: nothing may still be using the old ones when the next staged call cuts the buffer anew
        DeviceGuard guard(ctx);
        for (int i = 0; i < kMaxStagingSlots; ++i)
          if (ctx->free_valid[i]) { KV_CUDA(ctx, cudaEventSynchronize(ctx->ev_free[i])); ctx->free_valid[i] = false; }
      }
      ctx->staging_slots = (uint32_t)v;
      break;
    case KV_OPT_L2_HINT: if (v < 0 || v > 5) return KV_ERR_SIZE; ctx->l2_hint = (uint32_t)v; break;
    case KV_OPT_INLINE_TABLES: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->inline_tables = (uint32_t)v; break;
    case KV_OPT_DYNAMIC: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->dynamic = (uint32_t)v; break;
    case KV_OPT_TENSOR_MAPS: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->tensor_maps = (uint32_t)v; break;
    case KV_OPT_PDL: if (v < 0 || v > 1) return KV_ERR_SIZE; ctx->pdl = (uint32_t)v; break;
    case KV_OPT_LEAD_CHUNK: if (v < 0 || v > (1ll << 30)) return KV_ERR_SIZE; ctx->lead_chunk = (uint32_t)v; break;
    case KV_OPT_RESERVE_STAGING: {
      if (v < 0) return KV_ERR_SIZE;
      if (ctx->host_only) return KV_ERR_NO_DEVICE;
      if (ctx->staging) return (v == 0 || (size_t)v == ctx->staging_bytes) ? KV_OK : KV_ERR_SIZE;
      if (v) ctx->staging_bytes = (size_t)v;
      DeviceGuard guard(ctx);
      ctx->cur_capturing = false;
      return ensure_staging(ctx);
    }
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
    case KV_STAT_LAST_PLAIN: *out = ctx->last_plain; break;
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
  const size_t n1 = (size_t)n_sessions + 1;
  const uint64_t blocks = (total + 127) / 128;
  if (blocks > 0x7fffffffull) return KV_ERR_SIZE;
  kvt::ChainJob j{};
  j.ident = ident; j.out = out;
  j.default_root = KV_CHAIN_ROOT;
  j.total_pages = total; j.n_sessions = n_sessions; j.T = page_size;
  if (n_sessions <= (uint32_t)kvt::kChainInlineSessions) {  // tables inside the kernel parameters: capturable
    static thread_local kvt::ChainJobInline pi;
    pi.j = j;
    pi.j.roots = roots ? pi.roots : nullptr;  // non-null marks "roots present"; the kernel points it at its own copy
    std::memcpy(pi.tok_off, tok_offsets, n1 * 8);
    std::memcpy(pi.page_off, poff.data(), n1 * 8);
    if (roots) std::memcpy(pi.roots, roots, (size_t)n_sessions * 8);
    // one launch: a CTA per session digests its pages and then walks its chain (kv_chain.cuh)
    int64_t longest = 1;
    for (uint32_t q = 0; q < n_sessions; ++q) longest = std::max(longest, poff[q + 1] - poff[q]);
    const uint32_t threads = (uint32_t)std::min<int64_t>(1024, (longest + 31) / 32 * 32);
    kvt::kv_chain_fused<true><<<n_sessions, threads, 0, s>>>(pi);
    KV_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return KV_OK;
  }
  if (capturing(s)) return KV_ERR_CAPTURE;
  // larger batches: two launches, [tok_off: S+1][page_off: S+1][roots: S] staged through the pinned ring
  HostBlob hb;
  hb.bytes.resize((2 * n1 + (roots ? n_sessions : 0)) * 8);
  std::memcpy(hb.bytes.data(), tok_offsets, n1 * 8);
  std::memcpy(hb.bytes.data() + n1 * 8, poff.data(), n1 * 8);
  if (roots) std::memcpy(hb.bytes.data() + 2 * n1 * 8, roots, (size_t)n_sessions * 8);
  Blob b;
  int rc = upload_blob(ctx, hb, nullptr, true, s, &b);
  if (rc) return rc;
  BlobGuard guard_blob(ctx, &b, s);
  j.tok_off = (const int64_t *)b.slot->d;
  j.page_off = j.tok_off + n1;
  j.roots = roots ? (const uint64_t *)(j.page_off + n1) : nullptr;
  kvt::kv_chain_digest<false><<<(uint32_t)blocks, 128, 0, s>>>(j);
  KV_CUDA(ctx, cudaGetLastError());
  kvt::kv_chain_link<false><<<n_sessions, 32, 0, s>>>(j);
  KV_CUDA(ctx, cudaGetLastError());
  ctx->launches += 2;
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
  enter(ctx, stream);
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
  enter(ctx, stream);
  Call c;
  int rc = plan_unpack(ctx, srcs, nb, dst_page_ids, off, nt, 1, pools, layer_count, src_page_size,
                       dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, dst_page_ids, flags, (cudaStream_t)stream);
}

int kv_pack_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                    const int32_t *page_ids, const int64_t *req_offsets, uint32_t n_req, int layout,
                    void *const *dsts, const uint64_t *dst_bytes, uint32_t flags, kv_stream_t stream) {
  enter(ctx, stream);
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
  enter(ctx, stream);
  Call c;
  int rc = plan_unpack(ctx, srcs, src_bytes, dst_page_ids, req_offsets, n_tokens, n_req, pools,
                       layer_count, src_page_size, dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, dst_page_ids, flags, (cudaStream_t)stream);
}

int kv_submit(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const kv_op *ops, uint32_t n_ops,
              int layout, uint32_t flags, kv_stream_t stream) {
  enter(ctx, stream);
  Call c;
  std::vector<int32_t> ids;
  int rc = plan_submit(ctx, pools, layer_count, ops, n_ops, layout, flags, &c, &ids);
  if (rc) return rc;
  return run_device(ctx, pools, c, ids.data(), flags, (cudaStream_t)stream);
}

int kv_repage_batched(kv_ctx *ctx, const kv_pool_desc *src_pools, const int32_t *src_page_ids,
                      const int64_t *src_offsets, const kv_pool_desc *dst_pools,
                      const int32_t *dst_page_ids, const int64_t *dst_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, uint32_t layer_count, uint32_t flags,
                      kv_stream_t stream) {
  enter(ctx, stream);
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
  enter(ctx, stream);
  Call c;
  int rc = plan_cow(ctx, pools, layer_count, old_ids, new_ids, n_old, n_app, apps, n_sessions, flags, &c);
  if (rc) return rc;
  return run_device(ctx, pools, c, (flags & KV_FLAG_IDS_ON_DEVICE) ? old_ids : nullptr, flags, (cudaStream_t)stream);
}

int kv_cow_append(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, int32_t old_id,
                  int32_t new_id, uint32_t n_old, const void *app, uint32_t n_app, uint32_t flags,
                  kv_stream_t stream) {
  if (flags & KV_FLAG_IDS_ON_DEVICE) return KV_ERR_LAYOUT;  // the ids are passed by value here
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
  enter(ctx, stream);
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
  enter(ctx, stream);
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
  enter(ctx, stream);
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
  enter(ctx, stream);
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
  enter(ctx, stream);
  Call c;
  int rc = plan_unpack(ctx, host_srcs, host_bytes, dst_page_ids, req_offsets, n_tokens, n_req,
                       pools, layer_count, src_page_size, dst_page_size, layout, flags, &c);
  if (rc) return rc;
  return run_host(ctx, pools, c, dst_page_ids, mode, flags, (cudaStream_t)stream);
}

}  // extern "C"


// =============================================================================================
// kv_pack_static -- kv_pack for callers that must not allocate (include/kvtier.h, "kv_pack without any allocation").
//
// The tables-in-device-memory form of kv_move_shot_plain (JobT<0>) normally reads slab bases and page ids from the
// ctx's table arena, which upload_blob allocates (cudaMalloc + cudaMallocHost) inside the call.  Here the same kernel
// reads them from the array below, which is part of the library image: nobody allocates it, nobody frees it, and this
// code path contains no allocating CUDA call (its only working storage on the host is one thread_local parameter block).
// =============================================================================================
namespace {

static_assert(sizeof(void *) == 8, "slab bases are copied as 64-bit addresses");
constexpr uint32_t kStaticHeader = 256;  // bytes [0, 256): the kernels' status word (word 0) and padding, zero at kernel start
static_assert(KV_STATIC_TABLE_BYTES == kStaticHeader + KV_STATIC_MAX_SLABS * 8u + KV_STATIC_MAX_PAGES * 4u, "kvtier.h states this size");
static_assert(KV_STATIC_TABLE_BYTES % 16 == 0, "filled in 16-byte units");

// [header: 256 B][slab bases: LC x u64, padded to 16 B][page ids: n x i32, padded to 16 B] of the call in flight.
// One copy per GPU that loads this library, held until the process exits.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- never a device address; DEVICE code (kv_static_fill) may use it directly.
static __device__ __align__(256) unsigned char g_kv_static_tables[KV_STATIC_TABLE_BYTES];

// Writes one slice of the call's table image into the array.  The slice travels in the kernel parameters, so the
// caller's host arrays are consumed when the launch returns and no host-to-device copy (and no pinned staging) exists.
constexpr uint32_t kStaticFillChunk = 28672;  // with the 16-byte head: 28,688 B of the 32,764 B a parameter block may have
struct StaticFill {
  uint32_t off;    // byte offset in the array, multiple of 16
  uint32_t bytes;  // multiple of 16
  uint32_t pad_[2];
  alignas(16) uint8_t data[kStaticFillChunk];
};
__global__ void __launch_bounds__(256) kv_static_fill(const __grid_constant__ StaticFill p) {
  for (uint32_t i = threadIdx.x * 16; i < p.bytes; i += blockDim.x * 16)
    *reinterpret_cast<uint4 *>(g_kv_static_tables + p.off + i) = *reinterpret_cast<const uint4 *>(p.data + i);
}

// What the first call on a device learns and every later call reuses.  `tables` is written last (release) and read first
// (acquire); two threads racing through the set-up of one device compute the same values.
constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
  std::atomic<uint8_t *> tables{nullptr};  // THIS device's address of g_kv_static_tables
  int sm_count = 0;
};
StaticDevice g_static_device[kStaticMaxDevices];

// `device` is current.  No allocation: a symbol lookup, an attribute query, a function attribute.
cudaError_t static_setup(int device, uint8_t **tables, int *sm_count) {
  StaticDevice &d = g_static_device[device];
  uint8_t *t = d.tables.load(std::memory_order_acquire);
  if (!t) {
    void *sym = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&sym, g_kv_static_tables);
    if (e != cudaSuccess) return e;
    if (!sym) return cudaErrorInvalidSymbol;
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return e;
    // as many single-warp CTAs per SM as shared memory holds (what kv_ctx_create asks for, for the same kernel)
    if ((e = cudaFuncSetAttribute((const void *)kvt::kv_move_shot_plain<0, false>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                  cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return e;
    d.sm_count = sms;
    t = (uint8_t *)sym;
    d.tables.store(t, std::memory_order_release);
  }
  *tables = t;
  *sm_count = d.sm_count;
  return cudaSuccess;
}

}  // namespace

extern "C" int kv_pack_static(int device, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *page_ids,
                              uint32_t n, void *dst, size_t dst_bytes, kv_stream_t stream, int *cuda_error) {
  if (cuda_error) *cuda_error = 0;
  // ---- validation: all of it before the first CUDA call
  if (device < 0 || device >= kStaticMaxDevices) return KV_ERR_SIZE;
  int rc = check_desc(pools, layer_count);
  if (rc) return rc;
  const uint32_t LC = layer_count * pools->kv_count;
  if (LC > KV_STATIC_MAX_SLABS || n > KV_STATIC_MAX_PAGES) return KV_ERR_STATIC_LIMIT;
  if (pools->order == KV_ORDER_HND && pools->num_heads > 1 && pools->page_size > 1) return KV_ERR_LAYOUT;
  const uint64_t tokrow = (uint64_t)pools->num_heads * pools->head_dim * pools->elem_bytes;
  const uint64_t row = tokrow * pools->page_size;  // one page of one (layer, K|V); check_desc bounds it by 2^32-1
  if (!n) return KV_OK;
  if (!page_ids || !dst) return KV_ERR_NULL;
  if ((uint64_t)dst_bytes < (uint64_t)n * LC * row) return KV_ERR_SIZE;
  if ((tokrow | pools->page_stride_bytes | (uint64_t)(uintptr_t)dst) % 16) return KV_ERR_ALIGN;
  for (uint32_t i = 0; i < LC; ++i)
    if ((uint64_t)(uintptr_t)pools->base[i] % 16) return KV_ERR_ALIGN;
  rc = check_ids(page_ids, n, pools->num_pages);
  if (rc) return rc;

  // ---- device set-up (first call on this device) with the device current; restored on every way out
  struct Restore {
    int prev = -1;
    ~Restore() { if (prev >= 0) cudaSetDevice(prev); }
  } restore;
  auto fail = [&](cudaError_t e) {
    if (cuda_error) *cuda_error = (int)e;
    (void)cudaGetLastError();
    return (int)KV_ERR_CUDA;
  };
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return fail(e);
  if (cur != device) {
    if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(e);
    restore.prev = cur;
  }
  uint8_t *tables = nullptr;
  int sm_count = 0;
  if ((e = static_setup(device, &tables, &sm_count)) != cudaSuccess) return fail(e);

  // ---- segments: a page row of one (layer, K|V), cut like the library cuts it for kv_move_shot (kv_geom.inl)
  const uint32_t cap = 16384, chunk = (uint32_t)row;
  uint32_t sub = std::min(chunk, cap);
  if (chunk > cap) {  // equal pieces instead of full stages and a crumb
    const uint32_t k = (chunk + cap - 1) / cap, even = ((chunk + k - 1) / k + 127) / 128 * 128;
    if (even <= cap) sub = even;
  }
  while (sub >= 8192 && sub % 32 == 0 &&  // launch-sized calls: spread few segments over the chip
         (uint64_t)n * LC * ((chunk + sub - 1) / sub) * 2 <= (uint64_t)sm_count * 2)
    sub /= 2;
  const uint32_t subs = (chunk + sub - 1) / sub;
  const uint64_t total_items = (uint64_t)n * LC * subs;
  if (total_items > 0x7fffffffull) return KV_ERR_SIZE;

  // ---- the call's table image -> the array, slice by slice (header first: it re-zeroes the status word)
  const uint32_t off_bases = kStaticHeader;
  const uint32_t off_ids = off_bases + (LC * 8 + 15) / 16 * 16;
  cudaStream_t s = (cudaStream_t)stream;
  static thread_local StaticFill fill;
  uint32_t at = 0;       // array offset of fill.data[0]
  uint32_t have = 0;     // bytes of fill.data in use
  auto flush = [&]() -> cudaError_t {
    if (!have) return cudaSuccess;
    fill.off = at;
    fill.bytes = (have + 15) / 16 * 16;
    std::memset(fill.data + have, 0, fill.bytes - have);
    kv_static_fill<<<1, 256, 0, s>>>(fill);
    at += fill.bytes;
    have = 0;
    return cudaGetLastError();
  };
  auto emit = [&](const void *src, size_t bytes) -> cudaError_t {  // src == nullptr: zeros
    const uint8_t *q = (const uint8_t *)src;
    while (bytes) {
      const size_t m = std::min<size_t>(bytes, kStaticFillChunk - have);
      if (q) { std::memcpy(fill.data + have, q, m); q += m; }
      else std::memset(fill.data + have, 0, m);
      have += (uint32_t)m;
      bytes -= m;
      if (have == kStaticFillChunk) {
        cudaError_t fe = flush();
        if (fe != cudaSuccess) return fe;
      }
    }
    return cudaSuccess;
  };
  if ((e = emit(nullptr, kStaticHeader)) != cudaSuccess) return fail(e);
  if ((e = emit(pools->base, (size_t)LC * 8)) != cudaSuccess) return fail(e);
  if ((e = emit(nullptr, off_ids - off_bases - LC * 8)) != cudaSuccess) return fail(e);
  if ((e = emit(page_ids, (size_t)n * 4)) != cudaSuccess) return fail(e);
  if ((e = flush()) != cudaSuccess) return fail(e);

  // ---- the copy: kv_move_shot_plain, tables in device memory (JobT<0>), one request, every token valid
  kvt::JobT<0> p{};
  Job &j = p.j;
  j.bases = (const uint64_t *)(tables + off_bases);
  j.ids = (const int32_t *)(tables + off_ids);
  j.status = (uint32_t *)tables;
  j.total_items = total_items;
  j.page_stride = pools->page_stride_bytes;
  j.buf_row_bytes = row;
  j.buf_page_bytes = row * LC;
  j.n_pieces = 1; j.LC = LC; j.dir = 0; j.layout = KV_LAYOUT_PAGE_FIRST;
  j.g = pools->page_size; j.cpp_pool = 1; j.cpp_buf = 1;
  j.tokrow = (uint32_t)tokrow; j.chunk_bytes = chunk; j.sub_bytes = sub; j.subs = subs;
  j.num_pages = pools->num_pages;
  j.stage_bytes = (sub + 127) / 128 * 128;
  j.drow = pools->head_dim * pools->elem_bytes; j.H = pools->num_heads;
  j.one.item_begin = 0; j.one.buf = (uint64_t)(uintptr_t)dst; j.one.n_tokens = (uint64_t)n * pools->page_size;
  j.one.id_begin = 0; j.one.n_buf_pages = n; j.one.dir = 0;
  auto magic = [](uint32_t d) -> uint64_t { return d <= 1 ? 0ull : ~0ull / d + 1; };
  j.m_subs = magic(subs); j.m_LC = magic(LC); j.m_cpp_pool = 0; j.m_cpp_buf = 0;
  j.lean = 1;
  kvt::kv_move_shot_plain<0, false><<<(uint32_t)total_items, 32, j.stage_bytes, s>>>(p);
  if ((e = cudaGetLastError()) != cudaSuccess) return fail(e);
  return KV_OK;
}
