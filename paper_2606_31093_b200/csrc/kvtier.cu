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
