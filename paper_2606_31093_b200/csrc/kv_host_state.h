// kv_host_state.h -- the ctx: constants, staging ring, tensor-map cache, options, statistics
// Part of the host side of libkvtier.so; included by kvtier.cu only (one translation unit).
// Shares nothing with oracle/.
#pragma once

namespace {

using kvt::Job;
using kvt::Piece;

constexpr int kBlobSlots = 16;
// Inline tables.  Small: the WHOLE parameter block (Job header + blob) stays within the classic 4 KiB, so the launch does
// not take the large-parameter path; the size follows the header, whatever it grows to.  Large: CUDA 12.1+ kernel
// parameters (<= 32,764 B).
constexpr int kInlineSmall = (4096 - (int)offsetof(kvt::JobT<1>, blob)) / 64 * 64;
constexpr int kInlineLarge = 31744;
static_assert(kInlineSmall >= 2048 && sizeof(kvt::JobT<kInlineSmall>) <= 4096, "small inline tables: parameter block over 4 KiB");
static_assert(sizeof(kvt::JobT<kInlineLarge>) <= 32764, "large inline tables: parameter block over the 32,764-byte limit");
constexpr int kMaxStagingSlots = 4;
constexpr uint32_t kMaxLayersKv = 4096;  // layer_count * kv_count
constexpr uint64_t kAutoStagedMinBytes = 4ull << 20;
constexpr uint32_t kShotMinSegment = 4096;  // AUTO: kv_move_shot from this segment size (below it the SM's bulk-copy rate binds)
constexpr uint32_t kSchedSlots = 256;  // claim counters, handed out round-robin per launch
constexpr int kStaticSmemReserve = 8192;  // static shared memory of kv_move_bulk (barriers + stage metadata, 6 KiB) rounded up

enum KernelKind { KERNEL_AUTO = 0, KERNEL_BULK = 1, KERNEL_VEC = 2, KERNEL_ELEM = 3, KERNEL_SHOT = 4 };
inline bool is_async_kernel(int k) { return k == KERNEL_BULK || k == KERNEL_SHOT; }  // cp.async.bulk through shared-memory stages

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
  void *blob_arena_h = nullptr, *blob_arena_d = nullptr;  // the slots' backing store: one pinned, one device allocation
  uint32_t next_blob = 0;
  uint32_t *d_status = nullptr;
  // staging for KV_HOST_STAGED
  void *staging = nullptr;
  size_t staging_bytes = 0;
  // The staging allocation failed (the usual reason: the KV pools fill HBM).  KV_HOST_AUTO then takes DIRECT, which needs
  // no staging, and does not ask again -- a failing cudaMalloc still synchronises the device -- until a
  // KV_OPT_RESERVE_STAGING succeeds.  An explicit KV_HOST_STAGED keeps trying and keeps reporting KV_ERR_CUDA.
  bool staging_denied = false;
  // Slot i is ALWAYS the bytes [i * pitch, (i + 1) * pitch) of `staging`, pitch = staging_bytes / staging_slots: a
  // call whose chunks are smaller uses a prefix of each slot.  The per-slot events therefore guard the same memory for
  // every call, whatever its chunk size and whichever stream it runs on.
  cudaEvent_t ev_full[kMaxStagingSlots] = {};  // producer into the slot finished
  cudaEvent_t ev_free[kMaxStagingSlots] = {};  // consumer of the slot finished
  bool free_valid[kMaxStagingSlots] = {};
  // the same roles inside a stream capture: captured records are not real records, so they get events of their own
  // and never touch the bookkeeping of eager calls
  cudaEvent_t cap_entry = nullptr, cap_full[kMaxStagingSlots] = {}, cap_free[kMaxStagingSlots] = {};
  int last_cuda_error = 0;
  // options
  int kernel = KERNEL_AUTO;
  uint32_t stage_bytes = 16384, stages = 4, warps = 2, lag = 2, max_ctas = 0, host_max_ctas = 0;
  uint32_t lead_chunk = 32u << 20;  // KV_OPT_LEAD_CHUNK: bytes of the short leading (offload) / trailing (reload) chunk; 0 = equal chunks
  bool auto_geom = true;  // ring geometry follows the segment size until the caller sets stages / warps / stage bytes
  // bulk geometry of transposing transfers (an HND pool): rows are gathered with 16-byte cp.async by all
  // lanes, which wants more, shallower issuing warps (measured: 8 x 4 x 4 KiB)
  uint32_t t_stage_bytes = 4096, t_stages = 4, t_warps = 8;
  uint32_t staging_slots = 2, l2_hint = 0, inline_tables = 1, dynamic = 1, tensor_maps = 1, pdl = 1;
  uint32_t next_sched = 0;
  EncodeTiledFn encode_tiled = nullptr;  // cuTensorMapEncodeTiled, nullptr if the driver has none
  std::vector<MapSet> map_sets;
  cudaStream_t cur_stream = nullptr;     // stream of the entry point being served
  bool cur_capturing = false;            // ... and whether it is being captured (queried once per call)
  uint64_t last_tma = 0;
  uint64_t last_plain = 0;
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


}  // namespace
