/*
 * kvtier.h -- C ABI of the B200-native paged-KV tier transfer library (libkvtier.so).
 *
 * The one hot path of Omni-Flow's Data Flow layer: "Cross-tier migration converts between
 * compute-oriented layouts, including NHD block stacks, and the representation used by
 * lower-tier storage ... CUDA kernels ... copy and convert pages directly into destination
 * buffers" (sec. 4.1.2 Multi-Tier Slot Engine), over pools addressed by
 * (layer, page_idx, K|V slice) (sec. 4.1.1 Physical Paging Layer), between the
 * L1 GPU tier and the L2 CPU tier (sec. 4).  The lower-tier representation is the
 * dense page-first buffer [page][layer][K,V][token][head][dim] of BASELINE.json:configs[0].
 * Call shapes follow BASELINE.json:north_star; the scope table is SURVEY.md 8(a)/(b).
 *
 * Conventions that hold for EVERY entry point
 *   - Plain C types only.  `kv_stream_t` is a cudaStream_t / CUstream passed as an opaque
 *     pointer (NULL = the legacy default stream).
 *   - Return value: KV_OK (0) or a negative kv_status.  No exception crosses the ABI.
 *   - All argument validation happens before the first CUDA call that could write: a call that
 *     returns a validation error (anything but KV_ERR_CUDA) has written nothing.
 *   - Ownership: the caller owns pools, buffers and id arrays; the library never frees them.
 *     HOST arrays (page ids, offsets, token counts, pointer arrays, kv_pool_desc and its `base`
 *     array) are consumed before the call returns and may be reused immediately.
 *   - Asynchrony: work is enqueued on `stream` and the call returns.  Results (including the
 *     host-visible bytes of an offload) are defined once the caller has synchronised `stream`.
 *     Staged host transfers use a side stream owned by the ctx but are joined back to `stream`
 *     before the call returns control of ordering.
 *   - Aliasing: transfer buffers must not overlap any pool; destination page ids of one call
 *     must be distinct and free (the slot engine guarantees it).
 *   - Elements are opaque `elem_bytes`-wide bit patterns; nothing is ever interpreted as a number.
 *   - All byte offsets are 64-bit.
 *   - CUDA graphs: every transfer whose tables fit the kernel parameters is ONE kernel node and may be
 *     captured (cudaStreamBeginCapture on `stream`); page ids passed as host arrays are baked into the
 *     node, ids passed with KV_FLAG_IDS_ON_DEVICE are re-read from device memory at every replay.
 *     STAGED host transfers are capturable too (copy nodes on a forked branch + one kernel node per chunk, each
 *     with its tables in its parameters) once the ctx's staging exists (KV_OPT_RESERVE_STAGING, or any earlier
 *     staged call): KV_HOST_AUTO then captures what it would run eagerly; without staging it captures DIRECT.
 *     HND pools: a captured call whose pool has no tensor maps in device memory yet carries them in its kernel
 *     parameters (same kernels); if tables and maps together exceed the parameter space it takes the lane paths.
 *     A graph holding staged transfers uses the ctx's staging buffer at every replay: replay it on the stream on
 *     which the ctx's other staged transfers run, or not at the same time as them.  Otherwise: KV_ERR_CAPTURE.
 *     While a capture that holds a staged transfer of a ctx is still open (before cudaStreamEndCapture), the ctx's side
 *     stream belongs to it: an EAGER multi-chunk staged transfer of the same ctx on another stream is refused with
 *     KV_ERR_CAPTURE (explicit KV_HOST_STAGED) or runs DIRECT (KV_HOST_AUTO) instead of leaking into that graph.
 *   - A kv_ctx is not thread-safe: one ctx per calling thread.  Calls on different streams are
 *     independent when their destination page sets are disjoint; staged host transfers of ONE ctx issued on
 *     different streams share its staging slots and are ordered against one another slot by slot.
 */
#ifndef KVTIER_H
#define KVTIER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KVTIER_VERSION 0x00010000u /* major.minor.patch = 0.1.0 */

typedef struct kv_ctx kv_ctx;
typedef void *kv_stream_t;

/* One paged KV parameter: outer dim = layers, slice dim = K/V, a page size,
 * a shape and an element width.  Region (l, g, c) starts at base[l*kv_count + c] +
 * g*page_stride_bytes and holds page_size*num_heads*head_dim elements, in-page order `order`:
 * KV_ORDER_NHD [token][head][dim] ("NHD block stacks") or KV_ORDER_HND
 * [head][token][dim] ("compute-oriented layouts, INCLUDING NHD block stacks" -- NHD
 * is one of several).  The transfer buffer and the copy-on-write append block
 * are always NHD, so a transfer to or from an HND pool is a real transposition of [token] and [head].
 * Separate K and V allocations, one fused allocation per layer, or one allocation for everything are
 * all expressed by the base pointers and the stride; bytes between the dense row and the stride are
 * never read or written. */
typedef enum kv_order { KV_ORDER_NHD = 0, KV_ORDER_HND = 1 } kv_order;
typedef struct kv_pool_desc {
  void *const *base;          /* HOST array of layer_count*kv_count DEVICE pointers, [layer][kv], kv 0=K 1=V */
  uint32_t layer_count;       /* layers in the descriptor */
  uint32_t kv_count;          /* 2 for K and V; 1 for single-latent pools */
  uint32_t num_pages;         /* pages in each slab; valid page ids are 0 .. num_pages-1 */
  uint32_t page_size;         /* tokens per page */
  uint32_t num_heads;         /* KV heads held by THIS rank (a TP head partition has fewer) */
  uint32_t head_dim;
  uint32_t elem_bytes;        /* 1, 2, 4 or 8; bf16 = 2 */
  uint32_t order;             /* kv_order: in-page order of THIS pool (0 = NHD) */
  uint64_t page_stride_bytes; /* >= page_size*num_heads*head_dim*elem_bytes, multiple of elem_bytes */
} kv_pool_desc;

/* Layout of the transfer buffer (the "representation used by lower-tier storage"). */
typedef enum kv_layout {
  KV_LAYOUT_PAGE_FIRST = 0,  /* [page][layer][kv][token][head][dim]  (BASELINE.json:configs[0]) */
  KV_LAYOUT_LAYER_FIRST = 1, /* [layer][kv][page][token][head][dim] */
} kv_layout;

/* How a host-tier transfer crosses the host link (BASELINE.json:north_star item 3). */
typedef enum kv_host_mode {
  KV_HOST_AUTO = 0,   /* chosen from the measured table in DESIGN.md: STAGED from 4 MiB of payload (either layout), else DIRECT.
                         If the ctx has no staging buffer and cannot get one -- the allocation fails because the KV pools
                         fill HBM, or the stream is being captured -- AUTO runs DIRECT instead of failing, and after a
                         failed allocation it does not try again until KV_OPT_RESERVE_STAGING succeeds (the failure's
                         cudaError_t stays readable through kv_last_cuda_error) */
  KV_HOST_DIRECT = 1, /* the kernel stores to / loads from mapped pinned memory over the link */
  KV_HOST_STAGED = 2, /* device staging + copy-engine transfers (1-D, or 2-D for layer-first chunks) on the ctx's side stream,
                         chunk-pipelined.  Asked for explicitly, a staging allocation that fails is KV_ERR_CUDA */
} kv_host_mode;

typedef enum kv_status {
  KV_OK = 0,
  KV_ERR_NULL = -1,       /* a required pointer is NULL */
  KV_ERR_SIZE = -2,       /* buffer too small; page sizes / counts inconsistent; more than 2^32-1 items per request */
  KV_ERR_PAGE_RANGE = -3, /* a page id is < 0 or >= num_pages */
  KV_ERR_DUP_PAGE = -4,   /* duplicate destination page id (checked only under KV_FLAG_VALIDATE) */
  KV_ERR_LAYOUT = -5,     /* unknown kv_layout / kv_host_mode / option */
  KV_ERR_ALIGN = -6,      /* a pointer or stride is not elem_bytes-aligned */
  KV_ERR_CUDA = -7,       /* a CUDA call failed; see kv_last_cuda_error() */
  KV_ERR_HOST_MEM = -8,   /* host buffer of an offload/reload is not pinned (page-locked) memory */
  KV_ERR_DESC = -9,       /* malformed kv_pool_desc (zero dimension, bad elem_bytes or order, stride < row, layer_count too large) */
  KV_ERR_NO_DEVICE = -10, /* planning-only ctx (device < 0): arguments were valid, nothing was launched */
  KV_ERR_CAPTURE = -11,   /* `stream` is capturing a CUDA graph and this call is not replayable: its tables exceed
                             the kernel parameters (~31 KiB: about 7,500 page ids per launch), the element-wise
                             fallback kernel is needed, or mode is KV_HOST_STAGED and the ctx has no staging buffer
                             yet.  Also: an eager KV_HOST_STAGED transfer while another stream's open capture holds the
                             ctx's side stream.  Nothing was enqueued. */
  KV_ERR_STATIC_LIMIT = -12, /* kv_pack_static only: the request needs more table space than the library's fixed,
                             built-in device array holds (more than KV_STATIC_MAX_PAGES page ids or more than
                             KV_STATIC_MAX_SLABS layer x K/V slabs).  Nothing was enqueued; split the request. */
} kv_status;

/* flags (bit set) */
#define KV_FLAG_VALIDATE 0x1u      /* also check destination page ids for duplicates (unpack/reload) */
#define KV_FLAG_IDS_ON_DEVICE 0x2u /* page_ids is a DEVICE pointer; range errors skip the page and set the device status word */

/* kv_ctx_set_option keys (tuning; defaults are the measured best) */
typedef enum kv_option {
  KV_OPT_KERNEL = 0,         /* 0 auto, 1 bulk (cp.async.bulk ring, persistent CTAs), 2 vec (16-byte LDG/STG), 3 elem (any
                                alignment), 4 shot (cp.async.bulk, one segment per single-warp CTA) */
  KV_OPT_STAGE_BYTES = 1,    /* bulk: bytes per shared-memory stage (multiple of 16, 1 KiB .. 64 KiB) */
  KV_OPT_STAGES_PER_WARP = 2,/* bulk: ring depth per issuing warp (2 .. 16) */
  KV_OPT_WARPS = 3,          /* bulk: issuing warps per CTA (1 .. 8).  Until options 1-3 are set the ring follows the row
                                width: ~128 KiB of stages per SM (2 x 4 x 16 KiB ... 8 x 16 x 1 KiB); setting any pins it */
  KV_OPT_STORE_LAG = 4,      /* bulk: stores left in flight before a stage is refilled (1 .. 3) */
  KV_OPT_MAX_CTAS = 5,       /* cap on the grid (0 = SM count x CTAs per SM) */
  KV_OPT_CHUNK_BYTES = 6,    /* staged host transfers: bytes per pipeline chunk (0 = automatic: equal chunks, at least two per
                                transfer where that leaves 64 MiB each, at most one staging slot each) */
  KV_OPT_HOST_MAX_CTAS = 7,  /* grid cap for DIRECT host transfers (0 = automatic: 64 CTAs up to 16 MiB of payload -- the link
                                saturates with far fewer CTAs than HBM and small transfers finish sooner, 1 MiB 39 -> 34 us --
                                and the device grid above) */
  KV_OPT_STAGING_SLOTS = 8,  /* staged host transfers: pipeline slots the staging buffer is cut into (2 .. 4) */
  KV_OPT_L2_HINT = 9,        /* bulk: L2 cache hints, a bit set: 1 = loads evict_first, 2 = stores evict_first, 4 = stores
                                evict_last (2 and 4 exclude each other: 0 .. 5) */
  KV_OPT_INLINE_TABLES = 10, /* 1 (default): page ids / slab bases ride in the kernel parameters when they fit (<= 31 KiB);
                                0: always stage them through the ctx's pinned ring with one H2D copy */
  KV_OPT_DYNAMIC = 11,       /* bulk: 1 (default) large launches claim segments from a device counter (guided chunks);
                                0: static round-robin only */
  KV_OPT_TENSOR_MAPS = 12,   /* HND pools: 1 (default) whole-token boxes move with cp.async.bulk.tensor through per-slab
                                tensor maps (cached per pool in the ctx; the copy engine transposes [head][token]);
                                0: row-gather / 16-byte store paths only */
  KV_OPT_PDL = 13,           /* bulk: 1 (default) = launch with programmatic stream serialization: the grid may become resident
                                and run its prologue while the previous kernel of the stream drains; it touches no
                                global memory before that kernel has completed (griddepcontrol.wait) */
  KV_OPT_RESERVE_STAGING = 14, /* allocate the staging buffer of STAGED host transfers NOW (value = bytes; 0 = the size given
                                to kv_ctx_create, else 1 GiB) instead of on the first staged call -- required before a
                                first staged transfer can be captured.  Already allocated: KV_OK if value is 0 or the
                                same size, else KV_ERR_SIZE. */
  KV_OPT_LEAD_CHUNK = 15,    /* staged page-first host transfers of 128 MiB or more: bytes of the short chunk that leads an
                                offload / ends a reload, so that the one kernel no copy hides is a short one (default
                                32 MiB; 0 = equal chunks; ignored with KV_OPT_CHUNK_BYTES) */
} kv_option;

/* kv_ctx_get_stat keys */
typedef enum kv_stat {
  KV_STAT_LAUNCHES = 0,     /* kernels launched by this ctx since creation */
  KV_STAT_MEMCPYS = 1,      /* copy-engine memcpys issued by this ctx since creation (id staging + staged host transfers) */
  KV_STAT_LAST_ITEMS = 2,   /* work items (segments) planned by the last call */
  KV_STAT_LAST_PAYLOAD = 3, /* payload bytes of the last call (bytes written at the destination) */
  KV_STAT_LAST_KERNEL = 4,  /* kernel variant the last call used (KV_OPT_KERNEL values) */
  KV_STAT_LAST_HOST_MODE = 5,/* host mode the last offload/reload used (kv_host_mode) */
  KV_STAT_LAST_GRID = 6,    /* CTAs of the last launch */
  KV_STAT_LAST_SEGMENT = 7, /* bytes per work item of the last call */
  KV_STAT_LAST_TENSOR_MAPS = 8, /* 1 if the last call's launches used tensor maps for an HND pool side */
  KV_STAT_LAST_PLAIN = 9,   /* 1 if the last launch was the short kernel of the plain case (kv_move_shot_plain: one request,
                               equal page sizes, page-first, no zero fill, host ids) */
} kv_stat;

/* ---- library ------------------------------------------------------------------------------ */
uint32_t kv_version(void);          /* KVTIER_VERSION of the loaded library */
const char *kv_strerror(int status); /* static string, never NULL */

/* ---- context ------------------------------------------------------------------------------ */
/* Creates the per-thread context on CUDA device `device`: side stream, events, the ring that
 * stages page-id lists, a device status word and (lazily, on the first STAGED transfer)
 * `staging_bytes` of device staging (0 = 1 GiB = two 512 MiB pipeline slots).  `device` < 0 creates a PLANNING-ONLY ctx
 * that touches no CUDA API: every transfer call validates and plans, then returns
 * KV_ERR_NO_DEVICE instead of launching (used by host-side tests). */
int kv_ctx_create(kv_ctx **out, int device, size_t staging_bytes);
int kv_ctx_destroy(kv_ctx *ctx); /* synchronises the ctx's own work, frees everything it owns */
int kv_ctx_set_option(kv_ctx *ctx, int option, int64_t value); /* KV_ERR_LAYOUT on unknown key, KV_ERR_SIZE on bad value */
int kv_ctx_get_stat(kv_ctx *ctx, int stat, uint64_t *out);
int kv_last_cuda_error(kv_ctx *ctx); /* the cudaError_t behind the last KV_ERR_CUDA (0 if none) */
/* Reads (and clears) the device status word; synchronises the device.  Bit 0: a device-resident
 * page id was out of range (that page was skipped). */
int kv_device_status(kv_ctx *ctx, uint32_t *out);

/* ---- peer GPU as a tier --------------------------------------------- */
/* The single-box analogue of the provider-issued batched write of PAPER.md:L236 ("the consumer supplies
 * destination-buffer descriptors, and the provider issues batched RDMA writes"): after kv_peer_enable, any
 * pool slab or transfer buffer of a call may live on `peer_device`; the SAME kernels then load from / store
 * to it over NVLink (UVA addresses, one-sided, no collective, no copy on the peer).  The push direction
 * (kv_unpack / kv_repage from local memory into a peer pool: posted stores) is the fast one.
 * Errors: KV_ERR_SIZE if peer_device is the ctx's own device or negative; KV_ERR_CUDA if the device does
 * not exist, has no peer path to the ctx's device (cudaDeviceCanAccessPeer = 0) or enabling fails;
 * KV_ERR_NO_DEVICE on a planning-only ctx.  Enabling twice is KV_OK.  The mapping lasts for the process. */
int kv_peer_enable(kv_ctx *ctx, int peer_device);
/* kv_signal: enqueue on `stream` a release-ordered, system-scope store of `value` to the 8-byte-aligned
 * word `flag` (device memory of the ctx's device or of an enabled peer, or mapped pinned host memory).
 * Stream order puts it after every transfer enqueued on `stream` before it, so a consumer on the peer GPU
 * (or the host) that reads `flag` == value with an acquire load may read the transferred pages: the
 * availability notification of PAPER.md:L234, without a host round trip.  Capturable. */
int kv_signal(kv_ctx *ctx, uint64_t *flag, uint64_t value, kv_stream_t stream);

/* ---- chained paged hashing ------------------------------------------ */
/* "each page ID hashes its predecessor together with the current page's content
 * identities, thereby representing the complete page-aligned prefix" -- the 64-bit ids under which KV pages
 * are published and looked up (not the int32 pool slots the transfers take).  The paper names no hash;
 * this library fixes (readings H1-H4): one 64-bit content identity per token position; 64-bit
 * FNV-1a, byte-serial, little-endian encodings;
 *     digest_k = FNV1a(identities of page k, 8*page_size bytes)
 *     id_k     = FNV1a(LE64(id_{k-1}) || LE64(digest_k)),   id_{-1} = roots[s] (KV_CHAIN_ROOT if roots == NULL)
 * and only whole pages get ids: session s yields floor(len_s / page_size) of them.
 *   ident         DEVICE uint64[tok_offsets[n_sessions]], 8-byte aligned; session s owns
 *                 [tok_offsets[s], tok_offsets[s+1])
 *   tok_offsets   HOST int64[n_sessions+1], non-negative, non-decreasing (consumed before return)
 *   roots         HOST uint64[n_sessions] or NULL
 *   out           DEVICE uint64[out_capacity]; ids of session s start at page_offsets[s] (sessions back to back)
 *   page_offsets  HOST int64[n_sessions+1], written by the call (may be NULL)
 * Up to 128 sessions: ONE launch on `stream` (a CTA per session digests its pages, then its first warp walks the
 * chain), tables in the kernel parameters, capturable.  More: two launches (per-page digests of all sessions in
 * parallel, then one warp per session along the chain) with tables staged through the ctx's pinned ring.
 * Results are defined after the caller synchronises `stream`.  Errors: KV_ERR_NULL, KV_ERR_SIZE (page_size
 * 0, bad offsets, out_capacity too small), KV_ERR_ALIGN, KV_ERR_CAPTURE (more than 128 sessions), KV_ERR_NO_DEVICE
 * (planning-only ctx; page_offsets are still written), KV_ERR_CUDA.  n_sessions == 0 or no whole page:
 * KV_OK, nothing launched. */
#define KV_CHAIN_ROOT 0xcbf29ce484222325ull
int kv_chain_hash(kv_ctx *ctx, const uint64_t *ident, const int64_t *tok_offsets, uint32_t n_sessions,
                  uint32_t page_size, const uint64_t *roots, uint64_t *out, size_t out_capacity,
                  int64_t *page_offsets, kv_stream_t stream);

/* ---- pinned host memory (the L2 CPU tier) ----------------------------------- */
int kv_host_alloc(void **p, size_t bytes); /* page-locked, mapped, portable; free with kv_host_free */
int kv_host_free(void *p);
int kv_host_register(void *p, size_t bytes); /* pin + map an existing host range */
int kv_host_unregister(void *p);

/* ---- device-side pack / unpack -------------------------------------- */
/* kv_pack: gather pages page_ids[0..n) of the first `layer_count` layers of `pools` into the
 * transfer buffer `dst` (DEVICE-accessible memory, >= n*layer_count*kv_count*row bytes):
 *   page-first:  dst[p][l][c][t][h][d] = POOL[l][c][page_ids[p]][t][h][d]
 * (BASELINE.json:configs[0]).  page_ids order is sequence order and is never
 * changed; duplicates are allowed (read-only).  n == 0 is KV_OK with no launch. */
int kv_pack(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *page_ids,
            uint32_t n, int layout, void *dst, size_t dst_bytes, uint32_t flags, kv_stream_t stream);

/* kv_unpack: scatter a transfer buffer of `src_page_size`-token pages holding `n_tokens` valid
 * tokens into pages dst_page_ids[0..n_dst_pages) of `pools`, whose page size must equal
 * `dst_page_size`; n_dst_pages must be ceil(n_tokens / dst_page_size).  Sequence token
 * j = p*Ts + t lands in destination page j / Td, slot j % Td; slots j >= n_tokens of the touched
 * destination pages are set to all-bits-zero; source tokens >= n_tokens are ignored
 * (BASELINE.json:configs[4]; "total valid token length").  For a verbatim
 * whole-page copy pass n_tokens = n*Ts.  `src` must hold ceil(n_tokens/Ts) pages.
 * Nothing else in any pool is written. */
int kv_unpack(kv_ctx *ctx, const void *src, size_t src_bytes, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
              uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens, int layout,
              uint32_t flags, kv_stream_t stream);

/* Batched (CSR) variants (BASELINE.json:configs[3]): request r owns
 * page_ids[req_offsets[r] .. req_offsets[r+1]) and its own buffer dsts[r] / srcs[r] (HOST arrays
 * of device-accessible pointers).  ONE launch covers all requests.  `dst_bytes` / `src_bytes`
 * (per request) may be NULL to skip the size check.  For unpack, request r must own exactly
 * ceil(n_tokens[r] / dst_page_size) destination pages. */
int kv_pack_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                    const int32_t *page_ids, const int64_t *req_offsets, uint32_t n_req, int layout,
                    void *const *dsts, const uint64_t *dst_bytes, uint32_t flags, kv_stream_t stream);
int kv_unpack_batched(kv_ctx *ctx, const void *const *srcs, const uint64_t *src_bytes,
                      const int32_t *dst_page_ids, const int64_t *req_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                      uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                      int layout, uint32_t flags, kv_stream_t stream);

/* ---- kv_pack without any allocation (for callers that must not allocate) ----------------------
 * Who this is for.  Every other entry point needs a kv_ctx, and a ctx allocates: kv_ctx_create takes device memory,
 * a stream and events, and a transfer whose lookup tables (slab bases + page ids) outgrow the kernel parameters
 * (about 7,500 page ids) makes the ctx grow a pinned + device table arena INSIDE the call.  Some callers cannot live
 * with that:
 *   - a serving engine that has handed (nearly) all HBM to its KV pools: cudaMalloc would fail, or succeed only by
 *     evicting something the engine counted on;
 *   - a latency-critical step: cudaMalloc / cudaFree synchronise the whole device, so one allocation in a transfer
 *     call stalls every stream of the process, not only the caller's;
 *   - a process whose memory is owned by a pool allocator (or a sandbox / MPS client with a fixed memory budget) and
 *     whose rules forbid raw CUDA allocations from a library.
 * kv_pack_static is kv_pack for them: same bytes, no ctx, and neither it nor anything it calls ever calls cudaMalloc,
 * cudaMallocHost, cudaFree, cudaStreamCreate, cudaEventCreate or any other allocating routine.
 *
 * What it does.  dst[p][l][c][t][h][d] = POOL[l][c][page_ids[p]][t][h][d] for p < n, the first `layer_count` layers of
 * `pools`, page-first (KV_LAYOUT_PAGE_FIRST): byte for byte what kv_pack writes.  The kernel is the library's
 * kv_move_shot_plain in its tables-in-device-memory form -- the form that otherwise reads its tables from the ctx's
 * allocated arena.  Here the tables live in ONE fixed array that is part of the library image (a file-scope
 * `static __device__` array in kvtier.cu, 256-byte aligned, KV_STATIC_TABLE_BYTES = 270,592 bytes, about 264 KiB).  The
 * driver places a copy of it on every GPU on which this process uses the library, when the library's device code is
 * loaded there, and that copy stays until the process exits; no call allocates or frees it.
 *   device      CUDA device that owns `pools`, `dst` and `stream` (0 .. 63).  Made current for the call and restored.
 *   pools       as kv_pack.  Restrictions of this entry point: NHD pools only (KV_ERR_LAYOUT for an HND pool), and every
 *               slab base, the page stride, the token row (num_heads*head_dim*elem_bytes) and `dst` must be multiples
 *               of 16 bytes (KV_ERR_ALIGN): there is no element-wise fallback here.
 *   page_ids    HOST int32[n], sequence order, duplicates allowed; consumed before the call returns.
 *   dst         device-accessible memory (device, or mapped pinned host), >= n*layer_count*kv_count*row bytes.
 *   cuda_error  may be NULL; receives the cudaError_t behind a KV_ERR_CUDA (there is no ctx to ask).
 * Limits: n <= KV_STATIC_MAX_PAGES (65,536 page ids: a 1M-token prefix at 16 tokens per page) and
 * layer_count*kv_count <= KV_STATIC_MAX_SLABS (1,024).  Anything larger is refused with KV_ERR_STATIC_LIMIT before
 * anything is enqueued -- the array cannot grow; split the request into several calls on the same stream.
 *
 * First call on a device.  The array's name is not a device address in host code; the first call on each device asks
 * the runtime for that device's address of it (cudaGetSymbolAddress, with the device current), reads the SM count and
 * sets the kernel's shared-memory preference, and remembers the result for the life of the process.  This may make the
 * driver load the library's device code onto that GPU.  Make this first call (n = 1 is enough) during start-up, BEFORE
 * the stream is put into CUDA-graph capture: the set-up calls are not stream work and do not belong in a capture.
 *
 * Sharing.  All calls on one device use the SAME array.  A call overwrites the table prefix it needs (header, slab
 * bases, page ids) with small fill launches ahead of its copy kernel, all on `stream`; whatever a previous call left
 * behind that prefix is never read, and the one word that has to be zero at kernel start (the kernels' status word, in
 * the header) is rewritten as zero by every call.  Calls on ONE stream are therefore safe back to back.  Calls whose
 * GPU work can overlap -- two streams without an event between them, two host threads, two graphs replayed at once --
 * race on the tables and copy the wrong pages: order them (one stream, or events) yourself.  Nothing detects it.
 * Other errors as kv_pack: KV_ERR_NULL, KV_ERR_DESC, KV_ERR_SIZE (dst_bytes too small, device out of range,
 * more than 2^31-1 segments), KV_ERR_PAGE_RANGE, KV_ERR_CUDA.  A call that returns a validation error (anything but
 * KV_ERR_CUDA) has written nothing.  n == 0: KV_OK, nothing enqueued. */
#define KV_STATIC_MAX_PAGES 65536u
#define KV_STATIC_MAX_SLABS 1024u
#define KV_STATIC_TABLE_BYTES (256u + KV_STATIC_MAX_SLABS * 8u + KV_STATIC_MAX_PAGES * 4u)
int kv_pack_static(int device, const kv_pool_desc *pools, uint32_t layer_count, const int32_t *page_ids, uint32_t n,
                   void *dst, size_t dst_bytes, kv_stream_t stream, int *cuda_error);

/* ---- several independent transfers in ONE launch ----------
 * A serving turn issues small transfers back to back -- scatter a matched prefix into fresh pages, extend the
 * retained partial page copy-on-write (the append follows the reload in every turn), gather the
 * pages that became full -- and below ~100 MiB each of them is bound by launch latency, not by HBM.  kv_submit
 * runs a list of such operations on ONE pool as one persistent launch: the direction is a property of the piece,
 * not of the launch.
 *   KV_OP_PACK        buf[p][l][c][..] = POOL[l][c][page_ids[p]]          (kv_pack; n_pages ids, buf written)
 *   KV_OP_UNPACK      POOL[l][c][page_ids[q]] = buf[q][l][c][..], slots >= n_tokens zero  (kv_unpack with the buffer's
 *                     page size equal to the pool's; n_pages must be ceil(n_tokens / page_size))
 *   KV_OP_COW_APPEND  kv_cow_append with old_id = page_ids[0], new_id = page_ids[1], append block `buf`
 * The operations of one call are UNORDERED among themselves: no operation may read a page or buffer that another
 * one writes, and all written pages must be distinct (both checked under KV_FLAG_VALIDATE -> KV_ERR_DUP_PAGE for
 * pages; buffers are the caller's responsibility).  The result equals the single calls issued in any order.
 * Errors as the single calls; KV_FLAG_IDS_ON_DEVICE is not supported here (KV_ERR_LAYOUT).  n_ops == 0 or nothing
 * to move: KV_OK, no launch. */
typedef enum kv_op_kind { KV_OP_PACK = 0, KV_OP_UNPACK = 1, KV_OP_COW_APPEND = 3 } kv_op_kind;
typedef struct kv_op {
  uint32_t kind;           /* kv_op_kind */
  uint32_t n_pages;        /* PACK: pages gathered; UNPACK: destination pages; COW_APPEND: ignored */
  const int32_t *page_ids; /* HOST array: PACK source ids / UNPACK destination ids (n_pages of them); COW_APPEND: {old, new} */
  void *buf;               /* device-accessible: PACK destination buffer; UNPACK source buffer; COW_APPEND append block (NULL if n_app == 0) */
  uint64_t buf_bytes;      /* PACK / UNPACK: size of buf for the bounds check (0 = unchecked) */
  uint64_t n_tokens;       /* UNPACK: valid tokens (n_pages * page_size = verbatim whole pages) */
  uint32_t n_old, n_app;   /* COW_APPEND: tokens kept from the old page, tokens appended; n_old + n_app <= page_size */
} kv_op;
int kv_submit(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const kv_op *ops, uint32_t n_ops,
              int layout, uint32_t flags, kv_stream_t stream);

/* ---- fused pool -> pool re-paging (8(c) reading 11) ------------------
 * kv_repage: kv_pack followed by kv_unpack without the transfer buffer, for cross-role reuse on one
 * device (a diffusion role reuses the LLM role's conditioning KV;
 * BASELINE.json:configs[4]: destination page size differs).  With Ts = src_pools->page_size and
 * Td = dst_pools->page_size, sequence token j of the request lives in source page
 * src_page_ids[j / Ts], slot j % Ts, and lands in destination page dst_page_ids[j / Td], slot j % Td;
 * slots j >= n_tokens of the touched destination pages are all-bits-zero; source tokens >= n_tokens
 * are ignored.  n_src_pages must be ceil(n_tokens/Ts) and n_dst_pages ceil(n_tokens/Td).  The two
 * descriptors must agree in kv_count, num_heads, head_dim and elem_bytes (KV_ERR_DESC otherwise);
 * page counts, page sizes and strides are their own; `layer_count` layers of both are used.  Ts == Td
 * makes it a page migration inside or between pools.  The source pool is never written; destination
 * pages must be distinct and must not be source pages.  HBM traffic is 2 x payload instead of the
 * 4 x of pack + unpack.  With KV_FLAG_IDS_ON_DEVICE both id lists are DEVICE arrays (offsets and token counts
 * stay on the host); an out-of-range id of either list skips its piece and sets the device status word. */
int kv_repage(kv_ctx *ctx, const kv_pool_desc *src_pools, const int32_t *src_page_ids,
              uint32_t n_src_pages, const kv_pool_desc *dst_pools, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, uint32_t layer_count, uint64_t n_tokens, uint32_t flags,
              kv_stream_t stream);
/* Batched: request r re-pages src_page_ids[src_offsets[r] .. src_offsets[r+1]) into
 * dst_page_ids[dst_offsets[r] .. dst_offsets[r+1]) with n_tokens[r] valid tokens.  ONE launch. */
int kv_repage_batched(kv_ctx *ctx, const kv_pool_desc *src_pools, const int32_t *src_page_ids,
                      const int64_t *src_offsets, const kv_pool_desc *dst_pools,
                      const int32_t *dst_page_ids, const int64_t *dst_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, uint32_t layer_count, uint32_t flags,
                      kv_stream_t stream);

/* ---- copy-on-write partial-page append ----------------
 * "When incremental data extends a retained partial page, the system copies its existing contents
 * into a writable slot and appends the new data there.  The updated page is published under a new
 * page ID, preserving the old published identity" (sec. 4.1.4).  For every (layer, K|V):
 *   NEW[new_id][t] = OLD[old_id][t]        for t <  n_old
 *                  = app[l][c][t - n_old]  for n_old <= t < n_old + n_app
 *   slots t >= n_old + n_app of the new page, the old page and every other page are not written.
 * `app` is DEVICE-accessible memory (device, or mapped pinned host), dense
 * [layer][K,V][token][head][dim] with n_app tokens and `layer_count` layers; it may be NULL when
 * n_app == 0 (a plain page copy).  n_old + n_app <= page_size and old_id != new_id (KV_ERR_SIZE).
 * The batched call covers all sessions in ONE launch; new ids must be distinct and must not be any
 * session's old id (checked under KV_FLAG_VALIDATE -> KV_ERR_DUP_PAGE).  With KV_FLAG_IDS_ON_DEVICE (batched entry)
 * old_ids / new_ids are DEVICE arrays of n_sessions ids (n_old, n_app and apps stay on the host); a session whose
 * ids are out of range or equal is skipped and raises the device status word.  kv_cow_append itself takes its two
 * ids by value, so the flag has no meaning there and is refused (KV_ERR_LAYOUT). */
int kv_cow_append(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, int32_t old_id,
                  int32_t new_id, uint32_t n_old, const void *app, uint32_t n_app, uint32_t flags,
                  kv_stream_t stream);
int kv_cow_append_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                          const int32_t *old_ids, const int32_t *new_ids, const uint32_t *n_old,
                          const uint32_t *n_app, const void *const *apps, uint32_t n_sessions,
                          uint32_t flags, kv_stream_t stream);

/* ---- host tier: offload (device -> pinned host) and reload (pinned host -> device) ----------
 * Same semantics and bytes as kv_pack / kv_unpack with the transfer buffer in PINNED HOST memory
 * (from kv_host_alloc, kv_host_register, cudaHostAlloc or torch pin_memory); a pageable pointer
 * is KV_ERR_HOST_MEM.  `mode` must not change a single byte of the result.
 * Appending to a session's host buffer is a call with host_dst advanced by the pages already
 * there (page-first makes append a tail write). */
int kv_offload(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
               const int32_t *page_ids, uint32_t n, int layout, void *host_dst, size_t host_bytes,
               int mode, uint32_t flags, kv_stream_t stream);
int kv_reload(kv_ctx *ctx, const void *host_src, size_t host_bytes, const int32_t *dst_page_ids,
              uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
              uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens, int layout,
              int mode, uint32_t flags, kv_stream_t stream);
/* kv_reload_layerwise[_batched]: kv_reload of a LAYER-FIRST host buffer [layer][K,V][page][token][head][dim]
 * that publishes its progress per layer ("layer-first buffer ... enables per-layer
 * streaming reload overlapped with prefill").  Arguments as kv_reload[_batched]; the layout is
 * KV_LAYOUT_LAYER_FIRST by definition.  `layer_flags` is an 8-byte-aligned array of `layer_count` words in
 * device memory or mapped pinned host memory: once every page of layer l (all requests) is in the pool,
 * layer_flags[l] = flag_value is stored with release semantics at system scope, in stream order -- a consumer
 * that acquires the flag may read the layer: the host (which then launches layer l's attention), a kernel on
 * ANOTHER GPU, or a kernel that checks the flag once and does not spin.  Do NOT park a kernel of the same GPU in a
 * loop on these flags: nothing guarantees that it and the transfer's kernels run at the same time (measured on
 * this B200 / driver 580: a spinning kernel on one stream kept a kernel of another stream from starting).
 * Flags are stored in ascending layer order.  KV_HOST_STAGED (AUTO's choice from 4 MiB) streams the buffer
 * through the ctx's staging in chunks of whole layers (a layer wider than a staging slot is cut by page
 * ranges), copy engine and scatter kernel pipelined, so layer 0 is usable after ~1/layer_count of the
 * transfer; KV_HOST_DIRECT is one launch over all layers followed by all flags.  n_req == 0 or no pages:
 * the flags are still stored.  Errors as kv_reload, plus KV_ERR_NULL / KV_ERR_ALIGN / KV_ERR_HOST_MEM for
 * `layer_flags`. */
int kv_reload_layerwise(kv_ctx *ctx, const void *host_src, size_t host_bytes, const int32_t *dst_page_ids,
                        uint32_t n_dst_pages, const kv_pool_desc *pools, uint32_t layer_count,
                        uint32_t src_page_size, uint32_t dst_page_size, uint64_t n_tokens,
                        uint64_t *layer_flags, uint64_t flag_value, int mode, uint32_t flags,
                        kv_stream_t stream);
int kv_reload_layerwise_batched(kv_ctx *ctx, const void *const *host_srcs, const uint64_t *host_bytes,
                                const int32_t *dst_page_ids, const int64_t *req_offsets,
                                const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                                uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                                uint64_t *layer_flags, uint64_t flag_value, int mode, uint32_t flags,
                                kv_stream_t stream);
int kv_offload_batched(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count,
                       const int32_t *page_ids, const int64_t *req_offsets, uint32_t n_req,
                       int layout, void *const *host_dsts, const uint64_t *host_bytes, int mode,
                       uint32_t flags, kv_stream_t stream);
int kv_reload_batched(kv_ctx *ctx, const void *const *host_srcs, const uint64_t *host_bytes,
                      const int32_t *dst_page_ids, const int64_t *req_offsets,
                      const uint64_t *n_tokens, uint32_t n_req, const kv_pool_desc *pools,
                      uint32_t layer_count, uint32_t src_page_size, uint32_t dst_page_size,
                      int layout, int mode, uint32_t flags, kv_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* KVTIER_H */
