// kv_kernels.cuh -- sm_100a kernels of the paged-KV tier transfer.
//
// Every transfer (pack, unpack, re-page, copy-on-write append, batched, kv_submit, direct host offload/reload, every chunk
// of a staged host transfer) is ONE launch of one of the kernels below over a flat list of work items ("segments").  A
// segment is a run of bytes that is contiguous on BOTH sides: g = gcd(Tpool, Tbuf) tokens of one (layer, K|V) of one
// page, cut into pieces of at most `sub_bytes`.  The pool side hops between 2*L slabs by page id (PAPER.md:L207
// addressing); the buffer side is the dense lower-tier representation (BASELINE.json:configs[0]).
//
//   kv_move_shot        the B200 path, AUTO's choice for segments of 4 KiB or more (every shape of the paper): ONE
//                       segment per single-warp CTA, moved global -> shared -> global by cp.async.bulk (SASS UBLKCP) or,
//                       for an HND pool, by cp.async.bulk.tensor through per-slab tensor maps (UTMALDG / UTMASTG: the
//                       copy engine does the [head][token] transposition).  13 CTAs = 208 KiB in flight per SM; the CTA
//                       scheduler is the work distributor.  No payload byte passes through registers.
//   kv_move_shot_plain  its short form for the plain case (equal page sizes, page-first, nothing to zero-fill, host ids;
//                       one request or a batch): ~170 instructions, lane 0 alone works.  What small calls and the
//                       headline config run.
//   kv_move_bulk        persistent CTAs, a per-warp ring of mbarrier-tracked stages, 32 segments decoded per warp at
//                       once, guided claiming from a device counter: AUTO's choice for 2-4 KiB segments, where the rate
//                       at which one SM retires bulk copies binds the one-shot kernel.
//   kv_move_vec         16-byte LDG/STG, one warp per segment, 8 loads in flight per lane (strided HND destinations
//                       without tensor maps, large copy-on-write batches on narrow rows).
//   kv_move_small       segments <= 1 KiB: 32 segments decoded per warp, copied eight at a time (16-byte LDG/STG).
//   kv_move_elem        any alignment: unit-wide (1/2/4/8 B) coalesced copy.  Correctness fallback.
//
// This file shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kvt {

// One contiguous transfer buffer: a request, or one pipeline chunk of a request.
//   dir 2 (pool -> pool): `buf` is the index of the request's first SOURCE page id in ids[].
//   dir 3 (copy-on-write append, one piece per session): `buf` = append block address,
//         n_tokens = n_old | n_app << 32, id_begin = old page id | new page id << 32.
//   dir 4 (kv_submit: a mixed launch): every piece carries its own direction (0, 1 or 3) in `dir`.
struct Piece {
  uint64_t item_begin;   // first flat item index of this piece within the launch
  uint64_t buf;          // buffer base address (device memory or mapped pinned host memory)
  uint64_t n_tokens;     // valid tokens; destination slots >= n_tokens are zero-filled (unpack)
  uint64_t id_begin;     // index of this piece's first page id in ids[]
  uint64_t n_buf_pages;  // pages in this piece's buffer (layer-first page stride)
  uint32_t dir;          // Job::dir == 4 only: this piece's direction (0 pack, 1 unpack, 3 copy-on-write append)
  uint32_t pad_;
};

struct Job {
  const uint64_t *bases;  // [LC] slab base addresses, order [layer][kv]
  const int32_t *ids;     // page ids (device)
  const Piece *pieces;    // pieces of THIS launch
  uint32_t *status;       // device status word (bit 0: page id out of range)
  uint64_t total_items;
  uint64_t page_stride;     // pool bytes between pages
  uint64_t buf_row_bytes;   // Tbuf * tokrow
  uint64_t buf_page_bytes;  // LC * buf_row_bytes (page-first)
  uint32_t n_pieces;
  uint32_t LC;            // layer_count * kv_count
  uint32_t dir;           // 0 pack (pool -> buffer), 1 unpack (buffer -> pool), 2 re-page (pool -> pool),
                          // 3 copy-on-write append (old page + append block -> new page),
                          // 4 mixed (kv_submit): the direction is a property of the piece (Piece::dir)
  uint32_t layout;        // 0 page-first, 1 layer-first
  uint32_t g;             // tokens per chunk = gcd(Tpool, Tbuf)
  uint32_t cpp_pool;      // chunks per pool page  = Tpool / g
  uint32_t cpp_buf;       // chunks per buffer page = Tbuf / g
  uint32_t tokrow;        // bytes per token row = H*D*e
  uint32_t chunk_bytes;   // g * tokrow
  uint32_t sub_bytes;     // bytes per item (last item of a chunk may be shorter)
  uint32_t subs;          // items per chunk
  uint32_t num_pages;     // pool pages (range check of device-resident ids)
  // bulk kernel geometry
  uint32_t stage_bytes;
  uint32_t stages;        // per warp
  uint32_t lag;           // stores left in flight before a stage is refilled
  uint32_t zero_bytes;    // size of the shared zero region
  uint32_t l2_hint;
  // inline tables (JobT<N>, N > 0): byte offsets into the kernel-parameter blob
  uint32_t off_pieces, off_ids;
  // dynamic work distribution of kv_move_bulk (nullptr = static round-robin)
  unsigned long long *sched;  // global claim counter (items beyond the static first blocks)
  uint32_t *sched_done;       // warps finished; the last one resets both counters to 0
  uint32_t first_batch;       // B0: static items per warp before claiming starts
  uint32_t src_num_pages;     // dir 2: pages of the SOURCE pool (range check of device-resident ids)
  uint64_t src_page_stride;   // dir 2: source pool bytes between pages; its slab bases are bases[LC..2LC)
  // transposing transfers (an HND pool on either side; kTrans kernels only).  A side is either
  // contiguous in the item's NHD-linear order or "strided": row r = t*H + h of the chunk (one
  // head_dim row of `drow` bytes) sits at side_base + t*ts + h*hs.
  uint32_t drow;              // head_dim * elem_bytes
  uint32_t H;                 // num_heads
  uint32_t pool_hnd;          // the (destination) pool is HND
  uint32_t src_hnd;           // dir 2: the source pool is HND
  uint64_t p_ts, p_hs;        // strides of the pool side when it is HND (ts = drow, hs = Tpool*drow)
  uint64_t q_ts, q_hs;        // dir 2: strides of the source pool when it is HND
  // TMA tensor maps of HND pools (one 128-byte CUtensorMap per slab, device memory): the slab is the
  // rank-4 tensor (dim, head, token, page) with strides (1, T*drow, drow, page_stride) -- token and
  // head swapped against memory order -- so ONE cp.async.bulk.tensor with the box (drow, H, tb, 1)
  // moves tb whole tokens between the HND page and an NHD-linear shared-memory stage: the copy
  // engine does the [head][token] <-> [token][head] transposition.
  const uint8_t *maps_pool;   // nullptr: the pool side does not use tensor copies
  const uint8_t *maps_src;    // dir 2: the source pool's maps
  // The maps may instead ride INSIDE the kernel parameters (JobT<N>::blob, 64-byte aligned; 0 = they do not): a call
  // captured into a CUDA graph before its pool's maps exist in device memory cannot build them there (an allocation
  // and a blocking copy), but encoding a map is pure host work, and the copy engine reads a map from parameter space
  // as well as from global memory.
  uint32_t off_maps_pool, off_maps_src;
  uint32_t tb;                // tokens per box; a "full" item has bytes == valid == tb * tokrow
  // dir 2 with KV_FLAG_IDS_ON_DEVICE: the caller's device array of SOURCE page ids (then `ids` is the
  // caller's destination array and Piece::buf indexes this one); nullptr: both lists sit in `ids`
  const int32_t *src_ids;
  // n_pieces == 1 (every single-request call, every chunk of a staged single request): the piece itself.  It arrives
  // with the header, so a CTA's first load waits for one table level fewer (header -> ids / bases -> data instead of
  // header -> piece -> ids / bases -> data; each level is a first-touch constant-bank or L2 miss on every SM).
  Piece one;
  // Exact n / d for n < 2^32 by ONE 64-bit multiply-high: m = floor(2^64 / d) + 1 (0 stands for d == 1).  The divisors
  // are launch constants; a hardware-less 32-bit division costs ~20 dependent instructions, and decode chains three.
  uint64_t m_subs, m_LC, m_cpp_pool, m_cpp_buf;
  // The plain case -- pack or unpack between equal page sizes, page-first buffer(s), every token valid, page ids
  // validated on the host; 1 = ONE request (its piece rides in `one`), 2 = a batch of such requests (the plain kernel
  // finds an item's piece by binary search; the general kernel ignores the value 2): decode takes a short straight path
  // (two multiply-highs, two table reads, six multiply-adds).  A single-warp CTA hides no latency, so the ~300 dependent instructions of the general decode are
  // ~0.7 us in front of the first load of every CTA -- nothing at 768 MiB (13 CTAs per SM overlap), a quarter of a
  // 1 MiB call.
  uint32_t lean;
  uint32_t pad2_;
};
__device__ __forceinline__ uint32_t fdiv(uint32_t n, uint64_t m) {
  return m ? (uint32_t)__umul64hi((uint64_t)n, m) : n;
}

// The lookup tables of a launch: slab bases, page ids, pieces.  They live either in device memory
// (staged through the ctx's pinned ring, JobT<0>) or, for calls whose tables fit, INSIDE the kernel
// parameters (JobT<N>): one launch, no H2D copy, tables read through the constant bank.
struct Tables {
  const uint64_t *bases;
  const int32_t *ids;
  const Piece *pieces;
};
template <int N>
struct JobT {
  Job j;
  alignas(64) uint8_t blob[N];  // [bases: LC x u64][pieces][ids][64-byte aligned: tensor maps, if they travel here]
};
template <>
struct JobT<0> {
  Job j;
};
template <int N>
__device__ __forceinline__ Tables tables_of(const JobT<N> &p) {
  if constexpr (N == 0) {
    return Tables{p.j.bases, p.j.ids, p.j.pieces};
  } else {  // j.ids != nullptr: device-resident ids supplied by the caller
    return Tables{reinterpret_cast<const uint64_t *>(p.blob),
                  p.j.ids ? p.j.ids : reinterpret_cast<const int32_t *>(p.blob + p.j.off_ids),
                  reinterpret_cast<const Piece *>(p.blob + p.j.off_pieces)};
  }
}
template <bool kGlobal, typename T>
__device__ __forceinline__ T ldt(const T *p) {
  if constexpr (kGlobal) return __ldg(p);
  else return *p;
}

struct Item {
  uint64_t src, dst;
  uint32_t bytes;  // bytes written at dst
  uint32_t valid;  // first `valid` bytes come from src, the rest is zero fill
  // kTrans only: bit 0 = src strided, bit 1 = dst strided, bit 2 = never by tensor copies (copy-on-write rows).
  // A strided side's address is the base of
  // the CHUNK (token 0, head 0) and the item covers rows [r0, r0 + bytes/drow) of it; a contiguous
  // side's address already points at the item's first byte.
  uint32_t mode;
  uint32_t r0;
  // kTrans only: slab index and (page, first token) of a strided side, the coordinates of a tensor copy
  uint32_t lc, s_pg, s_t, d_pg, d_t;
};

// SURVEY.md 8(a) a2 for the plain case (Job::lean): flat item -> (page, layer/kv, sub) -> addresses.
struct Lean { uint64_t src, dst; uint32_t bytes; };
// `item` counts within the piece; buf / id_begin are the piece's (Job::one for a one-request launch).
template <bool kGlobal>
__device__ __forceinline__ Lean decode_lean(const Job &j, const Tables &tb, uint32_t item, uint64_t buf, uint64_t id_begin) {
  const uint32_t r1 = fdiv(item, j.m_subs), sub = item - r1 * j.subs;
  const uint32_t pp = fdiv(r1, j.m_LC), lc = r1 - pp * j.LC;
  const uint32_t sub_off = sub * j.sub_bytes;
  const int32_t id = kGlobal ? __ldg(tb.ids + id_begin + pp) : tb.ids[id_begin + pp];
  const uint64_t paddr = ldt<kGlobal>(tb.bases + lc) + (uint64_t)(uint32_t)id * j.page_stride + sub_off;
  const uint64_t baddr = buf + (uint64_t)pp * j.buf_page_bytes + (uint64_t)lc * j.buf_row_bytes + sub_off;
  Lean l;
  l.bytes = min(j.sub_bytes, j.chunk_bytes - sub_off);
  l.src = j.dir == 0 ? paddr : baddr;
  l.dst = j.dir == 0 ? baddr : paddr;
  return l;
}

// flat item -> (piece, chunk k, layer/kv, sub) -> addresses.
template <bool kGlobal, bool kTrans = false>
// `hint`: the piece this thread's previous item fell into.  A thread's items only grow, so the search starts
// there and gallops forward: one or two probes where a search over all pieces takes log2(n) dependent loads
// (2,048 one-page requests in one call: unpack 5.43 -> 5.87 TB/s; 64 requests: unchanged at 6.6).
__device__ __forceinline__ Item decode(const Job &j, const Tables &tb, uint64_t item, uint32_t &hint) {
  if (!kTrans && j.lean == 1) {  // launch() sets it: dir 0 / 1, one piece, page-first, Tpool == Tbuf, no padding, host ids
    const Lean l = decode_lean<kGlobal>(j, tb, (uint32_t)item, j.one.buf, j.one.id_begin);
    Item it;
    it.mode = 0; it.r0 = 0; it.lc = 0; it.s_pg = it.s_t = it.d_pg = it.d_t = 0;
    it.src = l.src; it.dst = l.dst; it.bytes = it.valid = l.bytes;
    return it;
  }
  uint32_t r = 0;
  if (j.n_pieces > 1) {  // largest r with pieces[r].item_begin <= item
    uint32_t lo = hint < j.n_pieces ? hint : 0;
    if (lo && ldt<kGlobal>(&tb.pieces[lo].item_begin) > item) lo = 0;
    uint32_t step = 1, hi = lo + 1;
    while (hi < j.n_pieces && ldt<kGlobal>(&tb.pieces[hi].item_begin) <= item) {
      lo = hi;
      hi += step;
      step <<= 1;
    }
    hi = min(hi, j.n_pieces);
    while (hi - lo > 1) {
      uint32_t mid = (lo + hi) >> 1;
      if (ldt<kGlobal>(&tb.pieces[mid].item_begin) <= item) lo = mid; else hi = mid;
    }
    r = lo;
    hint = r;
  }
  uint64_t item_begin, buf, n_tokens, id_begin, n_buf_pages;
  uint32_t pdir;
  if (j.n_pieces > 1) {
    const Piece *pc = tb.pieces + r;
    item_begin = ldt<kGlobal>(&pc->item_begin); buf = ldt<kGlobal>(&pc->buf);
    n_tokens = ldt<kGlobal>(&pc->n_tokens); id_begin = ldt<kGlobal>(&pc->id_begin);
    n_buf_pages = j.layout ? ldt<kGlobal>(&pc->n_buf_pages) : 0;
    pdir = j.dir == 4 ? ldt<kGlobal>(&pc->dir) : 0;
  } else {  // the piece rides in the header
    item_begin = j.one.item_begin; buf = j.one.buf; n_tokens = j.one.n_tokens; id_begin = j.one.id_begin;
    n_buf_pages = j.one.n_buf_pages; pdir = j.one.dir;
  }
  const uint32_t local = (uint32_t)(item - item_begin);
  const uint32_t dir = j.dir == 4 ? pdir : j.dir;
  if (dir == 3) {  // copy-on-write append: per (layer,kv) s0 items copy the old
                     // page's first n_old tokens, s1 items append the session's new rows behind them
    const uint32_t n_old = (uint32_t)n_tokens, n_app = (uint32_t)(n_tokens >> 32);
    const uint32_t b_old = n_old * j.tokrow, b_app = n_app * j.tokrow;
    const uint32_t s0 = (b_old + j.sub_bytes - 1) / j.sub_bytes, s1 = (b_app + j.sub_bytes - 1) / j.sub_bytes;
    const uint32_t lc = local / (s0 + s1), k = local - lc * (s0 + s1);
    const uint64_t slab = ldt<kGlobal>(tb.bases + lc);
    uint32_t old_id = (uint32_t)id_begin, new_id = (uint32_t)(id_begin >> 32);
    Item it;
    it.mode = 0; it.r0 = 0;
    it.lc = lc; it.s_pg = it.s_t = it.d_pg = it.d_t = 0;
    if (j.src_ids) {  // KV_FLAG_IDS_ON_DEVICE: id_begin is the session index into the caller's device arrays
      old_id = (uint32_t)__ldg(j.ids + id_begin);
      new_id = (uint32_t)__ldg(j.src_ids + id_begin);
      if (old_id >= j.num_pages || new_id >= j.num_pages || old_id == new_id) {
        atomicOr(j.status, 1u);
        it.src = it.dst = 0; it.bytes = it.valid = 0;
        return it;
      }
    }
    const uint64_t old_pg = slab + (uint64_t)old_id * j.page_stride;
    const uint64_t new_pg = slab + (uint64_t)new_id * j.page_stride;
    if (k < s0) {
      const uint32_t o = k * j.sub_bytes;
      it.src = old_pg + o; it.dst = new_pg + o; it.bytes = min(j.sub_bytes, b_old - o);
      if (kTrans && j.pool_hnd) {  // rows of the first n_old tokens, same place in both pages
        it.src = old_pg; it.dst = new_pg; it.mode = 3 | 4; it.r0 = o / j.drow;
      }
    } else {
      const uint32_t o = (k - s0) * j.sub_bytes;
      it.src = buf + (uint64_t)lc * b_app + o; it.dst = new_pg + b_old + o; it.bytes = min(j.sub_bytes, b_app - o);
      if (kTrans && j.pool_hnd) {  // NHD append block -> token slots n_old.. of every head's run
        it.dst = new_pg + (uint64_t)n_old * j.p_ts; it.mode = 2 | 4; it.r0 = o / j.drow;
      }
    }
    it.valid = it.bytes;
    return it;
  }
  const uint32_t r1 = fdiv(local, j.m_subs), sub = local - r1 * j.subs;
  const uint32_t k = fdiv(r1, j.m_LC), lc = r1 - k * j.LC;
  const uint32_t pp = fdiv(k, j.m_cpp_pool), pk = k - pp * j.cpp_pool;
  const uint32_t bp = fdiv(k, j.m_cpp_buf), bk = k - bp * j.cpp_buf;
  const uint64_t sub_off = (uint64_t)sub * j.sub_bytes;
  Item it;
  it.mode = 0; it.r0 = 0;
  it.lc = lc; it.s_pg = it.s_t = it.d_pg = it.d_t = 0;
  it.bytes = min(j.sub_bytes, j.chunk_bytes - (uint32_t)sub_off);
  // caller-supplied device ids are global memory even when the other tables are inline
  const int32_t id = (kGlobal || j.ids) ? __ldg(tb.ids + id_begin + pp) : tb.ids[id_begin + pp];
  if ((uint32_t)id >= j.num_pages) {  // only reachable with KV_FLAG_IDS_ON_DEVICE
    atomicOr(j.status, 1u);
    it.src = it.dst = 0; it.bytes = it.valid = 0;
    return it;
  }
  uint64_t paddr = ldt<kGlobal>(tb.bases + lc) + (uint64_t)id * j.page_stride;
  uint32_t pmode = 0, bmode = 0;  // is the pool / buffer side strided?
  if (kTrans && j.pool_hnd) { paddr += (uint64_t)pk * j.g * j.p_ts; pmode = 1; }
  else paddr += (uint64_t)pk * j.chunk_bytes + sub_off;
  const uint64_t tok0 = (uint64_t)k * j.g;
  const uint64_t vt = n_tokens > tok0 ? min(n_tokens - tok0, (uint64_t)j.g) : 0;
  uint64_t baddr;
  if (dir == 2 && vt == 0) {  // wholly zero-padded chunk: there is no source page to look up
    baddr = 0;
  } else if (dir == 2) {  // pool -> pool: the "buffer" side is page src_ids[bp] of the source pool
    const int32_t sid = j.src_ids ? __ldg(j.src_ids + buf + bp)
                                  : ((kGlobal || j.ids) ? __ldg(tb.ids + buf + bp) : tb.ids[buf + bp]);
    if ((uint32_t)sid >= j.src_num_pages) {
      atomicOr(j.status, 1u);
      it.src = it.dst = 0; it.bytes = it.valid = 0;
      return it;
    }
    baddr = ldt<kGlobal>(tb.bases + j.LC + lc) + (uint64_t)sid * j.src_page_stride;
    if (kTrans) { it.s_pg = (uint32_t)sid; it.s_t = bk * j.g + (uint32_t)(sub_off / j.tokrow); }
    if (kTrans && j.src_hnd) { baddr += (uint64_t)bk * j.g * j.q_ts; bmode = 1; }
    else baddr += (uint64_t)bk * j.chunk_bytes + sub_off;
  } else {
    baddr = buf + (uint64_t)bk * j.chunk_bytes + sub_off;
    if (j.layout == 0) baddr += (uint64_t)bp * j.buf_page_bytes + (uint64_t)lc * j.buf_row_bytes;
    else baddr += ((uint64_t)lc * n_buf_pages + bp) * j.buf_row_bytes;
  }
  const uint64_t vbytes = vt * j.tokrow;
  it.valid = vbytes > sub_off ? (uint32_t)min(vbytes - sub_off, (uint64_t)it.bytes) : 0u;
  if (dir == 0) { it.src = paddr; it.dst = baddr; } else { it.src = baddr; it.dst = paddr; }
  if (kTrans) {
    it.mode = dir == 0 ? (pmode | bmode << 1) : (bmode | pmode << 1);
    it.r0 = (uint32_t)(sub_off / j.drow);
    const uint32_t pt = pk * j.g + (uint32_t)(sub_off / j.tokrow);
    if (dir == 0) { it.s_pg = (uint32_t)id; it.s_t = pt; } else { it.d_pg = (uint32_t)id; it.d_t = pt; }
  }
  return it;
}

// Strides of a strided side (kTrans).  Source side: the pool for pack and copy-on-write, the source
// pool for pool -> pool; destination side: always the pool.
struct Strides { uint64_t s_ts, s_hs, d_ts, d_hs; };
__device__ __forceinline__ Strides strides_of(const Job &j) {
  Strides s;
  s.s_ts = j.dir == 2 ? j.q_ts : j.p_ts; s.s_hs = j.dir == 2 ? j.q_hs : j.p_hs;
  s.d_ts = j.p_ts; s.d_hs = j.p_hs;
  return s;
}

// ---------------------------------------------------------------------------------------------
// PTX wrappers (async proxy: mbarrier + cp.async.bulk)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "KV_WAIT:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra KV_DONE;\n\t"
      "bra KV_WAIT;\n\t"
      "KV_DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, uint64_t src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst_smem, uint64_t src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(uint64_t dst, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               ::"l"(dst), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(uint64_t dst, uint32_t src_smem, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(dst), "r"(src_smem), "r"(bytes), "l"(pol) : "memory");
}
// Tensor copies (SASS UTMALDG / UTMASTG) of the rank-4 box at coordinates (0, 0, token, page).
__device__ __forceinline__ void tensor_g2s(uint32_t dst_smem, const void *map, uint32_t t, uint32_t pg, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
               ::"r"(dst_smem), "l"(map), "r"(0), "r"(0), "r"(t), "r"(pg), "r"(bar) : "memory");
}
__device__ __forceinline__ void tensor_s2g(const void *map, uint32_t t, uint32_t pg, uint32_t src_smem) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
               ::"l"(map), "r"(0), "r"(0), "r"(t), "r"(pg), "r"(src_smem) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// 16-byte asynchronous global -> shared copy (SASS LDGSTS), L2 only; completion is reported to an
// mbarrier by cp_async_arrive (the arrival is pre-counted in the barrier's init count: .noinc).
__device__ __forceinline__ void cp_async16(uint32_t dst_smem, uint64_t src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_arrive(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(uint4 *p, const uint4 &v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
               ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// Address of the u-th unit (U bytes) of a kTrans item on one side.
template <uint32_t U>
__device__ __forceinline__ uint64_t trans_addr(uint64_t base, bool strided, uint32_t r0, uint32_t u,
                                               uint32_t upr, uint32_t H, uint64_t ts, uint64_t hs) {
  if (!strided) return base + (uint64_t)u * U;
  const uint32_t rr = u / upr, dd = u - rr * upr;
  const uint32_t row = r0 + rr, t = row / H, h = row - t * H;
  return base + t * ts + h * hs + (uint64_t)dd * U;
}

constexpr int kMaxWarps = 8;
constexpr int kMaxStages = 16;

struct StageMeta {
  uint64_t dst;
  uint32_t bytes, valid;
  uint32_t mode, r0;  // kTrans only
  uint32_t lc, d_pg, d_t;
};

// ---------------------------------------------------------------------------------------------
// kv_move_bulk: persistent CTAs (one per SM); every warp owns `stages` shared-memory stages.
//   load  item i  into stage i % K           at iteration i
//   store item i  from stage i % K           at iteration i + K - lag   (after its mbarrier flips)
//   refill stage  at iteration i + K         after cp.async.bulk.wait_group.read <lag>
// so K - lag loads and lag stores are in flight per warp.  Dynamic shared memory:
//   [zero region: zero_bytes][warp 0 stages][warp 1 stages]...   all 128-byte aligned.
// ---------------------------------------------------------------------------------------------
//
// kTrans (an HND pool on either side): a stage holds the item in NHD-linear order and every lane of
// the warp works.  A contiguous side moves it with one bulk copy as above.  A strided SOURCE is
// gathered row by row with 16-byte cp.async (SASS LDGSTS) by all 32 lanes, each lane's arrival on the
// stage's mbarrier (count 32) firing when its own copies have landed; the stage then leaves with one
// bulk store after a fence.proxy.async.  A strided DESTINATION is written with LDS.128 + STG.128.
// (Per-row bulk copies of head_dim*elem_bytes = 256 B were measured first: 3.1-4.3 TB/s, bound by the
// rate at which one SM retires small bulk copies.)
template <int N, bool kTrans>
__global__ void __launch_bounds__(kMaxWarps * 32, 1) kv_move_bulk(const __grid_constant__ JobT<N> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[kMaxWarps][kMaxStages];
  __shared__ StageMeta meta[kMaxWarps][kMaxStages];

  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t warps = blockDim.x >> 5;
  const uint32_t K = j.stages, lag = j.lag;

  // zero region (generic-proxy writes) + barrier init, then make both visible to the async proxy
  for (uint32_t o = threadIdx.x * 16; o < j.zero_bytes; o += blockDim.x * 16)
    *reinterpret_cast<uint4 *>(smem + o) = make_uint4(0, 0, 0, 0);
  if (lane == 0)
    for (uint32_t s = 0; s < K; ++s) mbar_init(smem_u32(&full_bar[warp][s]), kTrans ? 32 : 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  // Programmatic dependent launch (KV_OPT_PDL): let the next kernel of the stream become resident now, and
  // touch no global memory until the previous one has completed and flushed.  Both are no-ops for a
  // launch without the attribute.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");

  const uint64_t G = (uint64_t)gridDim.x * warps;
  const uint64_t gw = (uint64_t)blockIdx.x * warps + warp;
  // Work distribution.
  //   static  (j.sched == nullptr): this warp's my-th item is gw + my*G.
  //   dynamic (large launches): the first B0 items of every warp are the static block
  //           [gw*B0, gw*B0+B0); the rest is claimed from a global counter in guided chunks
  //           (remaining / 2G, clamped to 1..32), each claim issued one batch ahead so its
  //           latency hides behind the batch in flight.  SMs that run fast take more segments,
  //           so the launch ends when the work does, not when the slowest SM does.
  const bool dyn = j.sched != nullptr;
  const uint32_t B0 = j.first_batch;
  const uint64_t dyn_base = G * B0;
  const uint64_t dyn_total = dyn ? j.total_items - dyn_base : 0;
  const uint64_t n_my = dyn ? 0 : (gw < j.total_items ? (j.total_items - gw + G - 1) / G : 0);
  if (!dyn && n_my == 0) return;

  // L2 hints (KV_OPT_L2_HINT): bit 0 = loads evict_first (the source is read once), bit 1 = stores evict_first,
  // bit 2 = stores evict_last (keep what was just written resident for whoever reads it next)
  uint64_t pol = 0, pol_st = 0;
  if (j.l2_hint & 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  if (j.l2_hint & 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_st));
  if (j.l2_hint & 4) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_st));

  const uint32_t stage0 = smem_u32(smem) + j.zero_bytes + warp * K * j.stage_bytes;
  const uint32_t zero0 = smem_u32(smem);
  const uint32_t depth = K - lag;
  Item mine;
  mine.src = mine.dst = 0; mine.bytes = mine.valid = 0;
  uint32_t hint = 0;  // piece of this lane's previous item (decode)

  unsigned long long pre_start = 0;  // lane 0: result of the claim issued one batch ahead
  uint32_t pre_count = 0;            // warp-uniform: size of that claim (0 = none outstanding)
  auto guided = [&](uint64_t claimed) -> uint32_t {
    const uint64_t rem = dyn_total > claimed ? dyn_total - claimed : 0;
    return (uint32_t)min((uint64_t)32, max((uint64_t)1, rem / (2 * G)));
  };
  if (dyn) {
    pre_count = guided(0);
    if (lane == 0) pre_start = atomicAdd(j.sched, (unsigned long long)pre_count);
  }

  uint64_t n_known = 0;      // items of this warp claimed so far
  uint64_t batch_first = 0;  // my-index of the first item of the batch held in `mine`
  bool exhausted = false;
  for (uint64_t it = 0;; ++it) {
    if (it == n_known && !exhausted) {  // ---- next batch: warp-level lookup, <= 32 segments at once
      uint64_t first_item = 0, stride = 1;
      uint32_t cnt = 0;
      if (!dyn) {
        cnt = (uint32_t)min((uint64_t)32, n_my - n_known);
        first_item = gw + n_known * G;
        stride = G;
      } else if (n_known == 0) {
        cnt = B0;
        first_item = gw * B0;
      } else if (pre_count) {
        const uint64_t st = __shfl_sync(0xffffffffu, pre_start, 0);
        if (st < dyn_total) {
          cnt = (uint32_t)min((uint64_t)pre_count, dyn_total - st);
          first_item = dyn_base + st;
          const uint64_t claimed = st + pre_count;
          pre_count = claimed < dyn_total ? guided(claimed) : 0;
          if (pre_count && lane == 0) pre_start = atomicAdd(j.sched, (unsigned long long)pre_count);
        } else {
          pre_count = 0;
        }
      }
      if (cnt == 0) {
        exhausted = true;
      } else {
        if (lane < cnt) mine = decode<N == 0, kTrans>(j, tb, first_item + lane * stride, hint);
        batch_first = n_known;
        n_known += cnt;
      }
    }
    const bool have = it < n_known;
    if (!have && it >= n_known + depth) break;
    const uint32_t sel = (uint32_t)(it - batch_first) & 31;
    const uint64_t src = __shfl_sync(0xffffffffu, mine.src, sel);
    const uint64_t dst = __shfl_sync(0xffffffffu, mine.dst, sel);
    const uint32_t bytes = __shfl_sync(0xffffffffu, mine.bytes, sel);
    const uint32_t valid = __shfl_sync(0xffffffffu, mine.valid, sel);
    if constexpr (kTrans) {
      const uint32_t mode = __shfl_sync(0xffffffffu, mine.mode, sel);
      const uint32_t r0 = __shfl_sync(0xffffffffu, mine.r0, sel);
      const uint32_t lc = __shfl_sync(0xffffffffu, mine.lc, sel);
      const uint32_t s_pg = __shfl_sync(0xffffffffu, mine.s_pg, sel), s_t = __shfl_sync(0xffffffffu, mine.s_t, sel);
      const uint32_t d_pg = __shfl_sync(0xffffffffu, mine.d_pg, sel), d_t = __shfl_sync(0xffffffffu, mine.d_t, sel);
      const Strides st = strides_of(j);
      const uint32_t upr = j.drow >> 4;  // 16-byte units per head_dim row
      // tensor copies serve whole boxes only; ragged tails (and copy-on-write rows) take the lane paths
      const uint32_t box_bytes = j.tb * j.tokrow;
      // (a mixed launch has one pool: whichever side of an item is strided is that pool; bit 2 of the mode keeps
      // copy-on-write rows on the lane paths)
      const uint8_t *mp = j.maps_pool, *ms = j.maps_src;
      if constexpr (N > 0) {  // maps carried in the parameters (a first-ever captured call)
        if (j.off_maps_pool) mp = p.blob + j.off_maps_pool;
        if (j.off_maps_src) ms = p.blob + j.off_maps_src;
      }
      const uint8_t *maps_s = j.dir == 2 ? ms : ((j.dir == 0 || j.dir == 4) ? mp : nullptr);
      const uint8_t *maps_d = (j.dir == 1 || j.dir == 2 || j.dir == 4) ? mp : nullptr;
      if (it >= depth && it - depth < n_known) {  // ---- store side: item si
        const uint64_t si = it - depth;
        const uint32_t s = (uint32_t)(si % K);
        mbar_wait(smem_u32(&full_bar[warp][s]), (uint32_t)(si / K) & 1);
        const StageMeta m = meta[warp][s];
        const uint32_t sbase = stage0 + s * j.stage_bytes;
        if ((m.mode & 6) == 2 && maps_d && m.bytes == box_bytes && m.valid == box_bytes) {
          // strided destination, whole box: one tensor store scatters the NHD stage into the HND page.
          // The stage may have been written through the generic proxy (cp.async row gathers by all lanes): every
          // writing lane fences its own writes into the async proxy before lane 0 issues the store.
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) tensor_s2g(maps_d + (size_t)m.lc * 128, m.d_t, m.d_pg, sbase);
        } else if (m.mode & 2) {  // strided destination: LDS.128 from the stage, STG.128 to the row's place
          const uint32_t nb = m.bytes >> 4, nv = m.valid >> 4;
          for (uint32_t u0 = lane; u0 < nb; u0 += 128) {
            uint4 v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint32_t u = u0 + 32 * q;
              v[q] = make_uint4(0, 0, 0, 0);
              if (u < nv) v[q] = lds128(sbase + (u << 4));
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint32_t u = u0 + 32 * q;
              if (u < nb)
                st_stream(reinterpret_cast<uint4 *>(trans_addr<16>(m.dst, true, m.r0, u, upr, j.H, st.d_ts, st.d_hs)), v[q]);
            }
          }
        } else {
          // rows gathered by cp.async (generic proxy, all 32 lanes) -> bulk store (async proxy): the PTX memory model
          // wants the WRITING threads' accesses fenced into the async proxy, so every lane fences, then the warp meets
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) {
            if (m.valid) bulk_s2g(m.dst, sbase, m.valid);
            for (uint32_t z = m.valid; z < m.bytes; z += j.zero_bytes)
              bulk_s2g(m.dst + z, zero0, min(j.zero_bytes, m.bytes - z));
          }
        }
        bulk_commit();  // every lane, every item: the per-thread group counts stay in step
      }
      if (have) {  // ---- load side: item it
        const uint32_t s = (uint32_t)(it % K);
        if (it >= K) {
          if (lag == 1) bulk_wait_read<1>();
          else if (lag == 2) bulk_wait_read<2>();
          else bulk_wait_read<3>();
        }
        __syncwarp();  // every lane has finished reading this stage (bulk store or LDS)
        const uint32_t bar = smem_u32(&full_bar[warp][s]);
        const uint32_t sbase = stage0 + s * j.stage_bytes;
        if (lane == 0) {
          StageMeta &m = meta[warp][s];
          m.dst = dst; m.bytes = bytes; m.valid = valid; m.mode = mode; m.r0 = r0;
          m.lc = lc; m.d_pg = d_pg; m.d_t = d_t;
        }
        if ((mode & 5) == 1 && maps_s && bytes == box_bytes && valid == box_bytes) {
          // strided source, whole box: one tensor load gathers the HND page's rows in NHD order
          if (lane == 0) {
            mbar_expect_tx(bar, box_bytes);
            tensor_g2s(sbase, maps_s + (size_t)lc * 128, s_t, s_pg, bar);
          } else {
            mbar_arrive(bar);
          }
        } else if (mode & 1) {  // strided source: 16-byte cp.async (LDGSTS) gathers the rows in NHD order;
                         // each lane's arrival fires when its own copies have landed
          const uint32_t nv = valid >> 4;
          for (uint32_t u = lane; u < nv; u += 32)
            cp_async16(sbase + (u << 4), trans_addr<16>(src, true, r0, u, upr, j.H, st.s_ts, st.s_hs));
          cp_async_arrive(bar);
        } else if (lane == 0 && valid) {
          mbar_expect_tx(bar, valid);
          bulk_g2s(sbase, src, valid, bar);
        } else {
          mbar_arrive(bar);
        }
      }
      __syncwarp();  // meta[] written by lane 0 is read by every lane `depth` iterations later
    } else
    if (lane == 0) {
      auto store_side = [&]() {
        if (it >= depth && it - depth < n_known) {  // ---- store side: item si
          const uint64_t si = it - depth;
          const uint32_t s = (uint32_t)(si % K);
          mbar_wait(smem_u32(&full_bar[warp][s]), (uint32_t)(si / K) & 1);
          const StageMeta m = meta[warp][s];
          if (m.valid) {
            if (j.l2_hint & 6) bulk_s2g_hint(m.dst, stage0 + s * j.stage_bytes, m.valid, pol_st);
            else bulk_s2g(m.dst, stage0 + s * j.stage_bytes, m.valid);
          }
          for (uint32_t z = m.valid; z < m.bytes; z += j.zero_bytes)  // zero-padded tail (a5)
            bulk_s2g(m.dst + z, zero0, min(j.zero_bytes, m.bytes - z));
          bulk_commit();
        }
      };
      // Ramp: the first K loads of a warp go into stages nobody has used, so they are issued BEFORE this warp blocks on
      // its first store (all K x stage bytes of the warp in flight from the start: a transfer of a few segments per
      // warp never waits for a load it could already have issued).  From iteration K on a stage is refilled once the
      // store that last read it has finished reading: the store of this iteration is committed first, so that store
      // was committed `lag` groups ago.
      if (it >= K) store_side();
      if (have) {  // ---- load side: item it
        const uint32_t s = (uint32_t)(it % K);
        if (it >= K) {  // the store that last read this stage was committed `lag` groups ago
          if (lag == 1) bulk_wait_read<1>();
          else if (lag == 2) bulk_wait_read<2>();
          else bulk_wait_read<3>();
        }
        meta[warp][s].dst = dst; meta[warp][s].bytes = bytes; meta[warp][s].valid = valid;
        const uint32_t bar = smem_u32(&full_bar[warp][s]);
        if (valid) {
          mbar_expect_tx(bar, valid);
          if (j.l2_hint & 1) bulk_g2s_hint(stage0 + s * j.stage_bytes, src, valid, bar, pol);
          else bulk_g2s(stage0 + s * j.stage_bytes, src, valid, bar);
        } else {
          mbar_arrive(bar);
        }
      }
      if (it < K) store_side();
    }
  }
  if (dyn && lane == 0) {  // last warp out re-arms the counters for the next launch
    __threadfence();
    if (atomicAdd(j.sched_done, 1u) == (uint32_t)G - 1) {
      *j.sched = 0ull;
      *j.sched_done = 0u;
      __threadfence();
    }
  }
  // The stages must outlive the bulk stores' READS; their global writes complete with the grid (what a later kernel
  // or copy on the stream, or the host after a sync, observes), so a warp need not sit out the write acknowledgements.
  if (lane == 0 || kTrans) bulk_wait_read<0>();
}

// ---------------------------------------------------------------------------------------------
// kv_move_shot: ONE segment per single-warp CTA; the hardware's CTA scheduler is the work distributor.
//   load the segment into the CTA's one stage (cp.async.bulk / cp.async.bulk.tensor / row gathers), wait on the
//   mbarrier, store it (bulk / tensor / 16-byte stores), wait until the store has READ the stage, exit.
// A CTA owns `stage_bytes` of shared memory (16 KiB at the paper's shapes) and 32 threads, so an SM holds as many
// segments in flight as its shared memory takes (13-14 x 16 KiB: ~220 KiB per SM, 32 MB per chip, against the ~128 KiB
// per SM of the persistent ring), loads and stores of different CTAs overlap freely, a finished CTA is replaced at
// once, and there is no ring, no claim counter and no tail to balance.  Measured on B200 against a plain contiguous
// cudaMemcpyAsync of the same size under the same conditions (isolated call, cold clean L2; a one-off probe of round 2):
// a minimal kernel of this shape equals the plain copy from 1 MiB to 768 MiB (64 MiB 21.8 vs 21.5 us, 768 MiB 239 vs
// 242 us) where the ring needed 27.7 / 249 us.  DESIGN.md "Kernels".
// gridDim.x may be capped (KV_OPT_MAX_CTAS): a CTA then walks items blockIdx.x, + gridDim.x, ... reusing its stage.
// ---------------------------------------------------------------------------------------------
template <int N, bool kTrans>
__global__ void __launch_bounds__(32) kv_move_shot(const __grid_constant__ JobT<N> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar;
  const uint32_t lane = threadIdx.x;
  const uint32_t bar = smem_u32(&full_bar), sbase = smem_u32(smem);
  if (lane == 0) {
    mbar_init(bar, kTrans ? 32 : 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncwarp();
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // no-ops without the launch attribute (KV_OPT_PDL)
  asm volatile("griddepcontrol.wait;" ::: "memory");               // nothing global is touched before this
  uint64_t pol = 0, pol_st = 0;
  if (j.l2_hint & 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  if (j.l2_hint & 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_st));
  if (j.l2_hint & 4) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_st));
  uint32_t hint = 0, phase = 0;
  for (uint64_t item = blockIdx.x; item < j.total_items; item += gridDim.x) {
    // every lane decodes the CTA's segment (uniform: no shuffles, no divergence)
    const Item it = decode<N == 0, kTrans>(j, tb, item, hint);
    if (it.bytes == 0) continue;  // skipped: a device-resident page id was out of range
    if constexpr (kTrans) {
      const Strides st = strides_of(j);
      const uint32_t upr = j.drow >> 4;  // 16-byte units per head_dim row
      const uint32_t box_bytes = j.tb * j.tokrow;
      const uint8_t *mp = j.maps_pool, *ms = j.maps_src;
      if constexpr (N > 0) {  // maps carried in the parameters (a first-ever captured call)
        if (j.off_maps_pool) mp = p.blob + j.off_maps_pool;
        if (j.off_maps_src) ms = p.blob + j.off_maps_src;
      }
      const uint8_t *maps_s = j.dir == 2 ? ms : ((j.dir == 0 || j.dir == 4) ? mp : nullptr);
      const uint8_t *maps_d = (j.dir == 1 || j.dir == 2 || j.dir == 4) ? mp : nullptr;
      const bool whole = it.bytes == box_bytes && it.valid == box_bytes;
      if (it.valid) {  // ---- load
        if ((it.mode & 5) == 1 && maps_s && whole) {  // strided source, whole box: the copy engine gathers it in NHD order
          if (lane == 0) {
            mbar_expect_tx(bar, box_bytes);
            tensor_g2s(sbase, maps_s + (size_t)it.lc * 128, it.s_t, it.s_pg, bar);
          } else {
            mbar_arrive(bar);
          }
        } else if (it.mode & 1) {  // strided source: 16-byte cp.async row gathers by all lanes
          const uint32_t nv = it.valid >> 4;
          for (uint32_t u = lane; u < nv; u += 32)
            cp_async16(sbase + (u << 4), trans_addr<16>(it.src, true, it.r0, u, upr, j.H, st.s_ts, st.s_hs));
          cp_async_arrive(bar);
        } else if (lane == 0) {
          mbar_expect_tx(bar, it.valid);
          bulk_g2s(sbase, it.src, it.valid, bar);
        } else {
          mbar_arrive(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
      }
      // ---- store
      if ((it.mode & 6) == 2 && maps_d && whole) {  // strided destination, whole box: one tensor store
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the stage may hold generic-proxy writes of every lane
        __syncwarp();
        if (lane == 0) tensor_s2g(maps_d + (size_t)it.lc * 128, it.d_t, it.d_pg, sbase);
      } else if (it.mode & 2) {  // strided destination: LDS.128 from the stage, STG.128 to each row's place
        const uint32_t nb = it.bytes >> 4, nv = it.valid >> 4;
        for (uint32_t u0 = lane; u0 < nb; u0 += 128) {
          uint4 v[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const uint32_t u = u0 + 32 * q;
            v[q] = make_uint4(0, 0, 0, 0);
            if (u < nv) v[q] = lds128(sbase + (u << 4));
          }
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const uint32_t u = u0 + 32 * q;
            if (u < nb)
              st_stream(reinterpret_cast<uint4 *>(trans_addr<16>(it.dst, true, it.r0, u, upr, j.H, st.d_ts, st.d_hs)), v[q]);
          }
        }
      } else {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0 && it.valid) bulk_s2g(it.dst, sbase, it.valid);
        for (uint32_t z = it.valid + (lane << 4); z < it.bytes; z += 512)  // zero-padded tail (a5)
          st_stream(reinterpret_cast<uint4 *>(it.dst + z), make_uint4(0, 0, 0, 0));
      }
      bulk_commit();
      bulk_wait_read<0>();  // the stage may be refilled (next item of a capped grid) or released (exit)
      __syncwarp();
    } else {
      if (lane == 0 && it.valid) {
        mbar_expect_tx(bar, it.valid);
        if (j.l2_hint & 1) bulk_g2s_hint(sbase, it.src, it.valid, bar, pol);
        else bulk_g2s(sbase, it.src, it.valid, bar);
        mbar_wait(bar, phase);
        if (j.l2_hint & 6) bulk_s2g_hint(it.dst, sbase, it.valid, pol_st);
        else bulk_s2g(it.dst, sbase, it.valid);
        bulk_commit();
      }
      if (it.valid) phase ^= 1;
      for (uint32_t z = it.valid + (lane << 4); z < it.bytes; z += 512)  // zero-padded tail (a5): plain 16-byte stores
        st_stream(reinterpret_cast<uint4 *>(it.dst + z), make_uint4(0, 0, 0, 0));
      if (lane == 0) bulk_wait_read<0>();
    }
  }
}

// ---------------------------------------------------------------------------------------------
// kv_move_shot_plain: kv_move_shot for the plain case only (Job::lean, no L2 hints) -- one request, pack or unpack
// between equal page sizes, page-first buffer, nothing to zero-fill.  Same copy, a fraction of the code: a single-warp
// CTA hides no latency, so what sits between its start and its bulk load is paid in full by every small call (measured
// in CUDA-graph replays of 1-16 MiB packs).  Lane 0 alone works; the other lanes leave at once.
// ---------------------------------------------------------------------------------------------
// kTrans: the pool is HND and its whole-token boxes move by tensor copies (Job::tb, the per-slab maps): the pool side of an
// item is (slab lc, first token, page) instead of an address; the buffer side is the same contiguous run.
template <int N, bool kTrans>
__global__ void __launch_bounds__(32) kv_move_shot_plain(const __grid_constant__ JobT<N> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // no-ops without the launch attribute (KV_OPT_PDL)
  if (threadIdx.x != 0) return;
  const uint32_t bar = smem_u32(&full_bar), sbase = smem_u32(smem);
  mbar_init(bar, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");  // nothing global is touched before this
  uint32_t phase = 0;
  for (uint64_t item = blockIdx.x; item < j.total_items; item += gridDim.x) {
    uint64_t item_begin = 0, buf = j.one.buf, id_begin = j.one.id_begin;
    if (j.n_pieces > 1) {  // a batch (Job::lean == 2): largest r with pieces[r].item_begin <= item
      uint32_t lo = 0, hi = j.n_pieces;
      while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (ldt<N == 0>(&tb.pieces[mid].item_begin) <= item) lo = mid; else hi = mid;
      }
      const Piece *pc = tb.pieces + lo;
      item_begin = ldt<N == 0>(&pc->item_begin); buf = ldt<N == 0>(&pc->buf); id_begin = ldt<N == 0>(&pc->id_begin);
    }
    if constexpr (kTrans) {
      const uint8_t *maps = j.maps_pool;
      if constexpr (N > 0) { if (j.off_maps_pool) maps = p.blob + j.off_maps_pool; }  // a first-ever captured call
      const uint32_t local = (uint32_t)(item - item_begin);
      const uint32_t r1 = fdiv(local, j.m_subs), sub = local - r1 * j.subs;
      const uint32_t pp = fdiv(r1, j.m_LC), lc = r1 - pp * j.LC;
      const int32_t id = (N == 0) ? __ldg(tb.ids + id_begin + pp) : tb.ids[id_begin + pp];
      const uint64_t baddr = buf + (uint64_t)pp * j.buf_page_bytes + (uint64_t)lc * j.buf_row_bytes + (uint64_t)sub * j.sub_bytes;
      const uint32_t bytes = j.sub_bytes, t = sub * j.tb;  // whole boxes only (Job::lean)
      mbar_expect_tx(bar, bytes);
      if (j.dir == 0) tensor_g2s(sbase, maps + (size_t)lc * 128, t, (uint32_t)id, bar);  // the copy engine gathers the box in NHD order
      else bulk_g2s(sbase, baddr, bytes, bar);
      mbar_wait(bar, phase);
      phase ^= 1;
      if (j.dir == 0) bulk_s2g(baddr, sbase, bytes);
      else tensor_s2g(maps + (size_t)lc * 128, t, (uint32_t)id, sbase);  // ... and scatters it back into the HND page
    } else {
      const Lean l = decode_lean<N == 0>(j, tb, (uint32_t)(item - item_begin), buf, id_begin);
      mbar_expect_tx(bar, l.bytes);
      bulk_g2s(sbase, l.src, l.bytes, bar);
      mbar_wait(bar, phase);
      phase ^= 1;
      bulk_s2g(l.dst, sbase, l.bytes);
    }
    bulk_commit();
    bulk_wait_read<0>();  // the stage may be refilled (next item of a capped grid) or released (exit)
  }
}

// ---------------------------------------------------------------------------------------------
// kv_move_vec: one warp per segment, 16-byte streaming loads/stores, UNROLL loads in flight.
// ---------------------------------------------------------------------------------------------
template <int UNROLL, int N, bool kTrans>
__global__ void __launch_bounds__(256) kv_move_vec(const __grid_constant__ JobT<N> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t G = (uint64_t)gridDim.x * (blockDim.x >> 5);
  uint32_t hint = 0;
  for (uint64_t item = (uint64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
       item < j.total_items; item += G) {
    const Item it = decode<N == 0, kTrans>(j, tb, item, hint);
    const uint4 *s = reinterpret_cast<const uint4 *>(it.src);
    uint4 *d = reinterpret_cast<uint4 *>(it.dst);
    const uint32_t nv = it.valid >> 4, nb = it.bytes >> 4;
    if constexpr (kTrans) {
      if (it.mode) {  // [token] x [head] transposition in 16-byte units of head_dim rows
        const Strides st = strides_of(j);
        const uint32_t upr = j.drow >> 4;
        for (uint32_t i0 = lane; i0 < nb; i0 += 32 * UNROLL) {
          uint4 v[UNROLL];
#pragma unroll
          for (int u = 0; u < UNROLL; ++u) {
            const uint32_t i = i0 + 32 * u;
            v[u] = make_uint4(0, 0, 0, 0);
            if (i < nv)
              v[u] = ld_stream(reinterpret_cast<const uint4 *>(
                  trans_addr<16>(it.src, it.mode & 1, it.r0, i, upr, j.H, st.s_ts, st.s_hs)));
          }
#pragma unroll
          for (int u = 0; u < UNROLL; ++u) {
            const uint32_t i = i0 + 32 * u;
            if (i < nb)
              st_stream(reinterpret_cast<uint4 *>(
                            trans_addr<16>(it.dst, it.mode & 2, it.r0, i, upr, j.H, st.d_ts, st.d_hs)),
                        v[u]);
          }
        }
        continue;
      }
    }
    uint32_t i = lane;
    for (; i + 32 * (UNROLL - 1) < nv; i += 32 * UNROLL) {
      uint4 v[UNROLL];
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) v[u] = ld_stream(s + i + 32 * u);
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) st_stream(d + i + 32 * u, v[u]);
    }
    if (i < nv) {  // ragged remainder (copy-on-write pieces): its loads are issued together too, not one by one
      uint4 v[UNROLL];
#pragma unroll
      for (int u = 0; u < UNROLL; ++u)
        if (i + 32 * u < nv) v[u] = ld_stream(s + i + 32 * u);
#pragma unroll
      for (int u = 0; u < UNROLL; ++u)
        if (i + 32 * u < nv) st_stream(d + i + 32 * u, v[u]);
    }
    for (i = nv + lane; i < nb; i += 32) st_stream(d + i, make_uint4(0, 0, 0, 0));
  }
}

// ---------------------------------------------------------------------------------------------
// kv_move_small: segments of at most 1 KiB (one-token pages; re-paging between page sizes with no common
// divisor).  A segment is too short to pay for a warp-wide address computation of its own, so the 32 lanes
// decode 32 segments at once (as kv_move_bulk does) and the warp then copies them eight at a time: two
// 16-byte vectors per lane and segment, sixteen loads in flight per lane before the first store.
// ---------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(256) kv_move_small(const __grid_constant__ JobT<N> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t G = (uint64_t)gridDim.x * (blockDim.x >> 5);
  uint32_t hint = 0;
  for (uint64_t base = ((uint64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32; base < j.total_items;
       base += G * 32) {
    const uint32_t cnt = (uint32_t)min((uint64_t)32, j.total_items - base);
    Item mine;
    mine.src = mine.dst = 0; mine.bytes = mine.valid = 0;
    if (lane < cnt) mine = decode<N == 0, false>(j, tb, base + lane, hint);
    for (uint32_t k0 = 0; k0 < cnt; k0 += 8) {
      uint4 v[8][2];
      uint64_t dst[8];
      uint32_t nb[8], nv[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const uint32_t k = min(k0 + q, 31u);
        const uint64_t src = __shfl_sync(0xffffffffu, mine.src, k);
        dst[q] = __shfl_sync(0xffffffffu, mine.dst, k);
        nb[q] = k0 + q < cnt ? __shfl_sync(0xffffffffu, mine.bytes, k) >> 4 : 0;
        nv[q] = k0 + q < cnt ? __shfl_sync(0xffffffffu, mine.valid, k) >> 4 : 0;
        const uint4 *sp = reinterpret_cast<const uint4 *>(src);
        v[q][0] = lane < nv[q] ? ld_stream(sp + lane) : make_uint4(0, 0, 0, 0);
        v[q][1] = lane + 32 < nv[q] ? ld_stream(sp + lane + 32) : make_uint4(0, 0, 0, 0);
      }
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        uint4 *dp = reinterpret_cast<uint4 *>(dst[q]);
        if (lane < nb[q]) st_stream(dp + lane, v[q][0]);
        if (lane + 32 < nb[q]) st_stream(dp + lane + 32, v[q][1]);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// kv_move_elem: any elem_bytes-aligned pointers; U is the widest unit dividing every address
// and length of the call (1, 2, 4 or 8 bytes).
// ---------------------------------------------------------------------------------------------
template <typename U, bool kTrans>
__global__ void __launch_bounds__(256) kv_move_elem(const __grid_constant__ JobT<0> p) {
  const Job &j = p.j;
  const Tables tb = tables_of(p);
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t G = (uint64_t)gridDim.x * (blockDim.x >> 5);
  uint32_t hint = 0;
  for (uint64_t item = (uint64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
       item < j.total_items; item += G) {
    const Item it = decode<true, kTrans>(j, tb, item, hint);
    const U *s = reinterpret_cast<const U *>(it.src);
    U *d = reinterpret_cast<U *>(it.dst);
    const uint32_t nv = it.valid / sizeof(U), nb = it.bytes / sizeof(U);
    if constexpr (kTrans) {
      if (it.mode) {
        const Strides st = strides_of(j);
        const uint32_t upr = j.drow / sizeof(U);
        for (uint32_t i = lane; i < nb; i += 32) {
          U v = U(0);
          if (i < nv)
            v = *reinterpret_cast<const U *>(
                trans_addr<sizeof(U)>(it.src, it.mode & 1, it.r0, i, upr, j.H, st.s_ts, st.s_hs));
          *reinterpret_cast<U *>(
              trans_addr<sizeof(U)>(it.dst, it.mode & 2, it.r0, i, upr, j.H, st.d_ts, st.d_hs)) = v;
        }
        continue;
      }
    }
    uint32_t i = lane;
    for (; i + 32 * 7 < nv; i += 32 * 8) {  // eight loads in flight per lane before the first store
      U v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = s[i + 32 * u];
#pragma unroll
      for (int u = 0; u < 8; ++u) d[i + 32 * u] = v[u];
    }
    for (; i < nv; i += 32) d[i] = s[i];
    for (i = nv + lane; i < nb; i += 32) d[i] = U(0);
  }
}

// ---------------------------------------------------------------------------------------------
// kv_signal: the availability flag that follows a transfer in stream order (kvtier.h kv_signal).
// fence.sc.sys orders every write this GPU performed before the launch (the previous kernels of the
// stream have completed) ahead of the flag for observers anywhere in the system: a peer GPU or the host.
// ---------------------------------------------------------------------------------------------
__global__ void kv_signal_kernel(uint64_t *flag, uint64_t value) {
  __threadfence_system();
  asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(flag), "l"(value) : "memory");
}

// n <= 32 consecutive flags at once (kv_reload_layerwise: the layers whose pages have just landed)
__global__ void kv_signal_range(uint64_t *flags, uint32_t n, uint64_t value) {
  __threadfence_system();
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x)
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(flags + i), "l"(value) : "memory");
}

}  // namespace kvt
