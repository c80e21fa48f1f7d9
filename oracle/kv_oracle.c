/*
 * oracle/kv_oracle.c -- CPU ORACLE for the paged-KV tier transfer.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * build, link or call this file.  It shares no code, header, table or helper with the CUDA
 * path under paper_2606_31093_b200/csrc/, and neither side includes the other.
 *
 * What it computes (the method is an exact permutation copy, so the oracle is the definition
 * written out; citations are PAPER.md line + section, BASELINE.json key):
 *
 *   pool addressing   PAPER.md:L207 (sec. 4.1.1 Physical Paging Layer): a parameter has outer
 *                     dims (layers), slice dims (K/V), a page size, shape and dtype; a region is
 *                     fetched by (sub_names=layer, page_idx, slice_idx=K|V).  Here:
 *                       POOL[l][c][g][t][h][d] = *(elem*)(base[l*C+c] + g*page_stride_bytes
 *                                                         + ((t*H + h)*D + d)*e)
 *                     in-page order NHD = [token][head][dim] ("NHD block stacks").
 *   HND pools         PAPER.md:L214 "compute-oriented layouts, INCLUDING NHD block stacks" (so
 *                     others exist); SURVEY.md 8(f) NEXT-2 "HND pools".  `order` 1 stores a page
 *                     as [head][token][dim]:
 *                       POOL[l][c][g][t][h][d] at in-page element ((h*T + t)*D + d)
 *                     The transfer buffer and the CoW append block stay NHD.
 *   lower-tier layout BASELINE.json:configs[0]: page-first [page][layer][K,V][token][head][dim],
 *                     dense.  (reading R1.)
 *   O-pack            PAPER.md:L214 (sec. 4.1.2) "copy and convert pages directly into
 *                     destination buffers"; SURVEY.md 8(c) Definition O-pack.
 *   O-unpack          SURVEY.md 8(c) Definition O-unpack; BASELINE.json:configs[4] (re-paging,
 *                     "sequence order preserved, tail page partially filled and zero-padded");
 *                     PAPER.md:L238 (session metadata "records the total valid token length").
 *   layer-first       SURVEY.md 8(f) NEXT-2: buffer [layer][K,V][page][token][head][dim].
 *
 * Elements are opaque e-byte bit patterns; nothing is ever interpreted as a float.
 * All byte offsets are 64-bit.  Loops are in the paper's/SURVEY's index order
 * (page, layer, K/V, token, head, dim); there is no blocking, fusion or memcpy of rows.
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): hand-computed worked examples W1/W2,
 * numpy take/transpose/reshape special cases, an independently written "pull" formulation,
 * round trip, write-once bijectivity, untouched bytes, zero-pad count, 64-bit offsets.
 * Parity status: PINNED for every function in this file.
 *
 * `threads` > 1 splits the OUTER page loop across OpenMP threads (pages are independent);
 * it exists for the reported CPU baseline and changes no result.
 */
#include <stddef.h>
#include <stdint.h>

#define KVO_OK 0
#define KVO_ERR_ARG (-1)
#define KVO_ERR_PAGE_RANGE (-2)

/* copy one element of e bytes, as raw bytes */
static inline void kvo_copy_elem(uint8_t *dst, const uint8_t *src, uint32_t e) {
  for (uint32_t b = 0; b < e; ++b) dst[b] = src[b];
}
static inline void kvo_zero_elem(uint8_t *dst, uint32_t e) {
  for (uint32_t b = 0; b < e; ++b) dst[b] = 0;
}

/* In-page element index of POOL[..][t][h][d] (T = page size of THAT pool).
 *   order 0, NHD: (t*H + h)*D + d        order 1, HND: (h*T + t)*D + d */
static inline uint64_t kvo_in_page(int order, uint64_t t, uint64_t T, uint64_t h, uint64_t H,
                                   uint64_t d, uint64_t D) {
  if (order == 0) return (t * H + h) * D + d;
  return (h * T + t) * D + d;
}

static int kvo_ids_in_range(const int32_t *ids, uint64_t n, uint32_t num_pages) {
  for (uint64_t i = 0; i < n; ++i)
    if (ids[i] < 0 || (uint32_t)ids[i] >= num_pages) return 0;
  return 1;
}

/* Buffer element index for the two buffer layouts.
 *   layout 0, page-first : ((((p*L + l)*C + c)*T + t)*H + h)*D + d
 *   layout 1, layer-first: ((((l*C + c)*n + p)*T + t)*H + h)*D + d      (n = pages in buffer)
 */
static inline uint64_t kvo_buf_index(int layout, uint64_t p, uint64_t n, uint64_t l, uint64_t L,
                                     uint64_t c, uint64_t C, uint64_t t, uint64_t T, uint64_t h,
                                     uint64_t H, uint64_t d, uint64_t D) {
  if (layout == 0) return ((((p * L + l) * C + c) * T + t) * H + h) * D + d;
  return ((((l * C + c) * n + p) * T + t) * H + h) * D + d;
}

/* O-pack: buf[p][l][c][t][h][d] = POOL[l][c][ids[p]][t][h][d] */
int kvo_pack(const void *const *base, uint32_t L, uint32_t C, uint32_t num_pages, uint32_t T,
             uint32_t H, uint32_t D, uint32_t e, uint64_t page_stride_bytes, int order,
             const int32_t *ids, uint64_t n, int layout, void *buf, int threads) {
  if (!base || (!ids && n) || (!buf && n) || !L || !C || !T || !H || !D || !e) return KVO_ERR_ARG;
  if ((layout != 0 && layout != 1) || (order != 0 && order != 1)) return KVO_ERR_ARG;
  if (!kvo_ids_in_range(ids, n, num_pages)) return KVO_ERR_PAGE_RANGE;
  uint8_t *out = (uint8_t *)buf;
#pragma omp parallel for num_threads(threads) if (threads > 1) schedule(static)
  for (int64_t p = 0; p < (int64_t)n; ++p)
    for (uint64_t l = 0; l < L; ++l)
      for (uint64_t c = 0; c < C; ++c)
        for (uint64_t t = 0; t < T; ++t)
          for (uint64_t h = 0; h < H; ++h)
            for (uint64_t d = 0; d < D; ++d) {
              const uint8_t *src = (const uint8_t *)base[l * C + c] +
                                   (uint64_t)ids[p] * page_stride_bytes +
                                   kvo_in_page(order, t, T, h, H, d, D) * e;
              uint64_t o = kvo_buf_index(layout, (uint64_t)p, n, l, L, c, C, t, T, h, H, d, D);
              kvo_copy_elem(out + o * e, src, e);
            }
  return KVO_OK;
}

/* O-unpack (general re-paging; same-size is Ts == Td, n_tokens = n*Ts):
 *   n_dst = ceil(n_tokens / Td)
 *   for q,l,c,u,h,d:  j = q*Td + u
 *     DST[l][c][dst_ids[q]][u][h][d] = (j < n_tokens) ? src[(j/Ts) ...][j%Ts] : 0
 * n_src = ceil(n_tokens / Ts) is the number of pages in the source buffer (layer-first needs it).
 * Nothing else in any destination pool is written.  dst_ids must be distinct (caller checks).
 */
int kvo_unpack(const void *src, const int32_t *dst_ids, uint64_t n_dst, void *const *base,
               uint32_t L, uint32_t C, uint32_t num_pages, uint32_t H, uint32_t D, uint32_t e,
               uint64_t page_stride_bytes, int order, uint32_t Ts, uint32_t Td, uint64_t n_tokens,
               int layout, int threads) {
  if (!base || !L || !C || !Ts || !Td || !H || !D || !e) return KVO_ERR_ARG;
  if ((layout != 0 && layout != 1) || (order != 0 && order != 1)) return KVO_ERR_ARG;
  if (n_dst != (n_tokens + Td - 1) / Td) return KVO_ERR_ARG;
  if ((!src || !dst_ids) && n_dst) return KVO_ERR_ARG;
  if (!kvo_ids_in_range(dst_ids, n_dst, num_pages)) return KVO_ERR_PAGE_RANGE;
  const uint8_t *in = (const uint8_t *)src;
  const uint64_t n_src = (n_tokens + Ts - 1) / Ts;
#pragma omp parallel for num_threads(threads) if (threads > 1) schedule(static)
  for (int64_t q = 0; q < (int64_t)n_dst; ++q)
    for (uint64_t l = 0; l < L; ++l)
      for (uint64_t c = 0; c < C; ++c)
        for (uint64_t u = 0; u < Td; ++u)
          for (uint64_t h = 0; h < H; ++h)
            for (uint64_t d = 0; d < D; ++d) {
              uint64_t j = (uint64_t)q * Td + u; /* sequence position, order preserved */
              uint8_t *dst = (uint8_t *)base[l * C + c] +
                             (uint64_t)dst_ids[q] * page_stride_bytes +
                             kvo_in_page(order, u, Td, h, H, d, D) * e;
              if (j < n_tokens) {
                uint64_t o = kvo_buf_index(layout, j / Ts, n_src, l, L, c, C, j % Ts, Ts, h, H, d, D);
                kvo_copy_elem(dst, in + o * e, e);
              } else {
                kvo_zero_elem(dst, e);
              }
            }
  return KVO_OK;
}

/* O-batched (BASELINE.json:configs[3]): O-pack per request r over
 * ids[off[r] .. off[r+1]) into its own buffer dsts[r]. */
int kvo_pack_batched(const void *const *base, uint32_t L, uint32_t C, uint32_t num_pages,
                     uint32_t T, uint32_t H, uint32_t D, uint32_t e, uint64_t page_stride_bytes,
                     int order, const int32_t *ids, const int64_t *off, uint32_t R, int layout,
                     void *const *dsts, int threads) {
  if (R && (!off || !dsts)) return KVO_ERR_ARG;
  for (uint32_t r = 0; r < R; ++r) {
    if (off[r + 1] < off[r]) return KVO_ERR_ARG;
    if (!kvo_ids_in_range(ids + off[r], (uint64_t)(off[r + 1] - off[r]), num_pages))
      return KVO_ERR_PAGE_RANGE;
  }
  for (uint32_t r = 0; r < R; ++r) {
    int rc = kvo_pack(base, L, C, num_pages, T, H, D, e, page_stride_bytes, order, ids + off[r],
                      (uint64_t)(off[r + 1] - off[r]), layout, dsts[r], threads);
    if (rc) return rc;
  }
  return KVO_OK;
}

/* O-batched unpack: O-unpack per request r with its own source buffer srcs[r], its own
 * n_tokens[r] and destination ids dst_ids[off[r] .. off[r+1]) (count must be ceil(n_tokens/Td)). */
int kvo_unpack_batched(const void *const *srcs, const int32_t *dst_ids, const int64_t *off,
                       const uint64_t *n_tokens, uint32_t R, void *const *base, uint32_t L,
                       uint32_t C, uint32_t num_pages, uint32_t H, uint32_t D, uint32_t e,
                       uint64_t page_stride_bytes, int order, uint32_t Ts, uint32_t Td, int layout,
                       int threads) {
  if (R && (!off || !srcs || !n_tokens)) return KVO_ERR_ARG;
  if (!Td) return KVO_ERR_ARG;
  for (uint32_t r = 0; r < R; ++r) {
    if (off[r + 1] < off[r]) return KVO_ERR_ARG;
    if ((uint64_t)(off[r + 1] - off[r]) != (n_tokens[r] + Td - 1) / Td) return KVO_ERR_ARG;
    if (!kvo_ids_in_range(dst_ids + off[r], (uint64_t)(off[r + 1] - off[r]), num_pages))
      return KVO_ERR_PAGE_RANGE;
  }
  for (uint32_t r = 0; r < R; ++r) {
    int rc = kvo_unpack(srcs[r], dst_ids + off[r], (uint64_t)(off[r + 1] - off[r]), base, L, C,
                        num_pages, H, D, e, page_stride_bytes, order, Ts, Td, n_tokens[r], layout,
                        threads);
    if (rc) return rc;
  }
  return KVO_OK;
}

/* Copy-on-write partial-page append ("copies its existing contents into a
 * writable slot and appends the new data there"):
 *   for l,c,t,h,d:
 *     NEW[l][c][new_id][t] = OLD[l][c][old_id][t]            for t <  n_old
 *                          = app[l][c][t - n_old][h][d]      for n_old <= t < n_old + n_app
 *                          = untouched                       for t >= n_old + n_app
 * `app` is dense [layer][K,V][token][head][dim] with n_app tokens.  OLD page is never written.
 */
int kvo_cow_append(void *const *base, uint32_t L, uint32_t C, uint32_t num_pages, uint32_t T,
                   uint32_t H, uint32_t D, uint32_t e, uint64_t page_stride_bytes, int order,
                   int32_t old_id, int32_t new_id, uint32_t n_old, const void *app, uint32_t n_app) {
  if (!base || !L || !C || !T || !H || !D || !e || (order != 0 && order != 1)) return KVO_ERR_ARG;
  if ((uint64_t)n_old + n_app > T || old_id == new_id) return KVO_ERR_ARG;
  if (old_id < 0 || new_id < 0 || (uint32_t)old_id >= num_pages || (uint32_t)new_id >= num_pages)
    return KVO_ERR_PAGE_RANGE;
  if (!app && n_app) return KVO_ERR_ARG;
  for (uint64_t l = 0; l < L; ++l)
    for (uint64_t c = 0; c < C; ++c)
      for (uint64_t t = 0; t < (uint64_t)n_old + n_app; ++t)
        for (uint64_t h = 0; h < H; ++h)
          for (uint64_t d = 0; d < D; ++d) {
            uint8_t *slab = (uint8_t *)base[l * C + c];
            uint64_t in_page = kvo_in_page(order, t, T, h, H, d, D) * e;
            uint8_t *dst = slab + (uint64_t)new_id * page_stride_bytes + in_page;
            if (t < n_old) {
              kvo_copy_elem(dst, slab + (uint64_t)old_id * page_stride_bytes + in_page, e);
            } else {
              uint64_t o = ((((l * C + c) * n_app) + (t - n_old)) * H + h) * D + d;
              kvo_copy_elem(dst, (const uint8_t *)app + o * e, e);
            }
          }
  return KVO_OK;
}

/* Batched copy-on-write append (SURVEY.md 8(f) NEXT-1 "batched over sessions"):
 * kvo_cow_append once per session s, in order, with its own (old_ids[s], new_ids[s], n_old[s],
 * n_app[s], apps[s]).  All arguments are checked for every session before anything is written.
 * new_ids must be distinct and must not appear among old_ids (caller checks, like unpack). */
int kvo_cow_append_batched(void *const *base, uint32_t L, uint32_t C, uint32_t num_pages,
                           uint32_t T, uint32_t H, uint32_t D, uint32_t e,
                           uint64_t page_stride_bytes, int order, const int32_t *old_ids,
                           const int32_t *new_ids, const uint32_t *n_old, const uint32_t *n_app,
                           const void *const *apps, uint32_t S) {
  if (S && (!old_ids || !new_ids || !n_old || !n_app || !apps)) return KVO_ERR_ARG;
  for (uint32_t s = 0; s < S; ++s) {
    if ((uint64_t)n_old[s] + n_app[s] > T || old_ids[s] == new_ids[s]) return KVO_ERR_ARG;
    if (old_ids[s] < 0 || new_ids[s] < 0 || (uint32_t)old_ids[s] >= num_pages ||
        (uint32_t)new_ids[s] >= num_pages)
      return KVO_ERR_PAGE_RANGE;
    if (!apps[s] && n_app[s]) return KVO_ERR_ARG;
  }
  for (uint32_t s = 0; s < S; ++s) {
    int rc = kvo_cow_append(base, L, C, num_pages, T, H, D, e, page_stride_bytes, order, old_ids[s],
                            new_ids[s], n_old[s], apps[s], n_app[s]);
    if (rc) return rc;
  }
  return KVO_OK;
}

/* O-repage, pool -> pool (SURVEY.md 8(c) reading 11 "fused pool->pool is an optional extra";
 * 8(f) NEXT-2; PAPER.md:L298 cross-role reuse; BASELINE.json:configs[4] "sequence order preserved,
 * tail page partially filled and zero-padded"): the transfer buffer of O-pack/O-unpack is skipped,
 *   n_src = ceil(n_tokens / Ts), n_dst = ceil(n_tokens / Td)
 *   for q,l,c,u,h,d:  j = q*Td + u
 *     DST[l][c][dst_ids[q]][u][h][d] = (j < n_tokens) ? SRC[l][c][src_ids[j / Ts]][j % Ts][h][d] : 0
 * Source and destination pools have the same L, C, H, D, e; page sizes Ts / Td, page counts and
 * strides are their own.  Nothing else in the destination pool is written; SRC is never written. */
int kvo_repage(const void *const *src_base, uint32_t src_num_pages, uint64_t src_stride_bytes,
               int src_order, uint32_t Ts, const int32_t *src_ids, uint64_t n_src,
               void *const *dst_base, uint32_t dst_num_pages, uint64_t dst_stride_bytes,
               int dst_order, uint32_t Td, const int32_t *dst_ids, uint64_t n_dst, uint32_t L,
               uint32_t C, uint32_t H, uint32_t D, uint32_t e, uint64_t n_tokens, int threads) {
  if (!src_base || !dst_base || !L || !C || !Ts || !Td || !H || !D || !e) return KVO_ERR_ARG;
  if ((src_order != 0 && src_order != 1) || (dst_order != 0 && dst_order != 1)) return KVO_ERR_ARG;
  if (n_src != (n_tokens + Ts - 1) / Ts || n_dst != (n_tokens + Td - 1) / Td) return KVO_ERR_ARG;
  if ((!src_ids || !dst_ids) && n_tokens) return KVO_ERR_ARG;
  if (!kvo_ids_in_range(src_ids, n_src, src_num_pages)) return KVO_ERR_PAGE_RANGE;
  if (!kvo_ids_in_range(dst_ids, n_dst, dst_num_pages)) return KVO_ERR_PAGE_RANGE;
#pragma omp parallel for num_threads(threads) if (threads > 1) schedule(static)
  for (int64_t q = 0; q < (int64_t)n_dst; ++q)
    for (uint64_t l = 0; l < L; ++l)
      for (uint64_t c = 0; c < C; ++c)
        for (uint64_t u = 0; u < Td; ++u)
          for (uint64_t h = 0; h < H; ++h)
            for (uint64_t d = 0; d < D; ++d) {
              uint64_t j = (uint64_t)q * Td + u; /* sequence position, order preserved */
              uint8_t *dst = (uint8_t *)dst_base[l * C + c] +
                             (uint64_t)dst_ids[q] * dst_stride_bytes +
                             kvo_in_page(dst_order, u, Td, h, H, d, D) * e;
              if (j < n_tokens) {
                const uint8_t *src = (const uint8_t *)src_base[l * C + c] +
                                     (uint64_t)src_ids[j / Ts] * src_stride_bytes +
                                     kvo_in_page(src_order, j % Ts, Ts, h, H, d, D) * e;
                kvo_copy_elem(dst, src, e);
              } else {
                kvo_zero_elem(dst, e);
              }
            }
  return KVO_OK;
}

/* Batched O-repage: request r re-pages src_ids[src_off[r] .. src_off[r+1]) into
 * dst_ids[dst_off[r] .. dst_off[r+1]) with its own n_tokens[r]. */
int kvo_repage_batched(const void *const *src_base, uint32_t src_num_pages,
                       uint64_t src_stride_bytes, int src_order, uint32_t Ts,
                       const int32_t *src_ids, const int64_t *src_off, void *const *dst_base,
                       uint32_t dst_num_pages, uint64_t dst_stride_bytes, int dst_order,
                       uint32_t Td, const int32_t *dst_ids,
                       const int64_t *dst_off, const uint64_t *n_tokens, uint32_t R, uint32_t L,
                       uint32_t C, uint32_t H, uint32_t D, uint32_t e, int threads) {
  if (R && (!src_off || !dst_off || !n_tokens)) return KVO_ERR_ARG;
  if (!Ts || !Td) return KVO_ERR_ARG;
  for (uint32_t r = 0; r < R; ++r) {
    if (src_off[r + 1] < src_off[r] || dst_off[r + 1] < dst_off[r]) return KVO_ERR_ARG;
    if ((uint64_t)(src_off[r + 1] - src_off[r]) != (n_tokens[r] + Ts - 1) / Ts) return KVO_ERR_ARG;
    if ((uint64_t)(dst_off[r + 1] - dst_off[r]) != (n_tokens[r] + Td - 1) / Td) return KVO_ERR_ARG;
    if (!kvo_ids_in_range(src_ids + src_off[r], (uint64_t)(src_off[r + 1] - src_off[r]), src_num_pages))
      return KVO_ERR_PAGE_RANGE;
    if (!kvo_ids_in_range(dst_ids + dst_off[r], (uint64_t)(dst_off[r + 1] - dst_off[r]), dst_num_pages))
      return KVO_ERR_PAGE_RANGE;
  }
  for (uint32_t r = 0; r < R; ++r) {
    int rc = kvo_repage(src_base, src_num_pages, src_stride_bytes, src_order, Ts,
                        src_ids + src_off[r], (uint64_t)(src_off[r + 1] - src_off[r]), dst_base,
                        dst_num_pages, dst_stride_bytes, dst_order, Td, dst_ids + dst_off[r],
                        (uint64_t)(dst_off[r + 1] - dst_off[r]), L, C, H, D, e, n_tokens[r], threads);
    if (rc) return rc;
  }
  return KVO_OK;
}
