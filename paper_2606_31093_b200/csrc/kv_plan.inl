// kv_plan.inl -- validation and planning of every entry point: all of it precedes the first CUDA call, a failing call writes nothing
// Part of the host side of libkvtier.so; included by kvtier.cu only (one translation unit).
// Shares nothing with oracle/.
#pragma once

namespace {

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
  const bool dev_ids = flags & KV_FLAG_IDS_ON_DEVICE;  // old_ids / new_ids are device arrays, read by the kernel
  if (n_sessions && (!old_ids || !new_ids || !n_old || !n_app || !apps)) return KV_ERR_NULL;
  const uint64_t tokrow = (uint64_t)pools->num_heads * pools->head_dim * pools->elem_bytes;
  const uint64_t lc = (uint64_t)layer_count * pools->kv_count;
  c->reqs.clear();
  for (uint32_t s = 0; s < n_sessions; ++s) {
    if ((uint64_t)n_old[s] + n_app[s] > pools->page_size) return KV_ERR_SIZE;
    if (!dev_ids) {
      if (old_ids[s] == new_ids[s]) return KV_ERR_SIZE;
      if (old_ids[s] < 0 || new_ids[s] < 0 || (uint32_t)old_ids[s] >= pools->num_pages ||
          (uint32_t)new_ids[s] >= pools->num_pages)
        return KV_ERR_PAGE_RANGE;
    }
    if (n_app[s] && !apps[s]) return KV_ERR_NULL;
    if (!n_old[s] && !n_app[s]) continue;
    Req q;
    q.buf = (uint64_t)(uintptr_t)apps[s];
    q.n_tokens = (uint64_t)n_old[s] | ((uint64_t)n_app[s] << 32);
    q.id_begin = dev_ids ? (uint64_t)s : (uint64_t)(uint32_t)old_ids[s] | ((uint64_t)(uint32_t)new_ids[s] << 32);
    c->reqs.push_back(q);
  }
  if ((flags & KV_FLAG_VALIDATE) && !dev_ids) {  // new pages distinct, and none of them is some session's old page
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
  if (dev_ids) c->geom.dev_src_ids = new_ids;
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

// kv_submit: several independent pack / unpack / copy-on-write operations on one pool -> ONE launch in which the
// direction is a property of the piece (Job::dir == 4, Piece::dir).  Page ids of all pack / unpack operations are
// gathered into `all_ids` in operation order.
int plan_submit(kv_ctx *ctx, const kv_pool_desc *pools, uint32_t layer_count, const kv_op *ops, uint32_t n_ops,
                int layout, uint32_t flags, Call *c, std::vector<int32_t> *all_ids) {
  if (!ctx) return KV_ERR_NULL;
  int rc = check_desc(pools, layer_count);
  if (rc) return rc;
  if (flags & KV_FLAG_IDS_ON_DEVICE) return KV_ERR_LAYOUT;
  if (n_ops && !ops) return KV_ERR_NULL;
  const uint32_t T = pools->page_size;
  const uint64_t tokrow = (uint64_t)pools->num_heads * pools->head_dim * pools->elem_bytes;
  const uint64_t lc = (uint64_t)layer_count * pools->kv_count;
  const uint64_t page = lc * T * tokrow;
  c->reqs.clear();
  all_ids->clear();
  for (uint32_t i = 0; i < n_ops; ++i) {
    const kv_op &op = ops[i];
    Req q;
    q.dir = op.kind;
    if (op.kind == KV_OP_PACK || op.kind == KV_OP_UNPACK) {
      const uint64_t n = op.n_pages;
      if (op.kind == KV_OP_UNPACK) {
        if (n != (op.n_tokens + T - 1) / T) return KV_ERR_SIZE;
      }
      if (!n) continue;
      if (!op.page_ids || !op.buf) return KV_ERR_NULL;
      if (op.buf_bytes && op.buf_bytes < n * page) return KV_ERR_SIZE;
      rc = check_ids(op.page_ids, n, pools->num_pages);
      if (rc) return rc;
      q.buf = (uint64_t)(uintptr_t)op.buf;
      q.n_tokens = op.kind == KV_OP_PACK ? n * T : op.n_tokens;
      q.id_begin = all_ids->size(); q.n_ids = n; q.n_buf_pages = n;
      all_ids->insert(all_ids->end(), op.page_ids, op.page_ids + n);
    } else if (op.kind == KV_OP_COW_APPEND) {
      if (!op.page_ids) return KV_ERR_NULL;
      if ((uint64_t)op.n_old + op.n_app > T) return KV_ERR_SIZE;
      const int32_t o = op.page_ids[0], nw = op.page_ids[1];
      if (o == nw) return KV_ERR_SIZE;
      if (o < 0 || nw < 0 || (uint32_t)o >= pools->num_pages || (uint32_t)nw >= pools->num_pages) return KV_ERR_PAGE_RANGE;
      if (op.n_app && !op.buf) return KV_ERR_NULL;
      if (!op.n_old && !op.n_app) continue;
      q.buf = (uint64_t)(uintptr_t)op.buf;
      q.n_tokens = (uint64_t)op.n_old | ((uint64_t)op.n_app << 32);
      q.id_begin = (uint64_t)(uint32_t)o | ((uint64_t)(uint32_t)nw << 32);
    } else {
      return KV_ERR_LAYOUT;
    }
    c->reqs.push_back(q);
  }
  if (flags & KV_FLAG_VALIDATE) {  // written pages distinct; nothing read that the same call writes
    std::vector<uint8_t> written((size_t)(pools->num_pages + 7) / 8, 0);
    auto test = [&](uint32_t g) { return (written[g >> 3] >> (g & 7)) & 1u; };
    for (const Req &q : c->reqs) {
      if (q.dir == KV_OP_UNPACK) {
        for (uint64_t k = 0; k < q.n_ids; ++k) {
          const uint32_t g = (uint32_t)(*all_ids)[q.id_begin + k];
          if (test(g)) return KV_ERR_DUP_PAGE;
          written[g >> 3] |= (uint8_t)(1u << (g & 7));
        }
      } else if (q.dir == KV_OP_COW_APPEND) {
        const uint32_t g = (uint32_t)(q.id_begin >> 32);
        if (test(g)) return KV_ERR_DUP_PAGE;
        written[g >> 3] |= (uint8_t)(1u << (g & 7));
      }
    }
    for (const Req &q : c->reqs) {
      if (q.dir == KV_OP_PACK) {
        for (uint64_t k = 0; k < q.n_ids; ++k)
          if (test((uint32_t)(*all_ids)[q.id_begin + k])) return KV_ERR_DUP_PAGE;
      } else if (q.dir == KV_OP_COW_APPEND) {
        if (test((uint32_t)q.id_begin)) return KV_ERR_DUP_PAGE;
      }
    }
  }
  c->n_ids = all_ids->size();
  rc = make_geom(ctx, pools, layer_count, T, /*dir=*/4, layout, c->reqs, &c->geom);
  if (rc) return rc;
  c->total_items = 0; c->payload = 0;
  const uint64_t sub = c->geom.sub_bytes;
  for (Req &q : c->reqs) {
    if (q.dir == KV_OP_COW_APPEND) {
      const uint64_t b_old = (q.n_tokens & 0xffffffffull) * tokrow, b_app = (q.n_tokens >> 32) * tokrow;
      q.items = lc * ((b_old + sub - 1) / sub + (b_app + sub - 1) / sub);
      c->payload += lc * (b_old + b_app);
    } else {
      q.items = items_of(c->geom, q.n_ids);
      c->payload += q.n_ids * page;
    }
    if (q.items > 0xFFFFFFFFull) return KV_ERR_SIZE;
    c->total_items += q.items;
  }
  return KV_OK;
}

void note_plan(kv_ctx *ctx, const Call &c) {
  ctx->last_items = c.total_items;
  ctx->last_payload = c.payload;
  ctx->last_kernel = (uint64_t)c.geom.kernel;
  ctx->last_segment = c.geom.sub_bytes;
}

}  // namespace
