/* Plain-C consumer of include/kvtier.h: proves the boundary is a C ABI (no C++ or torch types in the
 * signatures) by compiling as C99 and driving a planning-only context (device = -1: no CUDA call is made).
 * Built and run by tests/test_abi_host.py::test_header_is_c_and_links_from_c. */
#include <stdio.h>
#include <string.h>

#include "kvtier.h"

#define CHECK(cond)                                              \
  do {                                                           \
    if (!(cond)) {                                               \
      fprintf(stderr, "abi_smoke: %s failed (line %d)\n", #cond, __LINE__); \
      return 1;                                                  \
    }                                                            \
  } while (0)

int main(void) {
  kv_ctx *ctx = NULL;
  CHECK(kv_version() == KVTIER_VERSION);
  CHECK(strcmp(kv_strerror(KV_OK), "ok") == 0);
  CHECK(kv_ctx_create(&ctx, -1, 0) == KV_OK && ctx != NULL);

  /* Tiny pool of BASELINE.json:configs[0]: 4 layers x (K, V), 256 pages of 16 tokens x 2 heads x 64 dims, bf16 */
  void *bases[8];
  int i;
  for (i = 0; i < 8; ++i) bases[i] = (void *)(size_t)(0x100000000ull + (unsigned long long)i * 0x1000000ull);
  kv_pool_desc pool;
  memset(&pool, 0, sizeof pool);
  pool.base = bases;
  pool.layer_count = 4; pool.kv_count = 2; pool.num_pages = 256; pool.page_size = 16;
  pool.num_heads = 2; pool.head_dim = 64; pool.elem_bytes = 2; pool.order = KV_ORDER_NHD;
  pool.page_stride_bytes = 16u * 2u * 64u * 2u;

  int32_t ids[3] = {7, 200, 31};
  void *buf = (void *)(size_t)0x200000000ull;
  const size_t page = 4u * 2u * 4096u;
  uint64_t stat = 0;

  /* valid call on a planning-only ctx: validated and planned, nothing launched */
  CHECK(kv_pack(ctx, &pool, 4, ids, 3, KV_LAYOUT_PAGE_FIRST, buf, 3 * page, 0, NULL) == KV_ERR_NO_DEVICE);
  CHECK(kv_ctx_get_stat(ctx, KV_STAT_LAST_PAYLOAD, &stat) == KV_OK && stat == 3 * page);
  /* errors precede everything else */
  CHECK(kv_pack(ctx, &pool, 4, ids, 3, KV_LAYOUT_PAGE_FIRST, buf, 3 * page - 1, 0, NULL) == KV_ERR_SIZE);
  ids[1] = 256;
  CHECK(kv_pack(ctx, &pool, 4, ids, 3, KV_LAYOUT_PAGE_FIRST, buf, 3 * page, 0, NULL) == KV_ERR_PAGE_RANGE);
  ids[1] = 7;
  CHECK(kv_unpack(ctx, buf, 3 * page, ids, 3, &pool, 4, 16, 16, 48, KV_LAYOUT_PAGE_FIRST, KV_FLAG_VALIDATE, NULL) ==
        KV_ERR_DUP_PAGE);
  CHECK(kv_pack(ctx, &pool, 4, ids, 0, KV_LAYOUT_PAGE_FIRST, buf, 0, 0, NULL) == KV_OK); /* n == 0 */
  {
    int64_t tok_off[3] = {0, 40, 75}, page_off[3] = {-1, -1, -1};
    CHECK(kv_chain_hash(ctx, (const uint64_t *)buf, tok_off, 2, 16, NULL, (uint64_t *)buf, 4, page_off, NULL) ==
          KV_ERR_NO_DEVICE);
    CHECK(page_off[0] == 0 && page_off[1] == 2 && page_off[2] == 4);
  }
  CHECK(kv_ctx_destroy(ctx) == KV_OK);
  puts("abi_smoke ok");
  return 0;
}
