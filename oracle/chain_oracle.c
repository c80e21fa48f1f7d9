/* oracle/chain_oracle.c -- CPU ORACLE for chained paged hashing.  TEST INFRASTRUCTURE ONLY
 * (only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may build, load or call it;
 * it shares nothing with paper_2606_31093_b200/).
 *
 * PAPER.md:L276 (Sec. 5.1, Multimodal Prefix Matching): "Both paths use Chained Paged Hashing: each page ID hashes its
 * predecessor together with the current page's content identities, thereby representing the complete
 * page-aligned prefix."  The paper names no hash function and no encoding; reading H1-H4:
 *
 *   H1  a content identity is one 64-bit word per token position (a token id, or the content hash id
 *       of the multimodal item a placeholder position belongs to);
 *   H2  the hash is 64-bit FNV-1a (Fowler/Noll/Vo; offset basis 0xcbf29ce484222325, prime
 *       0x100000001b3), byte-serial: h = (h XOR byte) * prime mod 2^64;
 *   H3  digest_k = FNV-1a of the 8*T little-endian bytes of page k's T identities;
 *       id_k     = FNV-1a of the 16 bytes  LE64(id_{k-1}) || LE64(digest_k),  id_{-1} = root;
 *   H4  only whole pages get ids: a session of n tokens has floor(n / T) ids ("page-aligned prefix").
 *
 * Plain loops, in that order; no blocking, no vectorisation.  Pinned by tests/test_chain_oracle_pins.py.
 */
#include <stdint.h>

#define CHO_BASIS 0xcbf29ce484222325ull
#define CHO_PRIME 0x100000001b3ull

/* FNV-1a over a byte string (H2). */
uint64_t cho_fnv1a64(const uint8_t *msg, uint64_t n) {
  uint64_t h = CHO_BASIS;
  for (uint64_t i = 0; i < n; ++i) {
    h ^= (uint64_t)msg[i];
    h *= CHO_PRIME;
  }
  return h;
}

static void cho_le64(uint64_t v, uint8_t out[8]) {
  for (int b = 0; b < 8; ++b) out[b] = (uint8_t)(v >> (8 * b));
}

/* Page ids of ONE session (H3, H4): ident[0..n_tokens), page size T, chain root `root`;
 * writes floor(n_tokens / T) ids to out and returns that count. */
uint64_t cho_chain(const uint64_t *ident, uint64_t n_tokens, uint32_t T, uint64_t root, uint64_t *out) {
  const uint64_t n_pages = T ? n_tokens / T : 0;
  uint64_t prev = root;
  for (uint64_t k = 0; k < n_pages; ++k) {
    uint64_t d = CHO_BASIS; /* digest of the page's identities, byte by byte */
    for (uint32_t t = 0; t < T; ++t) {
      uint8_t le[8];
      cho_le64(ident[k * T + t], le);
      for (int b = 0; b < 8; ++b) {
        d ^= (uint64_t)le[b];
        d *= CHO_PRIME;
      }
    }
    uint8_t msg[16];
    cho_le64(prev, msg);
    cho_le64(d, msg + 8);
    prev = cho_fnv1a64(msg, 16);
    out[k] = prev;
  }
  return n_pages;
}

/* Batched over sessions: identities of session s are ident[tok_off[s] .. tok_off[s+1]); its ids go to
 * out[page_off[s] ..) where page_off is the running sum of floor(len_s / T) (written to page_off[0..S]).
 * roots == NULL: every chain starts from `default_root`.  Sessions are independent; OpenMP only over
 * the session loop.  Returns the total number of ids, or -1 on a negative / decreasing offset. */
int64_t cho_chain_batched(const uint64_t *ident, const int64_t *tok_off, uint32_t n_sessions, uint32_t T,
                          const uint64_t *roots, uint64_t default_root, uint64_t *out, int64_t *page_off,
                          int threads) {
  if (!T) return -1;
  page_off[0] = 0;
  for (uint32_t s = 0; s < n_sessions; ++s) {
    if (tok_off[s] < 0 || tok_off[s + 1] < tok_off[s]) return -1;
    page_off[s + 1] = page_off[s] + (tok_off[s + 1] - tok_off[s]) / (int64_t)T;
  }
  (void)threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : 1)
#endif
  for (int64_t s = 0; s < (int64_t)n_sessions; ++s)
    cho_chain(ident + tok_off[s], (uint64_t)(tok_off[s + 1] - tok_off[s]), T,
              roots ? roots[s] : default_root, out + page_off[s]);
  return page_off[n_sessions];
}
