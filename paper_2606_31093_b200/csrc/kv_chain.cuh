// kv_chain.cuh -- chained paged hashing on the GPU (kvtier.h
// kv_chain_hash).  id_k = FNV1a64(LE64(id_{k-1}) || LE64(digest_k)), digest_k = FNV1a64 of the 8*T
// little-endian bytes of page k's T content identities; id_{-1} = the session's root.
//
// The work splits where the dependence does (two launches for large batches; kv_chain_fused does both phases in one
// launch for up to 128 sessions):
//   kv_chain_digest  one THREAD per page, all pages of all sessions at once: 8*T dependent
//                    xor/multiply steps per page, no dependence between pages -- the parallel 8/9ths.
//   kv_chain_link    one WARP per session: the chain proper, 16 dependent steps per page.  The 32 lanes
//                    fetch 32 digests with one coalesced load, every lane then walks the same 32 links
//                    (digest handed round by shuffle), lane i keeps link i, and the 32 ids leave with
//                    one coalesced store.  Serial along the chain, parallel across sessions -- as the
//                    definition is.
// Both are bound by the latency of dependent integer multiplies, not by memory (8 B read per token
// against 98,304 B of KV the same token owns).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kvt {

constexpr uint64_t kFnvBasis = 0xcbf29ce484222325ull;
constexpr uint64_t kFnvPrime = 0x100000001b3ull;

// One FNV-1a step on the two 32-bit halves of h:  h' = (h ^ b) * (2^40 + 0x1b3)  mod 2^64, i.e. with
// x = lo ^ b:   lo' = low32(x * 0x1b3),   hi' = hi * 0x1b3 + [ high32(x * 0x1b3) + (x << 8) ].
// The bracket depends on the LOW chain only, so the high half advances by ONE multiply-add per step
// and the step is bound by the low chain: LOP3 (alu pipe) -> IMAD.WIDE (fma pipe) -> LOP3.  Bare chains measured on
// B200 (one warp, clock64 around 1.6 M dependent steps, round 2): xor -> mul.wide 12.4 cycles per step, xor -> 32-bit
// mul.lo 10.1 -- so 12.4 cycles = 6.3 ns per step, 101 ns per 16-step link at 1,965 MHz is the floor of THIS step, and a
// 2,875-link chain runs at 102 ns per link (round 1 quoted 15.7 cycles: its probe also carried the high-half chain in
// program order).  Left to itself nvcc chains three dependent ops through the high half (171 ns per link); the asm
// below pins the association.  Taking the 32-bit multiply alone onto the chain (high word by a separate mul.hi) would
// be 19 % shorter, but ptxas fuses the pair back into one IMAD.WIDE, and hiding the pairing from it (an operand it
// cannot prove equal) moved the whole chain onto the uniform datapath: 427 instead of 288 us.  Not pursued.
__device__ __forceinline__ void fnv1a_step(uint32_t &lo, uint32_t &hi, uint32_t byte) {
  const uint32_t x = lo ^ byte;
  uint64_t w;
  uint32_t t;
  asm("mul.wide.u32 %0, %1, 0x1b3;" : "=l"(w) : "r"(x));
  asm("mad.lo.u32 %0, %1, 0x100, %2;" : "=r"(t) : "r"(x), "r"((uint32_t)(w >> 32)));
  asm("mad.lo.u32 %0, %1, 0x1b3, %2;" : "=r"(hi) : "r"(hi), "r"(t));
  lo = (uint32_t)w;
}

// eight byte-serial FNV-1a steps over the little-endian bytes of w
__device__ __forceinline__ uint64_t fnv1a_word(uint64_t h, uint64_t w) {
  uint32_t lo = (uint32_t)h, hi = (uint32_t)(h >> 32);
  const uint32_t w0 = (uint32_t)w, w1 = (uint32_t)(w >> 32);
#pragma unroll
  for (int b = 0; b < 4; ++b) fnv1a_step(lo, hi, (w0 >> (8 * b)) & 0xffu);
#pragma unroll
  for (int b = 0; b < 4; ++b) fnv1a_step(lo, hi, (w1 >> (8 * b)) & 0xffu);
  return ((uint64_t)hi << 32) | lo;
}

struct ChainJob {
  const uint64_t *ident;     // device: identities of all sessions
  uint64_t *out;             // device: digests (after kv_chain_digest), then ids (after kv_chain_link)
  const int64_t *tok_off;    // device [S+1]
  const int64_t *page_off;   // device [S+1]
  const uint64_t *roots;     // device [S] or nullptr
  uint64_t default_root;
  uint64_t total_pages;
  uint32_t n_sessions;
  uint32_t T;
};

// Tables of small batches ride inside the kernel parameters (kInline): no staging copy, so the call is two
// self-contained launches and can be captured into a CUDA graph.  [tok_off: S+1][page_off: S+1][roots: S]
constexpr int kChainInlineSessions = 128;
struct ChainJobInline {
  ChainJob j;
  int64_t tok_off[kChainInlineSessions + 1];
  int64_t page_off[kChainInlineSessions + 1];
  uint64_t roots[kChainInlineSessions];
};
template <bool kInline> struct ChainParam { typedef ChainJob type; };
template <> struct ChainParam<true> { typedef ChainJobInline type; };
template <bool kInline, typename P>
__device__ __forceinline__ ChainJob chain_job(const P &p) {
  if constexpr (kInline) {
    ChainJob j = p.j;
    j.tok_off = p.tok_off; j.page_off = p.page_off;
    if (j.roots) j.roots = p.roots;
    return j;
  } else {
    return p;
  }
}

// digest of page k of session s (8*T dependent steps; four identity loads in flight ahead of the arithmetic)
__device__ __forceinline__ uint64_t chain_digest_page(const ChainJob &j, uint32_t s, uint64_t k) {
  const uint64_t *src = j.ident + (uint64_t)j.tok_off[s] + k * j.T;
  uint64_t h = kFnvBasis;
  uint32_t t = 0;
  for (; t + 4 <= j.T; t += 4) {
    const uint64_t w0 = __ldg(src + t), w1 = __ldg(src + t + 1), w2 = __ldg(src + t + 2), w3 = __ldg(src + t + 3);
    h = fnv1a_word(fnv1a_word(fnv1a_word(fnv1a_word(h, w0), w1), w2), w3);
  }
  for (; t < j.T; ++t) h = fnv1a_word(h, __ldg(src + t));
  return h;
}

// the chain of session s, walked by one warp: digests in j.out[p0, p1) are replaced by the ids
__device__ __forceinline__ void chain_link_session(const ChainJob &j, uint32_t s, uint32_t lane) {
  const uint64_t p0 = (uint64_t)j.page_off[s], p1 = (uint64_t)j.page_off[s + 1];
  uint64_t prev = j.roots ? j.roots[s] : j.default_root;
  uint64_t next_d = p0 + lane < p1 ? j.out[p0 + lane] : 0;
  for (uint64_t base = p0; base < p1; base += 32) {
    const uint64_t d = next_d;
    if (base + 32 + lane < p1) next_d = j.out[base + 32 + lane];  // prefetch the next 32 digests
    const uint32_t n = (uint32_t)min((uint64_t)32, p1 - base);
    uint64_t mine = 0;
    uint64_t di = __shfl_sync(0xffffffffu, d, 0);
    for (uint32_t i = 0; i < n; ++i) {  // every lane walks the same links: no divergence, no broadcast of ids
      const uint64_t dn = __shfl_sync(0xffffffffu, d, (i + 1) & 31);  // next link's digest, off the chain
      prev = fnv1a_word(fnv1a_word(kFnvBasis, prev), di);
      if (i == lane) mine = prev;
      di = dn;
    }
    if (lane < n) j.out[base + lane] = mine;
  }
}

template <bool kInline>
__global__ void __launch_bounds__(128) kv_chain_digest(const __grid_constant__ typename ChainParam<kInline>::type prm) {
  const ChainJob j = chain_job<kInline>(prm);
  const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= j.total_pages) return;
  uint32_t lo = 0, hi = j.n_sessions;  // largest s with page_off[s] <= p
  while (hi - lo > 1) {
    const uint32_t mid = (lo + hi) >> 1;
    if ((uint64_t)j.page_off[mid] <= p) lo = mid; else hi = mid;
  }
  j.out[p] = chain_digest_page(j, lo, p - (uint64_t)j.page_off[lo]);
}

template <bool kInline>
__global__ void __launch_bounds__(32) kv_chain_link(const __grid_constant__ typename ChainParam<kInline>::type prm) {
  const ChainJob j = chain_job<kInline>(prm);
  if (blockIdx.x >= j.n_sessions) return;
  chain_link_session(j, blockIdx.x, threadIdx.x);
}

// Batches of up to kChainInlineSessions sessions: ONE launch, one CTA per session.  All threads of the CTA digest the
// session's pages (one page per thread and pass), the CTA meets, warp 0 walks the chain.  The digest phase of even the
// longest paper-shaped history (2,875 pages on 1,024 threads: three passes of 128 steps) is ~3 us against the 377 us of
// its chain, and a turn's incremental hash of a few dozen pages is one launch instead of two.
template <bool kInline>
__global__ void __launch_bounds__(1024) kv_chain_fused(const __grid_constant__ typename ChainParam<kInline>::type prm) {
  const ChainJob j = chain_job<kInline>(prm);
  const uint32_t s = blockIdx.x;
  if (s >= j.n_sessions) return;
  const uint64_t p0 = (uint64_t)j.page_off[s], p1 = (uint64_t)j.page_off[s + 1];
  for (uint64_t p = p0 + threadIdx.x; p < p1; p += blockDim.x) j.out[p] = chain_digest_page(j, s, p - p0);
  __syncthreads();  // the digests (global memory) are visible to warp 0
  if (threadIdx.x < 32) chain_link_session(j, s, threadIdx.x);
}

}  // namespace kvt
