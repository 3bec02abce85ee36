// f3: HOST-side block hasher and block pool - the step before block tables exist.  No device code.
//
// Eq. 1: the engine's chained block hash with two markers that act only when they are the FIRST token of a
// KV block:  h_i = H(h_0, x_i) if x_i starts with SSEP (detached from the chain: the span is cacheable wherever it appears),
//            h_i = H(h_0, x_{<=i}) if x_i starts with PDEP (depends on the whole prompt: no false hits for the task suffix),
//            h_i = H(h_{i-1}, x_i) otherwise.
// H = SHA-256 over (parent digest || tokens as little-endian int32); h_0 = SHA-256(seed as 8 little-endian bytes).
// The pool maps digests to physical blocks, so token streams turn into block tables, slot mappings (of the tokens that
// still have to be written) and the visibility descriptor q_vis_lo (reading A6) that the attention calls take.
#include <cstdint>
#include <cstring>
#include <deque>
#include <list>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/minipic.h"

namespace {

// ---- SHA-256 (FIPS 180-4), restated
struct Sha256 {
  uint32_t h[8];
  uint8_t buf[64];
  uint64_t len = 0;
  size_t fill = 0;
  Sha256() {
    static const uint32_t init[8] = {0x6a09e667u, 0xbb67ae85u, 0x3c6ef372u, 0xa54ff53au, 0x510e527fu, 0x9b05688cu, 0x1f83d9abu, 0x5be0cd19u};
    std::memcpy(h, init, sizeof(h));
  }
  static uint32_t rotr(uint32_t x, int n) { return (x >> n) | (x << (32 - n)); }
  void block(const uint8_t* p) {
    static const uint32_t K[64] = {
        0x428a2f98u, 0x71374491u, 0xb5c0fbcfu, 0xe9b5dba5u, 0x3956c25bu, 0x59f111f1u, 0x923f82a4u, 0xab1c5ed5u, 0xd807aa98u, 0x12835b01u,
        0x243185beu, 0x550c7dc3u, 0x72be5d74u, 0x80deb1feu, 0x9bdc06a7u, 0xc19bf174u, 0xe49b69c1u, 0xefbe4786u, 0x0fc19dc6u, 0x240ca1ccu,
        0x2de92c6fu, 0x4a7484aau, 0x5cb0a9dcu, 0x76f988dau, 0x983e5152u, 0xa831c66du, 0xb00327c8u, 0xbf597fc7u, 0xc6e00bf3u, 0xd5a79147u,
        0x06ca6351u, 0x14292967u, 0x27b70a85u, 0x2e1b2138u, 0x4d2c6dfcu, 0x53380d13u, 0x650a7354u, 0x766a0abbu, 0x81c2c92eu, 0x92722c85u,
        0xa2bfe8a1u, 0xa81a664bu, 0xc24b8b70u, 0xc76c51a3u, 0xd192e819u, 0xd6990624u, 0xf40e3585u, 0x106aa070u, 0x19a4c116u, 0x1e376c08u,
        0x2748774cu, 0x34b0bcb5u, 0x391c0cb3u, 0x4ed8aa4au, 0x5b9cca4fu, 0x682e6ff3u, 0x748f82eeu, 0x78a5636fu, 0x84c87814u, 0x8cc70208u,
        0x90befffau, 0xa4506cebu, 0xbef9a3f7u, 0xc67178f2u};
    uint32_t w[64];
    for (int i = 0; i < 16; ++i) w[i] = (uint32_t)p[4 * i] << 24 | (uint32_t)p[4 * i + 1] << 16 | (uint32_t)p[4 * i + 2] << 8 | p[4 * i + 3];
    for (int i = 16; i < 64; ++i) {
      const uint32_t s0 = rotr(w[i - 15], 7) ^ rotr(w[i - 15], 18) ^ (w[i - 15] >> 3);
      const uint32_t s1 = rotr(w[i - 2], 17) ^ rotr(w[i - 2], 19) ^ (w[i - 2] >> 10);
      w[i] = w[i - 16] + s0 + w[i - 7] + s1;
    }
    uint32_t a = h[0], b = h[1], c = h[2], d = h[3], e = h[4], f = h[5], g = h[6], hh = h[7];
    for (int i = 0; i < 64; ++i) {
      const uint32_t t1 = hh + (rotr(e, 6) ^ rotr(e, 11) ^ rotr(e, 25)) + ((e & f) ^ (~e & g)) + K[i] + w[i];
      const uint32_t t2 = (rotr(a, 2) ^ rotr(a, 13) ^ rotr(a, 22)) + ((a & b) ^ (a & c) ^ (b & c));
      hh = g; g = f; f = e; e = d + t1; d = c; c = b; b = a; a = t1 + t2;
    }
    h[0] += a; h[1] += b; h[2] += c; h[3] += d; h[4] += e; h[5] += f; h[6] += g; h[7] += hh;
  }
  void update(const void* data, size_t n) {
    const uint8_t* p = (const uint8_t*)data;
    len += n;
    while (n) {
      const size_t take = n < 64 - fill ? n : 64 - fill;
      std::memcpy(buf + fill, p, take);
      fill += take; p += take; n -= take;
      if (fill == 64) { block(buf); fill = 0; }
    }
  }
  void finish(uint8_t out[32]) {
    const uint64_t bits = len * 8;
    const uint8_t one = 0x80, zero = 0;
    update(&one, 1);
    while (fill != 56) update(&zero, 1);
    uint8_t lb[8];
    for (int i = 0; i < 8; ++i) lb[i] = (uint8_t)(bits >> (56 - 8 * i));
    update(lb, 8);
    for (int i = 0; i < 8; ++i) { out[4 * i] = h[i] >> 24; out[4 * i + 1] = h[i] >> 16; out[4 * i + 2] = h[i] >> 8; out[4 * i + 3] = h[i]; }
  }
};

typedef std::string Digest;   // 32 raw bytes

void put_tokens(Sha256& s, const int32_t* t, size_t n) {   // little-endian int32, whatever the host byte order
  for (size_t i = 0; i < n; ++i) {
    const uint32_t v = (uint32_t)t[i];
    const uint8_t b[4] = {(uint8_t)v, (uint8_t)(v >> 8), (uint8_t)(v >> 16), (uint8_t)(v >> 24)};
    s.update(b, 4);
  }
}
Digest H(const Digest& parent, const int32_t* t, size_t n) {
  Sha256 s;
  s.update(parent.data(), parent.size());
  put_tokens(s, t, n);
  uint8_t out[32];
  s.finish(out);
  return Digest((const char*)out, 32);
}
Digest seed_hash(uint64_t seed) {
  uint8_t b[8];
  for (int i = 0; i < 8; ++i) b[i] = (uint8_t)(seed >> (8 * i));
  Sha256 s;
  s.update(b, 8);
  uint8_t out[32];
  s.finish(out);
  return Digest((const char*)out, 32);
}
// Eq. 1 over the full blocks of a token stream
std::vector<Digest> block_hashes(const int32_t* tok, int n, int B, int ssep, int pdep, uint64_t seed) {
  const Digest h0 = seed_hash(seed);
  std::vector<Digest> out;
  Digest prev = h0;
  for (int i = 0; i < n / B; ++i) {
    const int32_t* x = tok + (size_t)i * B;
    Digest h;
    if (x[0] == ssep) h = H(h0, x, B);
    else if (x[0] == pdep) h = H(h0, tok, (size_t)(i + 1) * B);
    else h = H(prev, x, B);
    out.push_back(h);
    prev = h;
  }
  return out;
}

}  // namespace

// A block pool keyed by the Eq. 1 digest.  Blocks come off a free list in increasing id order; a block whose reference
// count is zero stays cached (it can still hit) until the free list is empty, then the least recently released one is
// evicted and its digest forgotten.  Not thread safe.
struct minipic_pool {
  int num_blocks, B, ssep, pdep;
  uint64_t seed;
  std::deque<int> free_list;
  std::unordered_map<Digest, int> by_hash;
  std::vector<Digest> hash_of;      // digest of a cached block ("" = none: partial / never hashed)
  std::vector<int> refs;
  std::list<int> lru;               // unreferenced cached blocks, least recently released first
  std::vector<std::list<int>::iterator> lru_it;
  std::vector<char> in_lru;
  uint64_t hits = 0, misses = 0, evictions = 0;

  int take_block() {
    if (!free_list.empty()) { const int b = free_list.front(); free_list.pop_front(); return b; }
    if (lru.empty()) return -1;
    const int b = lru.front();
    lru.pop_front(); in_lru[b] = 0;
    if (!hash_of[b].empty()) { by_hash.erase(hash_of[b]); hash_of[b].clear(); }
    ++evictions;
    return b;
  }
};

extern "C" {

int minipic_block_hashes(const int32_t* tokens_host, int32_t num_tokens, int32_t block_size, int32_t ssep_id,
                         int32_t pdep_id, uint64_t seed, uint8_t* hashes_out_host) {
  if (num_tokens < 0 || block_size <= 0 || (num_tokens > 0 && !tokens_host) || (num_tokens >= block_size && !hashes_out_host))
    return MINIPIC_ERR_INVALID_ARG;
  const std::vector<Digest> hs = block_hashes(tokens_host, num_tokens, block_size, ssep_id, pdep_id, seed);
  for (size_t i = 0; i < hs.size(); ++i) std::memcpy(hashes_out_host + 32 * i, hs[i].data(), 32);
  return MINIPIC_OK;
}

minipic_pool* minipic_pool_create(int32_t num_blocks, int32_t block_size, int32_t ssep_id, int32_t pdep_id, uint64_t seed) {
  if (num_blocks <= 0 || block_size <= 0) return nullptr;
  minipic_pool* p = new minipic_pool();
  p->num_blocks = num_blocks; p->B = block_size; p->ssep = ssep_id; p->pdep = pdep_id; p->seed = seed;
  for (int i = 0; i < num_blocks; ++i) p->free_list.push_back(i);
  p->hash_of.resize(num_blocks); p->refs.assign(num_blocks, 0);
  p->lru_it.resize(num_blocks); p->in_lru.assign(num_blocks, 0);
  return p;
}
void minipic_pool_destroy(minipic_pool* p) { delete p; }

int minipic_pool_admit(minipic_pool* p, const int32_t* tokens_host, int32_t num_tokens, int32_t* block_table_out,
                       uint8_t* hit_out, int64_t* slot_mapping_out, int32_t* q_vis_lo_out, int32_t* num_new_tokens_out) {
  if (!p || num_tokens < 0 || (num_tokens > 0 && (!tokens_host || !block_table_out || !hit_out || !slot_mapping_out || !q_vis_lo_out)))
    return MINIPIC_ERR_INVALID_ARG;
  const int B = p->B, nblk = (num_tokens + B - 1) / B;
  const std::vector<Digest> hs = block_hashes(tokens_host, num_tokens, B, p->ssep, p->pdep, p->seed);
  int n_new = 0, cur_lo = 0;
  for (int i = 0; i < nblk; ++i) {
    const int lo = i * B, hi = (i + 1) * B < num_tokens ? (i + 1) * B : num_tokens;
    // visibility (reading A6): SSEP opens a span that sees from its own start; PDEP (and what follows) sees from 0
    if (tokens_host[lo] == p->ssep) cur_lo = lo;
    else if (tokens_host[lo] == p->pdep) cur_lo = 0;
    for (int t = lo; t < hi; ++t) q_vis_lo_out[t] = cur_lo;
    int blk = -1;
    if (i < (int)hs.size()) {
      auto it = p->by_hash.find(hs[i]);
      if (it != p->by_hash.end()) blk = it->second;
    }
    if (blk >= 0) {   // cache hit: nothing to write
      if (p->in_lru[blk]) { p->lru.erase(p->lru_it[blk]); p->in_lru[blk] = 0; }
      ++p->refs[blk]; ++p->hits;
      block_table_out[i] = blk; hit_out[i] = 1;
      for (int t = lo; t < hi; ++t) slot_mapping_out[t] = -1;
      continue;
    }
    blk = p->take_block();
    if (blk < 0) {   // out of blocks: undo this request's references and report
      for (int k = 0; k < i; ++k) {
        const int b = block_table_out[k];
        if (--p->refs[b] == 0) { p->lru.push_back(b); p->lru_it[b] = std::prev(p->lru.end()); p->in_lru[b] = 1; }
      }
      return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
    }
    if (i < (int)hs.size()) { p->by_hash[hs[i]] = blk; p->hash_of[blk] = hs[i]; }
    p->refs[blk] = 1; ++p->misses;
    block_table_out[i] = blk; hit_out[i] = 0;
    for (int t = lo; t < hi; ++t) slot_mapping_out[t] = (int64_t)blk * B + (t - lo);
    n_new += hi - lo;
  }
  if (num_new_tokens_out) *num_new_tokens_out = n_new;
  return MINIPIC_OK;
}

int minipic_pool_release(minipic_pool* p, const int32_t* block_table_host, int32_t num_blocks) {
  if (!p || num_blocks < 0 || (num_blocks > 0 && !block_table_host)) return MINIPIC_ERR_INVALID_ARG;
  for (int i = 0; i < num_blocks; ++i) {
    const int b = block_table_host[i];
    if (b < 0 || b >= p->num_blocks || p->refs[b] <= 0) return MINIPIC_ERR_INVALID_ARG;
    if (--p->refs[b] == 0) {
      if (p->hash_of[b].empty()) p->free_list.push_back(b);          // an unhashed (partial) block cannot hit again
      else { p->lru.push_back(b); p->lru_it[b] = std::prev(p->lru.end()); p->in_lru[b] = 1; }
    }
  }
  return MINIPIC_OK;
}

void minipic_pool_stats(const minipic_pool* p, uint64_t* hits, uint64_t* misses, uint64_t* evictions, int32_t* free_blocks) {
  if (!p) return;
  if (hits) *hits = p->hits;
  if (misses) *misses = p->misses;
  if (evictions) *evictions = p->evictions;
  if (free_blocks) *free_blocks = (int32_t)(p->free_list.size() + p->lru.size());
}

}  // extern "C"
