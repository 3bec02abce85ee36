// extern "C" boundary of libminipic.so: argument validation, dispatch, host-buffer entry points.
// See include/minipic.h for the contract of every call.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "internal.h"

namespace minipic {

static std::atomic<uint64_t> g_launches{0};
static thread_local char g_cuda_err[256] = "";
static thread_local const char* g_variant = "";

void note_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }
void note_error(const char* what) { snprintf(g_cuda_err, sizeof(g_cuda_err), "%s", what); }
int current_sm_count() {   // SM count of the CURRENT device (cached per device ordinal)
  static std::atomic<int> cache[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  int sms = cache[dev].load(std::memory_order_relaxed);
  if (sms == 0) {
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
    cache[dev].store(sms, std::memory_order_relaxed);
  }
  return sms;
}
bool check_launch(const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) return true;
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  return false;
}

static int validate_cfg(const minipic_config* cfg) {
  if (!cfg) return MINIPIC_ERR_INVALID_ARG;
  if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->num_blocks <= 0) return MINIPIC_ERR_INVALID_ARG;
  if (cfg->num_q_heads % cfg->num_kv_heads) return MINIPIC_ERR_INVALID_ARG;
  if (!(cfg->rope_theta > 0.0)) return MINIPIC_ERR_INVALID_ARG;
  if (cfg->rope_table_len < 0 || (cfg->rope_table_len > 0 && !cfg->rope_table)) return MINIPIC_ERR_INVALID_ARG;
  if (cfg->block_size != kBlock) return MINIPIC_ERR_UNSUPPORTED;
  if (cfg->head_dim != 64 && cfg->head_dim != 128) return MINIPIC_ERR_UNSUPPORTED;
  if (cfg->dtype != MINIPIC_BF16 && cfg->dtype != MINIPIC_F32) return MINIPIC_ERR_UNSUPPORTED;
  return MINIPIC_OK;
}

static void make_rope(const minipic_config* cfg, RopeParams* rp) {
  const int half = cfg->head_dim / 2;
  const long double two_pi = 6.283185307179586476925286766559L;
  for (int i = 0; i < 64; ++i) rp->phase_inc[i] = 0;
  for (int i = 0; i < half; ++i) {
    // f_i = theta^(-2i/D) (reading A2); F_i = f_i / 2pi in 0.64 fixed point
    const long double f = powl((long double)cfg->rope_theta, -2.0L * (long double)i / (long double)cfg->head_dim);
    const long double turns = f / two_pi;  // in (0, 0.16]
    rp->phase_inc[i] = (unsigned long long)ldexpl(turns, 64);
  }
  rp->table = (const float2*)cfg->rope_table;
  rp->table_len = cfg->rope_table ? cfg->rope_table_len : 0;
  rp->half = half;
}

static void make_ctx(const minipic_config* cfg, void* stream, Ctx* c) {
  c->hq = cfg->num_q_heads; c->hkv = cfg->num_kv_heads; c->d = cfg->head_dim; c->group = c->hq / c->hkv;
  c->num_blocks = cfg->num_blocks; c->dtype = cfg->dtype; c->flags = cfg->flags;
  c->scale = cfg->softmax_scale > 0.f ? cfg->softmax_scale : (float)(1.0 / std::sqrt((double)cfg->head_dim));
  c->scale_log2 = (float)((double)c->scale * 1.4426950408889634);
  make_rope(cfg, &c->rope);
  for (int i = 0; i < 64; ++i) {
    const double f = i < cfg->head_dim / 2 ? std::pow(cfg->rope_theta, -2.0 * (double)i / (double)cfg->head_dim) : 0.0;
    c->rope_step_cos[i] = std::cos(f); c->rope_step_sin[i] = std::sin(f);
  }
  c->stream = (cudaStream_t)stream;
}

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
static inline int itemsize(const minipic_config* cfg) { return cfg->dtype == MINIPIC_BF16 ? 2 : 4; }

SplitPlan decode_split_plan(const Ctx& c, int num_seqs, int max_kv_len) {
  // Fixed-length splits (a multiple of 64 keys) so every CTA streams the same number of bytes; chosen from host
  // scalars only so that the grid has >= ~8 waves of (sequence, split) slices when the batch allows it (swept 3..16 on
  // config 4: 1.15 / 1.15 / 1.12 / 1.10 / 1.10 / 1.13 ms for 3 / 4 / 6 / 8 / 12 / 16).
  SplitPlan sp;
  const int sms = current_sm_count();
  const long long want_ctas = (long long)sms * 2 * 8;
  long long per_seq = (want_ctas + num_seqs - 1) / (num_seqs > 0 ? num_seqs : 1);
  if (per_seq < 1) per_seq = 1;
  long long len = (max_kv_len + per_seq - 1) / per_seq;
  len = (len + 63) / 64 * 64;
  if (len < 256) len = 256;
  if (len > 2048) len = 2048;
  sp.split_len = (int)len;
  sp.max_splits = max_kv_len > 0 ? (max_kv_len + sp.split_len - 1) / sp.split_len : 1;
  return sp;
}
size_t decode_workspace_bytes(const Ctx& c, int num_seqs, int max_kv_len) {
  const SplitPlan sp = decode_split_plan(c, num_seqs, max_kv_len);
  const size_t rows = (size_t)num_seqs * c.hq * sp.max_splits;
  return align_up(rows * c.d * sizeof(float)) + align_up(rows * sizeof(float));
}

}  // namespace minipic

using namespace minipic;

extern "C" {

const char* minipic_status_string(int status) {
  switch (status) {
    case MINIPIC_OK: return "MINIPIC_OK";
    case MINIPIC_ERR_INVALID_ARG: return "MINIPIC_ERR_INVALID_ARG";
    case MINIPIC_ERR_UNSUPPORTED: return "MINIPIC_ERR_UNSUPPORTED";
    case MINIPIC_ERR_WORKSPACE_TOO_SMALL: return "MINIPIC_ERR_WORKSPACE_TOO_SMALL";
    case MINIPIC_ERR_CUDA: return "MINIPIC_ERR_CUDA";
    case MINIPIC_ERR_KERNEL_TIMEOUT: return "MINIPIC_ERR_KERNEL_TIMEOUT";
    default: return "MINIPIC_ERR_UNKNOWN";
  }
}
const char* minipic_last_cuda_error(void) { return g_cuda_err; }
uint64_t minipic_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
const char* minipic_last_variant(void) { return g_variant; }

int minipic_prefill_status(const void* workspace, void* cuda_stream) {
  if (!workspace) return MINIPIC_ERR_INVALID_ARG;
  // the health word lives in the workspace header, tagged by the kernel that keeps one: the answer does not depend on
  // which thread asks or on what this thread called in between
  int word = 0;
  const int e = prefill_sm100_error_word(workspace, (cudaStream_t)cuda_stream, &word);
  if (e != 0) { std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s", cudaGetErrorString((cudaError_t)e)); return MINIPIC_ERR_CUDA; }
  return word == 0 ? MINIPIC_OK : MINIPIC_ERR_KERNEL_TIMEOUT;
}

size_t minipic_rope_table_bytes(const minipic_config* cfg, int32_t num_positions) {
  if (validate_cfg(cfg) != MINIPIC_OK || num_positions < 0) return 0;
  return (size_t)num_positions * (cfg->head_dim / 2) * sizeof(float2);
}
int minipic_rope_table_build(const minipic_config* cfg, int32_t num_positions, void* table, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_positions < 0 || (num_positions > 0 && !table)) return MINIPIC_ERR_INVALID_ARG;
  RopeParams rp;
  make_rope(cfg, &rp);
  rp.table = nullptr; rp.table_len = 0;
  launch_rope_table(rp, num_positions, (float2*)table, (cudaStream_t)cuda_stream);
  return check_launch("rope_table") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

int minipic_cache_write(const minipic_config* cfg, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                        int32_t num_tokens, void* k_cache, void* v_cache, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_tokens < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_tokens == 0) return MINIPIC_OK;
  if (!k_new || !v_new || !slot_mapping || !k_cache || !v_cache) return MINIPIC_ERR_INVALID_ARG;
  if (((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)k_cache | (uintptr_t)v_cache) & 15) return MINIPIC_ERR_INVALID_ARG;
  launch_cache_write(itemsize(cfg), cfg->num_kv_heads, cfg->head_dim, k_new, v_new, slot_mapping, num_tokens, k_cache,
                     v_cache, (cudaStream_t)cuda_stream);
  return check_launch("cache_write") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

int minipic_preattn_fused(const minipic_config* cfg, const void* qkv, const int64_t* slot_mapping, const int32_t* positions,
                          int32_t num_tokens, void* q_out, void* k_cache, void* v_cache, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_tokens < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_tokens == 0) return MINIPIC_OK;
  if (!qkv || !slot_mapping || !positions || !q_out || !k_cache || !v_cache) return MINIPIC_ERR_INVALID_ARG;
  if (((uintptr_t)qkv | (uintptr_t)q_out | (uintptr_t)k_cache | (uintptr_t)v_cache) & 15) return MINIPIC_ERR_INVALID_ARG;
  Ctx c; make_ctx(cfg, cuda_stream, &c);
  launch_preattn_fused(c, qkv, slot_mapping, positions, num_tokens, q_out, k_cache, v_cache);
  return check_launch("preattn_fused") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

int minipic_block_rerotate(const minipic_config* cfg, void* k_cache, void* v_cache, const int32_t* src_blocks,
                           const int32_t* dst_blocks, const int32_t* delta, int32_t num_pairs, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_pairs < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_pairs == 0) return MINIPIC_OK;
  if (!k_cache || !v_cache || !src_blocks || !dst_blocks || !delta) return MINIPIC_ERR_INVALID_ARG;
  if (((uintptr_t)k_cache | (uintptr_t)v_cache) & 15) return MINIPIC_ERR_INVALID_ARG;
  Ctx c; make_ctx(cfg, cuda_stream, &c);
  launch_block_rerotate(c, k_cache, v_cache, src_blocks, dst_blocks, delta, num_pairs);
  return check_launch("block_rerotate") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

size_t minipic_prefill_workspace_bytes(const minipic_config* cfg, int32_t num_reqs, int32_t num_q_tokens) {
  if (validate_cfg(cfg) != MINIPIC_OK || num_reqs < 0 || num_q_tokens < 0) return 0;
  Ctx c; make_ctx(cfg, nullptr, &c);
  size_t b = 256;
  if (prefill_sm100_supported(c)) b += prefill_sm100_workspace_bytes(c, num_reqs, num_q_tokens);
  return b;
}

int minipic_prefill_attention(const minipic_config* cfg, const void* q, const void* k_cache, const void* v_cache,
                              const int32_t* block_tables, int32_t max_blocks_per_req, const int32_t* cu_q_lens,
                              const int32_t* kv_lens, const int32_t* cu_kv_lens, const int32_t* kv_positions,
                              const int32_t* q_seq_idx, const int32_t* q_vis_lo, int32_t num_reqs, int32_t num_q_tokens,
                              int32_t max_kv_len, void* out, float* lse, void* workspace, size_t workspace_bytes,
                              void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_reqs < 0 || num_q_tokens < 0 || max_kv_len < 0 || max_blocks_per_req < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_q_tokens == 0 || num_reqs == 0) return MINIPIC_OK;
  if (!q || !k_cache || !v_cache || !block_tables || !cu_q_lens || !kv_lens || !cu_kv_lens || !kv_positions ||
      !q_seq_idx || !q_vis_lo || !out || !lse)
    return MINIPIC_ERR_INVALID_ARG;
  if ((long long)max_blocks_per_req * kBlock < max_kv_len) return MINIPIC_ERR_INVALID_ARG;
  if (((uintptr_t)q | (uintptr_t)k_cache | (uintptr_t)v_cache | (uintptr_t)out) & 15) return MINIPIC_ERR_INVALID_ARG;
  Ctx c; make_ctx(cfg, cuda_stream, &c);
  // required: the planning part.  minipic_prefill_workspace_bytes() asks for more on small inputs (partial rows of KV-range
  // splits); a caller that sized the workspace for a larger call simply runs those inputs unsplit.
  const size_t need = 256 + (prefill_sm100_supported(c) ? prefill_sm100_workspace_min_bytes(c, num_reqs, num_q_tokens) : 0);
  if (workspace_bytes < need || !workspace) return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
  if ((uintptr_t)workspace & 255) return MINIPIC_ERR_INVALID_ARG;
  PrefillArgs a{q, k_cache, v_cache, block_tables, max_blocks_per_req, cu_q_lens, kv_lens, cu_kv_lens, kv_positions,
                q_seq_idx, q_vis_lo, num_reqs, num_q_tokens, max_kv_len, out, lse, workspace, workspace_bytes};
  if (!(c.flags & MINIPIC_FORCE_SIMT) && prefill_sm100_supported(c)) {
    g_variant = "prefill_sm100_tcgen05";
    if (!launch_prefill_sm100(c, a)) return MINIPIC_ERR_CUDA;
  } else {
    g_variant = "prefill_simt";
    launch_prefill_simt(c, a);
  }
  return check_launch("prefill_attention") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

size_t minipic_decode_workspace_bytes(const minipic_config* cfg, int32_t num_seqs, int32_t max_kv_len) {
  if (validate_cfg(cfg) != MINIPIC_OK || num_seqs < 0 || max_kv_len < 0) return 0;
  Ctx c; make_ctx(cfg, nullptr, &c);
  return decode_workspace_bytes(c, num_seqs, max_kv_len);
}

int minipic_decode_attention(const minipic_config* cfg, const void* q, const void* k_cache, const void* v_cache,
                             const int32_t* block_tables, int32_t max_blocks_per_req, const int32_t* kv_lens,
                             const int32_t* cu_kv_lens, const int32_t* kv_positions, const int32_t* q_vis_lo,
                             int32_t num_seqs, int32_t max_kv_len, void* out, float* lse, void* workspace,
                             size_t workspace_bytes, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_seqs < 0 || max_kv_len < 0 || max_blocks_per_req < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_seqs == 0) return MINIPIC_OK;
  if (!q || !k_cache || !v_cache || !block_tables || !kv_lens || !cu_kv_lens || !kv_positions || !out || !lse)
    return MINIPIC_ERR_INVALID_ARG;
  if ((long long)max_blocks_per_req * kBlock < max_kv_len) return MINIPIC_ERR_INVALID_ARG;
  if (((uintptr_t)q | (uintptr_t)k_cache | (uintptr_t)v_cache | (uintptr_t)out) & 15) return MINIPIC_ERR_INVALID_ARG;
  Ctx c; make_ctx(cfg, cuda_stream, &c);
  const size_t need = decode_workspace_bytes(c, num_seqs, max_kv_len);
  if (workspace_bytes < need || !workspace) return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
  if ((uintptr_t)workspace & 255) return MINIPIC_ERR_INVALID_ARG;
  const SplitPlan sp = decode_split_plan(c, num_seqs, max_kv_len);
  if ((long long)num_seqs * sp.max_splits > 0x7fffffffLL) return MINIPIC_ERR_UNSUPPORTED;   // (sequence, split) is grid.x
  const size_t rows = (size_t)num_seqs * c.hq * sp.max_splits;
  float* o_part = (float*)workspace;
  float* lse_part = (float*)((char*)workspace + align_up(rows * c.d * sizeof(float)));
  DecodeArgs a{q, k_cache, v_cache, block_tables, max_blocks_per_req, kv_lens, cu_kv_lens, kv_positions, q_vis_lo,
               num_seqs, max_kv_len, out, lse, workspace, workspace_bytes};
  if (!(c.flags & MINIPIC_FORCE_SIMT) && decode_mma_supported(c)) {
    g_variant = "decode_mma";
    if (!launch_decode_mma(c, a, sp, o_part, lse_part)) return MINIPIC_ERR_CUDA;
  } else {
    g_variant = "decode_simt";
    launch_decode_simt(c, a, sp, o_part, lse_part);
  }
  if (!check_launch("decode_partial")) return MINIPIC_ERR_CUDA;
  launch_lse_merge(c, a, sp, o_part, lse_part);
  return check_launch("lse_merge") ? MINIPIC_OK : MINIPIC_ERR_CUDA;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ host-buffer steps
namespace {
struct Arena {
  char* base; size_t size; size_t off = 0; bool ok = true;
  void* take(size_t bytes) {
    size_t o = align_up(off);
    if (o + bytes > size) { ok = false; return nullptr; }
    off = o + bytes;
    return base + o;
  }
};
struct ArenaSizer {
  size_t off = 0;
  void take(size_t bytes) { off = align_up(off) + bytes; }
};
template <typename A>
void* up(A& ar, const void* host, size_t bytes, cudaStream_t s, bool* ok) {
  if (bytes == 0) return nullptr;
  void* d = ar.take(bytes);
  if (!d) { *ok = false; return nullptr; }
  if (cudaMemcpyAsync(d, host, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) *ok = false;
  return d;
}
// ---- chunked overlap of the prefill host step: Q goes up and out / lse come down in token-range chunks on two auxiliary
//      streams (forked from and joined back into the caller's stream), so that H2D of chunk i + 1, attention of chunk i and D2H
//      of chunk i - 1 run at the same time: the step is PCIe bound and the link is full duplex.
constexpr int kHostChunkMin = 8192, kHostChunksMax = 16;
int host_chunk_tokens(int num_q_tokens) {
  const int per = (num_q_tokens + kHostChunksMax - 1) / kHostChunksMax;
  return per > kHostChunkMin ? per : kHostChunkMin;
}
struct AuxStreams { cudaStream_t h2d = nullptr, d2h = nullptr; };
bool aux_streams(AuxStreams* out) {   // per device, created once
  static std::mutex mu;
  static AuxStreams per_dev[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
  std::lock_guard<std::mutex> lk(mu);
  AuxStreams& a = per_dev[dev];
  if (!a.h2d) {
    if (cudaStreamCreateWithFlags(&a.h2d, cudaStreamNonBlocking) != cudaSuccess) { a.h2d = nullptr; return false; }
    if (cudaStreamCreateWithFlags(&a.d2h, cudaStreamNonBlocking) != cudaSuccess) { cudaStreamDestroy(a.h2d); a.h2d = a.d2h = nullptr; return false; }
  }
  *out = a;
  return true;
}
// `to` waits for everything enqueued on `from` so far
bool stream_after(cudaStream_t to, cudaStream_t from) {
  cudaEvent_t e;
  if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return false;
  const bool ok = cudaEventRecord(e, from) == cudaSuccess && cudaStreamWaitEvent(to, e, 0) == cudaSuccess;
  cudaEventDestroy(e);   // released once the enqueued record / wait have completed
  return ok;
}
}  // namespace

extern "C" {

size_t minipic_prefill_host_arena_bytes(const minipic_config* cfg, int32_t num_reqs, int32_t num_q_tokens,
                                        int32_t num_new_tokens, int32_t max_blocks_per_req, int32_t total_kv_len) {
  if (validate_cfg(cfg) != MINIPIC_OK) return 0;
  const size_t is = itemsize(cfg), d = cfg->head_dim;
  ArenaSizer a;
  a.take((size_t)num_new_tokens * cfg->num_kv_heads * d * is); a.take((size_t)num_new_tokens * cfg->num_kv_heads * d * is);
  a.take((size_t)num_new_tokens * 8);
  a.take((size_t)num_q_tokens * cfg->num_q_heads * d * is);
  a.take((size_t)num_reqs * max_blocks_per_req * 4);
  a.take((size_t)(num_reqs + 1) * 4); a.take((size_t)num_reqs * 4); a.take((size_t)(num_reqs + 1) * 4);
  a.take((size_t)total_kv_len * 4); a.take((size_t)num_q_tokens * 4); a.take((size_t)num_q_tokens * 4);
  a.take((size_t)num_q_tokens * cfg->num_q_heads * d * is); a.take((size_t)num_q_tokens * cfg->num_q_heads * 4);
  const int chunk = host_chunk_tokens(num_q_tokens), n_chunks = num_q_tokens > 0 ? (num_q_tokens + chunk - 1) / chunk : 1;
  a.take(minipic_prefill_workspace_bytes(cfg, num_reqs, num_q_tokens < chunk ? num_q_tokens : chunk));
  a.take((size_t)n_chunks * (num_reqs + 1) * 4);   // cu_q_lens of every chunk, rebased to its first token
  return align_up(a.off) + 256;
}

int minipic_prefill_step_host(const minipic_config* cfg, const void* k_new_host, const void* v_new_host,
                              const int64_t* slot_mapping_host, int32_t num_new_tokens, const void* q_host, void* k_cache,
                              void* v_cache, const int32_t* block_tables_host, int32_t max_blocks_per_req,
                              const int32_t* cu_q_lens_host, const int32_t* kv_lens_host, const int32_t* cu_kv_lens_host,
                              const int32_t* kv_positions_host, const int32_t* q_seq_idx_host,
                              const int32_t* q_vis_lo_host, int32_t num_reqs, int32_t num_q_tokens, int32_t max_kv_len,
                              void* out_host, float* lse_host, void* arena, size_t arena_bytes, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_reqs <= 0 || num_q_tokens <= 0 || num_new_tokens < 0 || !arena || ((uintptr_t)arena & 255)) return MINIPIC_ERR_INVALID_ARG;
  if (!q_host || !cu_kv_lens_host || !out_host || !lse_host) return MINIPIC_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t is = itemsize(cfg), d = cfg->head_dim;
  const int total_kv = cu_kv_lens_host[num_reqs];
  Arena ar{(char*)arena, arena_bytes};
  bool ok = true;
  const size_t kvb = (size_t)num_new_tokens * cfg->num_kv_heads * d * is;
  void* dk = up(ar, k_new_host, kvb, s, &ok);
  void* dv = up(ar, v_new_host, kvb, s, &ok);
  void* dslots = up(ar, slot_mapping_host, (size_t)num_new_tokens * 8, s, &ok);
  const size_t qb = (size_t)num_q_tokens * cfg->num_q_heads * d * is;
  const size_t row_b = (size_t)cfg->num_q_heads * d * is;          // one query / output token
  char* dq = (char*)ar.take(qb);                                     // filled chunk by chunk below
  void* dbt = up(ar, block_tables_host, (size_t)num_reqs * max_blocks_per_req * 4, s, &ok);
  void* dcuq = up(ar, cu_q_lens_host, (size_t)(num_reqs + 1) * 4, s, &ok);
  void* dkvl = up(ar, kv_lens_host, (size_t)num_reqs * 4, s, &ok);
  void* dcukv = up(ar, cu_kv_lens_host, (size_t)(num_reqs + 1) * 4, s, &ok);
  void* dpos = up(ar, kv_positions_host, (size_t)total_kv * 4, s, &ok);
  void* didx = up(ar, q_seq_idx_host, (size_t)num_q_tokens * 4, s, &ok);
  void* dlo = up(ar, q_vis_lo_host, (size_t)num_q_tokens * 4, s, &ok);
  char* dout = (char*)ar.take(qb);
  float* dlse = (float*)ar.take((size_t)num_q_tokens * cfg->num_q_heads * 4);
  const int chunk = host_chunk_tokens(num_q_tokens), n_chunks = (num_q_tokens + chunk - 1) / chunk;
  const size_t wsb = minipic_prefill_workspace_bytes(cfg, num_reqs, num_q_tokens < chunk ? num_q_tokens : chunk);
  void* ws = ar.take(wsb);
  int* dcu_chunks = (int*)ar.take((size_t)n_chunks * (num_reqs + 1) * 4);
  if (!ar.ok || !dq || !dout || !dlse || !ws || !dcu_chunks) return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
  (void)dcuq;
  // ---- token-range chunks: chunk i = query tokens [t0, t1) and the requests r0 .. r1 - 1 they belong to; its cu_q_lens are
  //      the global ones clipped to the range and rebased to t0.  Rows are independent, so any cut is legal.
  struct Chunk { int t0, t1, r0, nr; };
  std::vector<Chunk> chunks;
  std::vector<int> cu_host;
  {
    int r = 0;
    for (int i = 0; i < n_chunks; ++i) {
      Chunk c{i * chunk, std::min(num_q_tokens, (i + 1) * chunk), 0, 0};
      while (r + 1 < num_reqs && cu_q_lens_host[r + 1] <= c.t0) ++r;
      c.r0 = r;
      int r1 = r;
      while (r1 < num_reqs && cu_q_lens_host[r1] < c.t1) ++r1;
      c.nr = r1 - c.r0;
      for (int k = 0; k <= c.nr; ++k) cu_host.push_back(std::min(std::max(cu_q_lens_host[c.r0 + k] - c.t0, 0), c.t1 - c.t0));
      cu_host.resize((size_t)(i + 1) * (num_reqs + 1), c.t1 - c.t0);
      chunks.push_back(c);
    }
  }
  // pageable source: the driver stages it before the call returns, the vector may go
  if (cudaMemcpyAsync(dcu_chunks, cu_host.data(), cu_host.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) ok = false;
  if (!ok) { check_launch("h2d"); return MINIPIC_ERR_CUDA; }
  if (num_new_tokens) {
    st = minipic_cache_write(cfg, dk, dv, (const int64_t*)dslots, num_new_tokens, k_cache, v_cache, cuda_stream);
    if (st != MINIPIC_OK) return st;
  }
  AuxStreams aux;
  const bool overlap = n_chunks > 1 && aux_streams(&aux);
  cudaStream_t s_in = overlap ? aux.h2d : s, s_out = overlap ? aux.d2h : s;
  if (overlap && !stream_after(s_in, s)) return MINIPIC_ERR_CUDA;   // the arena may still be in use by earlier work on s
  if (overlap && !stream_after(s_out, s)) return MINIPIC_ERR_CUDA;
  std::vector<cudaEvent_t> landed(n_chunks, nullptr);
  bool cuda_ok = true;
  for (int i = 0; i < n_chunks && cuda_ok; ++i) {   // all uploads are enqueued first: the copy engine never waits for compute
    const Chunk& c = chunks[i];
    cuda_ok = cudaMemcpyAsync(dq + (size_t)c.t0 * row_b, (const char*)q_host + (size_t)c.t0 * row_b, (size_t)(c.t1 - c.t0) * row_b,
                              cudaMemcpyHostToDevice, s_in) == cudaSuccess;
    if (overlap && cuda_ok)
      cuda_ok = cudaEventCreateWithFlags(&landed[i], cudaEventDisableTiming) == cudaSuccess && cudaEventRecord(landed[i], s_in) == cudaSuccess;
  }
  for (int i = 0; i < n_chunks && cuda_ok && st == MINIPIC_OK; ++i) {
    const Chunk& c = chunks[i];
    const int nt = c.t1 - c.t0;
    if (overlap) cuda_ok = cudaStreamWaitEvent(s, landed[i], 0) == cudaSuccess;
    if (!cuda_ok) break;
    st = minipic_prefill_attention(cfg, dq + (size_t)c.t0 * row_b, k_cache, v_cache, (const int*)dbt + (size_t)c.r0 * max_blocks_per_req,
                                   max_blocks_per_req, dcu_chunks + (size_t)i * (num_reqs + 1), (const int*)dkvl + c.r0,
                                   (const int*)dcukv + c.r0, (const int*)dpos, (const int*)didx + c.t0, (const int*)dlo + c.t0, c.nr, nt,
                                   max_kv_len, dout + (size_t)c.t0 * row_b, dlse + (size_t)c.t0 * cfg->num_q_heads, ws, wsb, cuda_stream);
    if (st != MINIPIC_OK) break;
    if (overlap) cuda_ok = stream_after(s_out, s);
    cuda_ok = cuda_ok &&
              cudaMemcpyAsync((char*)out_host + (size_t)c.t0 * row_b, dout + (size_t)c.t0 * row_b, (size_t)nt * row_b, cudaMemcpyDeviceToHost, s_out) == cudaSuccess &&
              cudaMemcpyAsync(lse_host + (size_t)c.t0 * cfg->num_q_heads, dlse + (size_t)c.t0 * cfg->num_q_heads,
                              (size_t)nt * cfg->num_q_heads * 4, cudaMemcpyDeviceToHost, s_out) == cudaSuccess;
  }
  for (cudaEvent_t e : landed) if (e) cudaEventDestroy(e);
  if (overlap) {   // join: the caller's stream has drained only when every copy has
    if (!stream_after(s, s_in) || !stream_after(s, s_out)) cuda_ok = false;
  }
  if (st != MINIPIC_OK) return st;
  if (!cuda_ok) { check_launch("host step copies"); return MINIPIC_ERR_CUDA; }
  return MINIPIC_OK;
}

size_t minipic_decode_host_arena_bytes(const minipic_config* cfg, int32_t num_seqs, int32_t num_new_tokens,
                                       int32_t max_blocks_per_req, int32_t total_kv_len, int32_t max_kv_len) {
  if (validate_cfg(cfg) != MINIPIC_OK) return 0;
  const size_t is = itemsize(cfg), d = cfg->head_dim;
  ArenaSizer a;
  a.take((size_t)num_new_tokens * cfg->num_kv_heads * d * is); a.take((size_t)num_new_tokens * cfg->num_kv_heads * d * is);
  a.take((size_t)num_new_tokens * 8);
  a.take((size_t)num_seqs * cfg->num_q_heads * d * is);
  a.take((size_t)num_seqs * max_blocks_per_req * 4);
  a.take((size_t)num_seqs * 4); a.take((size_t)(num_seqs + 1) * 4); a.take((size_t)total_kv_len * 4); a.take((size_t)num_seqs * 4);
  a.take((size_t)num_seqs * cfg->num_q_heads * d * is); a.take((size_t)num_seqs * cfg->num_q_heads * 4);
  a.take(minipic_decode_workspace_bytes(cfg, num_seqs, max_kv_len));
  return align_up(a.off) + 256;
}

int minipic_decode_step_host(const minipic_config* cfg, const void* k_new_host, const void* v_new_host,
                             const int64_t* slot_mapping_host, int32_t num_new_tokens, const void* q_host, void* k_cache,
                             void* v_cache, const int32_t* block_tables_host, int32_t max_blocks_per_req,
                             const int32_t* kv_lens_host, const int32_t* cu_kv_lens_host, const int32_t* kv_positions_host,
                             const int32_t* q_vis_lo_host, int32_t num_seqs, int32_t max_kv_len, void* out_host,
                             float* lse_host, void* arena, size_t arena_bytes, void* cuda_stream) {
  int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_seqs <= 0 || num_new_tokens < 0 || !arena || ((uintptr_t)arena & 255)) return MINIPIC_ERR_INVALID_ARG;
  if (!q_host || !cu_kv_lens_host || !out_host || !lse_host) return MINIPIC_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t is = itemsize(cfg), d = cfg->head_dim;
  const int total_kv = cu_kv_lens_host[num_seqs];
  Arena ar{(char*)arena, arena_bytes};
  bool ok = true;
  const size_t kvb = (size_t)num_new_tokens * cfg->num_kv_heads * d * is;
  void* dk = up(ar, k_new_host, kvb, s, &ok);
  void* dv = up(ar, v_new_host, kvb, s, &ok);
  void* dslots = up(ar, slot_mapping_host, (size_t)num_new_tokens * 8, s, &ok);
  const size_t qb = (size_t)num_seqs * cfg->num_q_heads * d * is;
  void* dq = up(ar, q_host, qb, s, &ok);
  void* dbt = up(ar, block_tables_host, (size_t)num_seqs * max_blocks_per_req * 4, s, &ok);
  void* dkvl = up(ar, kv_lens_host, (size_t)num_seqs * 4, s, &ok);
  void* dcukv = up(ar, cu_kv_lens_host, (size_t)(num_seqs + 1) * 4, s, &ok);
  void* dpos = up(ar, kv_positions_host, (size_t)total_kv * 4, s, &ok);
  void* dlo = q_vis_lo_host ? up(ar, q_vis_lo_host, (size_t)num_seqs * 4, s, &ok) : nullptr;
  void* dout = ar.take(qb);
  float* dlse = (float*)ar.take((size_t)num_seqs * cfg->num_q_heads * 4);
  const size_t wsb = minipic_decode_workspace_bytes(cfg, num_seqs, max_kv_len);
  void* ws = ar.take(wsb);
  if (!ar.ok || !dout || !dlse || !ws) return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
  if (!ok) { check_launch("h2d"); return MINIPIC_ERR_CUDA; }
  if (num_new_tokens) {
    st = minipic_cache_write(cfg, dk, dv, (const int64_t*)dslots, num_new_tokens, k_cache, v_cache, cuda_stream);
    if (st != MINIPIC_OK) return st;
  }
  st = minipic_decode_attention(cfg, dq, k_cache, v_cache, (const int*)dbt, max_blocks_per_req, (const int*)dkvl,
                                (const int*)dcukv, (const int*)dpos, (const int*)dlo, num_seqs, max_kv_len, dout, dlse, ws,
                                wsb, cuda_stream);
  if (st != MINIPIC_OK) return st;
  if (cudaMemcpyAsync(out_host, dout, qb, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaMemcpyAsync(lse_host, dlse, (size_t)num_seqs * cfg->num_q_heads * 4, cudaMemcpyDeviceToHost, s) != cudaSuccess) {
    check_launch("d2h");
    return MINIPIC_ERR_CUDA;
  }
  return MINIPIC_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ decode without a workspace
// The split-KV partials of minipic_decode_attention_static live in this file-scope device array.  In HOST code the name is a
// host-side stand-in, not a device address: the address is looked up per device with cudaGetSymbolAddress (below).
namespace {
static __device__ __align__(256) unsigned char g_static_scratch[MINIPIC_STATIC_SCRATCH_BYTES];

// device address of g_static_scratch on the CURRENT device; looked up once per device ordinal
void* static_scratch_ptr() {
  static std::mutex mu;
  static void* per_dev[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
    note_error("minipic_decode_attention_static: cudaGetDevice failed or device ordinal >= 64");
    return nullptr;
  }
  std::lock_guard<std::mutex> lk(mu);
  if (!per_dev[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      char msg[200];
      snprintf(msg, sizeof(msg), "minipic_decode_attention_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
      note_error(msg);
      return nullptr;
    }
    per_dev[dev] = p;
  }
  return per_dev[dev];
}
}  // namespace

extern "C" {

size_t minipic_static_scratch_bytes(void) { return (size_t)MINIPIC_STATIC_SCRATCH_BYTES; }

int minipic_decode_attention_static(const minipic_config* cfg, const void* q, const void* k_cache, const void* v_cache,
                                    const int32_t* block_tables, int32_t max_blocks_per_req, const int32_t* kv_lens,
                                    const int32_t* cu_kv_lens, const int32_t* kv_positions, const int32_t* q_vis_lo,
                                    int32_t num_seqs, int32_t max_kv_len, void* out, float* lse, void* cuda_stream) {
  const int st = validate_cfg(cfg);
  if (st != MINIPIC_OK) return st;
  if (num_seqs < 0 || max_kv_len < 0 || max_blocks_per_req < 0) return MINIPIC_ERR_INVALID_ARG;
  if (num_seqs == 0) return MINIPIC_OK;
  Ctx c; make_ctx(cfg, cuda_stream, &c);
  const size_t need = decode_workspace_bytes(c, num_seqs, max_kv_len);
  if (need > (size_t)MINIPIC_STATIC_SCRATCH_BYTES) {   // before anything is launched or any pointer is looked at
    char msg[200];
    snprintf(msg, sizeof(msg), "minipic_decode_attention_static: %zu bytes of split-KV partials needed, the static scratch holds %zu",
             need, (size_t)MINIPIC_STATIC_SCRATCH_BYTES);
    note_error(msg);
    return MINIPIC_ERR_WORKSPACE_TOO_SMALL;
  }
  void* scratch = static_scratch_ptr();
  if (!scratch) return MINIPIC_ERR_CUDA;
  return minipic_decode_attention(cfg, q, k_cache, v_cache, block_tables, max_blocks_per_req, kv_lens, cu_kv_lens, kv_positions,
                                  q_vis_lo, num_seqs, max_kv_len, out, lse, scratch, (size_t)MINIPIC_STATIC_SCRATCH_BYTES, cuda_stream);
}

}  // extern "C"
