// Launcher declarations shared by the translation units of libminipic.so.
#pragma once
#include <cuda.h>

#include "common.cuh"

// decode (a10) launch shape: blocks in flight per warp and resident warps per SM (kStages * 8 KB of shared memory per warp)
#ifndef MINIPIC_DECODE_STAGES
#define MINIPIC_DECODE_STAGES 2
#endif
#ifndef MINIPIC_DECODE_WARPS_PER_SM
#define MINIPIC_DECODE_WARPS_PER_SM 12
#endif

namespace minipic {

// a0
void launch_rope_table(const RopeParams& rp, int num_positions, float2* table, cudaStream_t s);
// a1
void launch_cache_write(int itemsize, int hkv, int d, const void* k_new, const void* v_new, const int64_t* slots,
                        int num_tokens, void* k_cache, void* v_cache, cudaStream_t s);

// f1 / f4 (preattn.cu)
void launch_preattn_fused(const Ctx& c, const void* qkv, const int64_t* slots, const int* positions, int num_tokens,
                          void* q_out, void* k_cache, void* v_cache);
void launch_block_rerotate(const Ctx& c, void* k_cache, void* v_cache, const int* src, const int* dst, const int* delta,
                           int num_pairs);

struct PrefillArgs {
  const void* q; const void* k_cache; const void* v_cache;
  const int* block_tables; int max_blocks;
  const int* cu_q_lens; const int* kv_lens; const int* cu_kv_lens; const int* kv_positions;
  const int* q_seq_idx; const int* q_vis_lo;
  int num_reqs, num_q_tokens, max_kv_len;
  void* out; float* lse;
  void* workspace; size_t workspace_bytes;
};
struct DecodeArgs {
  const void* q; const void* k_cache; const void* v_cache;
  const int* block_tables; int max_blocks;
  const int* kv_lens; const int* cu_kv_lens; const int* kv_positions; const int* q_vis_lo;
  int num_seqs, max_kv_len;
  void* out; float* lse;
  void* workspace; size_t workspace_bytes;
};

// split-KV geometry, a pure function of host scalars (shared by workspace sizing and launch)
struct SplitPlan { int split_len; int max_splits; };
SplitPlan decode_split_plan(const Ctx& c, int num_seqs, int max_kv_len);
size_t decode_workspace_bytes(const Ctx& c, int num_seqs, int max_kv_len);

// generic fp32 CUDA-core kernels (any supported dtype / head_dim)
void launch_prefill_simt(const Ctx& c, const PrefillArgs& a);
void launch_decode_simt(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part);
// a11
void launch_lse_merge(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, const float* o_part, const float* lse_part);
// a10 tensor-core (mma.sync, register operands) split-KV kernel: bf16, D=128, G<=8
bool decode_mma_supported(const Ctx& c);
bool launch_decode_mma(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part);
// the paged cache as a 4-D bf16 tensor map whose box is one (block, head): 16 tokens x 128 dims land as
// [row group (2)][half of head_dim (halves)][8 rows x 128 B], SWIZZLE_128B (defined in prefill_sm100.cu)
bool make_cache_tensor_map(CUtensorMap* m, const void* cache, int num_blocks, int hkv, int halves);
// a2-a9 tcgen05 / TMEM / TMA prefill: bf16, D=128, G in {1,2,4,8}
bool prefill_sm100_supported(const Ctx& c);
size_t prefill_sm100_workspace_bytes(const Ctx& c, int num_reqs, int num_q_tokens);       // with room for KV-range splits
size_t prefill_sm100_workspace_min_bytes(const Ctx& c, int num_reqs, int num_q_tokens);   // what a call needs at least
bool launch_prefill_sm100(const Ctx& c, const PrefillArgs& a);
int prefill_sm100_error_word(const void* workspace, cudaStream_t s, int* word);   // cudaError as int; *word = 0 if healthy

}  // namespace minipic
