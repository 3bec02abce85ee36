/*
 * minipic.h - C ABI of the MiniPIC hot path for NVIDIA B200 (sm_100a).
 *
 * Paged attention over a position-encoding-free KV cache (arxiv/paper_2606_13126, "MiniPIC";
 * citations below are PAPER.md:<line>):
 *
 *   - keys are stored UNROTATED in fixed-size physical blocks shared across requests
 *     (PAPER.md:14, :47, :100, :105);
 *   - RoPE is applied to every K tile inside the attention kernel at the request's per-token
 *     logical position pi(j); Q is rotated at its own logical position
 *     (Eq. 2:  score(t,j) = (R_t q_t)^T (R_pi(j) k~_j) / sqrt(d));
 *   - scores are masked by the block-level causal structure the span primitives induce
 *     (PAPER.md:57, :90, :123-128, :143): query row t sees sequence index j iff
 *     q_vis_lo[t] <= j <= q_seq_idx[t]  (span token: vis_lo = first index of its span;
 *     system / suffix token: vis_lo = 0).
 *
 * Conventions (every entry point):
 *   * All array arguments are DEVICE pointers owned by the caller unless the name ends in
 *     `_host` (see the *_host entry points at the end).  The library allocates nothing on the
 *     device path, keeps no state between calls (beyond the diagnostics at the end of this file: a launch counter
 *     and per-thread last-error / last-variant strings) and never synchronises the stream.
 *   * `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   * The return value is a minipic_status.  Argument errors are detected on the host before
 *     any launch.  Out-of-range block ids / slots / positions are undefined behaviour.
 *   * Layouts (row-major, innermost last):
 *       k_cache, v_cache : [num_blocks, num_kv_heads, block_size, head_dim]   (library-defined;
 *                          one (block, head) is one contiguous 16*head_dim*sizeof chunk)
 *       k_new, v_new, q, out : [tokens, heads, head_dim]
 *       lse              : float32 [tokens, num_q_heads], natural log of the sum of exp of the
 *                          SCALED scores over the visible keys
 *       block_tables     : int32 [num_reqs, max_blocks_per_req]; sequence index j of request r
 *                          lives in block block_tables[r][j / block_size], row j % block_size
 *       kv_positions     : int32 [sum kv_lens]; kv_positions[cu_kv_lens[r] + j] = pi_r(j) >= 0
 *   * Causality is by SEQUENCE INDEX, RoPE by LOGICAL POSITION ("position exists only
 *     as per-request metadata consumed inside attention").
 *   * The same physical block id may appear in many block tables and several times in one
 *     (PAPER.md:145, :232): attention only reads the caches.
 *   * A query row with no visible key returns out = 0, lse = -inf.
 *   * Supported: block_size 16; head_dim 64 or 128; num_q_heads % num_kv_heads == 0;
 *     dtype bf16 or f32 (q, k, v, caches and out share it).  Anything else returns
 *     MINIPIC_ERR_UNSUPPORTED.  There is no CPU fallback.
 */
#ifndef MINIPIC_H_
#define MINIPIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  MINIPIC_OK = 0,
  MINIPIC_ERR_INVALID_ARG = 1,
  MINIPIC_ERR_UNSUPPORTED = 2,
  MINIPIC_ERR_WORKSPACE_TOO_SMALL = 3,
  MINIPIC_ERR_CUDA = 4,
  MINIPIC_ERR_KERNEL_TIMEOUT = 5 /* a hand-off barrier inside the prefill kernel was never signalled (internal fault) */
} minipic_status;

typedef enum { MINIPIC_BF16 = 0, MINIPIC_F32 = 1 } minipic_dtype;

enum {
  MINIPIC_Q_PREROTATED = 1u, /* caller already applied R(pos) to Q (the paper's own flow) */
  MINIPIC_K_PREROTATED = 2u, /* CONTROL ONLY: the cache holds rotated K, kernels skip the K RoPE step   */
  MINIPIC_FORCE_SIMT   = 4u, /* DEBUG: run the generic fp32 CUDA-core attention kernels instead of the  */
                             /* tensor-core ones (bf16, head_dim 128 normally take the latter)          */
  MINIPIC_KEY_MASK     = 8u  /* mask variant for marker / padding tokens (the "key-vector zeroing" that */
                             /* PAPER.md:294 defers): a key with kv_positions[...] < 0 is invisible to  */
                             /* EVERY query row of its request (as if it were deleted from the sequence; */
                             /* sequence indices, q_seq_idx and q_vis_lo are unchanged).  Without the    */
                             /* flag positions must be >= 0.  A row that queries AT a masked index has   */
                             /* undefined output (such rows are discarded by the caller).               */
};

typedef struct {
  int32_t num_q_heads;   /* Hq                                                     */
  int32_t num_kv_heads;  /* Hkv, divides Hq (GQA group G = Hq / Hkv)               */
  int32_t head_dim;      /* D: 64 or 128                                           */
  int32_t block_size;    /* 16                                      */
  int32_t num_blocks;    /* physical pool size                                     */
  int32_t dtype;         /* minipic_dtype of q, k, v, caches, out                  */
  double  rope_theta;    /* RoPE base; f_i = theta^(-2i/D), rotate-half pairing    */
  float   softmax_scale; /* 0 => 1/sqrt(head_dim) (Eq. 2)                          */
  uint32_t flags;        /* MINIPIC_* bits                                         */
  /* Optional cos/sin table ("a cos/sin table lookup"): device float2
   * [rope_table_len][head_dim/2] = (cos, sin)(p * f_i), built by minipic_rope_table_build for this
   * (rope_theta, head_dim).  It is read ONLY by the generic fp32 CUDA-core kernels (fp32 I/O, head_dim 64,
   * MINIPIC_FORCE_SIMT); positions >= rope_table_len (or a NULL table) are computed there from a 64-bit
   * fixed-point phase to the same accuracy (~2e-7).  The bf16 tensor-core kernels (head_dim 128) IGNORE the
   * table: they always compute the phase in-kernel (a table read per K tile would cost as much on-chip
   * traffic as the tile itself), so callers of those shapes need not build one. */
  const void* rope_table;
  int32_t rope_table_len;
  int32_t reserved;
} minipic_config;

/* ---- a0: RoPE table (optional accelerator; not needed for correctness) ------------------------
 * Fills table[p][i] = (cos(p f_i), sin(p f_i)), p in [0, num_positions), i in [0, head_dim/2),
 * evaluated in fp64 on the device and rounded once to fp32.  Bytes = num_positions*head_dim/2*8. */
size_t minipic_rope_table_bytes(const minipic_config* cfg, int32_t num_positions);
int minipic_rope_table_build(const minipic_config* cfg, int32_t num_positions, void* table, void* cuda_stream);

/* ---- a1: paged cache write ("V vectors are unchanged" :113) -----------------
 * cache[slot / B, h, slot % B, :] = new[t, h, :] for every token t with slot_mapping[t] >= 0.
 * Raw byte copy: no rotation, no conversion - bit exact.  slot < 0 => the token is skipped.
 * Duplicate slots in one call are a caller error (undefined winner).  The caller orders this before
 * attention on the same stream. */
int minipic_cache_write(const minipic_config* cfg,
                        const void* k_new, const void* v_new,   /* [num_tokens, Hkv, D]            */
                        const int64_t* slot_mapping,            /* [num_tokens], block*B + offset  */
                        int32_t num_tokens,
                        void* k_cache, void* v_cache, void* cuda_stream);

/* ---- f1: fused pre-attention step ("rotated once by the model's RotaryEmbedding layer ... stores
 * unrotated key vectors"; Table 2 row rotary_embedding/base.py) ---------------------------------
 * ONE pass over the QKV-projection output of the new tokens, qkv [num_tokens, Hq + 2 Hkv, D] (heads [0, Hq) = Q,
 * [Hq, Hq + Hkv) = K, the rest V), instead of a rotary kernel over Q plus minipic_cache_write:
 *   k_cache / v_cache[slot / B, h, slot % B, :] = K / V rows of token t, raw byte copy (bit exact, slot < 0: skipped);
 *   q_out[t, h] = R(positions[t]) q[t, h], rotated in fp32 and rounded ONCE to the I/O dtype - the paper's own flow:
 *                 pass q_out to the attention calls with MINIPIC_Q_PREROTATED.  If cfg->flags has
 *                 MINIPIC_Q_PREROTATED the rows are copied unrotated.
 * positions: int32 [num_tokens], the tokens' logical positions (>= 0).  q_out: [num_tokens, Hq, D], must not overlap qkv. */
int minipic_preattn_fused(const minipic_config* cfg, const void* qkv, const int64_t* slot_mapping,
                          const int32_t* positions, int32_t num_tokens, void* q_out,
                          void* k_cache, void* v_cache, void* cuda_stream);

/* ---- f4: copy-and-re-rotate CONTROL ("block-by-block copy and repositioning"; App. A :284-286) ------
 * What a POSITION-DEPENDENT cache must do to reuse a span at another offset; MiniPIC never needs it (its blocks hold
 * unrotated keys) - it exists to measure the HBM traffic the position-free layout avoids.  For every i < num_pairs:
 *   k_cache[dst_blocks[i]] = R(delta[i]) k_cache[src_blocks[i]]  (all heads, all 16 rows; fp32 rotation, one RN),
 *   v_cache[dst_blocks[i]] = v_cache[src_blocks[i]]               (bit exact).
 * delta may be negative.  No block id may appear both as a source and as a destination in one call, destinations must
 * be distinct. */
int minipic_block_rerotate(const minipic_config* cfg, void* k_cache, void* v_cache, const int32_t* src_blocks,
                           const int32_t* dst_blocks, const int32_t* delta, int32_t num_pairs, void* cuda_stream);

/* ---- a2-a9: prefill attention (PAPER.md:100-113, Eq. 2; mask :57, :90, :123-128, :143) ---------
 * For every query row t of request r (rows cu_q_lens[r] .. cu_q_lens[r+1]) and head h:
 *   q' = R(pi_r(q_seq_idx[t])) q[t,h]      (skipped under MINIPIC_Q_PREROTATED)
 *   k_j = R(pi_r(j)) k~_j  gathered through block_tables[r]   (skipped under MINIPIC_K_PREROTATED)
 *   out[t,h] = softmax_j(q'.k_j * scale) V_j over q_vis_lo[t] <= j <= q_seq_idx[t];  lse[t,h].
 * Requires q_seq_idx[t] < kv_lens[r].  workspace: device scratch, 256-byte aligned; contents are overwritten.
 * minipic_prefill_workspace_bytes(...) bytes are always enough.  On small inputs (a few requests' questions over long
 * cached contexts) that figure includes up to 64 MiB for the partial rows of KV-RANGE SPLITS: an item whose KV range is too
 * long for a balanced grid is cut into chunks that run on different CTA pairs and are merged by a second kernel (same
 * result up to fp32 rounding order).  A workspace sized for a LARGER call (more tokens) is accepted for a smaller one: the
 * call then needs only the planning part and runs without splits.  Smaller than that: MINIPIC_ERR_WORKSPACE_TOO_SMALL. */
size_t minipic_prefill_workspace_bytes(const minipic_config* cfg, int32_t num_reqs, int32_t num_q_tokens);
int minipic_prefill_attention(const minipic_config* cfg,
                              const void* q,                    /* [Tq, Hq, D]                       */
                              const void* k_cache, const void* v_cache,
                              const int32_t* block_tables, int32_t max_blocks_per_req,
                              const int32_t* cu_q_lens,         /* [R+1]                             */
                              const int32_t* kv_lens,           /* [R]                               */
                              const int32_t* cu_kv_lens,        /* [R+1] offsets into kv_positions   */
                              const int32_t* kv_positions,      /* [sum kv_lens]                     */
                              const int32_t* q_seq_idx,         /* [Tq] sequence index of the query  */
                              const int32_t* q_vis_lo,          /* [Tq] lowest visible sequence idx  */
                              int32_t num_reqs, int32_t num_q_tokens, int32_t max_kv_len,
                              void* out, float* lse,            /* [Tq,Hq,D], [Tq,Hq]                */
                              void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- a10-a11: decode attention = split-KV partial kernel + LSE-merge kernel ------
 * One query per sequence, sitting at sequence index kv_lens[r]-1 (its K/V must already be in the
 * cache).  q_vis_lo may be NULL (=> 0).  Partials (o_s normalised over its split, lse_s) go to the
 * workspace and are merged by  lse = ln sum_s e^{lse_s},  o = sum_s e^{lse_s - lse} o_s. */
size_t minipic_decode_workspace_bytes(const minipic_config* cfg, int32_t num_seqs, int32_t max_kv_len);
int minipic_decode_attention(const minipic_config* cfg,
                             const void* q,                     /* [R, Hq, D]                        */
                             const void* k_cache, const void* v_cache,
                             const int32_t* block_tables, int32_t max_blocks_per_req,
                             const int32_t* kv_lens, const int32_t* cu_kv_lens, const int32_t* kv_positions,
                             const int32_t* q_vis_lo,           /* [R] or NULL                       */
                             int32_t num_seqs, int32_t max_kv_len,
                             void* out, float* lse, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- decode attention WITHOUT a caller workspace and without any allocation -------------------------------------
 * Same computation, arguments and result as minipic_decode_attention (Eq. 2), for callers that cannot
 * allocate device memory (code under CUDA graph capture, serving loops or harnesses that forbid cudaMalloc): the fp32
 * split-KV partials live in a file-scope static device array of MINIPIC_STATIC_SCRATCH_BYTES that every GPU which loads
 * the library holds until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree, no allocating library
 * routine); it looks the array's device address up once per device (cudaGetSymbolAddress) and enqueues the same kernels on
 * `cuda_stream`.
 *   - a problem that needs more than MINIPIC_STATIC_SCRATCH_BYTES of partials (minipic_decode_workspace_bytes says how
 *     much) is rejected with MINIPIC_ERR_WORKSPACE_TOO_SMALL and a message in minipic_last_cuda_error(); nothing is launched;
 *   - ALL calls on a device share the one array: two calls that overlap on the GPU (different streams, or concurrent graph
 *     branches) race on it - serialise them.  The array keeps the previous call's contents; nothing in it has to start at
 *     zero (a call writes every partial row that its merge kernel reads), so no clearing is done. */
#define MINIPIC_STATIC_SCRATCH_BYTES (16u << 20)
size_t minipic_static_scratch_bytes(void);   /* = MINIPIC_STATIC_SCRATCH_BYTES, for bindings without the macro */
int minipic_decode_attention_static(const minipic_config* cfg,
                                    const void* q, const void* k_cache, const void* v_cache,
                                    const int32_t* block_tables, int32_t max_blocks_per_req,
                                    const int32_t* kv_lens, const int32_t* cu_kv_lens,
                                    const int32_t* kv_positions, const int32_t* q_vis_lo /* or NULL */,
                                    int32_t num_seqs, int32_t max_kv_len,
                                    void* out, float* lse, void* cuda_stream);

/* ---- end-to-end entry points with HOST buffers ---------------------------------------------------
 * Same computation as cache_write followed by prefill / decode attention, but every per-step input
 * (new K/V rows, slot mapping, Q, index tables) is read from HOST memory and the result (out, lse)
 * is written to HOST memory; the resident KV cache stays on the device.  `arena` is caller-owned
 * DEVICE scratch of at least minipic_*_host_arena_bytes(...) bytes (256-byte aligned) that receives
 * the staged inputs, the workspace and the device-side result.  Copies and kernels are ordered by
 * `cuda_stream` (cudaMemcpyAsync: pin the host buffers for true asynchrony); the call does not
 * synchronise - outputs are valid once the stream has drained.  num_new_tokens may be 0.
 * The prefill step with more than 8192 query tokens runs as up to 16 token-range CHUNKS: Q goes up and
 * out / lse come down on two copy streams the library creates once per device (forked from and joined
 * back into `cuda_stream`), one attention call per chunk in between, so that the upload of chunk i + 1,
 * the attention of chunk i and the download of chunk i - 1 overlap (the step is PCIe bound and the link
 * is full duplex).  Rows are independent, so the cuts are invisible in the result up to rounding order. */
size_t minipic_prefill_host_arena_bytes(const minipic_config* cfg, int32_t num_reqs, int32_t num_q_tokens,
                                        int32_t num_new_tokens, int32_t max_blocks_per_req, int32_t total_kv_len);
int minipic_prefill_step_host(const minipic_config* cfg,
                              const void* k_new_host, const void* v_new_host, const int64_t* slot_mapping_host,
                              int32_t num_new_tokens,
                              const void* q_host,
                              void* k_cache, void* v_cache,     /* DEVICE */
                              const int32_t* block_tables_host, int32_t max_blocks_per_req,
                              const int32_t* cu_q_lens_host, const int32_t* kv_lens_host,
                              const int32_t* cu_kv_lens_host, const int32_t* kv_positions_host,
                              const int32_t* q_seq_idx_host, const int32_t* q_vis_lo_host,
                              int32_t num_reqs, int32_t num_q_tokens, int32_t max_kv_len,
                              void* out_host, float* lse_host,
                              void* arena, size_t arena_bytes, void* cuda_stream);

size_t minipic_decode_host_arena_bytes(const minipic_config* cfg, int32_t num_seqs, int32_t num_new_tokens,
                                       int32_t max_blocks_per_req, int32_t total_kv_len, int32_t max_kv_len);
int minipic_decode_step_host(const minipic_config* cfg,
                             const void* k_new_host, const void* v_new_host, const int64_t* slot_mapping_host,
                             int32_t num_new_tokens,
                             const void* q_host,
                             void* k_cache, void* v_cache,      /* DEVICE */
                             const int32_t* block_tables_host, int32_t max_blocks_per_req,
                             const int32_t* kv_lens_host, const int32_t* cu_kv_lens_host,
                             const int32_t* kv_positions_host, const int32_t* q_vis_lo_host /* or NULL */,
                             int32_t num_seqs, int32_t max_kv_len,
                             void* out_host, float* lse_host,
                             void* arena, size_t arena_bytes, void* cuda_stream);

/* Health of the last tcgen05 minipic_prefill_attention call that used `workspace` (DEVICE pointer, as passed to that call).
 * The tcgen05 prefill kernel is a pipeline of warp roles that hand tiles to each other through mbarriers; every wait is
 * bounded, and a wait that runs out records the barrier in the workspace header and drains the kernel instead of hanging
 * the GPU.  This call synchronises `cuda_stream`, reads the header's (error word, kernel tag) back and returns MINIPIC_OK,
 * MINIPIC_ERR_KERNEL_TIMEOUT (outputs of that call are then undefined) or MINIPIC_ERR_CUDA.  The state lives in the
 * workspace, not in the library: the answer is the same from any host thread and whatever was called in between.  The
 * other kernels keep no health word and never write the header; a workspace that no tcgen05 call has used reads as OK.
 * Optional: the attention calls themselves stay asynchronous. */
int minipic_prefill_status(const void* workspace, void* cuda_stream);

/* ---- f3: HOST-side block hasher and block pool (Eq. 1; request procedure :123-128) ----------------
 * The step before block tables exist.  Pure host code: every pointer below is a HOST pointer, nothing touches the GPU.
 *   h_i = H(h_0, x_i)      if block i STARTS WITH ssep_id   (SSEP: detached - the span hashes the same anywhere)
 *         H(h_0, x_{<=i})  if block i STARTS WITH pdep_id   (PDEP: depends on the whole prompt so far)
 *         H(h_{i-1}, x_i)  otherwise                        (the engine's ordinary chain; h_{-1} = h_0)
 * H = SHA-256(parent digest || tokens as little-endian int32), h_0 = SHA-256(seed as 8 little-endian bytes).
 * Only full blocks have a hash: hashes_out_host receives (num_tokens / block_size) digests of 32 bytes. */
int minipic_block_hashes(const int32_t* tokens_host, int32_t num_tokens, int32_t block_size, int32_t ssep_id,
                         int32_t pdep_id, uint64_t seed, uint8_t* hashes_out_host);

/* Block pool keyed by those digests (opaque host object, not thread safe; NULL on bad arguments). */
typedef struct minipic_pool minipic_pool;
minipic_pool* minipic_pool_create(int32_t num_blocks, int32_t block_size, int32_t ssep_id, int32_t pdep_id, uint64_t seed);
void minipic_pool_destroy(minipic_pool* pool);
/* Admit one request (a token stream, padded by the caller: PAPER.md:79).  For each of its ceil(n / B) blocks:
 *   a cached digest  -> block_table_out[i] = that block, hit_out[i] = 1, slot_mapping_out = -1 for its tokens;
 *   otherwise        -> a fresh block (free list in increasing id order, then the least recently released unreferenced
 *                       block, whose digest is forgotten), hit_out[i] = 0, slot_mapping_out[t] = block * B + offset -
 *                       exactly what minipic_cache_write / minipic_preattn_fused take for the tokens to be computed.
 * A trailing partial block is never cached.  q_vis_lo_out[t] is the visibility descriptor of the attention calls
 * (span token: first index of its SSEP block chain; before the first marker and from a PDEP block on: 0).
 * Every block of the table holds one reference until minipic_pool_release.  MINIPIC_ERR_WORKSPACE_TOO_SMALL if the pool
 * has no block left (the request's references are undone). */
int minipic_pool_admit(minipic_pool* pool, const int32_t* tokens_host, int32_t num_tokens, int32_t* block_table_out,
                       uint8_t* hit_out, int64_t* slot_mapping_out, int32_t* q_vis_lo_out, int32_t* num_new_tokens_out);
int minipic_pool_release(minipic_pool* pool, const int32_t* block_table_host, int32_t num_blocks);
void minipic_pool_stats(const minipic_pool* pool, uint64_t* hits, uint64_t* misses, uint64_t* evictions, int32_t* free_blocks);

/* ---- misc ---------------------------------------------------------------------------------------*/
const char* minipic_status_string(int status);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char* minipic_last_cuda_error(void);
/* Number of kernels the library has launched in this process since load (for bench accounting). */
uint64_t minipic_launch_count(void);
/* Name of the attention kernel variant the last prefill / decode call on this thread dispatched to
 * ("prefill_sm100_tcgen05", "prefill_simt", "decode_mma", "decode_simt", ...). */
const char* minipic_last_variant(void);

#ifdef __cplusplus
}
#endif
#endif /* MINIPIC_H_ */
