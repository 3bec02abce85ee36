// Generic CUDA-core attention kernels (fp32 math, any supported dtype / head_dim).
// They serve the fp32-I/O instantiation (BASELINE config 1), head_dim 64, GQA groups the tensor-core kernels do
// not cover, and MINIPIC_FORCE_SIMT.  One warp owns one (query row, query head): Eq. 2 is
// evaluated key by key - gather through the block table (:47-49), rotate K at pi(j) (:100-105), dot, online
// softmax (:111), PV.  The warp's lanes split head_dim; a lane holds both elements of every rotate-half pair.
#include "internal.h"

namespace minipic {

template <typename T, int D>
struct WarpAttn {
  static constexpr int E = D / 32;      // elements per lane: e = lane + 32*m
  static constexpr int HP = E / 2;      // rotate-half pairs per lane: (m, m + HP), frequency index lane + 32*m
  float q[E];
  float acc[E];
  float m_run, l_run;

  __device__ __forceinline__ void init(const T* qrow, const RopeParams& rp, int qpos, bool prerot, int lane) {
#pragma unroll
    for (int m = 0; m < E; ++m) { q[m] = IO<T>::load(qrow + lane + 32 * m); acc[m] = 0.f; }
    if (!prerot) {
#pragma unroll
      for (int m = 0; m < HP; ++m) {
        const float2 cs = rope_cs_precise(rp, qpos, lane + 32 * m);
        const float a = q[m], b = q[m + HP];
        q[m] = a * cs.x - b * cs.y;
        q[m + HP] = b * cs.x + a * cs.y;
      }
    }
    m_run = -INFINITY;
    l_run = 0.f;
  }

  // keys j in [j0, j1) of request with block table `bt`, positions `pos` (both already offset to the request)
  __device__ __forceinline__ void run(const T* kc, const T* vc, const int* bt, const int* pos, int hkv, int g,
                                      int j0, int j1, float scale, const RopeParams& rp, bool k_prerot, bool key_mask,
                                      int lane) {
    for (int j = j0; j < j1; ++j) {
      if (key_mask && __ldg(pos + j) < 0) continue;   // MINIPIC_KEY_MASK: invisible to every row
      const int blk = __ldg(bt + j / kBlock);
      const size_t row = (((size_t)blk * hkv + g) * kBlock + (j % kBlock)) * D;
      float k[E], v[E];
#pragma unroll
      for (int m = 0; m < E; ++m) { k[m] = IO<T>::load(kc + row + lane + 32 * m); v[m] = IO<T>::load(vc + row + lane + 32 * m); }
      if (!k_prerot) {
        const int p = __ldg(pos + j);
#pragma unroll
        for (int m = 0; m < HP; ++m) {
          const float2 cs = rope_cs_precise(rp, p, lane + 32 * m);
          const float a = k[m], b = k[m + HP];
          k[m] = a * cs.x - b * cs.y;
          k[m + HP] = b * cs.x + a * cs.y;
        }
      }
      float s = 0.f;
#pragma unroll
      for (int m = 0; m < E; ++m) s = fmaf(q[m], k[m], s);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      s *= scale;
      const float m_new = fmaxf(m_run, s);
      const float corr = expf(m_run - m_new);   // exp(-inf) = 0 on the first key
      const float p_ = expf(s - m_new);
      l_run = l_run * corr + p_;
#pragma unroll
      for (int m = 0; m < E; ++m) acc[m] = fmaf(p_, v[m], acc[m] * corr);
      m_run = m_new;
    }
  }
};

__device__ __forceinline__ int find_request(const int* cu, int num_reqs, int t) {
  int lo = 0, hi = num_reqs;  // largest r with cu[r] <= t
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(cu + mid) <= t) lo = mid; else hi = mid;
  }
  return lo;
}

template <typename T, int D>
__global__ void __launch_bounds__(128) prefill_simt_kernel(PrefillArgs a, int hq, int hkv, float scale, RopeParams rp,
                                                           unsigned flags) {
  const int lane = threadIdx.x & 31;
  const long long w = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (w >= (long long)a.num_q_tokens * hq) return;
  const int t = (int)(w / hq), h = (int)(w % hq);
  const int r = find_request(a.cu_q_lens, a.num_reqs, t);
  const int idx = __ldg(a.q_seq_idx + t), lo = max(__ldg(a.q_vis_lo + t), 0);
  const int* pos = a.kv_positions + __ldg(a.cu_kv_lens + r);
  const int* bt = a.block_tables + (size_t)r * a.max_blocks;
  WarpAttn<T, D> wa;
  wa.init((const T*)a.q + ((size_t)t * hq + h) * D, rp, __ldg(pos + idx), flags & MINIPIC_Q_PREROTATED, lane);
  const int hi = min(idx + 1, __ldg(a.kv_lens + r));
  wa.run((const T*)a.k_cache, (const T*)a.v_cache, bt, pos, hkv, h / (hq / hkv), lo, hi, scale, rp,
         flags & MINIPIC_K_PREROTATED, flags & MINIPIC_KEY_MASK, lane);
  T* o = (T*)a.out + ((size_t)t * hq + h) * D;
  const float inv = wa.l_run > 0.f ? 1.f / wa.l_run : 0.f;
#pragma unroll
  for (int m = 0; m < WarpAttn<T, D>::E; ++m) IO<T>::store(o + lane + 32 * m, wa.acc[m] * inv);
  if (lane == 0) a.lse[(size_t)t * hq + h] = wa.l_run > 0.f ? wa.m_run + logf(wa.l_run) : -INFINITY;
}

// decode partial: grid (seq * max_splits + split, head); one warp per CTA (the sequence count lives in grid.x: no 65535 limit)
template <typename T, int D>
__global__ void __launch_bounds__(32) decode_simt_kernel(DecodeArgs a, int hq, int hkv, float scale, RopeParams rp,
                                                         unsigned flags, int split_len, int max_splits,
                                                         float* __restrict__ o_part, float* __restrict__ lse_part) {
  const int lane = threadIdx.x, s = blockIdx.x % max_splits, r = blockIdx.x / max_splits, h = blockIdx.y;
  const int kv_len = __ldg(a.kv_lens + r);
  if (s * split_len >= kv_len) return;  // empty split: the merge kernel never reads it
  const int idx = kv_len - 1;
  const int lo = a.q_vis_lo ? max(__ldg(a.q_vis_lo + r), 0) : 0;
  const int* pos = a.kv_positions + __ldg(a.cu_kv_lens + r);
  const int* bt = a.block_tables + (size_t)r * a.max_blocks;
  WarpAttn<T, D> wa;
  wa.init((const T*)a.q + ((size_t)r * hq + h) * D, rp, __ldg(pos + idx), flags & MINIPIC_Q_PREROTATED, lane);
  const int j0 = max(lo, s * split_len), j1 = min(kv_len, (s + 1) * split_len);
  wa.run((const T*)a.k_cache, (const T*)a.v_cache, bt, pos, hkv, h / (hq / hkv), j0, j1, scale, rp,
         flags & MINIPIC_K_PREROTATED, flags & MINIPIC_KEY_MASK, lane);
  const size_t pr = ((size_t)r * hq + h) * max_splits + s;
  const float inv = wa.l_run > 0.f ? 1.f / wa.l_run : 0.f;
#pragma unroll
  for (int m = 0; m < WarpAttn<T, D>::E; ++m) o_part[pr * D + lane + 32 * m] = wa.acc[m] * inv;
  if (lane == 0) lse_part[pr] = wa.l_run > 0.f ? wa.m_run + logf(wa.l_run) : -INFINITY;
}

// a11: LSE merge.  lse = ln sum_s e^{lse_s};  o = sum_s e^{lse_s - lse} o_s.  One warp per (seq, head).
template <typename T, int D>
__global__ void __launch_bounds__(128) lse_merge_kernel(const float* __restrict__ o_part, const float* __restrict__ lse_part,
                                                        const int* __restrict__ kv_lens, int num_seqs, int hq,
                                                        int split_len, int max_splits, T* __restrict__ out,
                                                        float* __restrict__ lse) {
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (w >= num_seqs * hq) return;
  const int r = w / hq;
  const int kv_len = __ldg(kv_lens + r);
  const int ns = min((kv_len + split_len - 1) / split_len, max_splits);   // kv_len > max_kv_len is a caller error: stay inside the row
  const float* lp = lse_part + (size_t)w * max_splits;
  const float* op = o_part + (size_t)w * max_splits * D;
  float m = -INFINITY;
  for (int s = lane; s < ns; s += 32) m = fmaxf(m, __ldg(lp + s));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  constexpr int E = D / 32;
  float acc[E];
#pragma unroll
  for (int e = 0; e < E; ++e) acc[e] = 0.f;
  float z = 0.f;
  if (m > -INFINITY) {
    for (int s = 0; s < ns; ++s) {
      const float wgt = expf(__ldg(lp + s) - m);
      z += wgt;
#pragma unroll
      for (int e = 0; e < E; ++e) acc[e] = fmaf(wgt, __ldg(op + (size_t)s * D + lane + 32 * e), acc[e]);
    }
  }
  const float inv = z > 0.f ? 1.f / z : 0.f;
  T* o = out + (size_t)w * D;
#pragma unroll
  for (int e = 0; e < E; ++e) IO<T>::store(o + lane + 32 * e, acc[e] * inv);
  if (lane == 0) lse[w] = z > 0.f ? m + logf(z) : -INFINITY;
}

template <typename T, int D>
static void prefill_simt_t(const Ctx& c, const PrefillArgs& a) {
  const long long warps = (long long)a.num_q_tokens * c.hq;
  if (warps == 0) return;
  prefill_simt_kernel<T, D><<<(unsigned)((warps + 3) / 4), 128, 0, c.stream>>>(a, c.hq, c.hkv, c.scale, c.rope, c.flags);
  note_launch();
}
void launch_prefill_simt(const Ctx& c, const PrefillArgs& a) {
  if (c.dtype == MINIPIC_F32) { if (c.d == 64) prefill_simt_t<float, 64>(c, a); else prefill_simt_t<float, 128>(c, a); }
  else { if (c.d == 64) prefill_simt_t<__nv_bfloat16, 64>(c, a); else prefill_simt_t<__nv_bfloat16, 128>(c, a); }
}

template <typename T, int D>
static void decode_simt_t(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  dim3 grid((unsigned)sp.max_splits * (unsigned)a.num_seqs, c.hq);
  decode_simt_kernel<T, D><<<grid, 32, 0, c.stream>>>(a, c.hq, c.hkv, c.scale, c.rope, c.flags, sp.split_len,
                                                      sp.max_splits, o_part, lse_part);
  note_launch();
}
void launch_decode_simt(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  if (a.num_seqs == 0) return;
  if (c.dtype == MINIPIC_F32) { if (c.d == 64) decode_simt_t<float, 64>(c, a, sp, o_part, lse_part); else decode_simt_t<float, 128>(c, a, sp, o_part, lse_part); }
  else { if (c.d == 64) decode_simt_t<__nv_bfloat16, 64>(c, a, sp, o_part, lse_part); else decode_simt_t<__nv_bfloat16, 128>(c, a, sp, o_part, lse_part); }
}

template <typename T, int D>
static void merge_t(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, const float* o_part, const float* lse_part) {
  const int warps = a.num_seqs * c.hq;
  lse_merge_kernel<T, D><<<(warps + 3) / 4, 128, 0, c.stream>>>(o_part, lse_part, a.kv_lens, a.num_seqs, c.hq, sp.split_len,
                                                               sp.max_splits, (T*)a.out, a.lse);
  note_launch();
}
void launch_lse_merge(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, const float* o_part, const float* lse_part) {
  if (a.num_seqs == 0) return;
  if (c.dtype == MINIPIC_F32) { if (c.d == 64) merge_t<float, 64>(c, a, sp, o_part, lse_part); else merge_t<float, 128>(c, a, sp, o_part, lse_part); }
  else { if (c.d == 64) merge_t<__nv_bfloat16, 64>(c, a, sp, o_part, lse_part); else merge_t<__nv_bfloat16, 128>(c, a, sp, o_part, lse_part); }
}

}  // namespace minipic
