// Steps adjacent to the hot path, both HBM-bound elementwise kernels:
//
//  f1  preattn_fused_kernel    the step right before attention (PAPER.md:100; Table 2 row rotary_embedding/base.py, :207):
//                              one pass over the QKV-projection output of the new tokens writes K and V UNROTATED into the
//                              paged cache through the slot mapping (raw 16-byte copies: bit exact) and Q rotated at the
//                              token's logical position (fp32 rotation, one RN to the I/O dtype) - instead of a rotary
//                              kernel over Q plus a separate cache write.
//  f4  block_rerotate_kernel   CONTROL: what a position-dependent cache has to do to reuse a span at a new offset
//                              (PAPER.md:63 "block-by-block copy and repositioning", :284-286): dst block <- R(delta) src
//                              block for K, a plain copy for V.  MiniPIC itself never runs this; bench.py times it to put a
//                              number on the HBM traffic the position-free layout avoids.
//
// A thread owns one 16-byte vector position of the low half of head_dim and the matching one of the high half (the two
// elements of every rotate-half pair are then lane-local), for ALL heads of its token / block row: cos / sin of its VE
// frequencies are computed once (exact 64-bit fixed-point phase, common.cuh) and reused over the heads.
#include "internal.h"

namespace minipic {

namespace {

template <typename T> struct Vec;   // 16-byte vector of the I/O dtype <-> VE floats
template <> struct Vec<__nv_bfloat16> {
  static constexpr int VE = 8;
  static __device__ __forceinline__ void unpack(const uint4& v, float (&f)[8]) {
    const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) { f[2 * i] = bf16lo(w[i]); f[2 * i + 1] = bf16hi(w[i]); }
  }
  static __device__ __forceinline__ uint4 pack(const float (&f)[8]) {
    return make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
  }
};
template <> struct Vec<float> {
  static constexpr int VE = 4;
  static __device__ __forceinline__ void unpack(const uint4& v, float (&f)[4]) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  static __device__ __forceinline__ uint4 pack(const float (&f)[4]) {
    return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
  }
};

// cos / sin of frequencies i0 .. i0 + VE - 1 at a (possibly negative) position: the phase p * F_i wraps exactly in 64 bits
template <int VE>
__device__ __forceinline__ void trig(const RopeParams& rp, long long p, int i0, float (&c)[VE], float (&s)[VE]) {
#pragma unroll
  for (int e = 0; e < VE; ++e) {
    const unsigned long long ph = (unsigned long long)p * rp.phase_inc[i0 + e];
    sincospif((float)(int)(ph >> 32) * 4.656612873077393e-10f, &s[e], &c[e]);   // half-turns in [-1, 1); |err| ~ 1e-7
  }
}
template <typename T, int VE>
__device__ __forceinline__ void rotate_pair(uint4& lo, uint4& hi, const float (&c)[VE], const float (&s)[VE]) {
  float a[VE], b[VE], x[VE], y[VE];
  Vec<T>::unpack(lo, a); Vec<T>::unpack(hi, b);
#pragma unroll
  for (int e = 0; e < VE; ++e) { x[e] = a[e] * c[e] - b[e] * s[e]; y[e] = b[e] * c[e] + a[e] * s[e]; }
  lo = Vec<T>::pack(x); hi = Vec<T>::pack(y);
}

template <typename T>
__global__ void __launch_bounds__(256) preattn_fused_kernel(const uint4* __restrict__ qkv, const int64_t* __restrict__ slots,
                                                            const int* __restrict__ positions, long long num_tokens,
                                                            int hq, int hkv, int d, bool rotate_q, RopeParams rp,
                                                            uint4* __restrict__ q_out, uint4* __restrict__ k_cache,
                                                            uint4* __restrict__ v_cache) {
  constexpr int VE = Vec<T>::VE;
  const int vph = d / 2 / VE;          // vectors per half row
  const int vpr = 2 * vph;             // vectors per head row
  const long long total = num_tokens * vph;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const long long t = i / vph;
    const int ci = (int)(i % vph);
    const uint4* row = qkv + (size_t)t * (hq + 2 * hkv) * vpr;
    // ---- Q heads: q'[t, h] = R(positions[t]) q[t, h], one rounding to the I/O dtype
    float c[VE], s[VE];
    if (rotate_q) trig<VE>(rp, (long long)__ldg(positions + t), ci * VE, c, s);
    uint4* qo = q_out + (size_t)t * hq * vpr;
#pragma unroll 4
    for (int h = 0; h < hq; ++h) {
      uint4 lo = ldg_stream16(row + h * vpr + ci), hi = ldg_stream16(row + h * vpr + vph + ci);
      if (rotate_q) rotate_pair<T, VE>(lo, hi, c, s);
      qo[h * vpr + ci] = lo; qo[h * vpr + vph + ci] = hi;
    }
    // ---- K, V heads: raw copies into the paged cache [block][Hkv][16][D] (negative slot: skipped)
    const long long slot = __ldg(slots + t);
    if (slot >= 0) {
      const size_t base = ((size_t)(slot / kBlock) * hkv * kBlock + (size_t)(slot % kBlock)) * vpr;   // + h * 16 * vpr
#pragma unroll 2
      for (int h = 0; h < hkv; ++h) {
        const uint4 klo = ldg_stream16(row + (hq + h) * vpr + ci), khi = ldg_stream16(row + (hq + h) * vpr + vph + ci);
        const uint4 vlo = ldg_stream16(row + (hq + hkv + h) * vpr + ci), vhi = ldg_stream16(row + (hq + hkv + h) * vpr + vph + ci);
        const size_t o = base + (size_t)h * kBlock * vpr;
        k_cache[o + ci] = klo; k_cache[o + vph + ci] = khi;
        v_cache[o + ci] = vlo; v_cache[o + vph + ci] = vhi;
      }
    }
  }
}

// ncu (r2): with plain __launch_bounds__(256) the unrolled loop took 168 registers = ONE block per SM (12 % occupancy, 0.57 of
// HBM).  Now: at least 4 blocks per SM (<= 64 registers), the V copy issued as its own loads -> stores ahead of the K rotation.
template <typename T>
__global__ void __launch_bounds__(256, 4) block_rerotate_kernel(uint4* __restrict__ k_cache, uint4* __restrict__ v_cache,
                                                                const int* __restrict__ src, const int* __restrict__ dst,
                                                                const int* __restrict__ delta, long long num_pairs, int hkv,
                                                                int d, RopeParams rp) {
  constexpr int VE = Vec<T>::VE;
  const int vph = d / 2 / VE, vpr = 2 * vph;
  const int rows = hkv * kBlock;                       // (head, token) rows of one block
  const long long total = num_pairs * hkv * vph;        // a thread: one vector position of the 16 token rows of one head
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const long long p = i / (hkv * vph);
    const int h = (int)(i / vph % hkv), ci = (int)(i % vph);
    const size_t so = ((size_t)__ldg(src + p) * rows + (size_t)h * kBlock) * vpr + ci, dofs = ((size_t)__ldg(dst + p) * rows + (size_t)h * kBlock) * vpr + ci;
    // ---- V: a plain copy, four rows (8 vectors) in flight
#pragma unroll 1
    for (int r0 = 0; r0 < kBlock; r0 += 4) {
      uint4 t[8];
#pragma unroll
      for (int r = 0; r < 4; ++r) { t[2 * r] = ldg_stream16(v_cache + so + (size_t)(r0 + r) * vpr); t[2 * r + 1] = ldg_stream16(v_cache + so + (size_t)(r0 + r) * vpr + vph); }
#pragma unroll
      for (int r = 0; r < 4; ++r) { v_cache[dofs + (size_t)(r0 + r) * vpr] = t[2 * r]; v_cache[dofs + (size_t)(r0 + r) * vpr + vph] = t[2 * r + 1]; }
    }
    // ---- K: dst <- R(delta) src
    float c[VE], s[VE];
    trig<VE>(rp, (long long)__ldg(delta + p), ci * VE, c, s);
#pragma unroll 1
    for (int r0 = 0; r0 < kBlock; r0 += 4) {
      uint4 lo[4], hi[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) { lo[r] = ldg_stream16(k_cache + so + (size_t)(r0 + r) * vpr); hi[r] = ldg_stream16(k_cache + so + (size_t)(r0 + r) * vpr + vph); }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        rotate_pair<T, VE>(lo[r], hi[r], c, s);
        k_cache[dofs + (size_t)(r0 + r) * vpr] = lo[r]; k_cache[dofs + (size_t)(r0 + r) * vpr + vph] = hi[r];
      }
    }
  }
}

int grid_for(long long items) {
  const long long want = (items + 255) / 256, cap = (long long)current_sm_count() * 16;
  return (int)(want < 1 ? 1 : (want > cap ? cap : want));
}

}  // namespace

void launch_preattn_fused(const Ctx& c, const void* qkv, const int64_t* slots, const int* positions, int num_tokens,
                          void* q_out, void* k_cache, void* v_cache) {
  const bool rot = !(c.flags & MINIPIC_Q_PREROTATED);
  if (c.dtype == MINIPIC_BF16) {
    const long long items = (long long)num_tokens * (c.d / 16);
    preattn_fused_kernel<__nv_bfloat16><<<grid_for(items), 256, 0, c.stream>>>(
        (const uint4*)qkv, slots, positions, num_tokens, c.hq, c.hkv, c.d, rot, c.rope, (uint4*)q_out, (uint4*)k_cache, (uint4*)v_cache);
  } else {
    const long long items = (long long)num_tokens * (c.d / 8);
    preattn_fused_kernel<float><<<grid_for(items), 256, 0, c.stream>>>(
        (const uint4*)qkv, slots, positions, num_tokens, c.hq, c.hkv, c.d, rot, c.rope, (uint4*)q_out, (uint4*)k_cache, (uint4*)v_cache);
  }
  note_launch();
}

void launch_block_rerotate(const Ctx& c, void* k_cache, void* v_cache, const int* src, const int* dst, const int* delta,
                           int num_pairs) {
  if (c.dtype == MINIPIC_BF16) {
    const long long items = (long long)num_pairs * c.hkv * (c.d / 16);
    block_rerotate_kernel<__nv_bfloat16><<<grid_for(items), 256, 0, c.stream>>>((uint4*)k_cache, (uint4*)v_cache, src, dst,
                                                                                delta, num_pairs, c.hkv, c.d, c.rope);
  } else {
    const long long items = (long long)num_pairs * c.hkv * (c.d / 8);
    block_rerotate_kernel<float><<<grid_for(items), 256, 0, c.stream>>>((uint4*)k_cache, (uint4*)v_cache, src, dst, delta,
                                                                        num_pairs, c.hkv, c.d, c.rope);
  }
  note_launch();
}

}  // namespace minipic
