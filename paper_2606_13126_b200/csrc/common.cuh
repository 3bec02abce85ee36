// Shared device / host helpers of the MiniPIC CUDA path (sm_100a).  No code here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/minipic.h"

namespace minipic {

constexpr int kBlock = 16;  // KV block size

// ------------------------------------------------------------------------------------ RoPE phase
// Eq. 2 needs cos/sin(p * f_i), f_i = theta^(-2i/D).  fp32(p)*fp32(f_i) is off by up to
// 1.4e-3 rad at p = 33K, so the phase is carried in 64-bit fixed point instead:
//   turns(p, i) = frac(p * f_i / 2pi) = (p * F_i) mod 2^64 / 2^64,  F_i = round(f_i / 2pi * 2^64)
// The integer multiply wraps exactly; the top 32 bits, read as int32, are the angle in half-turns * 2^31.
struct RopeParams {
  unsigned long long phase_inc[64];  // F_i, i < D/2 <= 64   (host: long double)
  const float2* table;               // optional [table_len][half] (cos, sin), else nullptr
  int table_len;
  int half;                          // D/2
};

__device__ __forceinline__ float rope_half_turns(const RopeParams& rp, int pos, int i) {
  unsigned long long ph = (unsigned long long)(unsigned)pos * rp.phase_inc[i];
  return (float)(int)(ph >> 32) * 4.656612873077393e-10f;  // * 2^-31  -> [-1, 1)
}
// full-precision variant (SIMT / fp32 path): |err| ~ 1e-7
__device__ __forceinline__ float2 rope_cs_precise(const RopeParams& rp, int pos, int i) {
  if (pos < rp.table_len) return __ldg(rp.table + (size_t)pos * rp.half + i);
  float s, c;
  sincospif(rope_half_turns(rp, pos, i), &s, &c);
  return make_float2(c, s);
}
// fast variant (tensor-core paths, operands are rounded to bf16 afterwards): MUFU on the reduced angle, |err| < 1e-6
__device__ __forceinline__ float2 rope_cs_fast(const RopeParams& rp, int pos, int i) {
  if (pos < rp.table_len) return __ldg(rp.table + (size_t)pos * rp.half + i);
  float a = rope_half_turns(rp, pos, i) * 3.14159265358979f;
  return make_float2(__cosf(a), __sinf(a));
}

// ------------------------------------------------------------------------------------ dtype traits
template <typename T> struct IO;
template <> struct IO<float> {
  static __device__ __forceinline__ float load(const float* p) { return __ldg(p); }
  static __device__ __forceinline__ void store(float* p, float v) { *p = v; }
};
template <> struct IO<__nv_bfloat16> {
  static __device__ __forceinline__ float load(const __nv_bfloat16* p) {
    return __uint_as_float((unsigned)__ldg(reinterpret_cast<const unsigned short*>(p)) << 16);
  }
  static __device__ __forceinline__ void store(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
};

__device__ __forceinline__ float bf16lo(unsigned w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(unsigned w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ unsigned pack_bf16(float lo, float hi) {  // RN both, lo in bits [0,16)
  unsigned r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint4 ldg_stream16(const void* p) {  // 16-byte streaming load, no L1 allocation
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// packed fp32 pairs (one 64-bit register = two lanes of an FFMA2)
__device__ __forceinline__ uint64_t pk2(float a, float b) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ void upk2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// ------------------------------------------------------------------------------------ host side
struct Ctx {  // what every launcher needs, derived once from minipic_config
  int hq, hkv, d, group, num_blocks;
  int dtype;
  float scale;       // softmax scale
  float scale_log2;  // scale * log2(e)
  unsigned flags;
  RopeParams rope;
  double rope_step_cos[64], rope_step_sin[64];  // cos / sin of f_i: the one-position RoPE step (prefill recurrence)
  cudaStream_t stream;
};

void note_launch(int n = 1);
void note_error(const char* what);    // text for minipic_last_cuda_error() on non-CUDA failure paths
int current_sm_count();               // SMs of the current device
bool check_launch(const char* what);  // cudaGetLastError -> records text, returns ok

}  // namespace minipic
