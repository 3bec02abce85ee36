// a1: paged cache write (PAPER.md:47 paged blocks; :100 K stored UNROTATED; :113 V unchanged).
//   cache[slot / B, h, slot % B, :] = new[t, h, :]      raw 16-byte copies, bit exact, slot < 0 skipped.
// HBM-bound: algorithmic bytes = 2 * (K + V bytes of the written tokens) (read new + write cache).
#include "internal.h"

namespace minipic {

// One "row" is the D elements of one (token, head): row_vecs 16-byte vectors.  Work item = one vector of K
// and the matching vector of V.  kUnroll independent items per thread keep >= 2*kUnroll 16-byte loads in flight.
template <int kUnroll>
__global__ void __launch_bounds__(256) cache_write_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                                          const int64_t* __restrict__ slots, long long total_vecs,
                                                          int hkv, int row_vecs, uint4* __restrict__ k_cache,
                                                          uint4* __restrict__ v_cache) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  const int vecs_per_token = hkv * row_vecs;
  for (long long base = (long long)blockIdx.x * blockDim.x + threadIdx.x; base < total_vecs; base += stride * kUnroll) {
    uint4 kv[kUnroll], vv[kUnroll];
    long long dst[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const long long i = base + u * stride;
      dst[u] = -1;
      if (i < total_vecs) {
        const long long t = i / vecs_per_token;
        const int rem = (int)(i - t * vecs_per_token);
        const int h = rem / row_vecs, c = rem - h * row_vecs;
        const long long slot = __ldg(slots + t);
        if (slot >= 0) {
          const long long blk = slot / kBlock;
          const int off = (int)(slot - blk * kBlock);
          dst[u] = ((blk * hkv + h) * kBlock + off) * row_vecs + c;
          kv[u] = ldg_stream16(k_new + i);
          vv[u] = ldg_stream16(v_new + i);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      if (dst[u] >= 0) {
        k_cache[dst[u]] = kv[u];
        v_cache[dst[u]] = vv[u];
      }
    }
  }
}

void launch_cache_write(int itemsize, int hkv, int d, const void* k_new, const void* v_new, const int64_t* slots,
                        int num_tokens, void* k_cache, void* v_cache, cudaStream_t s) {
  if (num_tokens <= 0) return;
  const int row_vecs = d * itemsize / 16;
  const long long total = (long long)num_tokens * hkv * row_vecs;
  constexpr int kUnroll = 4;
  const int sms = current_sm_count();
  long long blocks = (total + 256LL * kUnroll - 1) / (256LL * kUnroll);
  const long long cap = (long long)sms * 16;  // 8 resident CTAs/SM x 2 waves; grid-stride beyond that
  if (blocks > cap) blocks = cap;
  cache_write_kernel<kUnroll><<<(unsigned)blocks, 256, 0, s>>>(
      (const uint4*)k_new, (const uint4*)v_new, slots, total, hkv, row_vecs, (uint4*)k_cache, (uint4*)v_cache);
  note_launch();
}

// a0: cos/sin table, evaluated in fp64 from the exact fixed-point phase and rounded once to fp32.
__global__ void rope_table_kernel(RopeParams rp, int num_positions, float2* __restrict__ table) {
  const long long n = (long long)num_positions * rp.half;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    const int p = (int)(e / rp.half), i = (int)(e - (long long)p * rp.half);
    const unsigned long long ph = (unsigned long long)(unsigned)p * rp.phase_inc[i];
    // signed half-turns in [-1, 1): keep 53 bits
    const double x = (double)(long long)ph * 1.0842021724855044e-19;  // * 2^-63
    double sn, cs;
    sincospi(x, &sn, &cs);
    table[e] = make_float2((float)cs, (float)sn);
  }
}

void launch_rope_table(const RopeParams& rp, int num_positions, float2* table, cudaStream_t s) {
  if (num_positions <= 0) return;
  const long long n = (long long)num_positions * rp.half;
  long long blocks = (n + 255) / 256;
  if (blocks > current_sm_count() * 8LL) blocks = current_sm_count() * 8LL;
  rope_table_kernel<<<(unsigned)blocks, 256, 0, s>>>(rp, num_positions, table);
  note_launch();
}

}  // namespace minipic
