// a10: split-KV decode partial kernel (bf16, head_dim 128, GQA group <= 8), HBM-bound.
//
// One warp owns one (sequence, KV head, split): it streams the split's 16-token blocks straight from the paged
// cache into registers with coalesced 16-byte loads (every 32-byte sector it touches is fully used), rotates K in
// registers at the request's logical positions (Eq. 2), and runs both contractions on the
// register-operand tensor path (mma.sync m16n8k16, bf16 x bf16 -> fp32) so that the CUDA cores are left for the
// bf16->fp32 conversion and the two FMAs per K element.  The G query heads of the group share the
// rotated K tile.  Online softmax uses warp shuffles across the 4 lanes that hold one head's scores.
// Partials (o_s normalised over the split, lse_s) go to the workspace; lse_merge_kernel (a11) combines them.
//
// Fragment trick: the dot products are sums over head_dim (QK^T) and over keys (PV), so any permutation of the
// summation index is legal as long as both operands use it.  That lets each lane feed the MMA fragments from
// whole 16-byte vectors:
//   QK^T as S^T[head, key] = Q'[head, d] K'^T[d, key]:  A = Q' (row g = head), B = K' (col g = key), and the lane
//     (g, q) loads for key rows g and g+8 the 16-byte chunks q, q+4, q+8, q+12 - chunk c and c+8 hold the two
//     halves of the rotate-half pairs, so the rotation is lane-local.
//   PV as O^T[d, head] = V^T[d, key] P[key, head]:  the S^T accumulator layout IS the B-fragment layout of P; the
//     lane loads chunk g (and g+8) of V rows 2q, 2q+1, 2q+8, 2q+9 and two byte-permutes per register pair build
//     the A fragments.
#include "internal.h"

namespace minipic {

namespace {

__device__ __forceinline__ void mma16816(float (&d)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0,
                                         unsigned b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// cos/sin of 8 consecutive frequencies i0..i0+7 at position p, computed in registers: exact 64-bit fixed-point phase
// (common.cuh) -> signed half-turns -> MUFU sin/cos on the reduced angle in [-pi, pi) (|err| < 1e-6, far below the
// bf16 rounding of the rotated operand).  No memory traffic: in this HBM-bound kernel a cos/sin table lookup
// costs as many L1 wavefronts as the KV stream itself (ncu: l1tex 92% with the table, profiles/).
__device__ __forceinline__ void rope_cs8(const unsigned long long* __restrict__ finc, int p, int i0, float (&c)[8],
                                         float (&s)[8]) {
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    const unsigned long long ph = (unsigned long long)(unsigned)p * finc[i0 + e];
    const float a = (float)(int)(ph >> 32) * 1.4629180792671596e-9f;  // * pi * 2^-31 -> radians in [-pi, pi)
    c[e] = __cosf(a);
    s[e] = __sinf(a);
  }
}

// rotate the pair of 16-byte chunks (lo = elements i0..i0+7, hi = elements i0+64..i0+71) in place -> bf16
__device__ __forceinline__ void rotate_chunks(uint4& lo, uint4& hi, const float (&c)[8], const float (&s)[8]) {
  unsigned* l = reinterpret_cast<unsigned*>(&lo);
  unsigned* h = reinterpret_cast<unsigned*>(&hi);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const float a0 = bf16lo(l[w]), a1 = bf16hi(l[w]), b0 = bf16lo(h[w]), b1 = bf16hi(h[w]);
    const float x0 = a0 * c[2 * w] - b0 * s[2 * w], x1 = a1 * c[2 * w + 1] - b1 * s[2 * w + 1];
    const float y0 = b0 * c[2 * w] + a0 * s[2 * w], y1 = b1 * c[2 * w + 1] + a1 * s[2 * w + 1];
    l[w] = pack_bf16(x0, x1);
    h[w] = pack_bf16(y0, y1);
  }
}

template <bool kRotK>
__global__ void __launch_bounds__(128, 4)   // 4-warp CTAs: 6 % faster than 8-warp CTAs at the same 16 warps / SM (finer-grained block scheduling)
decode_mma_kernel(DecodeArgs a, int hq, int hkv, int group, float scale_log2, RopeParams rp, unsigned flags,
                  int split_len, int max_splits, float* __restrict__ o_part, float* __restrict__ lse_part) {
  constexpr int D = 128;
  __shared__ unsigned long long finc[64];  // F_i: 64-bit fixed-point phase increments (turns per position)
  if (threadIdx.x < 64) finc[threadIdx.x] = rp.phase_inc[threadIdx.x];
  if (blockDim.x == 32) finc[threadIdx.x + 32] = rp.phase_inc[threadIdx.x + 32];   // a CTA can be a single warp (odd Hkv)
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 2, q4 = lane & 3;
  const int s = blockIdx.x, r = blockIdx.y;
  const int kvh = blockIdx.z * (blockDim.x >> 5) + warp;
  const int kv_len = __ldg(a.kv_lens + r);
  if (s * split_len >= kv_len) return;  // the merge kernel never reads empty splits
  const int vis_lo = a.q_vis_lo ? max(__ldg(a.q_vis_lo + r), 0) : 0;
  const int j_begin = max(vis_lo, s * split_len), j_end = min(kv_len, (s + 1) * split_len);
  const int* __restrict__ pos = a.kv_positions + __ldg(a.cu_kv_lens + r);
  const int* __restrict__ bt = a.block_tables + (size_t)r * a.max_blocks;
  const __nv_bfloat16* __restrict__ kc = (const __nv_bfloat16*)a.k_cache;
  const __nv_bfloat16* __restrict__ vc = (const __nv_bfloat16*)a.v_cache;

  // ---- Q' fragments (a3): head g of the group, chunks q4 + 4j, rotated at the query's logical position
  unsigned qf[8][2];
  {
    uint4 ch[4];
    if (g < group) {
      const __nv_bfloat16* qrow = (const __nv_bfloat16*)a.q + ((size_t)r * hq + (size_t)kvh * group + g) * D;
#pragma unroll
      for (int j = 0; j < 4; ++j) ch[j] = __ldg(reinterpret_cast<const uint4*>(qrow + (q4 + 4 * j) * 8));
      if (!(flags & MINIPIC_Q_PREROTATED)) {
        const int qpos = __ldg(pos + kv_len - 1);
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          float c[8], sn[8];
          rope_cs8(finc, qpos, (q4 + 4 * j) * 8, c, sn);
          rotate_chunks(ch[j], ch[j + 2], c, sn);
        }
      }
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) ch[j] = make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      qf[2 * j][0] = ch[j].x; qf[2 * j][1] = ch[j].y;
      qf[2 * j + 1][0] = ch[j].z; qf[2 * j + 1][1] = ch[j].w;
    }
  }

  float o[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
  float m_run = -INFINITY, l_run = 0.f;

  const int kb0 = j_begin / kBlock, kb1 = (j_end + kBlock - 1) / kBlock;
  int blk = __ldg(bt + kb0);
  for (int kb = kb0; kb < kb1; ++kb) {
    const size_t base = ((size_t)blk * hkv + kvh) * (kBlock * D);
    if (kb + 1 < kb1) blk = __ldg(bt + kb + 1);
    // ---- a4: K rows g and g+8, chunks q4 + 4j: 8 x 16-byte streaming loads
    uint4 kr[2][4];
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int j = 0; j < 4; ++j) kr[t][j] = ldg_stream16(kc + base + (g + 8 * t) * D + (q4 + 4 * j) * 8);
    // ---- a5: rotate in registers at pi_r(j)
    if (kRotK) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int jrow = kb * kBlock + g + 8 * t;
        const int p = __ldg(pos + min(jrow, kv_len - 1));
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          float c[8], sn[8];
          rope_cs8(finc, p, (q4 + 4 * j) * 8, c, sn);
          rotate_chunks(kr[t][j], kr[t][j + 2], c, sn);
        }
      }
    }
    // ---- a6: S^T[head, key] for the two 8-key halves of the block
    float st[2][4];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      st[t][0] = st[t][1] = st[t][2] = st[t][3] = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        mma16816(st[t], qf[2 * j][0], 0u, qf[2 * j][1], 0u, kr[t][j].x, kr[t][j].y);
        mma16816(st[t], qf[2 * j + 1][0], 0u, qf[2 * j + 1][1], 0u, kr[t][j].z, kr[t][j].w);
      }
    }
    // ---- V rows 2q, 2q+1, 2q+8, 2q+9, chunks g and g+8 (issued now, consumed after the softmax)
    uint4 vr[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int row = 2 * q4 + (i & 1) + 8 * (i >> 1);
      const int jrow = kb * kBlock + row;
      const bool ok = jrow >= j_begin && jrow < j_end;  // never multiply P = 0 with uninitialised cache bits
#pragma unroll
      for (int hf = 0; hf < 2; ++hf)
        vr[i][hf] = ok ? ldg_stream16(vc + base + row * D + (g + 8 * hf) * 8) : make_uint4(0, 0, 0, 0);
    }
    // ---- a7: mask + online softmax (row = head g; its 16 scores live in 4 lanes x 4 registers)
    float sc[2][2];
    float m_blk = -INFINITY;
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int j = kb * kBlock + 8 * t + 2 * q4 + e;
        sc[t][e] = (j >= j_begin && j < j_end) ? st[t][e] * scale_log2 : -INFINITY;
        m_blk = fmaxf(m_blk, sc[t][e]);
      }
    m_blk = fmaxf(m_blk, __shfl_xor_sync(0xffffffffu, m_blk, 1));
    m_blk = fmaxf(m_blk, __shfl_xor_sync(0xffffffffu, m_blk, 2));
    const float m_new = fmaxf(m_run, m_blk);
    // lazy rescale: P may grow up to 2^8 relative to the running max before O and l are rescaled
    if (__any_sync(0xffffffffu, m_new > m_run + 8.f)) {
      const float corr = (m_new == -INFINITY) ? 1.f : exp2f(m_run - m_new);
      l_run *= corr;
      m_run = m_new;
      const float ca = __shfl_sync(0xffffffffu, corr, (2 * q4) * 4), cb = __shfl_sync(0xffffffffu, corr, (2 * q4 + 1) * 4);
#pragma unroll
      for (int i = 0; i < 8; ++i) { o[i][0] *= ca; o[i][1] *= cb; o[i][2] *= ca; o[i][3] *= cb; }
    }
    const float m_use = (m_run == -INFINITY) ? 0.f : m_run;
    float p[2][2];
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int e = 0; e < 2; ++e) { p[t][e] = exp2f(sc[t][e] - m_use); l_run += p[t][e]; }
    const unsigned pb0 = pack_bf16(p[0][0], p[0][1]), pb1 = pack_bf16(p[1][0], p[1][1]);
    // ---- a8: O^T[d, head] += V^T[d, key] P[key, head]
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      const unsigned* v0 = reinterpret_cast<const unsigned*>(&vr[0][hf]);
      const unsigned* v1 = reinterpret_cast<const unsigned*>(&vr[1][hf]);
      const unsigned* v2 = reinterpret_cast<const unsigned*>(&vr[2][hf]);
      const unsigned* v3 = reinterpret_cast<const unsigned*>(&vr[3][hf]);
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) {
        const unsigned a0 = __byte_perm(v0[mt], v1[mt], 0x5410), a1 = __byte_perm(v0[mt], v1[mt], 0x7632);
        const unsigned a2 = __byte_perm(v2[mt], v3[mt], 0x5410), a3 = __byte_perm(v2[mt], v3[mt], 0x7632);
        mma16816(o[hf * 4 + mt], a0, a1, a2, a3, pb0, pb1);
      }
    }
  }

  // ---- partial epilogue: normalise over the split, lse_s = ln sum exp
  float l_tot = l_run + __shfl_xor_sync(0xffffffffu, l_run, 1);
  l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 2);
  const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;
  const float lse = l_tot > 0.f ? (m_run + log2f(l_tot)) * 0.6931471805599453f : -INFINITY;
  const float ia = __shfl_sync(0xffffffffu, inv, (2 * q4) * 4), ib = __shfl_sync(0xffffffffu, inv, (2 * q4 + 1) * 4);
  const size_t row0 = ((size_t)r * hq + (size_t)kvh * group) * max_splits;
  if (q4 == 0 && g < group) lse_part[row0 + (size_t)g * max_splits + s] = lse;
#pragma unroll
  for (int hh = 0; hh < 2; ++hh) {
    const int head = 2 * q4 + hh;
    if (head < group) {
      float* dst = o_part + (row0 + (size_t)head * max_splits + s) * D;
      const float sc_ = hh ? ib : ia;
#pragma unroll
      for (int hf = 0; hf < 2; ++hf)
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
          *reinterpret_cast<float2*>(dst + 64 * hf + 8 * g + 2 * mt) =
              make_float2(o[hf * 4 + mt][hh] * sc_, o[hf * 4 + mt][2 + hh] * sc_);
    }
  }
}

}  // namespace

bool decode_mma_supported(const Ctx& c) { return c.dtype == MINIPIC_BF16 && c.d == 128 && c.group <= 8; }

void launch_decode_mma(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  if (a.num_seqs == 0) return;
  int warps = 1;
  for (int w = 4; w >= 1; --w)
    if (c.hkv % w == 0) { warps = w; break; }
  dim3 grid(sp.max_splits, a.num_seqs, c.hkv / warps);
  if (c.flags & MINIPIC_K_PREROTATED)
    decode_mma_kernel<false><<<grid, 32 * warps, 0, c.stream>>>(a, c.hq, c.hkv, c.group, c.scale_log2, c.rope, c.flags,
                                                               sp.split_len, sp.max_splits, o_part, lse_part);
  else
    decode_mma_kernel<true><<<grid, 32 * warps, 0, c.stream>>>(a, c.hq, c.hkv, c.group, c.scale_log2, c.rope, c.flags,
                                                              sp.split_len, sp.max_splits, o_part, lse_part);
  note_launch();
}

}  // namespace minipic
