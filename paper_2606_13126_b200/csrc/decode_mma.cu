// a10: split-KV decode partial kernel (bf16, head_dim 128, GQA group <= 8), HBM-bound.
//
// One warp owns one (sequence, KV head, split): it streams the split's 16-token blocks straight from the paged
// cache into registers with coalesced 16-byte loads (every 32-byte sector it touches is fully used), rotates K in
// registers at the request's logical positions (Eq. 2), and runs both contractions on the
// register-operand tensor path (mma.sync m16n8k16, bf16 x bf16 -> fp32) so that the CUDA cores are left for the
// bf16->fp32 conversion and the two FMAs per K element.  The G query heads of the group share the
// rotated K tile.  Online softmax uses warp shuffles across the 4 lanes that hold one head's scores.
// Partials (o_s normalised over the split, lse_s) go to the workspace; lse_merge_kernel (a11) combines them.
// The W warps of a CTA are W KV heads of the SAME (sequence, split): they share the (cos, sin) tile of every 16-key block
// through a small shared-memory ring instead of each recomputing it (see "cos/sin ring" below).
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
// bf16 rounding of the rotated operand).  No global-memory traffic: in this HBM-bound kernel a cos/sin table lookup
// from global memory costs as many L1 wavefronts as the KV stream itself (ncu: l1tex 92% with the table).
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

// ---- cos/sin ring shared by the warps (KV heads) of a CTA ------------------------------------------------------------
// The warps of a CTA work on the SAME 16 key positions of the same (sequence, split); only the KV head differs.  The
// (cos, sin) tile of a block - 16 positions x 64 frequencies - is therefore computed ONCE per CTA: every warp computes 1/W
// of it for the block kLook iterations ahead (8 * 4/W exact evaluations per lane instead of 32), stores it to a ring of
// kSlots tiles in shared memory, and picks up its own 32 pairs with 16 LDS.128.  Hand-off is two mbarriers per slot
// (full / empty, one arrival per warp), so the warps stay loosely coupled (up to kLook blocks of skew) instead of running
// in lock step.  Tile layout: row r (512 B) x 8 chunks of 8 frequencies (64 B) x 4 pieces of 16 B = (c0, c1, s0, s1) of two
// neighbouring frequencies - the operand order of the packed f32x2 rotation; the piece index is XOR-swizzled with
// ((r & 1) << 1 | (chunk >> 1) & 1) so that both the writers' and the readers' quarter-warps touch 32 distinct banks.
constexpr int kSlots = 4, kLook = 2, kCsTileBytes = kBlock * 512;
constexpr unsigned kSpinLimit = 1u << 26;

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  unsigned spins = 0;
  for (;;) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (done) return;
    if (++spins > kSpinLimit) __trap();   // a protocol bug must fail loudly instead of hanging the GPU
  }
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, float a, float b, float c, float d) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
// rotate word w of a (lo, hi) chunk pair with the piece (c0, c1, s0, s1): packed f32x2 math, one RN to bf16
__device__ __forceinline__ void rotate_word(unsigned& l, unsigned& h, const uint4& cs) {
  const uint64_t a = pk2(bf16lo(l), bf16hi(l)), b = pk2(bf16lo(h), bf16hi(h));
  const uint64_t c = ((uint64_t)cs.y << 32) | cs.x, s = ((uint64_t)cs.w << 32) | cs.z;
  const uint64_t ns = mul2(s, pk2(-1.f, -1.f));
  float x0, x1, y0, y1;
  upk2(fma2(b, ns, mul2(a, c)), x0, x1);
  upk2(fma2(a, s, mul2(b, c)), y0, y1);
  l = pack_bf16(x0, x1);
  h = pack_bf16(y0, y1);
}

template <bool kRotK, int W>
__global__ void __launch_bounds__(32 * W, 16 / W)   // 16 warps / SM; 4-warp CTAs measured 6 % faster than 8-warp CTAs
decode_mma_kernel(DecodeArgs a, int hq, int hkv, int group, float scale_log2, RopeParams rp, unsigned flags,
                  int split_len, int max_splits, float* __restrict__ o_part, float* __restrict__ lse_part) {
  constexpr int D = 128;
  __shared__ unsigned long long finc[64];  // F_i: 64-bit fixed-point phase increments (turns per position)
  __shared__ __align__(128) unsigned char cs_ring[kRotK ? kSlots * kCsTileBytes : 16];
  __shared__ unsigned long long bars[2 * kSlots];
  for (int i = threadIdx.x; i < 64; i += 32 * W) finc[i] = rp.phase_inc[i];
  if (kRotK && threadIdx.x == 0) {
    for (int i = 0; i < 2 * kSlots; ++i) mbar_init(smem_addr(&bars[i]), W);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 2, q4 = lane & 3;
  const int s = blockIdx.x % max_splits, r = blockIdx.x / max_splits;   // the sequence count lives in grid.x: no 65535 limit
  const int kvh = blockIdx.y * W + warp;
  const int kv_len = __ldg(a.kv_lens + r);
  if (s * split_len >= kv_len) return;  // the merge kernel never reads empty splits (uniform over the CTA)
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

  // ---- this lane's share of a (cos, sin) tile: rows prow0 + 4 i (i < 4 / W), frequency chunk pc
  const int pc = (lane & 3) + 4 * ((lane >> 3) & 1);
  const int prow0 = warp * (kBlock / W) + ((lane >> 2) & 1) + 2 * (lane >> 4);
  const uint32_t ring0 = smem_addr(cs_ring), bar0 = smem_addr(bars);
  const uint32_t psw = (uint32_t)((((lane >> 2) & 1) << 1) | ((pc >> 1) & 1));   // row parity of prow0 + 4 i = (lane >> 2) & 1
  const uint32_t rsw = (uint32_t)(((g & 1) << 1) | (q4 >> 1));                   // reader: rows g, g + 8, chunks q4, q4 + 4
  auto produce = [&](int n) {   // tile of block kb0 + n -> slot n % kSlots
    const int slot = n % kSlots, kb = kb0 + n;
    if (n >= kSlots) mbar_wait(bar0 + 8u * (kSlots + slot), ((n / kSlots) & 1) ^ 1);   // every warp is done with block n - kSlots
    const uint32_t tile = ring0 + slot * kCsTileBytes;
#pragma unroll
    for (int i = 0; i < 4 / W; ++i) {
      const int row = prow0 + 4 * i;
      const int p = __ldg(pos + min(kb * kBlock + row, kv_len - 1));
      float c[8], sn[8];
      rope_cs8(finc, p, pc * 8, c, sn);
      const uint32_t base = tile + row * 512 + pc * 64;
#pragma unroll
      for (int k = 0; k < 4; ++k) sts128(base + ((k ^ psw) << 4), c[2 * k], c[2 * k + 1], sn[2 * k], sn[2 * k + 1]);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8u * slot);
  };
  if (kRotK) {
#pragma unroll 1
    for (int n = 0; n < kLook && kb0 + n < kb1; ++n) produce(n);
  }

  int blk = __ldg(bt + kb0);
#pragma unroll 1
  for (int kb = kb0; kb < kb1; ++kb) {
    const int n = kb - kb0;
    const size_t base = ((size_t)blk * hkv + kvh) * (kBlock * D);
    if (kb + 1 < kb1) blk = __ldg(bt + kb + 1);
    // ---- a4: K rows g and g+8, chunks q4 + 4j: 8 x 16-byte streaming loads
    uint4 kr[2][4];
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int j = 0; j < 4; ++j) kr[t][j] = ldg_stream16(kc + base + (g + 8 * t) * D + (q4 + 4 * j) * 8);
    // ---- a5: rotate in registers at pi_r(j); cos/sin from the CTA's shared tile (this warp's share of the tile kLook
    //      blocks ahead is computed first, under the latency of the loads above)
    if (kRotK) {
      if (kb + kLook < kb1) produce(n + kLook);
      const int slot = n % kSlots;
      mbar_wait(bar0 + 8u * slot, (n / kSlots) & 1);
      const uint32_t tile = ring0 + slot * kCsTileBytes;
#pragma unroll
      for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const uint32_t src = tile + (g + 8 * t) * 512 + (q4 + 4 * j) * 64;
          unsigned* l = reinterpret_cast<unsigned*>(&kr[t][j]);
          unsigned* h = reinterpret_cast<unsigned*>(&kr[t][j + 2]);
#pragma unroll
          for (int k = 0; k < 4; ++k) rotate_word(l[k], h[k], lds128(src + ((k ^ rsw) << 4)));
        }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8u * (kSlots + slot));   // this warp no longer needs the tile
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

template <int W>
void launch_w(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  dim3 grid((unsigned)sp.max_splits * (unsigned)a.num_seqs, c.hkv / W);
  if (c.flags & MINIPIC_K_PREROTATED)
    decode_mma_kernel<false, W><<<grid, 32 * W, 0, c.stream>>>(a, c.hq, c.hkv, c.group, c.scale_log2, c.rope, c.flags,
                                                               sp.split_len, sp.max_splits, o_part, lse_part);
  else
    decode_mma_kernel<true, W><<<grid, 32 * W, 0, c.stream>>>(a, c.hq, c.hkv, c.group, c.scale_log2, c.rope, c.flags,
                                                              sp.split_len, sp.max_splits, o_part, lse_part);
}

}  // namespace

bool decode_mma_supported(const Ctx& c) { return c.dtype == MINIPIC_BF16 && c.d == 128 && c.group <= 8; }

void launch_decode_mma(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  if (a.num_seqs == 0) return;
  // W warps = W KV heads of one (sequence, split) per CTA; they share the (cos, sin) tiles through shared memory
  if (c.hkv % 4 == 0) launch_w<4>(c, a, sp, o_part, lse_part);
  else if (c.hkv % 2 == 0) launch_w<2>(c, a, sp, o_part, lse_part);
  else launch_w<1>(c, a, sp, o_part, lse_part);
  note_launch();
}

}  // namespace minipic
