// a10: split-KV decode partial kernel (bf16, head_dim 128, GQA group <= 8), HBM-bound.
//
// One warp owns one (sequence, KV head, split).  It is its own producer and consumer: lane 0 keeps a ring of kStages
// 16-token blocks in flight with cp.async.bulk.tensor (one 4 KB box of K and one of V per physical block, looked up in the
// block table; SWIZZLE_128B, so the fragment reads below are bank-conflict free), the whole warp then rotates K in
// registers at the request's logical positions (Eq. 2) and runs both contractions on the register-operand
// tensor path (mma.sync m16n8k16, bf16 x bf16 -> fp32), so the CUDA cores are left for the bf16->fp32 conversion and the two
// FMAs per K element.  Staging through shared memory (instead of streaming straight into registers, the
// round-1 kernel) takes the HBM latency off the warp's critical path: with the loads decoupled the rotation's ~500 extra
// instructions per block overlap the stream instead of adding to it.  The G query heads of the group share the rotated K
// tile.  Online softmax uses warp shuffles across the 4 lanes that hold one head's scores.  Partials (o_s normalised over
// the split, lse_s) go to the workspace; lse_merge_kernel (a11) combines them.
//
// Fragment trick: the dot products are sums over head_dim (QK^T) and over keys (PV), so any permutation of the
// summation index is legal as long as both operands use it.  That lets each lane feed the MMA fragments from
// whole 16-byte vectors:
//   QK^T as S^T[head, key] = Q'[head, d] K'^T[d, key]:  A = Q' (row g = head), B = K' (col g = key), and the lane
//     (g, q) reads for key rows g and g+8 the 16-byte chunks 2q, 2q+1 of both halves of head_dim - chunk c of the low half
//     and chunk c of the high half hold the two elements of the rotate-half pairs, so the rotation is lane-local.
//   PV as O^T[d, head] = V^T[d, key] P[key, head]:  the S^T accumulator layout IS the B-fragment layout of P; the
//     lane reads chunk g of both halves of V rows 2q, 2q+1, 2q+8, 2q+9 and two byte-permutes per register pair build
//     the A fragments.
#include <cuda.h>

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
// finc is PADDED: the 8 increments of frequency chunk c start at finc + 10 c (80 bytes apart), so that the four lane groups
// of a warp (chunks 2 q4 + j) read four different bank groups instead of the same one (ncu: 4-way conflict otherwise).
constexpr int kFincStride = 10;
__device__ __forceinline__ void rope_cs8(const unsigned long long* __restrict__ finc, int p, int chunk, float (&c)[8],
                                         float (&s)[8]) {
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    const unsigned long long ph = (unsigned long long)(unsigned)p * finc[chunk * kFincStride + e];
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

constexpr int kStages = MINIPIC_DECODE_STAGES;   // blocks in flight per warp (internal.h)
constexpr int kStageBytes = 8192;                // K block (4 KB) | V block (4 KB) of one KV head
constexpr unsigned kSpinLimit = 1u << 26;

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
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
__device__ __forceinline__ void tma_block(uint32_t dst, const CUtensorMap* tmap, uint32_t bar, int grp) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %3, %3, %4}], [%2];"
      ::"r"(dst), "l"(tmap), "r"(bar), "r"(0), "r"(grp) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}

template <bool kRotK, bool kKeyMask, int W>
__global__ void __launch_bounds__(32 * W, MINIPIC_DECODE_WARPS_PER_SM / W)
decode_mma_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v, DecodeArgs a,
                  int hq, int hkv, int group, float scale_log2, RopeParams rp, unsigned flags, int split_len,
                  int max_splits, float* __restrict__ o_part, float* __restrict__ lse_part) {
  constexpr int D = 128;
  // dynamic shared memory only (the swizzled block images need a 1024-byte aligned base):
  // [W warps][kStages][K 4 KB | V 4 KB] | F_i[64] | barriers[W * kStages]
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned long long* finc = reinterpret_cast<unsigned long long*>(smem_raw + W * kStages * kStageBytes);  // 64-bit phase increments
  unsigned long long* bars = finc + 8 * kFincStride;
  for (int i = threadIdx.x; i < 64; i += 32 * W) finc[(i >> 3) * kFincStride + (i & 7)] = rp.phase_inc[i];
  if (threadIdx.x == 0) {
    if (smem_addr(smem_raw) & 1023u) __trap();
    for (int i = 0; i < W * kStages; ++i) mbar_init(smem_addr(&bars[i]), 1);
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

  // this lane's 16-byte chunks of a row: j = 0, 1 -> chunks 2 q4 + j of the low half, j = 2, 3 -> the same of the high half
  // ---- Q' fragments (a3): head g of the group, rotated at the query's logical position
  unsigned qf[8][2];
  {
    uint4 ch[4];
    if (g < group) {
      const __nv_bfloat16* qrow = (const __nv_bfloat16*)a.q + ((size_t)r * hq + (size_t)kvh * group + g) * D;
#pragma unroll
      for (int j = 0; j < 4; ++j) ch[j] = __ldg(reinterpret_cast<const uint4*>(qrow + (2 * q4 + (j & 1) + 8 * (j >> 1)) * 8));
      if (!(flags & MINIPIC_Q_PREROTATED)) {
        const int qpos = __ldg(pos + kv_len - 1);
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          float c[8], sn[8];
          rope_cs8(finc, qpos, 2 * q4 + j, c, sn);
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

  const int kb0 = j_begin / kBlock, kb1 = (j_end + kBlock - 1) / kBlock, nb = kb1 - kb0;
  const uint32_t ring = smem_addr(smem_raw) + (uint32_t)warp * (kStages * kStageBytes);
  const uint32_t bar0 = smem_addr(&bars[warp * kStages]);
  // a4: block n of the split -> stage n % kStages (lane 0 only): one 4 KB box of K and one of V through the block table
  auto issue = [&](int n, int blk) {
    const int st = n % kStages;
    const int grp = (blk * hkv + kvh) * 2;   // row-group coordinate of (block, head) in the cache tensor map
    mbar_expect_tx(bar0 + 8u * st, kStageBytes);
    tma_block(ring + st * kStageBytes, &tmap_k, bar0 + 8u * st, grp);
    tma_block(ring + st * kStageBytes + 4096, &tmap_v, bar0 + 8u * st, grp);
  };
  int blk_next = 0;   // lane 0: physical block of the next block to issue, read from the block table one iteration early
  if (lane == 0) {
    for (int n = 0; n < kStages - 1 && n < nb; ++n) issue(n, __ldg(bt + kb0 + n));
    if (kStages - 1 < nb) blk_next = __ldg(bt + kb0 + kStages - 1);
  }

  // swizzled offsets of this lane's chunks inside a 4 KB block image: [row group (2)][half (2)][8 rows x 128 B], SWIZZLE_128B
  uint32_t koff[2];   // K rows g (group 0) and g + 8 (group 1) share the in-group offset: chunk 2 q4 + j of row g
#pragma unroll
  for (int j = 0; j < 2; ++j) koff[j] = (uint32_t)(g * 128 + (((2 * q4 + j) ^ g) << 4));
  uint32_t voff[4];   // V rows 2 q4 + (i & 1) + 8 (i >> 1), chunk g
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = 2 * q4 + (i & 1);
    voff[i] = (uint32_t)((i >> 1) * 2048 + row * 128 + ((g ^ row) << 4));
  }

  int pcur[2] = {0, 0};   // logical positions of this lane's rows g, g + 8 of the current block
  if (kRotK) {
#pragma unroll
    for (int t = 0; t < 2; ++t) pcur[t] = __ldg(pos + min(kb0 * kBlock + g + 8 * t, kv_len - 1));
  }
#pragma unroll 1
  for (int n = 0; n < nb; ++n) {
    const int kb = kb0 + n;
    // every lane is done with the stage that block n + kStages - 1 reuses (it held block n - 1): refill it
    __syncwarp();
    if (lane == 0 && n + kStages - 1 < nb) {
      issue(n + kStages - 1, blk_next);
      if (n + kStages < nb) blk_next = __ldg(bt + kb0 + n + kStages);
    }
    // a5 (first half): cos/sin of this lane's two rows, computed while the block is still in flight
    float cs[2][2][8], sn[2][2][8];
    // Measured and dropped: row g + 8 from row g by one angle-addition step with a (cos 8 f, sin 8 f) table in shared
    // memory (-72 instructions per block): 1.14 -> 1.43 ms.  The loop is bound by dependent latency at 3 warps per
    // scheduler, not by issue slots, and the second row's cos/sin then wait for the first row's MUFU results.
    if (kRotK) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
#pragma unroll
        for (int j = 0; j < 2; ++j) rope_cs8(finc, pcur[t], 2 * q4 + j, cs[t][j], sn[t][j]);
      }
    }
    const uint32_t stg = ring + (n % kStages) * kStageBytes;
    mbar_wait(bar0 + 8u * (n % kStages), (n / kStages) & 1);
    // ---- K rows g and g+8: 8 x 16-byte conflict-free shared loads
    uint4 kr[2][4];
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int j = 0; j < 4; ++j) kr[t][j] = lds128(stg + t * 2048 + (j >> 1) * 1024 + koff[j & 1]);
    // ---- a5: rotate in registers at pi_r(j)
    if (kRotK) {
#pragma unroll
      for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int j = 0; j < 2; ++j) rotate_chunks(kr[t][j], kr[t][j + 2], cs[t][j], sn[t][j]);
    }
    // positions of the NEXT block's two rows: a global load whose latency would otherwise sit at the top of every iteration
    // (ncu: 12 % of the stall samples were long-scoreboard waits on it).  Issued here, where the cos / sin registers are dead
    // (issued before the rotation it spilled to local memory).
    if (kRotK) {
#pragma unroll
      for (int t = 0; t < 2; ++t) pcur[t] = __ldg(pos + min((kb + 1) * kBlock + g + 8 * t, kv_len - 1));
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
    // ---- V rows 2q, 2q+1, 2q+8, 2q+9, chunk g of both halves
    uint4 vr[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) vr[i][hf] = lds128(stg + 4096 + hf * 1024 + voff[i]);
    if (kb * kBlock < j_begin || (kb + 1) * kBlock > j_end) {   // only the first / last block of a split (warp-uniform):
#pragma unroll
      for (int i = 0; i < 4; ++i) {                              // never multiply P = 0 with uninitialised cache bits
        const int jrow = kb * kBlock + 2 * q4 + (i & 1) + 8 * (i >> 1);
        if (jrow < j_begin || jrow >= j_end) { vr[i][0] = make_uint4(0, 0, 0, 0); vr[i][1] = make_uint4(0, 0, 0, 0); }
      }
    }
    // ---- a7: mask + online softmax (row = head g; its 16 scores live in 4 lanes x 4 registers)
    float sc[2][2];
    float m_blk = -INFINITY;
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int j = kb * kBlock + 8 * t + 2 * q4 + e;
        bool vis = j >= j_begin && j < j_end;
        if (kKeyMask && vis) vis = __ldg(pos + j) >= 0;   // MINIPIC_KEY_MASK: invisible to every row
        sc[t][e] = vis ? st[t][e] * scale_log2 : -INFINITY;
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

template <bool kRotK, bool kKeyMask, int W>
bool launch_k(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, const CUtensorMap& mk, const CUtensorMap& mv,
              float* o_part, float* lse_part) {
  const size_t smem = (size_t)W * kStages * kStageBytes + 8 * kFincStride * 8 + (size_t)W * kStages * 8;
  static bool attr_done[64] = {};   // per (function, device)
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_done[dev]) {
    if (cudaFuncSetAttribute(decode_mma_kernel<kRotK, kKeyMask, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
      note_error("decode_mma: cudaFuncSetAttribute(MaxDynamicSharedMemorySize) failed");
      return false;
    }
    if (dev >= 0 && dev < 64) attr_done[dev] = true;
  }
  dim3 grid((unsigned)sp.max_splits * (unsigned)a.num_seqs, c.hkv / W);
  decode_mma_kernel<kRotK, kKeyMask, W><<<grid, 32 * W, smem, c.stream>>>(mk, mv, a, c.hq, c.hkv, c.group, c.scale_log2, c.rope,
                                                               c.flags, sp.split_len, sp.max_splits, o_part, lse_part);
  return true;
}
template <int W>
bool launch_w(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, const CUtensorMap& mk, const CUtensorMap& mv,
              float* o_part, float* lse_part) {
  if (c.flags & MINIPIC_KEY_MASK)
    return (c.flags & MINIPIC_K_PREROTATED) ? launch_k<false, true, W>(c, a, sp, mk, mv, o_part, lse_part)
                                            : launch_k<true, true, W>(c, a, sp, mk, mv, o_part, lse_part);
  return (c.flags & MINIPIC_K_PREROTATED) ? launch_k<false, false, W>(c, a, sp, mk, mv, o_part, lse_part)
                                          : launch_k<true, false, W>(c, a, sp, mk, mv, o_part, lse_part);
}

}  // namespace

bool decode_mma_supported(const Ctx& c) { return c.dtype == MINIPIC_BF16 && c.d == 128 && c.group <= 8; }

bool launch_decode_mma(const Ctx& c, const DecodeArgs& a, const SplitPlan& sp, float* o_part, float* lse_part) {
  if (a.num_seqs == 0) return true;
  CUtensorMap mk, mv;
  if (!make_cache_tensor_map(&mk, a.k_cache, c.num_blocks, c.hkv, 2) || !make_cache_tensor_map(&mv, a.v_cache, c.num_blocks, c.hkv, 2)) {
    note_error("decode_mma: cuTensorMapEncodeTiled failed (driver entry point missing or bad tensor geometry)");
    return false;
  }
  // W warps = W KV heads of one (sequence, split) per CTA
  bool ok;
  if (c.hkv % 4 == 0) ok = launch_w<4>(c, a, sp, mk, mv, o_part, lse_part);
  else if (c.hkv % 2 == 0) ok = launch_w<2>(c, a, sp, mk, mv, o_part, lse_part);
  else ok = launch_w<1>(c, a, sp, mk, mv, o_part, lse_part);
  if (ok) note_launch();
  return ok;
}

}  // namespace minipic
