// a2-a9: fused RoPE-in-attention prefill for sm_100a (bf16, head_dim 128, GQA group 1/2/4/8).
//
// Work item = (Q tile, KV head).  A Q tile is up to 128/G consecutive query tokens of one request that share
// vis_lo (one span, or suffix rows); its 128 MMA rows are (token, head-in-group) pairs, so one rotated K tile
// serves the whole GQA group.  A tiny plan kernel (a2) cuts the query rows into tiles, computes each tile's KV
// range [floor16(vis_lo), idx_last] (span-mask TILE SKIPPING: keys outside it are never touched) and sorts the
// tiles longest-first; a persistent kernel (one CTA per SM, 10 warps) then runs, per KV tile of 128 keys:
//
//   warp 8     TMA producer : gathers the tile's 8 physical blocks through the block table with
//                             cp.async.bulk.tensor (SWIZZLE_128B boxes of 16 keys x 64 dims) into smem  (a4)
//   warps 4-7  rotation     : Q load + RoPE once per item (a3); K tile RoPE in place, smem -> registers -> smem,
//                             one key per thread, cos/sin by table lookup or in-register phase (a5)
//   warp 9     MMA issuer   : tcgen05.mma S = Q' K'^T into TMEM (double-buffered), O += P V              (a6, a8)
//   warps 0-3  softmax      : tcgen05.ld S (one row per thread - no shuffles needed), mask, online softmax with
//                             lazy rescale, P -> bf16 -> smem; epilogue O / l -> out, LSE                 (a7, a9)
//
// All hand-offs are mbarriers; generic-proxy smem writes are fenced with fence.proxy.async before the MMA reads.
#include <cuda.h>
#include <cstdio>

#include "internal.h"

namespace minipic {

namespace {

constexpr int BM = 128, BN = 128, D = 128;
constexpr int kTileBytes = BN * D * 2;       // 32 KB: one K / V / Q / P tile
constexpr int kHalfBytes = kTileBytes / 2;   // [half of head_dim or keys][128 rows][128 B]
constexpr int kThreads = 320;
constexpr int kMaxBins = 4096;

struct TileDesc { int t0, ntok, r, idx0, lo, n_kv; };
struct PlanHeader { int n_tiles; int next_item; int pad[62]; };

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  unsigned long long spins = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (done) break;
    if (++spins > (1ull << 24)) {  // watchdog: a protocol bug must fault, not hang the GPU
      printf("minipic prefill: mbarrier wait timed out (block %d thread %d bar %u parity %u)\n", blockIdx.x, threadIdx.x,
             bar, parity);
      __trap();
    }
  }
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tmap, uint32_t bar, int x, int y) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"(tmap), "r"(bar), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* v) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
      "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float* v) {
  const uint32_t* r = reinterpret_cast<const uint32_t*>(v);
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
      "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]),
        "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]),
        "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
      : "memory");
}
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor (SWIZZLE_128B, version 1): start address, leading / stride byte offsets
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: D fp32, A/B bf16, M=128, N=128; b_mn = B operand is MN-major (V tile)
__host__ __device__ constexpr uint32_t instr_desc(bool b_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn ? 1u : 0u) << 16) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

// byte offset of 16-byte chunk `c` (0..15) of row `r` inside a [2][128 rows][128 B] SWIZZLE_128B tile
__device__ __forceinline__ uint32_t tile_off(int r, int c) {
  return (uint32_t)((c >> 3) * kHalfBytes + r * 128 + (((c & 7) ^ (r & 7)) << 4));
}

__device__ __forceinline__ void cs8(const RopeParams& rp, const unsigned long long* finc, int p, int i0, float (&c)[8],
                                    float (&s)[8]) {
  if (p < rp.table_len) {  // PAPER.md:113 "a cos/sin table lookup"
    const float4* t = reinterpret_cast<const float4*>(rp.table + (size_t)p * rp.half + i0);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const float4 v = __ldg(t + e);
      c[2 * e] = v.x; s[2 * e] = v.y; c[2 * e + 1] = v.z; s[2 * e + 1] = v.w;
    }
  } else {
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const unsigned long long ph = (unsigned long long)(unsigned)p * finc[i0 + e];
      const float a = (float)(int)(ph >> 32) * 1.4629180792671596e-9f;
      c[e] = __cosf(a); s[e] = __sinf(a);
    }
  }
}
__device__ __forceinline__ void rotate16(uint4& lo, uint4& hi, const float (&c)[8], const float (&s)[8]) {
  unsigned* l = reinterpret_cast<unsigned*>(&lo);
  unsigned* h = reinterpret_cast<unsigned*>(&hi);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const float a0 = bf16lo(l[w]), a1 = bf16hi(l[w]), b0 = bf16lo(h[w]), b1 = bf16hi(h[w]);
    l[w] = pack_bf16(a0 * c[2 * w] - b0 * s[2 * w], a1 * c[2 * w + 1] - b1 * s[2 * w + 1]);
    h[w] = pack_bf16(b0 * c[2 * w] + a0 * s[2 * w], b1 * c[2 * w + 1] + a1 * s[2 * w + 1]);
  }
}

// ------------------------------------------------------------------------------------------------ a2: plan
__device__ __forceinline__ bool tile_starts(const PrefillArgs& a, int t, int r, int tok) {
  if (t == __ldg(a.cu_q_lens + r)) return true;
  const int i1 = __ldg(a.q_seq_idx + t), i0 = __ldg(a.q_seq_idx + t - 1);
  const int l1 = __ldg(a.q_vis_lo + t), l0 = __ldg(a.q_vis_lo + t - 1);
  return i1 != i0 + 1 || l1 != l0 || ((i1 - max(l1, 0)) % tok) == 0;
}

__global__ void __launch_bounds__(1024) prefill_plan_kernel(PrefillArgs a, int tok, PlanHeader* hdr, TileDesc* sorted,
                                                            TileDesc* tmp) {
  __shared__ int hist[kMaxBins];
  __shared__ int n_tiles_s;
  for (int i = threadIdx.x; i < kMaxBins; i += blockDim.x) hist[i] = 0;
  if (threadIdx.x == 0) n_tiles_s = 0;
  __syncthreads();
  for (int t = threadIdx.x; t < a.num_q_tokens; t += blockDim.x) {
    int lo_r = 0, hi_r = a.num_reqs;
    while (hi_r - lo_r > 1) {
      const int mid = (lo_r + hi_r) >> 1;
      if (__ldg(a.cu_q_lens + mid) <= t) lo_r = mid; else hi_r = mid;
    }
    const int r = lo_r;
    if (!tile_starts(a, t, r, tok)) continue;
    const int t_end = __ldg(a.cu_q_lens + r + 1);
    int n = 1;
    while (n < tok && t + n < t_end && !tile_starts(a, t + n, r, tok)) ++n;
    TileDesc td;
    td.t0 = t; td.ntok = n; td.r = r; td.idx0 = __ldg(a.q_seq_idx + t); td.lo = max(__ldg(a.q_vis_lo + t), 0);
    const int kv_lo = td.lo & ~(kBlock - 1), kv_hi = min(td.idx0 + n, __ldg(a.kv_lens + r));
    td.n_kv = kv_hi > kv_lo ? (kv_hi - kv_lo + BN - 1) / BN : 0;
    const int slot = atomicAdd(&n_tiles_s, 1);
    tmp[slot] = td;
    atomicAdd(&hist[min(td.n_kv, kMaxBins - 1)], 1);
  }
  __syncthreads();
  // exclusive prefix over bins in DESCENDING cost order (longest-first), one warp
  if (threadIdx.x < 32) {
    int carry = 0;
    for (int base = kMaxBins - 32; base >= 0; base -= 32) {
      const int b = base + 31 - threadIdx.x;  // lane 0 takes the most expensive bin of the chunk
      const int v = hist[b];
      int incl = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, o);
        if ((int)threadIdx.x >= o) incl += n;
      }
      hist[b] = carry + incl - v;
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  const int n_tiles = n_tiles_s;
  for (int i = threadIdx.x; i < n_tiles; i += blockDim.x) {
    const TileDesc td = tmp[i];
    sorted[atomicAdd(&hist[min(td.n_kv, kMaxBins - 1)], 1)] = td;
  }
  if (threadIdx.x == 0) { hdr->n_tiles = n_tiles; hdr->next_item = 0; }
}

// ------------------------------------------------------------------------------------------------ main kernel
struct Smem {
  alignas(1024) unsigned char q[kTileBytes];
  alignas(1024) unsigned char k[2][kTileBytes];
  alignas(1024) unsigned char v[2][kTileBytes];
  alignas(1024) unsigned char p[kTileBytes];
  unsigned long long finc[64];
  unsigned long long bars[32];
  uint32_t tmem_base;
};
enum Bar { Q_FULL = 0, Q_EMPTY, K_FULL, K_READY = K_FULL + 2, K_EMPTY = K_READY + 2, V_FULL = K_EMPTY + 2,
           V_READY = V_FULL + 2, V_EMPTY = V_READY + 2, S_FULL = V_EMPTY + 2, S_EMPTY = S_FULL + 2, P_FULL = S_EMPTY + 2,
           PV_DONE, O_FREE, NUM_BARS };

struct Params {
  PrefillArgs a;
  int hq, hkv;
  float scale_log2;
  unsigned flags;
  const PlanHeader* hdr;
  const TileDesc* tiles;
  RopeParams rp;
};

template <int G>
__global__ void __launch_bounds__(kThreads, 1)
prefill_sm100_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
                     const __grid_constant__ Params prm) {
  extern __shared__ unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  constexpr int TOK = BM / G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const PrefillArgs& a = prm.a;
  const uint32_t bar0 = smem_u32(sm.bars);
  auto bar = [&](int b) { return bar0 + 8u * (uint32_t)b; };

  if (threadIdx.x < 64) sm.finc[threadIdx.x] = prm.rp.phase_inc[threadIdx.x];
  if (threadIdx.x == 0) {
    mbar_init(bar(Q_FULL), 128); mbar_init(bar(Q_EMPTY), 1);
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar(K_FULL + s), 1); mbar_init(bar(K_READY + s), 128); mbar_init(bar(K_EMPTY + s), 1);
      mbar_init(bar(V_FULL + s), 1); mbar_init(bar(V_READY + s), 128); mbar_init(bar(V_EMPTY + s), 1);
      mbar_init(bar(S_FULL + s), 1); mbar_init(bar(S_EMPTY + s), 128);
    }
    mbar_init(bar(P_FULL), 128); mbar_init(bar(PV_DONE), 1); mbar_init(bar(O_FREE), 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 9) {  // TMEM: 512 columns (S0, S1, O at 0, 128, 256)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;

  const int n_tiles = prm.hdr->n_tiles;
  const int n_items = n_tiles * prm.hkv;
  const int nctas = gridDim.x;
  // static longest-first assignment in snake order: round k gives CTA b item k*nctas + (k odd ? nctas-1-b : b)
  auto item_of = [&](int k) { return k * nctas + ((k & 1) ? nctas - 1 - (int)blockIdx.x : (int)blockIdx.x); };

  if (warp == 8) {
    // ============================================================ TMA producer (a4)
    uint32_t kv_it = 0;
    for (int k = 0;; ++k) {
      const int item = item_of(k);
      if (item >= n_items) break;
      const TileDesc td = prm.tiles[item / prm.hkv];
      const int kvh = item % prm.hkv;
      const int kv_lo = td.lo & ~(kBlock - 1), kv_hi = min(td.idx0 + td.ntok, __ldg(a.kv_lens + td.r));
      const int* bt = a.block_tables + (size_t)td.r * a.max_blocks;
      for (int i = 0; i < td.n_kv; ++i, ++kv_it) {
        const int st = kv_it & 1;
        const uint32_t par = ((kv_it >> 1) & 1) ^ 1;
        const int j0 = kv_lo + i * BN;
        const int nblk = min(BN / kBlock, (kv_hi - j0 + kBlock - 1) / kBlock);
        int y = 0;
        if (lane < nblk) y = (__ldg(bt + j0 / kBlock + lane) * prm.hkv + kvh) * kBlock;
        if (lane == 0) { mbar_wait(bar(K_EMPTY + st), par); mbar_expect_tx(bar(K_FULL + st), nblk * 4096); }
        __syncwarp();
        if (lane < nblk) {
          const uint32_t dst = smem_u32(sm.k[st]) + lane * 2048;
          tma_load_2d(dst, &tmap_k, bar(K_FULL + st), 0, y);
          tma_load_2d(dst + kHalfBytes, &tmap_k, bar(K_FULL + st), 64, y);
        }
        if (lane == 0) { mbar_wait(bar(V_EMPTY + st), par); mbar_expect_tx(bar(V_FULL + st), nblk * 4096); }
        __syncwarp();
        if (lane < nblk) {
          const uint32_t dst = smem_u32(sm.v[st]) + lane * 2048;
          tma_load_2d(dst, &tmap_v, bar(V_FULL + st), 0, y);
          tma_load_2d(dst + kHalfBytes, &tmap_v, bar(V_FULL + st), 64, y);
        }
      }
    }
  } else if (warp == 9) {
    // ============================================================ MMA issuer (a6, a8)
    const uint32_t idesc_qk = instr_desc(false), idesc_pv = instr_desc(true);
    const uint32_t q_addr = smem_u32(sm.q), p_addr = smem_u32(sm.p);
    uint32_t kv_it = 0, s_it = 0, pv_it = 0;
    int n_used = 0;   // items with at least one KV tile (only those touch the Q / O barriers)
    for (int k = 0;; ++k) {
      const int item = item_of(k);
      if (item >= n_items) break;
      const TileDesc td = prm.tiles[item / prm.hkv];
      if (td.n_kv == 0) continue;
      auto issue_qk = [&](uint32_t kv_i, uint32_t s_i) {
        const int st = kv_i & 1, sb = s_i & 1;
        mbar_wait(bar(K_READY + st), (kv_i >> 1) & 1);
        mbar_wait(bar(S_EMPTY + sb), ((s_i >> 1) & 1) ^ 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t k_addr = smem_u32(sm.k[st]);
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks) {
            const uint32_t off = (ks >> 2) * kHalfBytes + (ks & 3) * 32;
            umma_bf16(tmem + sb * BN, smem_desc(q_addr + off, 16, 1024), smem_desc(k_addr + off, 16, 1024), idesc_qk, ks > 0);
          }
          tc_commit(bar(S_FULL + sb));
          tc_commit(bar(K_EMPTY + st));
        }
        __syncwarp();
      };
      mbar_wait(bar(Q_FULL), n_used & 1);
      issue_qk(kv_it, s_it);
      for (int i = 0; i < td.n_kv; ++i) {
        if (i + 1 < td.n_kv) issue_qk(kv_it + i + 1, s_it + i + 1);
        if (i == max(td.n_kv - 2, 0) && lane == 0) tc_commit(bar(Q_EMPTY));  // the item's last QK has been issued
        const int st = (kv_it + i) & 1;
        mbar_wait(bar(P_FULL), pv_it & 1);
        mbar_wait(bar(V_READY + st), ((kv_it + i) >> 1) & 1);
        if (i == 0) mbar_wait(bar(O_FREE), (n_used & 1) ^ 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t v_addr = smem_u32(sm.v[st]);
#pragma unroll
          for (int ks = 0; ks < BN / 16; ++ks) {
            const uint32_t aoff = (ks >> 2) * kHalfBytes + (ks & 3) * 32;
            umma_bf16(tmem + 2 * BN, smem_desc(p_addr + aoff, 16, 1024), smem_desc(v_addr + ks * 2048, kHalfBytes, 1024),
                      idesc_pv, (i > 0 || ks > 0));
          }
          tc_commit(bar(PV_DONE));
          tc_commit(bar(V_EMPTY + st));
        }
        __syncwarp();
        ++pv_it;
      }
      kv_it += td.n_kv; s_it += td.n_kv;
      ++n_used;
    }
  } else if (warp >= 4) {
    // ============================================================ rotation warps: Q (a3) and K tiles (a5)
    const int row = threadIdx.x - 128;
    uint32_t kv_it = 0;
    int n_used = 0;
    for (int k = 0;; ++k) {
      const int item = item_of(k);
      if (item >= n_items) break;
      const TileDesc td = prm.tiles[item / prm.hkv];
      const int kvh = item % prm.hkv;
      if (td.n_kv == 0) continue;
      const int* pos = a.kv_positions + __ldg(a.cu_kv_lens + td.r);
      const int kv_lo = td.lo & ~(kBlock - 1), kv_hi = min(td.idx0 + td.ntok, __ldg(a.kv_lens + td.r));
      // ---- Q tile: row = token * G + head-in-group
      mbar_wait(bar(Q_EMPTY), (n_used & 1) ^ 1);
      {
        const int tok = row / G, hg = row % G;
        if (tok < td.ntok) {
          const __nv_bfloat16* qrow = (const __nv_bfloat16*)a.q + ((size_t)(td.t0 + tok) * prm.hq + kvh * G + hg) * D;
          const int qpos = __ldg(pos + td.idx0 + tok);
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            uint4 lo = __ldg(reinterpret_cast<const uint4*>(qrow + 8 * c));
            uint4 hi = __ldg(reinterpret_cast<const uint4*>(qrow + 64 + 8 * c));
            if (!(prm.flags & MINIPIC_Q_PREROTATED)) {
              float cs[8], sn[8];
              cs8(prm.rp, sm.finc, qpos, 8 * c, cs, sn);
              rotate16(lo, hi, cs, sn);
            }
            *reinterpret_cast<uint4*>(sm.q + tile_off(row, c)) = lo;
            *reinterpret_cast<uint4*>(sm.q + tile_off(row, c + 8)) = hi;
          }
        } else {
#pragma unroll
          for (int c = 0; c < 16; ++c) *reinterpret_cast<uint4*>(sm.q + tile_off(row, c)) = make_uint4(0, 0, 0, 0);
        }
      }
      fence_proxy_async();
      mbar_arrive(bar(Q_FULL));
      // ---- K tiles: one key per thread, rotated in place in the UMMA layout
      for (int i = 0; i < td.n_kv; ++i, ++kv_it) {
        const int st = kv_it & 1;
        const uint32_t par = (kv_it >> 1) & 1;
        const int j = kv_lo + i * BN + row;
        mbar_wait(bar(K_FULL + st), par);
        if (!(prm.flags & MINIPIC_K_PREROTATED) && j < kv_hi) {
          const int p = __ldg(pos + j);
          unsigned char* kt = sm.k[st];
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            uint4 lo = *reinterpret_cast<uint4*>(kt + tile_off(row, c));
            uint4 hi = *reinterpret_cast<uint4*>(kt + tile_off(row, c + 8));
            float cs[8], sn[8];
            cs8(prm.rp, sm.finc, p, 8 * c, cs, sn);
            rotate16(lo, hi, cs, sn);
            *reinterpret_cast<uint4*>(kt + tile_off(row, c)) = lo;
            *reinterpret_cast<uint4*>(kt + tile_off(row, c + 8)) = hi;
          }
        }
        fence_proxy_async();
        mbar_arrive(bar(K_READY + st));
        // V: rows at or beyond the item's last visible key get P = 0; make sure 0 * (stale / uninitialised bits) != NaN
        mbar_wait(bar(V_FULL + st), par);
        if (j >= kv_hi) {
#pragma unroll
          for (int c = 0; c < 16; ++c) *reinterpret_cast<uint4*>(sm.v[st] + tile_off(row, c)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async();
        mbar_arrive(bar(V_READY + st));
      }
      ++n_used;
    }
  } else {
    // ============================================================ softmax + epilogue warps (a7, a9): thread = row
    const int row = threadIdx.x;
    const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);
    uint32_t s_it = 0, pv_it = 0;
    for (int k = 0;; ++k) {
      const int item = item_of(k);
      if (item >= n_items) break;
      const TileDesc td = prm.tiles[item / prm.hkv];
      const int kvh = item % prm.hkv;
      const int tok = row / G, hg = row % G;
      const bool row_ok = tok < td.ntok;
      const int idx_row = td.idx0 + tok;
      const int kv_lo = td.lo & ~(kBlock - 1);
      float m_used = -INFINITY, l_run = 0.f;   // m in log2 units (score * scale * log2 e)
      for (int i = 0; i < td.n_kv; ++i, ++s_it) {
        const int sb = s_it & 1;
        const int j0 = kv_lo + i * BN;
        float s[BN];
        mbar_wait(bar(S_FULL + sb), (s_it >> 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32(t_lane + sb * BN + c * 32, s + c * 32);
        tmem_wait_ld();
        tc_fence_before();
        mbar_arrive(bar(S_EMPTY + sb));
        const bool full = (j0 >= td.lo) && (j0 + BN - 1 <= td.idx0);
        float mx = -INFINITY;
        if (full) {
#pragma unroll
          for (int c = 0; c < BN; ++c) mx = fmaxf(mx, s[c]);
        } else {
#pragma unroll
          for (int c = 0; c < BN; ++c) {
            const int j = j0 + c;
            s[c] = (j >= td.lo && j <= idx_row) ? s[c] : -INFINITY;
            mx = fmaxf(mx, s[c]);
          }
        }
        const float m_new = fmaxf(m_used, mx * prm.scale_log2);
        const bool grow = m_new > m_used + 8.f;   // lazy rescale: P may exceed 1 by up to 2^8 before O, l are rescaled
        bool pv_waited = (i == 0);
        if (i == 0) {
          m_used = m_new;
        } else if (__any_sync(0xffffffffu, grow)) {
          mbar_wait(bar(PV_DONE), pv_it & 1);     // O is stable once PV(i-1) has completed
          pv_waited = true;
          const float corr = grow ? fast_exp2(m_used - m_new) : 1.f;
          if (grow) { l_run *= corr; m_used = m_new; }
          tc_fence_after();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            float o[32];
            tmem_ld32(t_lane + 2 * BN + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] *= corr;
            tmem_st32(t_lane + 2 * BN + c * 32, o);
          }
          tmem_wait_st();
          tc_fence_before();
        }
        const float m_sub = (m_used == -INFINITY) ? 0.f : m_used;
        float lsum = 0.f;
        uint4 pk[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) {
          float pv[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) { pv[e] = fast_exp2(fmaf(s[8 * c + e], prm.scale_log2, -m_sub)); lsum += pv[e]; }
          pk[c].x = pack_bf16(pv[0], pv[1]); pk[c].y = pack_bf16(pv[2], pv[3]);
          pk[c].z = pack_bf16(pv[4], pv[5]); pk[c].w = pack_bf16(pv[6], pv[7]);
        }
        if (!pv_waited) mbar_wait(bar(PV_DONE), pv_it & 1);   // the single P buffer is free once PV(i-1) has read it
        if (i > 0) ++pv_it;
#pragma unroll
        for (int c = 0; c < 16; ++c) *reinterpret_cast<uint4*>(sm.p + tile_off(row, c)) = pk[c];
        l_run += lsum;
        fence_proxy_async();
        mbar_arrive(bar(P_FULL));
      }
      if (td.n_kv > 0) {
        mbar_wait(bar(PV_DONE), pv_it & 1);
        ++pv_it;
        tc_fence_after();
      }
      // ---- epilogue (a9): O / l -> out, LSE = ln sum exp of the scaled scores
      const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
      __nv_bfloat16* orow = (__nv_bfloat16*)a.out + ((size_t)(td.t0 + tok) * prm.hq + kvh * G + hg) * D;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        float o[32];
        if (td.n_kv > 0) { tmem_ld32(t_lane + 2 * BN + c * 32, o); tmem_wait_ld(); }
        else {
#pragma unroll
          for (int e = 0; e < 32; ++e) o[e] = 0.f;
        }
        if (row_ok) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            uint4 w;
            w.x = pack_bf16(o[8 * e] * inv, o[8 * e + 1] * inv); w.y = pack_bf16(o[8 * e + 2] * inv, o[8 * e + 3] * inv);
            w.z = pack_bf16(o[8 * e + 4] * inv, o[8 * e + 5] * inv); w.w = pack_bf16(o[8 * e + 6] * inv, o[8 * e + 7] * inv);
            *reinterpret_cast<uint4*>(orow + c * 32 + e * 8) = w;
          }
        }
      }
      if (row_ok)
        a.lse[(size_t)(td.t0 + tok) * prm.hq + kvh * G + hg] =
            l_run > 0.f ? (m_used + log2f(l_run)) * 0.6931471805599453f : -INFINITY;
      if (td.n_kv > 0) { tc_fence_before(); mbar_arrive(bar(O_FREE)); }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 9) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
  }
}

// ------------------------------------------------------------------------------------------------ host
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}
// cache viewed as a 2-D bf16 matrix [num_blocks * Hkv * 16 rows][128]; box = 16 rows x 64 columns, SWIZZLE_128B
bool make_cache_map(CUtensorMap* m, const void* cache, int num_blocks, int hkv) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[2] = {(cuuint64_t)D, (cuuint64_t)num_blocks * hkv * kBlock};
  cuuint64_t strides[1] = {(cuuint64_t)D * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)kBlock};
  cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(cache), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int G>
bool launch_g(const Ctx& c, const PrefillArgs& a, const CUtensorMap& mk, const CUtensorMap& mv, const Params& prm, int sms) {
  const size_t smem = sizeof(Smem) + 1024;
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(prefill_sm100_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return false;
    attr_done = true;
  }
  prefill_sm100_kernel<G><<<sms, kThreads, smem, c.stream>>>(mk, mv, prm);
  note_launch();
  return true;
}

}  // namespace

bool prefill_sm100_supported(const Ctx& c) {
  return c.dtype == MINIPIC_BF16 && c.d == 128 && (c.group == 1 || c.group == 2 || c.group == 4 || c.group == 8);
}

size_t prefill_sm100_workspace_bytes(const Ctx&, int, int num_q_tokens) {
  return sizeof(PlanHeader) + 2 * (size_t)(num_q_tokens + 1) * sizeof(TileDesc) + 512;
}

bool launch_prefill_sm100(const Ctx& c, const PrefillArgs& a) {
  CUtensorMap mk, mv;
  if (!make_cache_map(&mk, a.k_cache, c.num_blocks, c.hkv) || !make_cache_map(&mv, a.v_cache, c.num_blocks, c.hkv)) return false;
  PlanHeader* hdr = (PlanHeader*)a.workspace;
  TileDesc* sorted = (TileDesc*)((char*)a.workspace + sizeof(PlanHeader));
  TileDesc* tmp = sorted + (a.num_q_tokens + 1);
  prefill_plan_kernel<<<1, 1024, 0, c.stream>>>(a, BM / c.group, hdr, sorted, tmp);
  note_launch();
  Params prm;
  prm.a = a; prm.hq = c.hq; prm.hkv = c.hkv; prm.scale_log2 = c.scale_log2; prm.flags = c.flags;
  prm.hdr = hdr; prm.tiles = sorted; prm.rp = c.rope;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  switch (c.group) {
    case 1: return launch_g<1>(c, a, mk, mv, prm, sms);
    case 2: return launch_g<2>(c, a, mk, mv, prm, sms);
    case 4: return launch_g<4>(c, a, mk, mv, prm, sms);
    case 8: return launch_g<8>(c, a, mk, mv, prm, sms);
  }
  return false;
}

}  // namespace minipic
