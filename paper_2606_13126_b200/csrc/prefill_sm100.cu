// a2-a9: fused RoPE-in-attention prefill for sm_100a (bf16, head_dim 128, GQA group 1/2/4/8).
//
// Work item = (Q super-tile, KV head).  A super-tile is up to 2 * (128/G) consecutive query tokens of one request
// that share vis_lo (one span, or suffix rows); it is processed as TWO 128-row MMA tiles, A and B, whose rows are
// (token, head-in-group) pairs, so one gathered + rotated K tile serves 256 score rows (the whole GQA group of up
// to 2*128/G tokens).  Plan kernels (a2) cut the query rows into super-tiles, compute each one's KV range
// [floor16(vis_lo), idx_last] (span-mask TILE SKIPPING: keys outside it are never touched) and sort the tiles
// longest-first; a persistent kernel (one CTA per SM, 16 warps) pulls items from an atomic counter and runs, per
// KV tile of 128 keys:
//
//   warp 12      TMA producer  : scheduler ring; Q super-tile (3-D box) and the KV tile's 8 physical blocks through
//                                the block table with cp.async.bulk.tensor (SWIZZLE_128B boxes) into smem       (a4)
//   warps 8-11   rotation      : in-place RoPE of every K tile (a5): smem -> registers -> smem; a lane owns 8 frequencies
//                                (one 16-byte chunk of both halves of a row), cos/sin restarted exactly (64-bit fixed-point
//                                phase + MUFU) once per 32-key chunk / at every position jump and advanced by the
//                                angle-addition recurrence in between (packed f32x2 FMAs)
//   warp 13      MMA issuer    : tcgen05.mma S_X = Q_X K'^T (smem x smem -> TMEM), O_X += P_X V (TMEM x smem -> TMEM),
//                                X in {A, B} ping-pong so the tensor pipe runs while the other tile is in softmax (a6, a8)
//   warps 0-3 / 4-7 softmax A/B: in-place RoPE of their own Q tile at the start of an item (a3); tcgen05.ld S (one row per
//                                thread), mask, online softmax with lazy rescale of O, P -> bf16 -> TMEM (aliasing S);
//                                epilogue O / l -> out, LSE, deferred until the next item's Q is rotated       (a7, a9)
//
// All hand-offs are mbarriers; generic-proxy smem writes are fenced with fence.proxy.async before the MMA reads.
#include <cuda.h>
#include <algorithm>
#include <cstddef>

#include "internal.h"

namespace minipic {

namespace {

constexpr int BM = 128, BN = 128, D = 128;
constexpr int kTileBytes = BM * D * 2;       // 32 KB: one Q tile (128 rows)
constexpr int kHalfBytes = kTileBytes / 2;   // [half of head_dim][128 rows][128 B]
// CTA PAIR (cta_group::2): one tcgen05.mma covers M = 256 rows = the same tile (A or B) of BOTH CTAs of the cluster.  The B
// operand is split between the two CTAs: for QK^T by keys (each CTA gathers + rotates 64 of the tile's 128 keys), for PV
// by head_dim (each CTA holds its 64-column half of V for all 128 keys).  Per CTA a K stage and a V stage are 16 KB.
constexpr int kKeysCta = BN / 2;
constexpr int kKTileBytes = kKeysCta * D * 2;    // 8 row groups of [half (2)][8 rows x 128 B]
constexpr int kVTileBytes = BN * (D / 2) * 2;    // 16 row groups of [8 rows x 128 B] (this CTA's half of head_dim)
#ifndef MINIPIC_KSTAGES
#define MINIPIC_KSTAGES 2
#endif
#ifndef MINIPIC_VSTAGES
#define MINIPIC_VSTAGES 2
#endif
constexpr int kKStages = MINIPIC_KSTAGES, kVStages = MINIPIC_VSTAGES, kRing = 4;
// Measured and dropped (config 5, in-kernel RoPE; the kept version runs 2.24 ms):
//  * a ring of three Q tile slots (next item's tile A loaded + rotated during the current item, epilogue staged in the
//    finishing item's tile-B slot): parity-green, dense +3 %, but span items -7 % (2.30 ms): the four rotation warps are
//    saturated at item boundaries (K0', Q_A', Q_B', K1' = 4.5 tile rotations per ~3-tile item) and starting Q earlier only
//    takes issue slots from the current item's softmax;  a single V stage (needed for a full Q double buffer) costs 7 %;
//  * K rotation by the eight softmax warps in the gap where they wait for S_FULL (16 rows each, no dedicated rotation
//    warps): parity-green but 2.78 ms - the exact restart per 16 rows (~600 cycles of dependent latency) lands on the
//    softmax critical path instead of running ahead on separate warps;
//  * Q rotation unrolled like the K path, or two rows per iteration: 8 % / 7 % slower (instruction cache);
//  * L2 prefetch of the next item's Q tiles: no change;  MMA N / K trimmed to the visible columns of a diagonal tile: no
//    change (the tensor pipe is not the limiter on span items);
//  * speculative row max (exps against the running max at once, tile max tracked inside the exp loop, redo if it grew by
//    more than the lazy-rescale threshold): 2.41 ms - the exp loop is issue-bound, 64 more FMNMX in it cost more than the
//    separate max pass saves;  second half of S loaded from TMEM under the first half's max: no change;
//  * mbarrier.try_wait with a suspend-time hint (500 / 4000 ns) to take the wait loops (44 % of the issued instructions)
//    off the issue slots: no change on dense tiles, 2 % slower on config 5 - try_wait already sleeps in hardware.
// Measured and dropped on the CTA-pair kernel (config 5 at 2.04 ms, all parity-green):
//  * Q double buffer + Q rotation by the rotation warps one item ahead + epilogue staged in the finished item's Q buffer +
//    "resident" items (several 64-token sub-items over K tiles gathered and rotated once): 2.27 ms.  Four rotation warps
//    need ~7.5 K cycles for the 256 Q rows of a sub-item (latency-bound at ~470 cycles per 4-row step whether rolled or
//    unrolled), longer than a short sub-item lasts, and with Q and K both pre-rotated the structure still ran 2.04 ms;
//  * P in shared memory (SS-mode PV) so that QK^T of tile i + 1 is issued as soon as S(i) is in registers and runs under the
//    softmax of tile i: 2.05 ms, dense causal input 1058 -> 1025 TFLOP/s.  The softmax warps then wait for PV(i) (P buffer,
//    O rescale) instead of for S(i + 1): the two tile slots run in phase and share the scheduler's MUFU / issue rate, which
//    is what bounds the period, not the dependency chain;
//  * named-barrier ping-pong that makes the tile-A and tile-B warps of a scheduler take turns in the exp phase: 2.09 ms;
//  * 2, 3 or 4 K / V stages: 2.034 - 2.048 ms (no effect).
// Measured after the early P publish (config 5 at 2.00 ms):
//  * Q tile B rotated by the four K rotation warps as soon as the Q tile lands (they are idle then), tile A by its softmax
//    warps: 2.08 ms, config 3 0.353 -> 0.410 ms - the rotation warps then run late on K tile 2 of short items;
//  * mbarrier.test_wait (no suspend) in the issuer's waits for P: 2.014 ms - the spinning warp takes issue slots from the
//    softmax warps of its scheduler;  2 or 3 chunks of P published early instead of 1: 2.015 / 1.999 ms;
//  * Q double buffer in the 64 KB that the non-dual kernels do not need for the exchange buffer, the producer fetching the NEXT
//    item's Q tiles during the current item (rotation still at the boundary, by the softmax warps): config 5 2.012 -> 2.001 ms,
//    span-only input 2.310 -> 2.298 ms, dense causal 1.034 -> 1.048 ms; with Q and K pre-rotated 1.895 -> 1.840 ms - the boundary
//    is the Q rotation itself, not the load.  On top of that, rotating the next item's Q rows in the softmax warps' wait for their
//    next S tile ("idle" time): 2.198 ms - that wait is when the other tile slot's softmax has the sub-partition to itself;
//  * slot B writes the previous item's rows BEFORE it rotates its Q rows (slot A after), so that the two slots' softmaxes start
//    an item half a period apart instead of in phase: 2.13 ms (and the two-step loop that keeps one copy of each code path costs
//    3 % by itself, 2.08 ms, with the old order);
//  * Q rotation with the lane owning a TOKEN (row 8 rsub + k: for G = 8 one exact restart per item, no angle-addition steps, -sin
//    formed once; ~30 % fewer instructions in the loop that takes ~3.8 K of the ~8.4 K cycles of an item boundary): span-only
//    input 2.311 -> 2.271 ms, but dense causal 1.033 -> 1.058 ms and config 5 2.012 -> 2.027 ms; the Q rotation as a
//    __noinline__ function (to keep it from disturbing the tile loop's register allocation): dense 1.074 ms, with the
//    token-per-lane mapping inside 1.113 ms - the call's ABI costs the tile loop more than the inlined code did;
//  * (again, on this kernel, after ncu showed the exp phase waiting at the MUFU cadence) every 4th / 3rd / 2nd exp2 pair as a
//    packed-f32x2 cubic on the FMA pipe: dense causal 1.032 -> 1.148 / 1.149 / 1.294 ms, config 5 2.013 -> 2.106 / 2.137 / 2.198 ms;
//    only with K pre-rotated (idle rotation warps) does it gain (0.953 -> 0.939 ms): the FMA pipe is what the rotation needs;
//  * dual items: tile-A warps read O_B straight from TMEM (no 64 KB exchange buffer): config 3 0.375 -> 0.392 ms, slot B's
//    accumulator stays busy until the deferred epilogue; with the freed shared memory 3 - 4 K / V stages: no effect.
// Two restructurings of the softmax were measured on config 5 (2.38 ms at the time) and dropped:
//  * every 2nd / 3rd / 4th exp2 pair on the FMA pipe (Cody-Waite + cubic minimax) instead of MUFU: 2.59 / 2.56 / 2.45 ms -
//    the softmax warps are issue / latency bound, not MUFU bound, at this tile period;
//  * the two 64-column halves of S as a double buffer (QK of the next half issued right after the PV that frees it, softmax
//    in 64-column steps): 2.61 ms - the P -> PV -> QK -> S round trip (~1000 cycles) is as long as a 64-column softmax
//    step, so the softmax warps still wait (49 % of their samples) and A / B no longer alternate on the MUFU unit.
// K / V tile in shared memory: 16 row groups of [half of head_dim (2)][8 rows x 128 B] = 2048 B each, so one (block, head)
// of the cache (16 tokens x 256 B) is ONE 4-D TMA box of two groups.  Q tile: [half (2)][128 rows x 128 B].
constexpr int kGroupBytes = 2048, kKvHalfOff = 1024, kVGroupBytes = 1024;
constexpr int kStageBytes = 4096;            // epilogue staging per softmax warp: 32 rows x 128 B (64 bf16 columns)
// 16 warps = 4 warpgroups: softmax A, softmax B (184 registers each after setmaxnreg), rotation (96), control (TMA, MMA and
// two idle warps, 48).  setmaxnreg is a WARPGROUP-wide instruction (all four warps, same count), and the split must fit the
// launch pool of 512 * 128 registers or setmaxnreg.inc blocks forever: 256*184 + 128*96 + 128*48 = 65536.
constexpr int kThreads = 512;
constexpr int kRegsSoftmax = 184, kRegsRot = 96, kRegsCtl = 48;
static_assert(256 * kRegsSoftmax + 128 * kRegsRot + 128 * kRegsCtl <= 65536, "setmaxnreg split exceeds the CTA register pool");
#ifndef MINIPIC_PEARLY
#define MINIPIC_PEARLY 1
#endif
constexpr int kPEarly = MINIPIC_PEARLY;   // 32-key chunks of P published early (P_HALF): PV of those keys starts under the remaining exps
constexpr int kMaxBins = 4096;
constexpr int kDualMinTiles = 4;   // a "dual" item (see struct Item) needs at least this many KV tiles
constexpr unsigned kWaitMaxSpins = 1u << 26;   // x (>= 30 cycles per failed try_wait) = seconds

// kv_off = cu_kv_lens[r]; pad: dual item; part: see SplitGroup.  plan_kernel pass 1 reads ints 1, 5, 9 (ntok, n_kv, pad) by index
struct alignas(16) TileDesc { int t0, ntok, r, idx0, lo, n_kv, kv_hi, kv_len, kv_off, pad, part, rsv; };
static_assert(sizeof(TileDesc) == 48, "three 16-byte words");
// KV-RANGE SPLITS (small grids only): an item whose tile steps exceed what one CTA pair should get is cut into chunks over
// consecutive KV tiles; every chunk is an item of its own that writes (O normalised over the chunk, lse of the chunk) as fp32
// into partial token slots of the workspace - chunk s of a group owns slots [base + s ntok, base + (s + 1) ntok), part = 1 +
// its first slot - and split_merge_kernel combines them: the 64-token question of ONE request over a long cached context then
// runs on many CTA pairs instead of on hkv of them.
struct SplitGroup { int t0, ntok, nsplit, base; };
// magic tags a header written by THIS kernel family, so minipic_prefill_status() can tell it from a workspace that a call
// dispatched to another kernel never touched (err and magic are adjacent: one 8-byte read)
constexpr int kPlanMagic = 0x4d504943;   // "MPIC"
struct PlanHeader { int n_tiles; int next_item; int err; int magic; int err_info[4]; int ticket; int n_raw; int n_groups; int part_used; int pad[52]; };
static_assert(sizeof(PlanHeader) == 256, "header size");
struct ItemInfo { int t0, ntok, r, idx0, lo, kvh, n_kv, kv_hi, kv_len, kv_off, pad[2]; };   // 48 B ring entry; t0 < 0 = stop; pad = {dual, part}

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
// ---- cluster (CTA pair) helpers
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {   // shared::cta address -> shared::cluster address in CTA rank
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
// arrive on a barrier of any CTA of the pair.  Default semantics (release at CTA scope), as in CUTLASS' 2-SM pipelines: what
// the waiting MMA issuer hands on is consumed by the tensor core of the ARRIVING thread's own SM (its shared memory through
// the async proxy after fence.proxy.async, its TMEM after tcgen05.fence).  A cluster-scope release costs a MEMBAR.ALL.GPU
// per arrival (measured: config 5 2.19 -> 2.61 ms).
__device__ __forceinline__ void mbar_arrive_cl(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// the scheduler's arrive publishes ring entries written into the peer's shared memory: release at cluster scope
__device__ __forceinline__ void mbar_arrive_cl_release(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void st_cluster_v4(uint32_t cluster_addr, int a, int b, int c, int d) {
  asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(cluster_addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ bool mbar_try_cl(uint32_t bar, uint32_t parity) {   // acquire at cluster scope: remote arrivals
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  return done != 0;
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  return done != 0;
}
// A protocol bug must neither hang the GPU nor kill the context: a wait that exceeds the timeout records
// (barrier, parity, block, thread) in the plan header, and every thread that sees the flag stops waiting, so the
// kernel drains and the host can read the error word (minipic_prefill_status()).
struct Waiter {
  int* err;
  bool dead;
  // kept tiny on purpose: ~25 wait sites inline this, and the kernel is instruction-cache bound (four roles with
  // different code share an SM).  try_wait suspends in hardware for a bounded time, so spins are cheap to count.
  __device__ __forceinline__ void wait(uint32_t bar, uint32_t parity) {
    if (dead) return;
    unsigned spins = 0;
    while (!mbar_try(bar, parity)) {
      if ((++spins & 4095u) == 0 && (*(volatile int*)err != 0 || spins > kWaitMaxSpins)) {
        atomicCAS(err, 0, (int)(bar | 0x40000000u));   // records the barrier that timed out
        dead = true;
        return;
      }
    }
  }
  // same, for barriers that threads of the PEER CTA arrive on (acquire at cluster scope)
  __device__ __forceinline__ void wait_cl(uint32_t bar, uint32_t parity) {
    if (dead) return;
    unsigned spins = 0;
    while (!mbar_try_cl(bar, parity)) {
      if ((++spins & 4095u) == 0 && (*(volatile int*)err != 0 || spins > kWaitMaxSpins)) {
        atomicCAS(err, 0, (int)(bar | 0x20000000u));
        dead = true;
        return;
      }
    }
  }
};
// Debug-only event trace (-DMINIPIC_TRACE, never in the shipped library): CTA 0 records (tag, SM clock) per role.  One thread
// per role; its running count is a register (a global read-modify-write per event costs ~700 cycles and distorts the timeline).
// Roles: 0 scheduler, 1 MMA issuer, 2 rotation warp 0, 3 / 4 softmax warp 0 of tile slot A / B, 5 Q / K producer, 6 V producer.
// Tags: 40 S_FULL seen, 44 S in registers, 45 row max done, 46 exps done, 41 P_FULL; 48 / 49 before / after the Q_FULL wait, 47 Q rows
// rotated, 42 / 43 epilogue in / out, 1000 + 4 n + dual + 2 part = item start (n KV tiles).
#ifdef MINIPIC_TRACE
constexpr int kTraceRoles = 8, kTraceLen = 8192;
__device__ long long g_trace[kTraceRoles][kTraceLen][2];
__device__ int g_trace_n[kTraceRoles];
__device__ __forceinline__ void trace_ev(int role, int tag, int& n) {
  if (blockIdx.x != 0) return;
  if (n < kTraceLen) { g_trace[role][n][0] = tag; g_trace[role][n][1] = clock64(); ++n; g_trace_n[role] = n; }
}
#define TRACE(role, tag) trace_ev(role, tag, trace_n)
#define TRACE_L0(role, tag) do { if (lane == 0) trace_ev(role, tag, trace_n); } while (0)
#else
#define TRACE(role, tag) do { } while (0)
#define TRACE_L0(role, tag) do { } while (0)
#endif
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  // arrives on the barrier at this offset in BOTH CTAs of the pair once every MMA issued so far has completed
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"((unsigned short)3) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tmap, uint32_t bar, int x, int y, int z) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(tmap), "r"(bar), "r"(x), "r"(y), "r"(z) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tmap, uint32_t bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(tmap), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* tmap, uint32_t src, int x, int y, int z) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(tmap), "r"(src), "r"(x), "r"(y), "r"(z) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// Shared-memory matrix descriptors (SWIZZLE_128B): the low word carries the start address (>> 4) and the leading byte
// offset (>> 4, bits 16-29); the high word is the same for every operand of this kernel: stride byte offset 1024
// (8 rows x 128 B), descriptor version 1 (bit 46), swizzle mode 128B (2 << 61).
constexpr uint32_t kDescHiQ = (1024u >> 4) | (1u << 14) | (2u << 29);                    // Q tile: 8-row groups 1024 B apart
constexpr uint32_t kDescHiKV = ((uint32_t)kGroupBytes >> 4) | (1u << 14) | (2u << 29);   // K tile: 8-row groups 2048 B apart
constexpr uint32_t kDescHiV = ((uint32_t)kVGroupBytes >> 4) | (1u << 14) | (2u << 29);   // V half tile: 8-key groups 1024 B apart
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "mov.b64 da, {%1, %5};\n\tmov.b64 db, {%2, %6};\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], da, db, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(idesc), "r"(acc), "r"(kDescHiQ), "r"(kDescHiKV) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 db;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "mov.b64 db, {%2, %5};\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], db, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(idesc), "r"(acc), "r"(kDescHiV) : "memory");
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
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float max3(float a, float b, float c) {
  float d;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts128z(uint32_t addr) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0) : "memory");
}
__device__ __forceinline__ bool elect_one() {   // one lane of a converged warp (the same lane every time)
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

// instruction descriptor: D fp32, A/B bf16, M = 256 (128 rows in each CTA of the pair), N = 128; b_mn = B operand is
// MN-major (V tile)
__host__ __device__ constexpr uint32_t instr_desc(bool b_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn ? 1u : 0u) << 16) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(2 * BM >> 4) << 24);
}

// ------------------------------------------------------------------------------------------------ a2: plan
// A token starts a new item if it is the first of its request, if it does not continue the previous token (sequence index + 1,
// same vis_lo), or every `tok` tokens counted from its span start (plan_kernel evaluates this rule branch-free).

// ONE launch (a2).  Every block marks its 256 query tokens: the start flags of those tokens and of the next `tok` ones go
// into a shared bitmask, so a starting token finds the length of its item with a find-first-set instead of a sequential
// scan (which alone took 22 us on config 2), and appends its descriptor with an atomic.  The LAST block to finish (ticket)
// then sees every item: it adds up the tile steps, cuts items that are too long for a balanced grid into KV-range chunks
// (SplitGroup; only when the host allows it), and sorts all descriptors by DESCENDING cost - a counting sort in shared
// memory, longest item first - for the persistent kernel's atomic work counter to walk.
constexpr int kPlanThreads = 256, kPlanMaxTok = 512;   // tok = 4 * 128 / G <= 512
constexpr int kPlanSingleThreads = 1024, kPlanSingleMaxTok = 4096;   // one-block plan for small inputs (see plan_kernel)
constexpr int kPlanCache = 2560;                         // descriptors the last block keeps in shared memory when it may split
constexpr int kSplitMinSteps = 4, kSplitMax = 16;      // a chunk runs at least 4 tile steps; at most 16 chunks per item
__device__ __forceinline__ int tile_cost(const TileDesc& td) { return td.pad ? (td.n_kv + 1) >> 1 : td.n_kv; }   // tile steps
__device__ __forceinline__ int dual_flag(int dual_ok, int ntok, int tok, int n_kv) {   // dual item: at most 2 TOK tokens over a long KV range
  return (dual_ok && 2 * ntok <= tok && n_kv >= kDualMinTiles) ? 1 : 0;
}
// chunks an item of `cost` steps is cut into when a pair should not run more than `tsplit` steps of it (1 = not cut)
__device__ __forceinline__ int split_count(int cost, int n_kv, int tsplit, int* tiles_per_chunk) {
  *tiles_per_chunk = n_kv;
  if (2 * cost <= 3 * tsplit) return 1;   // not worth a second item (per-item overhead ~ one tile step, plus the merge)
  const int ns = min(kSplitMax, (cost + tsplit - 1) / tsplit);
  const int ct = (n_kv + ns - 1) / ns;
  *tiles_per_chunk = ct;
  return (n_kv + ct - 1) / ct;
}
struct PlanArgs {
  int tok, dual_ok;
  int split_pairs;    // 0: no KV-range splits; else the number of CTA pairs to balance for
  int hkv, part_cap;  // partial token slots the workspace has room for
  int sorted_cap;     // descriptors `sorted` has room for
  PlanHeader* hdr; TileDesc* tmp; TileDesc* sorted; SplitGroup* groups;
};
__device__ __forceinline__ TileDesc load_desc(const TileDesc* p) {   // written by other blocks of this launch: read through L2
  TileDesc td;
  const int* src = reinterpret_cast<const int*>(p);
  int* dst = reinterpret_cast<int*>(&td);
#pragma unroll
  for (int e = 0; e < (int)(sizeof(TileDesc) / sizeof(int)); ++e) dst[e] = __ldcg(src + e);
  return td;
}
// kSingle: ONE block of kT = 1024 threads does everything for a small input (the host decides: at most kPlanSingleMaxTok
// query tokens).  No ticket, no header memset before the launch, item count and (cost, tiles, tokens) of every item stay in shared
// memory: about half the dependent L2 round trips of the multi-block version, which are what a plan of a few hundred items costs.
#ifdef MINIPIC_PLAN_TIMES
__device__ long long g_plan_t[16];
#define PLAN_T(i) do { if (threadIdx.x == 0) g_plan_t[i] = clock64(); } while (0)
#else
#define PLAN_T(i) do { } while (0)
#endif
template <int kT, bool kSingle>
__global__ void __launch_bounds__(kT) plan_kernel(PrefillArgs a, PlanArgs pa) {
  constexpr int kRounds = ((kSingle ? kPlanSingleMaxTok : kT) + kPlanMaxTok + kT - 1) / kT;   // rounds of kT tokens that cover the block + the lookahead
  constexpr int kWords = kRounds * (kT / 32);
  __shared__ unsigned sflag[kWords];
  __shared__ int s_last, s_groups, s_slots, s_nraw;
  __shared__ int wsum[kT / 32];
  __shared__ int red[3], wred[3][32], cand_items[8], cand_max[8], s_nlong, long_idx[kT];
  __shared__ unsigned short s_cost[kPlanCache], s_nkv[kPlanCache], s_ntk[kPlanCache];
  __shared__ int shist[kMaxBins];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int tok = pa.tok;
  PlanHeader* hdr = pa.hdr;
  PLAN_T(0);
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the attention grid may start its prologue (see its scheduler)
  if (blockIdx.x == 0 && tid == 0) hdr->magic = kPlanMagic;
  if (kSingle && tid == 0) {   // no memset ran before this launch: the counters the other kernels read start here
    hdr->next_item = 0; hdr->err = 0; hdr->n_groups = 0; hdr->part_used = 0;
    s_nraw = 0;
  }
  if (kSingle) __syncthreads();
  int* const n_raw_ctr = kSingle ? &s_nraw : &hdr->n_raw;
  // the block's tokens: kT of them, or (kSingle) all - then a thread marks and makes items for several tokens, kT apart
  const int span = kSingle ? ((a.num_q_tokens + kT - 1) / kT) * kT : kT;
  const int b0 = kSingle ? 0 : (int)blockIdx.x * kT;
  auto request_of = [&](int t) {
    int lo_r = 0, hi_r = a.num_reqs;
    while (hi_r - lo_r > 1) {
      const int mid = (lo_r + hi_r) >> 1;
      if (__ldg(a.cu_q_lens + mid) <= t) lo_r = mid; else hi_r = mid;
    }
    return lo_r;
  };
  // straight-line on purpose: every round's loads are issued (clamped indices, no branches) before any of them is used, so that
  // the rounds cost one memory round trip together instead of two each
  bool fl[kRounds];
  {
    int tc[kRounds], rr[kRounds], tq[kRounds], i1[kRounds], i0[kRounds], l1[kRounds], l0[kRounds];
    const int t_last = max(a.num_q_tokens - 1, 0);
#pragma unroll
    for (int c = 0; c < kRounds; ++c) { tc[c] = min(b0 + c * kT + tid, t_last); rr[c] = request_of(tc[c]); }
#pragma unroll
    for (int c = 0; c < kRounds; ++c) {
      const int tm = max(tc[c] - 1, 0);
      tq[c] = __ldg(a.cu_q_lens + rr[c]);
      i1[c] = __ldg(a.q_seq_idx + tc[c]); i0[c] = __ldg(a.q_seq_idx + tm);
      l1[c] = __ldg(a.q_vis_lo + tc[c]); l0[c] = __ldg(a.q_vis_lo + tm);
    }
#pragma unroll
    for (int c = 0; c < kRounds; ++c) {
      const int t = b0 + c * kT + tid;
      // the item-start rule (above); tokens past the end count as starts (sentinel)
      fl[c] = t >= a.num_q_tokens || t == tq[c] || i1[c] != i0[c] + 1 || l1[c] != l0[c] || ((i1[c] - max(l1[c], 0)) % tok) == 0;
    }
  }
#pragma unroll
  for (int c = 0; c < kRounds; ++c) {
    if (c * kT < span + tok) {
      const unsigned m = __ballot_sync(0xffffffffu, fl[c]);
      if (lane == 0) sflag[c * (kT / 32) + wid] = m;
    }
  }
  __syncthreads();
#pragma unroll
  for (int c2 = 0; c2 < (kSingle ? kPlanSingleMaxTok / kT : 1); ++c2) {   // unrolled for the same reason
    const int li = c2 * kT + tid, t = b0 + li;   // li: index within the block's tokens = bit index in sflag
    if (c2 * kT < span && t < a.num_q_tokens && ((sflag[li >> 5] >> (li & 31)) & 1u)) {
      int nxt = -1;                        // index of the next start after li
      unsigned wbits = sflag[li >> 5] & ~((2u << (li & 31)) - 1u);
      for (int wi = li >> 5; nxt < 0; ++wi) {
        if (wbits) nxt = wi * 32 + __ffs(wbits) - 1;
        else wbits = sflag[wi + 1];        // a start exists within `tok` tokens (item length rule / end sentinel)
      }
      const int n = min(nxt - li, tok);
      const int r = request_of(t);
      TileDesc td;
      td.t0 = t; td.ntok = n; td.r = r; td.idx0 = __ldg(a.q_seq_idx + t); td.lo = max(__ldg(a.q_vis_lo + t), 0);
      td.kv_len = __ldg(a.kv_lens + r);
      td.kv_off = __ldg(a.cu_kv_lens + r);
      const int kv_lo = td.lo & ~(kBlock - 1);
      td.kv_hi = min(td.idx0 + n, td.kv_len);
      td.n_kv = td.kv_hi > kv_lo ? (td.kv_hi - kv_lo + BN - 1) / BN : 0;
      td.pad = dual_flag(pa.dual_ok, n, tok, td.n_kv);
      td.part = 0; td.rsv = 0;
      const int slot = atomicAdd(n_raw_ctr, 1);
      pa.tmp[slot] = td;
      if (kSingle && slot < kPlanCache) {
        s_cost[slot] = (unsigned short)min(tile_cost(td), 65535); s_nkv[slot] = (unsigned short)min(td.n_kv, 65535); s_ntk[slot] = (unsigned short)td.ntok;
      }
    }
  }
  if (kSingle) __syncthreads();
  // ---- last block: balance (KV-range splits) and counting sort of all descriptors, longest first
  if (!kSingle) {
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&hdr->ticket, 1) == (int)gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
  }
  const int n_raw = kSingle ? s_nraw : *(volatile int*)&hdr->n_raw;
  PLAN_T(1);
  auto block_reduce = [&](int v0, int v1, int vmax) {   // red[0], red[1] = block-wide sums, red[2] = block-wide max (>= 0)
    // two levels of shuffles through wred, no shared-memory atomics (32 warps on three addresses took ~3 us per call)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      v0 += __shfl_xor_sync(0xffffffffu, v0, o); v1 += __shfl_xor_sync(0xffffffffu, v1, o);
      vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    }
    __syncthreads();   // the previous call's red[] has been read by everyone
    if (lane == 0) { wred[0][wid] = v0; wred[1][wid] = v1; wred[2][wid] = vmax; }
    __syncthreads();
    if (wid == 0) {
      int a0 = lane < kT / 32 ? wred[0][lane] : 0, a1 = lane < kT / 32 ? wred[1][lane] : 0, am = lane < kT / 32 ? wred[2][lane] : 0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o);
        am = max(am, __shfl_xor_sync(0xffffffffu, am, o));
      }
      if (lane == 0) { red[0] = a0; red[1] = a1; red[2] = am; }
    }
    __syncthreads();
  };
  int tsplit = 0x3fffffff;
  PLAN_T(2);
  constexpr int kCand = 8;   // candidate chunk lengths
  if (pa.split_pairs > 0 && n_raw <= kPlanCache) {   // kPlanCache descriptors: more than any small grid has
    int steps = 0, cmax_all = 0;
    for (int i = tid; i < n_raw; i += kT) {
      int c;
      if (kSingle) c = s_cost[i];   // filled when the item was made
      else {
        const TileDesc td = load_desc(pa.tmp + i);
        c = tile_cost(td);
        s_cost[i] = (unsigned short)min(c, 65535); s_nkv[i] = (unsigned short)min(td.n_kv, 65535); s_ntk[i] = (unsigned short)td.ntok;
      }
      steps += c; cmax_all = max(cmax_all, c);
    }
    PLAN_T(3);
    block_reduce(steps, 0, cmax_all);
    PLAN_T(4);
    // float arithmetic on purpose: every thread evaluates this, and 64-bit integer divisions cost ~500 cycles each (they were
    // 4 us of a 13 us plan); it is a heuristic, and every thread gets the same bits
    const float all_steps = (float)red[0] * (float)pa.hkv;
    const int per_pair = max(kSplitMinSteps, (int)ceilf(all_steps / (float)pa.split_pairs));
    const int cstep = max(1, per_pair / 8);
    if (2 * red[2] > 3 * per_pair && red[2] < 32767) {   // at least one item is long enough to be cut (and n_kv <= 2 cost fits 16 bits)
      __syncthreads();
      if (tid < kCand) { cand_items[tid] = n_raw; cand_max[tid] = 0; }
      if (tid == 0) { s_nlong = 0; s_groups = 0; s_slots = 0; }
      __syncthreads();
      int short_max = 0;
      for (int i = tid; i < n_raw; i += kT) {
        const int c = s_cost[i];
        if (2 * c > 3 * per_pair) { const int j = atomicAdd(&s_nlong, 1); if (j < kT) long_idx[j] = i; }
        else short_max = max(short_max, c);
      }
      PLAN_T(5);
      block_reduce(0, 0, short_max);
      PLAN_T(6);
      short_max = red[2];
      const int n_long = s_nlong;
      if (n_long <= kT) {
        // a few candidate chunk lengths: keep the one with the shortest estimated makespan - rounds of items x mean item cost,
        // but at least the longest item - so that e.g. 8 long items become 72 chunks on 74 pairs rather than 80.  One task per
        // (long item, candidate); the short items count 1 each whatever the candidate.
        for (int task = tid; task < n_long * kCand; task += kT) {
          const int k = task % kCand, i = long_idx[task / kCand];
          int ct;
          const int ns = split_count(s_cost[i], s_nkv[i], per_pair + k * cstep, &ct);
          atomicAdd(&cand_items[k], ns - 1);
          atomicMax(&cand_max[k], dual_flag(pa.dual_ok, s_ntk[i], tok, ct) ? (ct + 1) >> 1 : ct);
        }
        __syncthreads();
        PLAN_T(7);
        {   // candidate k is evaluated by lane k of every warp (the serial loop with its divisions took ~5 K cycles)
          float est = 3.0e38f;
          if (lane < kCand) {
            const int n_it = cand_items[lane] * pa.hkv, rounds = (n_it + pa.split_pairs - 1) / pa.split_pairs;   // <= 2560 x 16 x hkv items
            // + rounds: the fixed cost of an item (Q load + rotation, pipeline fill, epilogue) is about one tile step
            est = fmaxf((float)max(cand_max[lane], short_max), (float)rounds * (all_steps / (float)n_it)) + (float)rounds;
          }
          float mn = est;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
          const unsigned eq = __ballot_sync(0xffffffffu, lane < kCand && est == mn);
          tsplit = per_pair + (__ffs(eq) - 1) * cstep;   // the first (shortest chunk) of equally good candidates
        }
        int slots = 0, extra = 0;
        if (tid < n_long) {
          const int i = long_idx[tid];
          int ct;
          const int ns = split_count(s_cost[i], s_nkv[i], tsplit, &ct);
          if (ns > 1) { slots = ns * s_ntk[i]; extra = ns - 1; }
        }
        block_reduce(slots, extra, 0);
        if (red[0] > pa.part_cap || n_raw + red[1] > pa.sorted_cap) tsplit = 0x3fffffff;   // no room: run unsplit
      }
    }
    __syncthreads();
  }
  PLAN_T(8);
  for (int i = tid; i < kMaxBins; i += kT) shist[i] = 0;
  if (tid == 0) { s_groups = 0; s_slots = 0; }
  __syncthreads();
  // pass 1: histogram of the (chunk) costs - from the shared-memory copy when pass 0 made one (only then can items be cut)
  const bool cached = pa.split_pairs > 0 && n_raw <= kPlanCache;
  if (cached) {
    for (int i = tid; i < n_raw; i += kT) {
      const int cost = s_cost[i], n_kv = s_nkv[i], ntok = s_ntk[i];
      int ct;
      const int ns = split_count(cost, n_kv, tsplit, &ct);
      if (ns == 1) { atomicAdd(&shist[min(cost, kMaxBins - 1)], 1); continue; }
      for (int sidx = 0; sidx < ns; ++sidx) {
        const int nk = min(ct, n_kv - sidx * ct);
        atomicAdd(&shist[min(dual_flag(pa.dual_ok, ntok, tok, nk) ? (nk + 1) >> 1 : nk, kMaxBins - 1)], 1);
      }
    }
  } else {   // large grids (thousands of items, nothing is cut): four descriptors in flight per thread, two words of each
    for (int i0 = tid; i0 < n_raw; i0 += 4 * kT) {
      int nk[4], pd[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = min(i0 + u * kT, n_raw - 1);
        const int* src = reinterpret_cast<const int*>(pa.tmp + i);
        nk[u] = __ldcg(src + 5); pd[u] = __ldcg(src + 9);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (i0 + u * kT < n_raw) atomicAdd(&shist[min(pd[u] ? (nk[u] + 1) >> 1 : nk[u], kMaxBins - 1)], 1);
    }
  }
  __syncthreads();
  PLAN_T(9);
  // exclusive prefix over the bins in DESCENDING cost order: rank = kMaxBins - 1 - bin
  constexpr int PER = kMaxBins / kT;   // 16 ranks per thread
  int v[PER], tot = 0;
#pragma unroll
  for (int e = 0; e < PER; ++e) { v[e] = shist[kMaxBins - 1 - (PER * tid + e)]; tot += v[e]; }
  int incl = tot;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int nb = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += nb;
  }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  int base = incl - tot;
  for (int w2 = 0; w2 < wid; ++w2) base += wsum[w2];
#pragma unroll
  for (int e = 0; e < PER; ++e) { shist[kMaxBins - 1 - (PER * tid + e)] = base; base += v[e]; }
  if (tid == kT - 1) hdr->n_tiles = base;   // total number of descriptors after the splits
  __syncthreads();
  PLAN_T(10);
  // pass 2: scatter
  if (!cached) {   // plain scatter, four 48-byte descriptors in flight per thread
    for (int i0 = tid; i0 < n_raw; i0 += 4 * kT) {
      uint4 v[4][3];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const uint4* src = reinterpret_cast<const uint4*>(pa.tmp + min(i0 + u * kT, n_raw - 1));
        v[u][0] = __ldcg(src); v[u][1] = __ldcg(src + 1); v[u][2] = __ldcg(src + 2);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (i0 + u * kT >= n_raw) continue;
        const int n_kv = (int)v[u][1].y, cost = v[u][2].y ? (n_kv + 1) >> 1 : n_kv;   // ints 5 (n_kv) and 9 (pad)
        uint4* dst = reinterpret_cast<uint4*>(pa.sorted + atomicAdd(&shist[min(cost, kMaxBins - 1)], 1));
        dst[0] = v[u][0]; dst[1] = v[u][1]; dst[2] = v[u][2];
      }
    }
    return;   // no groups: the header's counters stay 0
  }
  for (int i = tid; i < n_raw; i += kT) {
    const TileDesc td = load_desc(pa.tmp + i);
    int ct;
    const int ns = split_count(tile_cost(td), td.n_kv, tsplit, &ct);
    if (ns == 1) { pa.sorted[atomicAdd(&shist[min(tile_cost(td), kMaxBins - 1)], 1)] = td; continue; }
    const int g = atomicAdd(&s_groups, 1), slot0 = atomicAdd(&s_slots, ns * td.ntok);
    pa.groups[g] = SplitGroup{td.t0, td.ntok, ns, slot0};
    const int kv_lo = td.lo & ~(kBlock - 1);
    for (int sidx = 0; sidx < ns; ++sidx) {
      TileDesc ch = td;
      ch.n_kv = min(ct, td.n_kv - sidx * ct);
      if (sidx > 0) ch.lo = kv_lo + sidx * ct * BN;                    // a multiple of 128: no vis_lo mask inside the chunk
      if (sidx < ns - 1) ch.kv_hi = kv_lo + (sidx + 1) * ct * BN;       // < kv_hi: whole tiles, no partial last block
      ch.pad = dual_flag(pa.dual_ok, td.ntok, tok, ch.n_kv);
      ch.part = 1 + slot0 + sidx * td.ntok;
      pa.sorted[atomicAdd(&shist[min(tile_cost(ch), kMaxBins - 1)], 1)] = ch;
    }
  }
  __syncthreads();
  if (tid == 0) { hdr->n_groups = s_groups; hdr->part_used = s_slots; }
  PLAN_T(11);
}

// a9 for split items: out[t, h] = sum_s w_s O_s / sum_s w_s with w_s = e^{lse_s - max}, lse = max + ln sum_s w_s.  One warp
// per (token, head) row, a lane owns 4 of the 128 columns.  Launched after the attention kernel whenever splits were
// allowed; with no group in the header it returns at once.
__global__ void __launch_bounds__(256) split_merge_kernel(const PlanHeader* hdr, const SplitGroup* groups, const float* part_o,
                                                          const float* part_lse, int hq, __nv_bfloat16* out, float* lse) {
  asm volatile("griddepcontrol.wait;" ::: "memory");   // launched as a programmatic dependent of the attention grid
  const int n_groups = *(volatile const int*)&hdr->n_groups;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  if (n_groups == 0) return;
  // blocks are dealt out to the groups: bpg blocks share the rows of one group, all groups run side by side (one group: the
  // whole grid works on it; more groups than blocks: a block walks through several)
  const int bpg = max(1, (int)gridDim.x / n_groups), gstep = max(1, (int)gridDim.x / bpg), part = blockIdx.x % bpg;
  for (int g = blockIdx.x / bpg; g < n_groups; g += gstep) {
    const SplitGroup sg = groups[g];
    for (int rowi = part * 8 + wib; rowi < sg.ntok * hq; rowi += bpg * 8) {
      const int j = rowi / hq, h = rowi % hq;
      // all loads first (nsplit <= kSplitMax, fixed trip count): two memory round trips per row instead of one per chunk
      float ls[kSplitMax];
      float4 os[kSplitMax];
#pragma unroll
      for (int sidx = 0; sidx < kSplitMax; ++sidx) {
        const size_t prow = (size_t)(sg.base + min(sidx, sg.nsplit - 1) * sg.ntok + j) * hq + h;
        ls[sidx] = sidx < sg.nsplit ? __ldcg(part_lse + prow) : -INFINITY;
        os[sidx] = __ldcg(reinterpret_cast<const float4*>(part_o + prow * D + 4 * lane));
      }
      float mx = -INFINITY;
#pragma unroll
      for (int sidx = 0; sidx < kSplitMax; ++sidx) mx = fmaxf(mx, ls[sidx]);
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float wsum_ = 0.f;
      if (mx > -INFINITY) {
#pragma unroll
        for (int sidx = 0; sidx < kSplitMax; ++sidx) {   // fixed order: bit reproducible
          const float wgt = __expf(ls[sidx] - mx);       // e^{-inf} = 0: no such chunk, or a chunk with no visible key for this row
          if (sidx < sg.nsplit && wgt > 0.f) {            // (the guard keeps 0 x NaN of a never-written slot out)
            acc.x += wgt * os[sidx].x; acc.y += wgt * os[sidx].y; acc.z += wgt * os[sidx].z; acc.w += wgt * os[sidx].w;
            wsum_ += wgt;
          }
        }
      }
      const float inv = wsum_ > 0.f ? 1.f / wsum_ : 0.f;
      const size_t orow = (size_t)(sg.t0 + j) * hq + h;
      uint2 pk;
      pk.x = pack_bf16(acc.x * inv, acc.y * inv); pk.y = pack_bf16(acc.z * inv, acc.w * inv);
      *reinterpret_cast<uint2*>(out + orow * D + 4 * lane) = pk;
      if (lane == 0) lse[orow] = wsum_ > 0.f ? mx + logf(wsum_) : -INFINITY;
    }
  }
}

// ------------------------------------------------------------------------------------------------ main kernel
struct Smem {
  alignas(1024) unsigned char q[2][kTileBytes];
  alignas(1024) unsigned char k[kKStages][kKTileBytes];
  alignas(1024) unsigned char v[kVStages][kVTileBytes];
  alignas(1024) unsigned char ostage[8][kStageBytes];
  alignas(1024) float xchg[BM][D];                    // dual items: O_B rows (fp32) on their way to the A warps, 16-byte chunks XOR-swizzled by row
  float2 xml[BM];                                     // ... and (m_B, l_B)
  unsigned long long bars[36];
  alignas(16) ItemInfo ring[kRing];
  alignas(16) unsigned long long finc[64];   // F_i (common.cuh), read by the rotation lanes at every exact restart
  alignas(16) float2 step1[64];              // (cos f_i, sin f_i): one-position step, used by the Q rotation
  alignas(16) float2 step4[64];              // (cos 4 f_i, sin 4 f_i): four-position step, used by the K rotation
  uint32_t tmem_base;
};
// Barriers live at the same offset in both CTAs.  "local" ones are completed and waited on inside one CTA; "leader" ones
// are waited on only by the MMA issuer / scheduler of CTA rank 0 and collect arrivals from BOTH CTAs (mbar_arrive_cl);
// "multicast" ones are completed in both CTAs at once by a tcgen05.commit of the leader's MMA issuer.
enum Bar {
  SCHED_FULL = 0,                       // [kRing] local, 1 arrival by the leader's scheduler (remote for rank 1)
  SCHED_EMPTY = SCHED_FULL + kRing,     // [kRing] leader, 15 consumer warps per CTA
  Q_FULL = SCHED_EMPTY + kRing,         // local (TMA)
  Q_READY,                              // [2] leader, 4 softmax warps per CTA
  Q_EMPTY = Q_READY + 2,                // multicast
  K_FULL,                               // [kKStages] local (TMA)
  K_READY = K_FULL + kKStages,          // [kKStages] leader, 4 rotation warps per CTA
  K_EMPTY = K_READY + kKStages,         // [kKStages] multicast
  V_FULL = K_EMPTY + kKStages,          // [kVStages] local (TMA)
  V_PEER = V_FULL + kVStages,           // [kVStages] leader, 1 arrival by rank 1's forwarder warp: its half of V has landed
  V_EMPTY = V_PEER + kVStages,          // [kVStages] multicast
  V_FIX = V_EMPTY + kVStages,           // local, 128 rotation threads
  S_FULL,                               // [2] multicast
  P_FULL = S_FULL + 2,                  // [2] leader, 4 softmax warps per CTA
  O_FULL = P_FULL + 2,                  // [2] multicast
  O_FREE = O_FULL + 2,                  // [2] leader, 4 softmax warps per CTA
  P_HALF = O_FREE + 2,                  // [2] leader, 4 softmax warps per CTA: P of the tile's first 64 keys is in TMEM
  XCHG = P_HALF + 2,                    // local, 128 tile-B softmax threads: (O_B, m_B, l_B) of a dual item are in shared memory
  NUM_BARS
};
static_assert(NUM_BARS <= 36, "barrier array too small");
static_assert(sizeof(Smem) <= 232448, "shared memory budget");
static_assert(sizeof(ItemInfo) == 48, "ring entries are copied to the peer CTA as three 16-byte stores");

struct Params {
  PrefillArgs a;
  int hq, hkv;
  float scale_log2;
  unsigned flags;
  PlanHeader* hdr;
  const TileDesc* tiles;
  int oob_grp;                       // first row-group coordinate beyond the cache tensor map: TMA zero-fills
  int dual_ok;                       // the plan may make dual items (host decision from scalars: small grids only)
  float* part_o;                     // KV-range splits: partial O [token slot][hq][128] fp32 and the chunk's lse [token slot][hq]
  float* part_lse;
  unsigned long long phase_inc[64];  // F_i (common.cuh)
  float2 step1[64];                  // (cos f_i, sin f_i)
  float2 step4[64];                  // (cos 4 f_i, sin 4 f_i): the four-position RoPE step of the rotation lanes
};

// A work item as one CTA of the pair sees it.  The item covers up to 4 * TOK query tokens (TOK = 128 / G tokens fill one
// 128-row MMA tile): CTA rank c owns tokens [2 c TOK, 2 c TOK + 2 TOK) of it, tile A the first TOK of those, tile B the rest.
// Both CTAs run the SAME number of KV tiles for a tile slot (the MMA covers both); rows a CTA does not own are masked.
// DUAL items (short Q, long KV: ntok <= 2 TOK and n_kv >= kDualMinTiles, chosen by the plan): the two tile slots of a CTA hold
// the SAME query rows (CTA rank c owns tokens [c TOK, c TOK + TOK)) and split the KV range - slot A runs tiles [0, n_a), slot B
// tiles [n_a, n_kv) - so a 64-token suffix over a long context takes half as many tile steps and keeps both CTAs busy.  The
// K / V "uses" are interleaved in the order the MMA issuer consumes them: use u = 2 j + x is tile j of slot x.  At the end
// the B warps hand (O_B, m_B, l_B) to the A warps through shared memory and those merge the two partial softmaxes.
struct Item {
  int t0, ntok, r, idx0, lo, kvh, n_kv, kv_hi, kv_len, kv_off;
  int kv_lo, tb, ntok_a, ntok_b, n_a, n_b;
  int part;   // > 0: a KV-range chunk; its rows go to partial token slots part - 1 + (token within the item)
  bool dual;
  __device__ __forceinline__ int ntok_x(int x) const { return x ? ntok_b : ntok_a; }
  __device__ __forceinline__ int n_x(int x) const { return x ? n_b : n_a; }   // KV tiles slot x runs (0: the pair skips the slot)
  __device__ __forceinline__ int tile_x(int x, int i) const { return (dual && x) ? n_a + i : i; }      // i-th KV tile of slot x
  __device__ __forceinline__ int tile_of_use(int u) const { return dual ? ((u & 1) ? n_a + (u >> 1) : (u >> 1)) : u; }
  __device__ __forceinline__ int tok_x(int x, int tok_per_tile) const { return dual ? tb : tb + x * tok_per_tile; }   // first token of slot x
};
template <int TOK, bool kDual>
__device__ __forceinline__ Item load_item(const ItemInfo& ii, int rank) {
  Item it;
  it.t0 = ii.t0; it.ntok = ii.ntok; it.r = ii.r; it.idx0 = ii.idx0; it.lo = ii.lo; it.kvh = ii.kvh; it.n_kv = ii.n_kv;
  it.kv_hi = ii.kv_hi; it.kv_len = ii.kv_len; it.kv_off = ii.kv_off;
  it.kv_lo = it.lo & ~(kBlock - 1);
  it.dual = kDual && ii.pad[0] != 0;   // kDual = false: a compile-time constant, every dual branch folds away
  it.part = kDual ? ii.pad[1] : 0;     // splits are only made where dual items are
  if (it.dual) {
    it.tb = rank * TOK;
    it.ntok_a = it.ntok_b = min(max(it.ntok - it.tb, 0), TOK);
    it.n_a = (it.n_kv + 1) >> 1; it.n_b = it.n_kv - it.n_a;
  } else {
    it.tb = rank * 2 * TOK;
    const int mine = min(max(it.ntok - it.tb, 0), 2 * TOK);
    it.ntok_a = min(mine, TOK); it.ntok_b = mine - it.ntok_a;
    it.n_a = it.n_kv; it.n_b = it.ntok > TOK ? it.n_kv : 0;
  }
  return it;
}


// RoPE state of one rotation lane.  A warp covers 4 tile rows per step: lane = (row-in-step = lane >> 3, 16-byte
// chunk = lane & 7); the lane owns dims [8*chunk, 8*chunk + 8) of both halves of its row, i.e. 8 RoPE pairs (i, i + 64)
// and 8 frequencies, kept as four packed f32x2 (cos, sin) registers.  One 128-bit shared load / store per half.
struct Rot8 {
  uint64_t c[4], s[4];
  // exact restart at position p: 64-bit fixed-point phase (common.cuh) + MUFU on the reduced angle
  __device__ __forceinline__ void restart(int p, uint32_t finc_addr) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const uint4 f = lds128(finc_addr + 16 * e);   // F of frequencies 2e, 2e + 1 of this lane
      const unsigned long long f0 = ((unsigned long long)f.y << 32) | f.x, f1 = ((unsigned long long)f.w << 32) | f.z;
      const unsigned long long p0 = (unsigned long long)(unsigned)p * f0, p1 = (unsigned long long)(unsigned)p * f1;
      const float a0 = (float)(int)(p0 >> 32) * 1.4629180792671596e-9f;   // * pi * 2^-31
      const float a1 = (float)(int)(p1 >> 32) * 1.4629180792671596e-9f;
      c[e] = pk2(__cosf(a0), __cosf(a1));
      s[e] = pk2(__sinf(a0), __sinf(a1));
    }
  }
  // angle-addition step by a fixed position stride: (c, s) <- (c, s) * (cd, sd)
  __device__ __forceinline__ void advance(const uint64_t (&cd)[4], const uint64_t (&sd)[4], const uint64_t (&nsd)[4]) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const uint64_t cn = fma2(c[e], cd[e], mul2(s[e], nsd[e]));
      s[e] = fma2(s[e], cd[e], mul2(c[e], sd[e]));
      c[e] = cn;
    }
  }
  // rotate the lane's 8 + 8 elements of one 128-dim row (already loaded: lo / hi = its chunk of the two halves) and
  // store them back; addr = the lane's chunk in the low half, half_off = distance to the high half
  __device__ __forceinline__ void rotate_store(uint32_t addr, uint32_t half_off, const uint4& lo, const uint4& hi) const {
    const uint32_t wl[4] = {lo.x, lo.y, lo.z, lo.w}, wh[4] = {hi.x, hi.y, hi.z, hi.w};
    uint32_t ol[4], oh[4];
    const uint64_t neg1 = pk2(-1.f, -1.f);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const uint64_t a = pk2(bf16lo(wl[e]), bf16hi(wl[e])), b = pk2(bf16lo(wh[e]), bf16hi(wh[e]));
      const uint64_t ns = mul2(s[e], neg1);
      const uint64_t an = fma2(a, c[e], mul2(b, ns));
      const uint64_t bn = fma2(b, c[e], mul2(a, s[e]));
      float x0, x1, y0, y1;
      upk2(an, x0, x1); upk2(bn, y0, y1);
      ol[e] = pack_bf16(x0, x1); oh[e] = pack_bf16(y0, y1);
    }
    sts128(addr, make_uint4(ol[0], ol[1], ol[2], ol[3]));
    sts128(addr + half_off, make_uint4(oh[0], oh[1], oh[2], oh[3]));
  }
};

// kKeyMask: MINIPIC_KEY_MASK variant; kDual: dual items possible (the plan only makes them on small grids).  Both are their own
// instantiations, so the common path (config 5) pays nothing for either.
template <int G, bool kKeyMask, bool kDual>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
prefill_sm100_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
                     const __grid_constant__ CUtensorMap tmap_v, const __grid_constant__ CUtensorMap tmap_o,
                     const __grid_constant__ Params prm) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  constexpr int TOK = BM / G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)cluster_ctarank();   // 0 = leader: owns the scheduler, the MMA issuer and every "leader" barrier
  const PrefillArgs& a = prm.a;
  const uint32_t bar0 = smem_u32(sm.bars);
  const uint32_t lbar0 = mapa(bar0, 0);      // the leader's barrier array in the cluster window (== own array for rank 0)
  auto bar = [&](int b) { return bar0 + 8u * (uint32_t)b; };
  auto lbar = [&](int b) { return lbar0 + 8u * (uint32_t)b; };
  Waiter w{&prm.hdr->err, false};

  if (threadIdx.x >= 64 && threadIdx.x < 128) {
    sm.finc[threadIdx.x - 64] = prm.phase_inc[threadIdx.x - 64];
    sm.step1[threadIdx.x - 64] = prm.step1[threadIdx.x - 64];
    sm.step4[threadIdx.x - 64] = prm.step4[threadIdx.x - 64];
  }
#ifdef MINIPIC_TRACE
  int trace_n = 0;
#endif
  if (threadIdx.x == 0) {
    if (smem_u32(smem_raw) & 1023u) atomicCAS(&prm.hdr->err, 0, 2);   // swizzled tiles need a 1024-byte aligned base
    for (int s = 0; s < kRing; ++s) { mbar_init(bar(SCHED_FULL + s), 1); mbar_init(bar(SCHED_EMPTY + s), 30); }
    mbar_init(bar(Q_FULL), 1); mbar_init(bar(Q_READY), 8); mbar_init(bar(Q_READY + 1), 8); mbar_init(bar(Q_EMPTY), 1);
    for (int s = 0; s < kKStages; ++s) { mbar_init(bar(K_FULL + s), 1); mbar_init(bar(K_READY + s), 8); mbar_init(bar(K_EMPTY + s), 1); }
    for (int s = 0; s < kVStages; ++s) { mbar_init(bar(V_FULL + s), 1); mbar_init(bar(V_PEER + s), 1); mbar_init(bar(V_EMPTY + s), 1); }
    mbar_init(bar(V_FIX), 128);
    for (int x = 0; x < 2; ++x) {
      mbar_init(bar(S_FULL + x), 1); mbar_init(bar(P_FULL + x), 8); mbar_init(bar(O_FULL + x), 1); mbar_init(bar(O_FREE + x), 8);
    }
    mbar_init(bar(P_HALF), 8); mbar_init(bar(P_HALF + 1), 8);
    mbar_init(bar(XCHG), 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 13) {  // TMEM: 512 columns = S_A | S_B | O_A | O_B, 128 each; P_X aliases the first 64 columns of S_X.
                     // cta_group::2: the same warp of both CTAs allocates; both get all 512 columns (base 0)
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::);
  }
  tc_fence_before();
  cluster_sync_all();   // barriers of BOTH CTAs are initialised before anyone arrives remotely
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  if (kDual) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // split_merge_kernel (small grids) may queue up behind the tail

  if (warp >= 12) {
    reg_dec<kRegsCtl>();
    if (warp == 15 && rank == 0) {
      // ============================================================ scheduler (leader only): item ring of both CTAs
      const uint32_t ring_l = smem_u32(sm.ring), ring_p = mapa(ring_l, 1), full_p = mapa(bar(SCHED_FULL), 1);
      if (lane == 0) {
        // PROGRAMMATIC DEPENDENT LAUNCH: this grid may start while plan_kernel is still sorting (its blocks signal
        // launch_dependents at once), so the launch latency and the prologue above overlap the plan.  Only this thread reads
        // what the plan writes (item count, sorted descriptors): it waits here for the plan grid to complete and flush.
        asm volatile("griddepcontrol.wait;" ::: "memory");
        const int n_items = *(volatile const int*)&prm.hdr->n_tiles * prm.hkv;
        for (uint32_t it_n = 0;; ++it_n) {
          const int slot = it_n & (kRing - 1);
          w.wait(bar(SCHED_EMPTY + slot), ((it_n / kRing) & 1) ^ 1);
          const int item = w.dead ? n_items : atomicAdd(&prm.hdr->next_item, 1);
          ItemInfo ii;
          if (item >= n_items) {
            ii.t0 = -1; ii.ntok = 0; ii.r = 0; ii.idx0 = 0; ii.lo = 0; ii.kvh = 0; ii.n_kv = 0; ii.kv_hi = 0; ii.kv_len = 0; ii.kv_off = 0;
          } else {
            const TileDesc td = prm.tiles[item / prm.hkv];
            ii.t0 = td.t0; ii.ntok = td.ntok; ii.r = td.r; ii.idx0 = td.idx0; ii.lo = td.lo; ii.kvh = item % prm.hkv; ii.n_kv = td.n_kv;
            ii.kv_hi = td.kv_hi; ii.kv_len = td.kv_len; ii.kv_off = td.kv_off;
          }
          ii.pad[0] = ii.pad[1] = 0;
          if (item < n_items) { ii.pad[0] = prm.tiles[item / prm.hkv].pad; ii.pad[1] = prm.tiles[item / prm.hkv].part; }
          sm.ring[slot] = ii;
          const uint32_t dst = ring_p + (uint32_t)slot * (uint32_t)sizeof(ItemInfo);
          st_cluster_v4(dst, ii.t0, ii.ntok, ii.r, ii.idx0);
          st_cluster_v4(dst + 16, ii.lo, ii.kvh, ii.n_kv, ii.kv_hi);
          st_cluster_v4(dst + 32, ii.kv_len, ii.kv_off, ii.pad[0], ii.pad[1]);
          mbar_arrive_cl_release(lbar(SCHED_FULL + slot));
          mbar_arrive_cl_release(full_p + 8u * (uint32_t)slot);
          TRACE(0, 1);
          if (item >= n_items) break;
        }
      }
    } else if (warp == 15) {
      // ============================================================ V forwarder (rank 1): tells the leader's MMA issuer that
      // this CTA's half of a V tile has landed (and, for a partial last block, that its tail rows are zeroed)
      uint32_t vc = 0, fixc = 0;
      for (uint32_t it_n = 0;; ++it_n) {
        const int slot = it_n & (kRing - 1);
        w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
        if (__any_sync(0xffffffffu, w.dead) || sm.ring[slot].t0 < 0) break;
        const Item it = load_item<TOK, kDual>(sm.ring[slot], rank);
        const int n = it.n_kv;
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
        const bool vfix = (it.kv_hi & (kBlock - 1)) != 0;
        for (int i = 0; i < n; ++i, ++vc) {   // i = use index (see struct Item)
          const int st = vc % kVStages;
          w.wait(bar(V_FULL + st), (vc / kVStages) & 1);
          if (it.tile_of_use(i) == n - 1 && vfix) { w.wait(bar(V_FIX), fixc & 1); ++fixc; }
          __syncwarp();
          if (lane == 0) mbar_arrive_cl(lbar(V_PEER + st));
        }
      }
    } else if (warp == 12) {
      // ============================================================ Q / K TMA producer (a4): this CTA's 64 keys of every K tile
      uint32_t kc = 0, qc = 0;
      for (uint32_t it_n = 0;; ++it_n) {
        const int slot = it_n & (kRing - 1);
        w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
        if (__any_sync(0xffffffffu, w.dead) || sm.ring[slot].t0 < 0) break;
        const Item it = load_item<TOK, kDual>(sm.ring[slot], rank);
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
        if (it.n_kv == 0) continue;
        const int nblk_total = (it.kv_hi + kBlock - 1) / kBlock;   // blocks [0, nblk_total) of the request hold visible keys
        const int* bt = a.block_tables + (size_t)it.r * a.max_blocks;
        auto block_grp = [&](int i) {   // cache row-group coordinate of this lane's block (lanes 0-3) of KV tile i
          const int b = (it.kv_lo >> 4) + i * (BN / kBlock) + rank * (kKeysCta / kBlock) + lane;
          return (lane < kKeysCta / kBlock && b < nblk_total) ? (__ldg(bt + b) * prm.hkv + it.kvh) * 2 : prm.oob_grp;
        };
        int y = block_grp(it.tile_of_use(0));
        for (int i = 0; i < it.n_kv; ++i) {   // i = use index: tile it.tile_of_use(i)
          const int y_next = (i + 1 < it.n_kv) ? block_grp(it.tile_of_use(i + 1)) : 0;
          {  // one K tile: one 4 KB box per physical block
            const int st = kc % kKStages;
            if (lane == 0) { w.wait(bar(K_EMPTY + st), ((kc / kKStages) & 1) ^ 1); if (!w.dead) mbar_expect_tx(bar(K_FULL + st), kKTileBytes); }
            if (__any_sync(0xffffffffu, w.dead)) break;   // a timed-out wait: stop issuing, let the kernel drain
            if (lane < kKeysCta / kBlock) tma_load_4d(smem_u32(sm.k[st]) + lane * 4096, &tmap_k, bar(K_FULL + st), 0, 0, 0, y);
            ++kc;
            TRACE_L0(5, 2);
          }
          if (i == 0) {  // this CTA's Q rows: (token, head-in-group), tile A then tile B
            const int ntile = it.dual ? (it.ntok_a > 0 ? 1 : 0) : (it.ntok_b > 0 ? 2 : (it.ntok_a > 0 ? 1 : 0));   // dual: both slots read tile 0
            if (lane == 0) { w.wait(bar(Q_EMPTY), (qc & 1) ^ 1); if (!w.dead) mbar_expect_tx(bar(Q_FULL), ntile * kTileBytes); }
            if (__any_sync(0xffffffffu, w.dead)) break;
            if (lane < 2 * ntile) {
              const int x = lane >> 1, h = lane & 1;
              tma_load_3d(smem_u32(sm.q[x]) + h * kHalfBytes, &tmap_q, bar(Q_FULL), 64 * h, it.kvh * G, it.t0 + it.tb + x * TOK);
            }
            ++qc;
            TRACE_L0(5, 3);
          }
          y = y_next;
        }
      }
    } else if (warp == 14) {
      // ============================================================ V TMA producer (a4): this CTA's half of head_dim, all 128 keys
      uint32_t vc = 0;
      for (uint32_t it_n = 0;; ++it_n) {
        const int slot = it_n & (kRing - 1);
        w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
        if (__any_sync(0xffffffffu, w.dead) || sm.ring[slot].t0 < 0) break;
        const ItemInfo ii = sm.ring[slot];
        const Item itv = load_item<TOK, kDual>(sm.ring[slot], rank);
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
        if (ii.n_kv == 0) continue;
        const int kv_lo = ii.lo & ~(kBlock - 1);
        const int nblk_total = (ii.kv_hi + kBlock - 1) / kBlock;
        const int* bt = a.block_tables + (size_t)ii.r * a.max_blocks;
        auto block_grp = [&](int i) {
          const int b = (kv_lo >> 4) + i * (BN / kBlock) + lane;
          return (lane < BN / kBlock && b < nblk_total) ? (__ldg(bt + b) * prm.hkv + ii.kvh) * 2 : prm.oob_grp;
        };
        int y = block_grp(itv.tile_of_use(0));
        for (int i = 0; i < ii.n_kv; ++i) {   // i = use index
          const int y_next = (i + 1 < ii.n_kv) ? block_grp(itv.tile_of_use(i + 1)) : 0;
          const int st = vc % kVStages;
          if (lane == 0) { w.wait(bar(V_EMPTY + st), ((vc / kVStages) & 1) ^ 1); if (!w.dead) mbar_expect_tx(bar(V_FULL + st), kVTileBytes); }
          if (__any_sync(0xffffffffu, w.dead)) break;
          if (lane < BN / kBlock) tma_load_4d(smem_u32(sm.v[st]) + lane * 2048, &tmap_v, bar(V_FULL + st), 0, 0, rank, y);
          ++vc;
          TRACE_L0(6, 4);
          y = y_next;
        }
      }
    } else if (warp == 13 && rank == 0) {
      // ============================================================ MMA issuer (a6, a8), leader CTA only
      // The whole warp runs the control flow converged on warp-uniform values (item fields are broadcast from
      // lane 0, so descriptors, stages and phases live in uniform registers); one elected lane issues every
      // tcgen05.mma / tcgen05.commit for the PAIR.  This role lives in 48 registers: 32-bit descriptor words, running
      // stage / phase counters, no per-stage tables.
      constexpr uint32_t idesc_qk = instr_desc(false), idesc_pv = instr_desc(true);
      const uint32_t q_lo = ((smem_u32(sm.q[0]) >> 4) & 0x3FFF) | (1u << 16);          // + x * 2048
      const uint32_t k_lo = ((smem_u32(sm.k[0]) >> 4) & 0x3FFF) | (1u << 16);          // + stage * 1024
      const uint32_t v_lo = ((smem_u32(sm.v[0]) >> 4) & 0x3FFF) | (1u << 16);          // + stage * 1024
      uint32_t k_st = 0, k_ph = 0, v_st = 0, v_ph = 0;   // next K / V stage to consume and its full-barrier parity
      uint32_t ph = 0;   // bit 0,1: P_FULL parity of tile A,B; bit 2,3: O_FREE; bit 4: Q_READY; bit 5: V_FIX; bit 6,7: P_HALF
      for (uint32_t it_n = 0;; ++it_n) {
        const int slot = it_n & (kRing - 1);
        w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
        if (__any_sync(0xffffffffu, w.dead) || sm.ring[slot].t0 < 0) break;
        int n, nx1, kv_hi, dual;
        {
          const Item it = load_item<TOK, kDual>(sm.ring[slot], 0);
          n = __shfl_sync(0xffffffffu, it.n_kv, 0);
          nx1 = __shfl_sync(0xffffffffu, it.n_b, 0); kv_hi = __shfl_sync(0xffffffffu, it.kv_hi, 0);
          dual = __shfl_sync(0xffffffffu, (int)it.dual, 0);
        }
        const bool vfix = (kv_hi & (kBlock - 1)) != 0;
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
        if (n == 0) continue;
        // QK^T of tile x against K stage st: S_x = Q_x K'^T for both CTAs (elected lane only)
        auto qk = [&](int x, uint32_t st) {   // dual items: both slots read Q tile 0 (the same rows)
          const uint32_t a_lo = q_lo + (uint32_t)(dual ? 0 : x) * (kTileBytes >> 4), b_lo = k_lo + st * (kKTileBytes >> 4);
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks) {
            const uint32_t off_q = (ks >> 2) * (kHalfBytes >> 4) + (ks & 3) * 2, off_k = (ks >> 2) * (kKvHalfOff >> 4) + (ks & 3) * 2;
            umma_ss(tmem + x * BN, a_lo + off_q, b_lo + off_k, idesc_qk, ks > 0);
          }
          tc_commit(bar(S_FULL + x));
          TRACE(1, 10 + x);
        };
        if (dual) {
          // ---- dual item: K / V uses alternate between the slots (use u = 2 j + x is tile j of slot x); n_a = n - nx1 >= nx1
          const int n_a = n - nx1;
          auto k_next = [&]() { if (++k_st == kKStages) { k_st = 0; k_ph ^= 1; } };
          auto issue_qk = [&](int x, int u) {   // QK^T of slot x against K use u (the next one in the ring), then release it
            w.wait(bar(K_READY + k_st), k_ph);
            tc_fence_after();
            if (elect_one()) {
              qk(x, k_st);
              tc_commit(bar(K_EMPTY + k_st));
              if (u == n - 1) tc_commit(bar(Q_EMPTY));   // the item's last QK^T
            }
            __syncwarp();
            k_next();
          };
          w.wait(bar(Q_READY), (ph >> 4) & 1);
          w.wait(bar(Q_READY + 1), (ph >> 4) & 1); ph ^= 16u;
          issue_qk(0, 0);
          issue_qk(1, 1);
#pragma unroll 1
          for (int j = 0; j < n_a; ++j) {
#pragma unroll 1
            for (int x = 0; x < 2; ++x) {
              if (x == 1 && j >= nx1) break;
              const int u = 2 * j + x, nx = x ? nx1 : n_a;
              w.wait(bar(V_FULL + v_st), v_ph);
              w.wait(bar(V_PEER + v_st), v_ph);
              if (vfix && (x ? n_a + j : j) == n - 1) { w.wait(bar(V_FIX), (ph >> 5) & 1); ph ^= 32u; }
              w.wait(bar(P_HALF + x), (ph >> (6 + x)) & 1); ph ^= 64u << x;
              w.wait(bar(P_FULL + x), (ph >> x) & 1); ph ^= 1u << x;
              if (j == 0) { w.wait(bar(O_FREE + x), ((ph >> (2 + x)) & 1) ^ 1); ph ^= 4u << x; }
              tc_fence_after();
              if (elect_one()) {
                const uint32_t b_lo = v_lo + v_st * (kVTileBytes >> 4);
#pragma unroll
                for (int ks = 0; ks < BN / 16; ++ks)
                  umma_ts(tmem + (2 + x) * BN, tmem + x * BN + ks * 8, b_lo + ks * (2 * kVGroupBytes >> 4), idesc_pv, (j > 0 || ks > 0));
                if (j == nx - 1) tc_commit(bar(O_FULL + x));
                tc_commit(bar(V_EMPTY + v_st));
              }
              __syncwarp();
              if (++v_st == kVStages) { v_st = 0; v_ph ^= 1; }
              if (j + 1 < nx) issue_qk(x, u + 2);
            }
          }
          continue;
        }
        w.wait(bar(Q_READY), (ph >> 4) & 1);   // tile A of Q is rotated; tile B follows while QK_A already runs
        w.wait(bar(K_READY + k_st), k_ph);
        tc_fence_after();
        if (elect_one()) qk(0, k_st);
        __syncwarp();
        w.wait(bar(Q_READY + 1), (ph >> 4) & 1); ph ^= 16u;
        tc_fence_after();
        if (elect_one()) {
          if (nx1 > 0) qk(1, k_st);
          tc_commit(bar(K_EMPTY + k_st));
          if (n == 1) tc_commit(bar(Q_EMPTY));
        }
        __syncwarp();
        if (++k_st == kKStages) { k_st = 0; k_ph ^= 1; }
#pragma unroll 1
        for (int i = 0; i < n; ++i) {
          w.wait(bar(V_FULL + v_st), v_ph);
          w.wait(bar(V_PEER + v_st), v_ph);
          if (i == n - 1 && vfix) { w.wait(bar(V_FIX), (ph >> 5) & 1); ph ^= 32u; }
          bool k_waited = false;
#pragma unroll 1
          for (int x = 0; x < 2; ++x) {
            const int nx = x ? nx1 : n;
            const bool do_pv = i < nx, do_qk = i + 1 < nx;
            // PV in two halves: the first 64 keys' P is published (P_HALF) while the softmax warps still run the exps of the
            // other 64, so half of PV is off the P -> PV -> QK -> S chain that bounds a tile slot's period
            if (do_pv) {
              w.wait(bar(P_HALF + x), (ph >> (6 + x)) & 1); ph ^= 64u << x;
              if (i == 0) { w.wait(bar(O_FREE + x), ((ph >> (2 + x)) & 1) ^ 1); ph ^= 4u << x; }
            }
            tc_fence_after();
            const uint32_t b_lo_v = v_lo + v_st * (kVTileBytes >> 4);
            if (do_pv && elect_one()) {
#pragma unroll
              for (int ks = 0; ks < 2 * kPEarly; ++ks)
                umma_ts(tmem + (2 + x) * BN, tmem + x * BN + ks * 8, b_lo_v + ks * (2 * kVGroupBytes >> 4), idesc_pv, (i > 0 || ks > 0));
            }
            __syncwarp();
            // the next K tile is waited for HERE, while the softmax warps still work on P: off the P -> PV -> QK -> S chain
            if (do_qk && !k_waited) { w.wait(bar(K_READY + k_st), k_ph); k_waited = true; }
            if (do_pv) { w.wait(bar(P_FULL + x), (ph >> x) & 1); ph ^= 1u << x; }
            tc_fence_after();
            if (do_pv && elect_one()) {
#pragma unroll
              for (int ks = 2 * kPEarly; ks < BN / 16; ++ks)
                umma_ts(tmem + (2 + x) * BN, tmem + x * BN + ks * 8, b_lo_v + ks * (2 * kVGroupBytes >> 4), idesc_pv, 1);
              if (i == nx - 1) tc_commit(bar(O_FULL + x));
              TRACE(1, 20 + x);
            }
            __syncwarp();
            if (elect_one()) {
              if (x == 1) tc_commit(bar(V_EMPTY + v_st));
              if (do_qk) qk(x, k_st);
              if (x == 1 && i + 1 < n) {
                tc_commit(bar(K_EMPTY + k_st));
                if (i + 1 == n - 1) tc_commit(bar(Q_EMPTY));
              }
            }
            __syncwarp();
          }
          if (++v_st == kVStages) { v_st = 0; v_ph ^= 1; }
          if (i + 1 < n) { if (++k_st == kKStages) { k_st = 0; k_ph ^= 1; } }
        }
      }
    }
  } else if (warp >= 8) {
    // ============================================================ rotation warps: this CTA's 64 keys of every K tile (a5)
    // NOTE on code shape: the kernel is instruction-cache bound (four roles with different code share an SM), so only the
    // per-tile K path is unrolled.  The once-per-item Q rotation (a3) lives in the softmax warps as a rolled loop.
    reg_dec<kRegsRot>();
    const int rw = warp - 8, rot_tid = threadIdx.x - 256;
    const int rsub = lane >> 3, ch = lane & 7;
    Rot8 rot;
    uint64_t c4[4], s4[4], ns4[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const float2 u0 = prm.step4[8 * ch + 2 * e], u1 = prm.step4[8 * ch + 2 * e + 1];
      c4[e] = pk2(u0.x, u1.x); s4[e] = pk2(u0.y, u1.y); ns4[e] = pk2(-u0.y, -u1.y);
    }
    const uint32_t finc_addr = smem_u32(sm.finc) + 64 * ch;
    // byte offset of the lane's 16-byte chunk in row (4k + rsub) of a 16-row stretch: even k / odd k (SWIZZLE_128B)
    const uint32_t off_e = (uint32_t)(rsub * 128 + ((ch ^ rsub) << 4));
    const uint32_t off_o = (uint32_t)((4 + rsub) * 128 + ((ch ^ (4 + rsub)) << 4));
    const bool k_prerot = (prm.flags & MINIPIC_K_PREROTATED) != 0;
    constexpr int RW = kKeysCta / 4;   // 16 tile rows (= 2 row groups) per rotation warp
    uint32_t kc = 0, vc = 0;
    for (uint32_t it_n = 0;; ++it_n) {
      const int slot = it_n & (kRing - 1);
      w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
      if (w.dead || sm.ring[slot].t0 < 0) break;
      const Item it = load_item<TOK, kDual>(sm.ring[slot], rank);
      __syncwarp();
      if (lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
      if (it.n_kv == 0) continue;
      const int* pos = a.kv_positions + it.kv_off;
      const int jw = it.kv_lo + rank * kKeysCta + RW * rw;   // first key of this warp's rows in tile 0
      // lane l (< 16) holds the position of key jw + i * 128 + l (fetched one tile early)
      int myp = __ldg(pos + min(jw + it.tile_of_use(0) * BN + (lane & (RW - 1)), it.kv_len - 1));
      for (int i = 0; i < it.n_kv; ++i) {   // i = use index: tile it.tile_of_use(i)
        const int st = kc % kKStages;
        const int tile = it.tile_of_use(i);
        const int j0 = jw + tile * BN;
        const int myp_next = (i + 1 < it.n_kv) ? __ldg(pos + min(jw + it.tile_of_use(i + 1) * BN + (lane & (RW - 1)), it.kv_len - 1)) : 0;
        const int nrow = it.kv_hi - j0;                   // rows of this warp's chunk that hold visible keys
        const bool work = !k_prerot && nrow > 0;
        const int p0 = __shfl_sync(0xffffffffu, myp, 0);
        // consecutive positions (every workload the paper describes): one exact restart, then 4-position steps
        const bool contig = __all_sync(0xffffffffu, (lane & (RW - 1)) >= nrow || myp == p0 + (lane & (RW - 1)));
        if (work && contig) rot.restart(p0 + rsub, finc_addr);          // before the wait: overlaps the TMA latency
        w.wait(bar(K_FULL + st), (kc / kKStages) & 1);
        if (rw == 0) TRACE_L0(2, 30);
        if (work) {
          const uint32_t kt = smem_u32(sm.k[st]) + (uint32_t)rw * (2 * kGroupBytes);
          auto row_addr = [&](int k) { return kt + (k >> 1) * kGroupBytes + ((k & 1) ? off_o : off_e); };
          if (contig) {
            uint4 lo = lds128(row_addr(0)), hi = lds128(row_addr(0) + kKvHalfOff);
#pragma unroll
            for (int k = 0; k < RW / 4; ++k) {
              uint4 lo_n = lo, hi_n = hi;
              if (k < RW / 4 - 1) { lo_n = lds128(row_addr(k + 1)); hi_n = lds128(row_addr(k + 1) + kKvHalfOff); }
              rot.rotate_store(row_addr(k), kKvHalfOff, lo, hi);
              if (k < RW / 4 - 1) rot.advance(c4, s4, ns4);
              lo = lo_n; hi = hi_n;
            }
          } else {
#pragma unroll 1
            for (int k = 0; k < RW / 4; ++k) {
              if (4 * k >= nrow) break;
              rot.restart(__shfl_sync(0xffffffffu, myp, 4 * k + rsub), finc_addr);
              const uint4 lo = lds128(row_addr(k)), hi = lds128(row_addr(k) + kKvHalfOff);
              rot.rotate_store(row_addr(k), kKvHalfOff, lo, hi);
            }
          }
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(K_READY + st));
        if (rw == 0) TRACE_L0(2, 31);
        ++kc;
        myp = myp_next;
        // ---- V tile i: rows at or beyond kv_hi inside the last gathered block may hold anything (never written
        //      cache slots); their P is 0, make sure 0 * (those bits) is not NaN
        if (tile == it.n_kv - 1 && (it.kv_hi & (kBlock - 1)) != 0) {
          const int vs = (vc + i) % kVStages;
          w.wait(bar(V_FULL + vs), ((vc + i) / kVStages) & 1);
          const int first = it.kv_hi - (it.kv_lo + tile * BN), last = (first + kBlock - 1) & ~(kBlock - 1);
          if (rot_tid >= first && rot_tid < last) {
            const uint32_t vrow = smem_u32(sm.v[vs]) + (rot_tid >> 3) * kVGroupBytes + (rot_tid & 7) * 128;
#pragma unroll
            for (int c = 0; c < 8; ++c) sts128z(vrow + c * 16);
          }
          fence_proxy_async();
          mbar_arrive(bar(V_FIX));
        }
      }
      vc += it.n_kv;
    }
  } else {
    // ============================================================ softmax + epilogue warps (a7, a9): thread = row
    reg_inc<kRegsSoftmax>();
    const int x = warp >> 2;                 // 0: tile A, 1: tile B
    const int row = threadIdx.x & 127;
    const uint32_t t_lane = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t t_s = t_lane + x * BN, t_o = t_lane + (2 + x) * BN;
    const int tok_in = row / G, hg = row % G;
    uint32_t sc = 0, oc = 0, qc = 0, xc = 0;
    struct { bool valid, dual; int t0, kvh, ntok_x, n, pslot; float l, m; } pe;   // pslot >= 0: partial token slot of the tile's first token
    pe.valid = false;
    auto epilogue = [&]() {
      // ---- epilogue (a9): O / l -> out, LSE = ln sum exp of the scaled scores.  A thread owns a row in TMEM, but a row
      //      is 256 B in global memory: the warp transposes 64 columns at a time through its 4 KB staging buffer so
      //      that every store instruction writes four full 128-byte lines instead of 32 scattered 16-byte pieces
      if (pe.n > 0) { w.wait(bar(O_FULL + x), oc & 1); ++oc; tc_fence_after(); }
      // dual item (tile A warps only get here with pe.dual): merge slot B's partial softmax over the other half of the KV
      // range: m = max(m_A, m_B), O = O_A 2^(m_A - m) + O_B 2^(m_B - m), l likewise
      float wa = 1.f, wb = 0.f;
      const uint32_t xrow = smem_u32(sm.xchg[row]);
      if (pe.dual) {
        w.wait(bar(XCHG), xc & 1); ++xc;
        const float2 ml = sm.xml[row];
        const float m = fmaxf(pe.m, ml.x);
        wa = (pe.m == -INFINITY) ? 0.f : fast_exp2(pe.m - m);
        wb = (ml.x == -INFINITY) ? 0.f : fast_exp2(ml.x - m);
        pe.l = pe.l * wa + ml.y * wb;
        pe.m = m;
      }
      const float inv = pe.l > 0.f ? 1.f / pe.l : 0.f;
      if ((warp & 3) == 0) TRACE_L0(3 + x, 42);
      if (pe.ntok_x <= 0) {   // this CTA owns no row of the tile (the peer does): only release O
        if (pe.n > 0) { tc_fence_before(); __syncwarp(); if (lane == 0) mbar_arrive_cl(lbar(O_FREE + x)); }
        return;
      }
      {
        const uint32_t stg = smem_u32(sm.ostage[warp]);
        const int rr = lane >> 3, cc = lane & 7;
        const bool whole = pe.ntok_x == TOK;   // every row of the tile is a real query row: the warp's 32 rows go out
                                                  // as one TMA tensor store per pass (box = 64 columns x G heads x 32/G tokens)
        __nv_bfloat16* obase = (__nv_bfloat16*)a.out + ((size_t)pe.t0 * prm.hq + pe.kvh * G) * D + cc * 8;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
          float o[64];
          if (pe.n > 0) {
            tmem_ld32(t_o + pass * 64, o); tmem_ld32(t_o + pass * 64 + 32, o + 32);
            tmem_wait_ld();
            if (pass == 1) {   // O is in registers: the next item may start
              tc_fence_before(); __syncwarp();
              if (lane == 0) mbar_arrive_cl(lbar(O_FREE + x));
            }
          } else {
#pragma unroll
            for (int e = 0; e < 64; ++e) o[e] = 0.f;
          }
          if (pe.dual) {
#pragma unroll
            for (int c = 0; c < 16; ++c) {
              const uint4 u = lds128(xrow + (uint32_t)(((16 * pass + c) ^ (row & 31)) << 4));
              o[4 * c] = o[4 * c] * wa + __uint_as_float(u.x) * wb; o[4 * c + 1] = o[4 * c + 1] * wa + __uint_as_float(u.y) * wb;
              o[4 * c + 2] = o[4 * c + 2] * wa + __uint_as_float(u.z) * wb; o[4 * c + 3] = o[4 * c + 3] * wa + __uint_as_float(u.w) * wb;
            }
          }
          if (kDual && pe.pslot >= 0) {   // KV-range chunk: the row, normalised over the chunk, goes to its partial slot as fp32
            if (tok_in < pe.ntok_x) {
              float4* po = reinterpret_cast<float4*>(prm.part_o + ((size_t)(pe.pslot + tok_in) * prm.hq + pe.kvh * G + hg) * D + pass * 64);
#pragma unroll
              for (int c = 0; c < 16; ++c) po[c] = make_float4(o[4 * c] * inv, o[4 * c + 1] * inv, o[4 * c + 2] * inv, o[4 * c + 3] * inv);
            }
            continue;
          }
          if (lane == 0) tma_store_wait_read();   // the previous store out of this staging buffer has been read
          __syncwarp();
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            uint4 v;
            v.x = pack_bf16(o[8 * c] * inv, o[8 * c + 1] * inv); v.y = pack_bf16(o[8 * c + 2] * inv, o[8 * c + 3] * inv);
            v.z = pack_bf16(o[8 * c + 4] * inv, o[8 * c + 5] * inv); v.w = pack_bf16(o[8 * c + 6] * inv, o[8 * c + 7] * inv);
            sts128(stg + lane * 128 + ((c ^ (lane & 7)) << 4), v);
          }
          if (whole) {
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
              tma_store_3d(&tmap_o, stg, pass * 64, pe.kvh * G, pe.t0 + ((warp & 3) * 32) / G);
              tma_store_commit();
            }
          } else {
            __syncwarp();
#pragma unroll
            for (int itr = 0; itr < 8; ++itr) {
              const int r = itr * 4 + rr, rowg = (warp & 3) * 32 + r;
              const uint4 v = lds128(stg + r * 128 + ((cc ^ (r & 7)) << 4));
              if (rowg / G < pe.ntok_x)
                *reinterpret_cast<uint4*>(obase + ((size_t)(rowg / G) * prm.hq + rowg % G) * D + pass * 64) = v;
            }
            __syncwarp();
          }
        }
      }
      if ((warp & 3) == 0) TRACE_L0(3 + x, 43);
      if ((tok_in < pe.ntok_x)) {
        const float lse_row = pe.l > 0.f ? (pe.m + log2f(pe.l)) * 0.6931471805599453f : -INFINITY;
        if (kDual && pe.pslot >= 0) prm.part_lse[(size_t)(pe.pslot + tok_in) * prm.hq + pe.kvh * G + hg] = lse_row;
        else a.lse[(size_t)(pe.t0 + tok_in) * prm.hq + pe.kvh * G + hg] = lse_row;
      }
        };
    // Q rotation (a3) state of this lane: same row / chunk mapping as the K rotation lanes
    const int rw = warp & 3, rsub = lane >> 3, ch = lane & 7;
    const uint32_t finc_addr = smem_u32(sm.finc) + 64 * ch, step1_addr = smem_u32(sm.step1) + 64 * ch;
    const uint32_t off_e = (uint32_t)(rsub * 128 + ((ch ^ rsub) << 4));
    const uint32_t off_o = (uint32_t)((4 + rsub) * 128 + ((ch ^ (4 + rsub)) << 4));
    const bool q_prerot = (prm.flags & MINIPIC_Q_PREROTATED) != 0;
    constexpr int NTW = (32 / G) > 0 ? (32 / G) : 1;   // Q tokens per warp per tile
    for (uint32_t it_n = 0;; ++it_n) {
      const int slot = it_n & (kRing - 1);
      w.wait_cl(bar(SCHED_FULL + slot), (it_n / kRing) & 1);
      const bool stop = w.dead || sm.ring[slot].t0 < 0;   // one more trip for the deferred epilogue, then out
      const Item it = load_item<TOK, kDual>(sm.ring[slot], rank);
      __syncwarp();
      if (!stop && lane == 0) mbar_arrive_cl(lbar(SCHED_EMPTY + slot));
      const int n = stop ? 0 : it.n_x(x);      // KV tiles this tile slot runs (the same in both CTAs)
      const int tile_t = it.tok_x(x, TOK);     // first token (within the item) of this CTA's tile slot x
      if (!stop && it.n_kv > 0) {
        // ---- a3: rotate this warp's 32 rows of Q tile x in place: row = token * G + head-in-group, the G rows of a token
        //      share one position.  Exact restart at the first row, one-position steps while the positions are consecutive.
        //      The eight softmax warps do this (not the four K rotation warps): they would otherwise idle at the item
        //      boundary while K0, Q_A, Q_B queue up on the rotation warps.  Rolled loop: see the note on code size there.
        const int ntw = it.ntok_x(x) - (32 * rw) / G;   // tokens of this tile that this warp rotates
        int qpx = 0;
        const bool rot_q = !q_prerot && ntw > 0 && !(it.dual && x == 1);   // dual: slot B reads slot A's (rotated) Q tile
        if (rot_q) {
          const int tk = min((32 * rw) / G + min(lane, NTW - 1), it.ntok_x(x) - 1);
          qpx = __ldg(a.kv_positions + it.kv_off + min(it.idx0 + tile_t + tk, it.kv_len - 1));
        }
        if ((warp & 3) == 0) TRACE_L0(3 + x, 48);
        w.wait(bar(Q_FULL), qc & 1); ++qc;
        if ((warp & 3) == 0) TRACE_L0(3 + x, 49);
        if (rot_q) {
          Rot8 rot;
          uint64_t c1[4], s1[4], ns1[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const uint4 u = lds128(step1_addr + 16 * e);   // (cos, sin) of frequencies 2e, 2e + 1 of this lane
            c1[e] = pk2(__uint_as_float(u.x), __uint_as_float(u.z));
            s1[e] = pk2(__uint_as_float(u.y), __uint_as_float(u.w));
            ns1[e] = pk2(-__uint_as_float(u.y), -__uint_as_float(u.w));
          }
          const uint32_t qt = smem_u32(sm.q[x]) + (uint32_t)rw * 4096;
          int prev = 0;
#pragma unroll 1
          for (int k = 0; k < 8; ++k) {
            if ((4 * k) / G >= ntw) break;
            const uint32_t addr = qt + (k >> 1) * 1024 + ((k & 1) ? off_o : off_e);
            const uint4 lo = lds128(addr), hi = lds128(addr + kHalfBytes);
            const int p = __shfl_sync(0xffffffffu, qpx, ((32 * rw) % G + 4 * k + rsub) / G);
            if (k > 0 && p == prev + 1) rot.advance(c1, s1, ns1);
            else if (k == 0 || p != prev) rot.restart(p, finc_addr);
            prev = p;
            rot.rotate_store(addr, kHalfBytes, lo, hi);
          }
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(Q_READY + x));
      }
      if ((warp & 3) == 0) TRACE_L0(3 + x, 47);
      if (pe.valid) epilogue();   // previous item of this tile
      if (stop) break;
      if ((warp & 3) == 0) TRACE_L0(3 + x, 1000 + 4 * n + (it.dual ? 1 : 0) + (it.part > 0 ? 2 : 0));
      const bool row_ok = tok_in < it.ntok_x(x);
      const int idx_first = it.idx0 + tile_t;                               // lowest query index of this tile
      const int idx_row = min(it.idx0 + tile_t + tok_in, it.kv_len - 1);    // highest visible key of this row
      float m_used = -INFINITY, l_run = 0.f;   // m in log2 units (score * scale * log2 e)
      for (int i = 0; i < n; ++i, ++sc) {
        const int j0 = it.kv_lo + it.tile_x(x, i) * BN;
        float s[BN];
        // MINIPIC_KEY_MASK: keys with a negative logical position are invisible to every row.  Lane l looks
        // at the positions of columns l, l + 32, l + 64, l + 96 (fetched before the wait); four ballots give the tile's
        // 128-bit mask, warp-uniform, and tiles without a masked key (nearly all) pay nothing more.
        unsigned dead0 = 0, dead1 = 0, dead2 = 0, dead3 = 0;
        if (kKeyMask) {
          const int* pos = a.kv_positions + it.kv_off;
          const int jl = j0 + lane;
          dead0 = __ballot_sync(0xffffffffu, jl < it.kv_len && __ldg(pos + jl) < 0);
          dead1 = __ballot_sync(0xffffffffu, jl + 32 < it.kv_len && __ldg(pos + jl + 32) < 0);
          dead2 = __ballot_sync(0xffffffffu, jl + 64 < it.kv_len && __ldg(pos + jl + 64) < 0);
          dead3 = __ballot_sync(0xffffffffu, jl + 96 < it.kv_len && __ldg(pos + jl + 96) < 0);
        }
        w.wait(bar(S_FULL + x), sc & 1);
        if ((warp & 3) == 0) TRACE_L0(3 + x, 40);
        tc_fence_after();
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32(t_s + c * 32, s + c * 32);
        tmem_wait_ld();
        if ((warp & 3) == 0) TRACE_L0(3 + x, 44);
        // mask at 32-column chunk granularity (all bounds but c_hi are warp-uniform): a chunk that every row of the
        // tile sees needs no mask code, a chunk no row sees (above the causal diagonal) skips max / exp altogether
        const int c_lo = it.lo - j0;
        const int c_hi = row_ok ? idx_row - j0 : -1;
        const int c_hi_max = min(idx_first + TOK - 1, it.kv_len - 1) - j0;   // highest row of the tile (warp-uniform)
        if (j0 + BN - 1 > min(idx_first, it.kv_len - 1)) {   // tile reaches past the lowest row's last visible key
#pragma unroll
          for (int c = 0; c < BN; ++c) s[c] = (c <= c_hi) ? s[c] : -INFINITY;
        }
        if (kKeyMask && (dead0 | dead1 | dead2 | dead3)) {
#pragma unroll
          for (int c = 0; c < 32; ++c) {
            if ((dead0 >> c) & 1u) s[c] = -INFINITY;
            if ((dead1 >> c) & 1u) s[32 + c] = -INFINITY;
            if ((dead2 >> c) & 1u) s[64 + c] = -INFINITY;
            if ((dead3 >> c) & 1u) s[96 + c] = -INFINITY;
          }
        }
        if (c_lo > 0) {   // vis_lo inside the first gathered 16-token block (kv_lo = floor16(vis_lo)): c_lo < 16
#pragma unroll
          for (int c = 0; c < kBlock; ++c) s[c] = (c >= c_lo) ? s[c] : -INFINITY;
        }
        float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
        for (int c = 0; c < BN; c += 8) {
          mx0 = max3(mx0, s[c], s[c + 1]); mx1 = max3(mx1, s[c + 2], s[c + 3]);
          mx2 = max3(mx2, s[c + 4], s[c + 5]); mx3 = max3(mx3, s[c + 6], s[c + 7]);
        }
        const float m_new = fmaxf(m_used, fmaxf(max3(mx0, mx1, mx2), mx3) * prm.scale_log2);
        if ((warp & 3) == 0) TRACE_L0(3 + x, 45);
        if (i == 0) {
          m_used = m_new;
        } else {
          const bool grow = m_new > m_used + 8.f;   // lazy rescale: P may exceed 1 by up to 2^8 before O, l are rescaled
          if (__any_sync(0xffffffffu, grow)) {
            // S_FULL(i) was committed after PV(i-1): O is stable until this thread publishes P(i)
            const float corr = grow ? fast_exp2(m_used - m_new) : 1.f;
            if (grow) { l_run *= corr; m_used = m_new; }
#pragma unroll 1
            for (int c = 0; c < 8; ++c) {
              float o[16];
              tmem_ld16(t_o + c * 16, o);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 16; ++e) o[e] *= corr;
              tmem_st16(t_o + c * 16, reinterpret_cast<const uint32_t*>(o));
            }
          }
        }
        const float m_sub = (m_used == -INFINITY) ? 0.f : m_used;
        const uint64_t sc2 = pk2(prm.scale_log2, prm.scale_log2), nm2 = pk2(-m_sub, -m_sub);
        uint64_t lsum0 = pk2(0.f, 0.f), lsum1 = lsum0;
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          uint32_t pk[16];
          if (32 * h > c_hi_max) {   // keys above the causal diagonal for every row of the tile: P = 0, no exp
#pragma unroll
            for (int c = 0; c < 16; ++c) pk[c] = 0u;
            tmem_st16(t_s + 16 * h, pk);
            if (h == kPEarly - 1) { tmem_wait_st(); tc_fence_before(); __syncwarp(); if (lane == 0) mbar_arrive_cl(lbar(P_HALF + x)); }
            continue;
          }
#pragma unroll
          for (int c = 0; c < 16; ++c) {
            float x0, x1, p0, p1;
            upk2(fma2(pk2(s[32 * h + 2 * c], s[32 * h + 2 * c + 1]), sc2, nm2), x0, x1);
            p0 = fast_exp2(x0); p1 = fast_exp2(x1);
            if (c & 1) lsum1 = add2(lsum1, pk2(p0, p1)); else lsum0 = add2(lsum0, pk2(p0, p1));
            pk[c] = pack_bf16(p0, p1);
          }
          tmem_st16(t_s + 16 * h, pk);
          if (h == kPEarly - 1) { tmem_wait_st(); tc_fence_before(); __syncwarp(); if (lane == 0) mbar_arrive_cl(lbar(P_HALF + x)); }   // first keys: PV may start
        }
        {
          float a0, a1;
          upk2(add2(lsum0, lsum1), a0, a1);
          l_run += a0 + a1;
        }
        if ((warp & 3) == 0) TRACE_L0(3 + x, 46);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(P_FULL + x));
        if ((warp & 3) == 0) TRACE_L0(3 + x, 41);
      }
      // the epilogue of an item is DEFERRED until this tile's Q rows of the next item are rotated (below), so that QK of the
      // next item starts ~3 K cycles earlier; pe = what it needs.  A tile slot that ran KV tiles for the peer's rows only
      // (ntok_x = 0, n > 0) still has to consume O_FULL and release O.
      pe.valid = it.ntok_x(x) > 0 || n > 0; pe.t0 = it.t0 + tile_t; pe.kvh = it.kvh; pe.ntok_x = it.ntok_x(x); pe.n = n;
      pe.l = l_run; pe.m = m_used; pe.dual = it.dual; pe.pslot = it.part > 0 ? it.part - 1 + tile_t : -1;
      if (it.dual && x == 1) {
        // ---- dual item, slot B: hand (O_B, m_B, l_B) to the tile-A warps of this CTA right away (not deferred)
        w.wait(bar(O_FULL + 1), oc & 1); ++oc;
        tc_fence_after();
#pragma unroll 1
        for (int c = 0; c < 4; ++c) {
          float o[32];
          tmem_ld32(t_o + 32 * c, o);
          tmem_wait_ld();
#pragma unroll
          for (int q = 0; q < 8; ++q)
            sts128(smem_u32(sm.xchg[row]) + (uint32_t)(((8 * c + q) ^ (row & 31)) << 4),
                   make_uint4(__float_as_uint(o[4 * q]), __float_as_uint(o[4 * q + 1]), __float_as_uint(o[4 * q + 2]), __float_as_uint(o[4 * q + 3])));
        }
        sm.xml[row] = make_float2(m_used, l_run);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cl(lbar(O_FREE + 1));
        mbar_arrive(bar(XCHG));
        pe.valid = false;
      }
    }
    if (lane == 0) tma_store_wait_all();   // the staging buffers must outlive the last tensor stores
  }
  tc_fence_before();
  cluster_sync_all();   // no CTA may exit (or free TMEM) while its peer can still arrive on its barriers / run MMAs on it
  if (warp == 13) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
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
// cache viewed as a 4-D bf16 tensor (64 columns, 8 rows of a group [256 B apart], 2 halves of head_dim [128 B apart],
// row groups [2048 B apart]); box = (64, 8, 2, 2) = one (block, head) = 4 KB landing as [group][half][8 x 128 B], SWIZZLE_128B
// q viewed as [Tq][Hq][128]; box = (128/G tokens) x (G heads) x 64 columns: one half of an MMA tile, rows (token, head)
bool make_q_map(CUtensorMap* m, const void* q, int num_q_tokens, int hq, int group) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)hq, (cuuint64_t)num_q_tokens};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)hq * D * 2};
  cuuint32_t box[3] = {64, (cuuint32_t)group, (cuuint32_t)(BM / group)};
  cuuint32_t estr[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// out viewed as [Tq][Hq][128]; box = 64 columns x G heads x 32/G tokens = the 32 rows of one softmax warp, SWIZZLE_128B
bool make_out_map(CUtensorMap* m, void* out, int num_q_tokens, int hq, int group) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)hq, (cuuint64_t)num_q_tokens};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)hq * D * 2};
  cuuint32_t box[3] = {64, (cuuint32_t)group, (cuuint32_t)(32 / group > 0 ? 32 / group : 1)};
  cuuint32_t estr[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, out, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int G, bool kKeyMask, bool kDual>
bool launch_gk(const Ctx& c, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mo,
              const Params& prm, int sms) {
  const size_t smem = sizeof(Smem);
  static bool attr_done[64] = {};   // the attribute is per (function, device): track it per device ordinal
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_done[dev]) {
    if (cudaFuncSetAttribute(prefill_sm100_kernel<G, kKeyMask, kDual>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
      note_error("prefill_sm100: cudaFuncSetAttribute(MaxDynamicSharedMemorySize) failed");
      return false;
    }
    if (dev >= 0 && dev < 64) attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(sms); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = smem; cfg.stream = c.stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // overlap with the tail of plan_kernel (griddepcontrol)
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, prefill_sm100_kernel<G, kKeyMask, kDual>, mq, mk, mv, mo, prm) != cudaSuccess) {
    note_error("prefill_sm100: cudaLaunchKernelEx failed");
    return false;
  }
  note_launch();
  return true;
}

template <int G>
bool launch_g(const Ctx& c, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mo,
              const Params& prm, int sms) {
  if (c.flags & MINIPIC_KEY_MASK) return launch_gk<G, true, true>(c, mq, mk, mv, mo, prm, sms);
  return prm.dual_ok ? launch_gk<G, false, true>(c, mq, mk, mv, mo, prm, sms) : launch_gk<G, false, false>(c, mq, mk, mv, mo, prm, sms);
}

}  // namespace

// halves = 2: K (both halves of head_dim, 4 KB per block); halves = 1: V (the CTA's half, chosen by the box coordinate, 2 KB)
bool make_cache_tensor_map(CUtensorMap* m, const void* cache, int num_blocks, int hkv, int halves) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[4] = {64, 8, 2, (cuuint64_t)num_blocks * hkv * 2};
  cuuint64_t strides[3] = {(cuuint64_t)D * 2, 128, (cuuint64_t)kGroupBytes};
  cuuint32_t box[4] = {64, 8, (cuuint32_t)halves, 2};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(cache), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
#ifdef MINIPIC_PLAN_TIMES
extern "C" int minipic_debug_plan_times(long long* host) { cudaDeviceSynchronize(); return (int)cudaMemcpyFromSymbol(host, g_plan_t, sizeof(long long) * 16); }
#endif
#ifdef MINIPIC_TRACE
extern "C" int minipic_debug_trace_copy(long long* host, int* counts) {
  cudaDeviceSynchronize();
  if (cudaMemcpyFromSymbol(host, g_trace, sizeof(long long) * kTraceRoles * kTraceLen * 2) != cudaSuccess) return -1;
  if (cudaMemcpyFromSymbol(counts, g_trace_n, sizeof(int) * kTraceRoles) != cudaSuccess) return -1;
  int zero[kTraceRoles] = {0};
  cudaMemcpyToSymbol(g_trace_n, zero, sizeof(zero));
  return kTraceLen;
}
#endif

int prefill_sm100_error_word(const void* workspace, cudaStream_t st, int* word) {
  *word = 0;
  int pair[2] = {0, 0};   // {err, magic}
  static_assert(offsetof(PlanHeader, magic) == offsetof(PlanHeader, err) + sizeof(int), "err and magic must be adjacent");
  cudaError_t e = cudaMemcpyAsync(pair, (const char*)workspace + offsetof(PlanHeader, err), sizeof(pair), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e == cudaSuccess && pair[1] == kPlanMagic) *word = pair[0];   // any other tag: not a header of this kernel -> healthy
  return (int)e;
}

bool prefill_sm100_supported(const Ctx& c) {
  return c.dtype == MINIPIC_BF16 && c.d == 128 && (c.group == 1 || c.group == 2 || c.group == 4 || c.group == 8);
}

// Workspace: [PlanHeader][sorted descriptors][unsorted descriptors][split groups][partial lse][partial O].  The part up to the
// split groups is REQUIRED; the partial slots are optional: KV-range splits are made only if they fit in what the caller gave.
struct WsLayout { size_t sorted, tmp, groups, part, min_bytes; int sorted_cap; };
static size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }
static WsLayout ws_layout(int num_q_tokens) {
  WsLayout l;
  l.sorted_cap = 2 * (num_q_tokens + 1);   // room for the chunks of split items
  l.sorted = sizeof(PlanHeader);
  l.tmp = up256(l.sorted + (size_t)l.sorted_cap * sizeof(TileDesc));
  l.groups = up256(l.tmp + (size_t)(num_q_tokens + 1) * sizeof(TileDesc));
  l.part = up256(l.groups + (size_t)(num_q_tokens + 1) * sizeof(SplitGroup));
  l.min_bytes = l.part;
  return l;
}
static size_t slot_bytes(const Ctx& c) { return (size_t)c.hq * (D + 1) * sizeof(float); }   // one partial token slot: O row + lse per head
// small grids only (fewer than ~32 full items per CTA pair): there a few long items set the time, and dual items / KV-range
// splits pay; on large grids they would only add code to the hot loops.  Decided from host scalars.
static bool small_grid(const Ctx& c, int num_q_tokens, int num_reqs) {
  const int tok2 = 4 * BM / c.group;   // query tokens per work item: two 128-row tiles in each CTA of a pair
  const long long items_upper = ((long long)num_q_tokens / tok2 + num_reqs) * c.hkv;
  return items_upper < 32LL * (current_sm_count() / 2);
}
constexpr int kPartSlotsMax = 4096;                 // partial token slots asked for ...
constexpr size_t kPartBytesMax = (size_t)64 << 20;   // ... within this many bytes

size_t prefill_sm100_workspace_min_bytes(const Ctx&, int, int num_q_tokens) { return ws_layout(num_q_tokens).min_bytes + 512; }

size_t prefill_sm100_workspace_bytes(const Ctx& c, int, int num_q_tokens) {
  size_t b = ws_layout(num_q_tokens).min_bytes + 512;
  if (small_grid(c, num_q_tokens, 0)) {   // a superset of the launches that may split (num_reqs only makes the grid larger)
    const size_t slots = std::min<size_t>(kPartSlotsMax, kPartBytesMax / slot_bytes(c));
    b += slots * slot_bytes(c) + 256;
  }
  return b;
}

bool launch_prefill_sm100(const Ctx& c, const PrefillArgs& a) {
  CUtensorMap mq, mk, mv, mo;
  if (!make_cache_tensor_map(&mk, a.k_cache, c.num_blocks, c.hkv, 2) || !make_cache_tensor_map(&mv, a.v_cache, c.num_blocks, c.hkv, 1) ||
      !make_q_map(&mq, a.q, a.num_q_tokens, c.hq, c.group) || !make_out_map(&mo, a.out, a.num_q_tokens, c.hq, c.group)) {
    note_error("prefill_sm100: cuTensorMapEncodeTiled failed (driver entry point missing or bad tensor geometry)");
    return false;
  }
  const WsLayout wl = ws_layout(a.num_q_tokens);
  char* ws = (char*)a.workspace;
  PlanHeader* hdr = (PlanHeader*)ws;
  TileDesc* sorted = (TileDesc*)(ws + wl.sorted);
  TileDesc* tmp = (TileDesc*)(ws + wl.tmp);
  SplitGroup* groups = (SplitGroup*)(ws + wl.groups);
  const int tok2 = 4 * BM / c.group;
  // dual items (short Q over a long KV range split between the two tile slots, struct Item) and KV-range splits (SplitGroup):
  // small grids, or the key-mask variant (a cold path anyway)
  const int dual_ok = (c.flags & MINIPIC_KEY_MASK) || small_grid(c, a.num_q_tokens, a.num_reqs) ? 1 : 0;
  const int pairs = current_sm_count() / 2;
  int part_cap = 0;
  if (dual_ok && a.workspace_bytes > wl.part + 256)
    part_cap = (int)std::min<size_t>(kPartSlotsMax, (a.workspace_bytes - wl.part - 256) / slot_bytes(c));
  float* part_lse = (float*)(ws + wl.part);
  float* part_o = (float*)(ws + up256(wl.part + (size_t)part_cap * c.hq * sizeof(float)));
  const bool plan_single = a.num_q_tokens <= kPlanSingleMaxTok;
  if (!plan_single && cudaMemsetAsync(hdr, 0, sizeof(PlanHeader), c.stream) != cudaSuccess) return false;
  if (a.num_q_tokens > 0) {
    PlanArgs pa;
    pa.tok = tok2; pa.dual_ok = dual_ok; pa.split_pairs = part_cap > 0 ? pairs : 0; pa.hkv = c.hkv; pa.part_cap = part_cap;
    pa.sorted_cap = wl.sorted_cap; pa.hdr = hdr; pa.tmp = tmp; pa.sorted = sorted; pa.groups = groups;
    if (plan_single) plan_kernel<kPlanSingleThreads, true><<<1, kPlanSingleThreads, 0, c.stream>>>(a, pa);
    else plan_kernel<kPlanThreads, false><<<(a.num_q_tokens + kPlanThreads - 1) / kPlanThreads, kPlanThreads, 0, c.stream>>>(a, pa);
    note_launch(1);
  }
  Params prm;
  prm.a = a; prm.hq = c.hq; prm.hkv = c.hkv; prm.scale_log2 = c.scale_log2; prm.flags = c.flags;
  prm.hdr = hdr; prm.tiles = sorted;
  prm.oob_grp = c.num_blocks * c.hkv * 2;
  prm.dual_ok = dual_ok;
  prm.part_o = part_o; prm.part_lse = part_lse;
  for (int i = 0; i < 64; ++i) {
    prm.phase_inc[i] = c.rope.phase_inc[i];
    const double c1 = c.rope_step_cos[i], s1 = c.rope_step_sin[i];
    const double c2 = c1 * c1 - s1 * s1, s2 = 2.0 * s1 * c1;
    prm.step1[i] = make_float2((float)c1, (float)s1);
    prm.step4[i] = make_float2((float)(c2 * c2 - s2 * s2), (float)(2.0 * s2 * c2));
  }
  const int sms = current_sm_count() & ~1;   // CTA pairs (clusters of 2)
  bool ok = false;
  switch (c.group) {
    case 1: ok = launch_g<1>(c, mq, mk, mv, mo, prm, sms); break;
    case 2: ok = launch_g<2>(c, mq, mk, mv, mo, prm, sms); break;
    case 4: ok = launch_g<4>(c, mq, mk, mv, mo, prm, sms); break;
    case 8: ok = launch_g<8>(c, mq, mk, mv, mo, prm, sms); break;
  }
  if (ok && part_cap > 0) {   // the plan may have split items: combine their partial rows (no group: the kernel returns at once)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(sms); cfg.blockDim = dim3(256); cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // its blocks take the SMs the attention grid's tail frees
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, split_merge_kernel, (const PlanHeader*)hdr, (const SplitGroup*)groups, (const float*)part_o,
                           (const float*)part_lse, c.hq, (__nv_bfloat16*)a.out, a.lse) != cudaSuccess) {
      note_error("prefill_sm100: cudaLaunchKernelEx(split_merge) failed");
      return false;
    }
    note_launch(1);
  }
  return ok;
}

}  // namespace minipic
