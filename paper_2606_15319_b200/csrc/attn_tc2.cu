// attn_tc2.cu — A3 on CTA PAIRS: the same computation as attn_tc.cu (PAPER.md P:21, P:84 chunk attends to cached earlier
// chunks; P:86 rolling window / sink; P:251 paged pool; include/slack.h), with tcgen05.mma.cta_group::2.
//
// Why pairs.  attn_tc.cu keeps an item's two 128-row query tiles in ONE CTA (TMEM: S0 S1 O0 O1 = 512 columns).  P_j has to
// overwrite S_j, so each tile runs the serial chain softmax -> P V -> Q K^T -> softmax and the tensor pipe idles a third
// of the time; and every SM ingests every K/V tile whole and feeds both MMA operands from its own shared memory, which
// puts the 128 B/clk shared-memory port at the same cycle count as the tensor pipe.  Here a cluster of two
// CTAs (two SMs of one TPC) walks each item together, CTA rank r owning query rows [128 r, 128 r + 128):
//   * one tile per SM leaves TMEM room for a DOUBLE-BUFFERED S (Sa Sb O = 384 columns): Q K_{j+1}^T is in flight while the
//     softmax of step j runs, so the tensor pipe never waits for a softmax leg and the softmax has the SM to itself
//     (eight warps: two threads per query row, 64 key columns each);
//   * one `tcgen05.mma.cta_group::2` of M = 256 covers both CTAs' tiles and SPLITS the B operand between them (Q K^T: each
//     CTA holds 64 of the tile's 128 keys; P V: each holds 64 of V's 128 columns), so every SM stores and reads HALF of
//     every K/V tile: 96 KB of shared-memory traffic per 1024 MMA cycles instead of 162 KB, half the L2 -> SM bytes.
//
// Per CTA (384 threads):
//   warp 0        TMA producer: this CTA's Q tile once per item; per key step its K half (keys 64 r .. 64 r + 63 of the
//                 tile) and its V half (columns 64 r .. 64 r + 63 of all 128 keys) through a ring of 16 KB slots, in the
//                 order they are consumed: K_0, K_1, V_0, K_2, V_1, K_3, ...
//   warp 1        rank 0: MMA issuer for BOTH CTAs (one lane issues tcgen05.mma.cta_group::2); rank 1: relay - tells the
//                 issuer when this CTA's slots have landed.  Both zero the masked key rows of their own V half.
//   warps 4-7     softmax of key columns 0..63 of this CTA's 128 rows (thread = query row = TMEM lane), O columns 0..63
//   warps 8-11    the same for key columns 64..127 / O columns 64..127
// TMEM (512 columns in each CTA, allocated with cta_group::2): Sa [0,128) Sb [128,256) O [256,384); the bf16 P of column
// half h is written over the first 32 columns of that half of S.
//
// Barriers.  Local (same offset in both CTAs): Q_FULL, KV_FULL[s] (TMA transaction bytes of the CTA's own loads);
// Q_EMPTY, KV_EMPTY[s], S_FULL[b], PV_DONE, O_FINAL (one tcgen05.commit of the issuer, multicast to both CTAs).  In the
// issuer's CTA only: Q_PEER, KV_PEER[s] (one remote arrival of the rank-1 relay), P_LO[b] (16 arrivals: every softmax
// warp of both CTAs: "P of keys 0..63 is written and nobody touches O any more"), P_READY[b] (8: P of keys 64..127),
// O_FREE (16).
//
// Work comes from a PAIR plan (plan.cpp, kernel kind 2): sm_count / 2 queues of ordinary items (<= 256 rows); the pair
// of CTAs 2q, 2q+1 walks queue q.  An item with <= 128 rows leaves rank 1 computing rows that are never stored.
#include <cuda_bf16.h>

#include "kernels.h"
#include "ptx_sm100.cuh"

namespace slack {
using namespace ptx;

namespace {

constexpr int kSlots = 11;               // ring of 16 KB slots (K halves and V halves in consumption order)
constexpr uint32_t kSlotBytes = 16384;
constexpr uint32_t kQTileBytes = 32768;  // 128 rows x 128 d bf16: two 16 KB halves (d 0..63, d 64..127)
constexpr uint32_t kQHalfBytes = 16384;
constexpr uint32_t kKHalfBytes = 8192;   // K slot: [64 keys][d 0..63] then [64 keys][d 64..127], 128-byte rows
constexpr int kThreads = 384;

constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffKV = kQTileBytes;
constexpr uint32_t kOffBar = kOffKV + kSlots * kSlotBytes;

enum : int {
  BAR_Q_FULL = 0,
  BAR_Q_PEER = 1,
  BAR_Q_EMPTY = 2,
  BAR_KV_FULL = 3,
  BAR_KV_PEER = BAR_KV_FULL + kSlots,
  BAR_KV_EMPTY = BAR_KV_PEER + kSlots,
  BAR_S_FULL = BAR_KV_EMPTY + kSlots, // [buffer 2]
  BAR_P_LO = BAR_S_FULL + 2,          // [2] P of keys 0..63 written AND nobody touches O any more in this step
  BAR_P_READY = BAR_P_LO + 2,         // [2] P of keys 64..127 written
  BAR_PV_DONE = BAR_P_READY + 2,      // one completion per P V (the rare O rescale waits on it)
  BAR_O_FINAL = BAR_PV_DONE + 1,
  BAR_O_FREE = BAR_O_FINAL + 1,
  NUM_BARS = BAR_O_FREE + 1
};
constexpr uint32_t kOffTmemPtr = kOffBar + NUM_BARS * 8;
constexpr uint32_t kOffXch = (kOffTmemPtr + 16 + 15) & ~15u; // row-max exchange [parity 2][half 2][128 rows] fp32
constexpr uint32_t kOffXchL = kOffXch + 2048;                 // row-sum exchange [half 2][128 rows] fp32
constexpr uint32_t kSmemUsed = kOffXchL + 1024;
constexpr uint32_t kSmemBytes = kSmemUsed + 1024; // slack for manual 1024-byte alignment
static_assert(kSmemBytes <= 232448, "shared memory budget of one CTA per SM");

constexpr uint32_t kIdescQK = make_idesc_bf16(256, 128, 0, 0);
constexpr uint32_t kIdescPV = make_idesc_bf16(256, 128, 0, 1);

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
#ifndef SLACK_EMU_OF_8
#define SLACK_EMU_OF_8 2
#endif
constexpr int kEmuOf8 = SLACK_EMU_OF_8;
constexpr float kRescaleThreshold = 8.0f;

struct ItemView {
  int tb, te, T, ns, st0, s_lo, s_hi, w_lo, w_hi;
  __device__ __forceinline__ int tile_of(int j) const { return j < ns ? st0 + j : tb + (j - ns); }
  __device__ __forceinline__ int lo_of(int j) const { return j < ns ? s_lo : w_lo; }
  __device__ __forceinline__ int hi_of(int j) const { return j < ns ? s_hi : w_hi; }
};
__device__ __forceinline__ ItemView view_of(const DevItem &it) {
  ItemView v;
  v.tb = it.kv_tile_begin;
  v.te = it.kv_tile_end;
  v.ns = it.sink_tiles;
  v.st0 = it.sink_tile0;
  v.s_lo = it.sink_lo;
  v.s_hi = it.sink_hi;
  v.w_lo = it.pos_lo;
  v.w_hi = it.pos_hi;
  v.T = v.ns + v.te - v.tb;
  return v;
}
__device__ __forceinline__ ItemView uniform_view_of(const DevItem &it) {
  ItemView v = view_of(it);
  v.tb = uni(v.tb);
  v.te = uni(v.te);
  v.ns = uni(v.ns);
  v.st0 = uni(v.st0);
  v.s_lo = uni(v.s_lo);
  v.s_hi = uni(v.s_hi);
  v.w_lo = uni(v.w_lo);
  v.w_hi = uni(v.w_hi);
  v.T = uni(v.T);
  return v;
}

// ---- cluster-scope PTX used only here ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
// Arrival on a barrier of another CTA of the cluster.  Deliberately the plain form (release at CTA scope, what CUTLASS'
// ClusterBarrier::arrive emits): `.release.cluster` / `.acquire.cluster` make ptxas bracket every arrive and wait with
// MEMBAR.ALL.GPU + CCTL.IVALL, measured at +50 % cycles per key step.  What the barriers order here needs no such fence:
// TMEM writes are complete at tcgen05.wait::st, shared-memory bytes come from the TMA (transaction barrier) or are
// published with fence.proxy.async + an explicit cluster fence on the rare masked-V path, and each CTA's tensor core
// reads only its own CTA's TMEM and shared memory.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void fence_cluster() { asm volatile("fence.acq_rel.cluster;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc2(uint32_t smem_result, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_result), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish2() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem of both CTAs] (+)= A[smem of each CTA: its 128 rows] * B[smem: each CTA holds half of N]
__device__ __forceinline__ void mma2_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// D[tmem] (+)= A[tmem of each CTA] * B[smem: each CTA holds half of N]
__device__ __forceinline__ void mma2_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// the barrier at offset `bar` in BOTH CTAs of the pair gets one arrival once every tcgen05 operation issued so far is done
__device__ __forceinline__ void mma2_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
               "h"((uint16_t)3)
               : "memory");
}

} // namespace

// SLACK_DIAGNOSTICS builds: clock64() stamps of the first item of CTA 0 / CTA 1 into p.dbg_t (slack_debug_set key 1):
// word ((role * 64 + step) * 8 + slot), role 0 / 1 = first warp of the lower / upper column half of CTA 0, 2 = MMA issuer,
// 3 / 4 = the same softmax warps of CTA 1.  The default build has no trace code.
#ifdef SLACK_DIAGNOSTICS
#define SLACK_TRACE2(role, step, slot)                                                                   \
  if ((role) >= 0 && p.dbg_t != nullptr && queue == 0 && k == item_begin && (step) < 64 && lane == 0)                  \
    p.dbg_t[((role) * 64 + (step)) * 8 + (slot)] = (uint32_t)clock64();
#else
#define SLACK_TRACE2(role, step, slot)
#endif

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
attn_tc2_kernel(const TcParams p, const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                const __grid_constant__ CUtensorMap tm_v) {
  extern __shared__ uint8_t smem_raw[];
  // both CTAs of the pair use the SAME offsets (multicast commits and MMA descriptors name offsets, not CTAs)
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base + kOffQ;
  const uint32_t sKV = smem_base + kOffKV;
  const uint32_t bars = smem_base + kOffBar;
  const uint32_t tmem_ptr_smem = smem_base + kOffTmemPtr;
  auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const int rank = (int)cluster_ctarank(); // this CTA owns query rows [128 rank, 128 rank + 128) of every item
  const int queue = blockIdx.x >> 1;       // the pair's planned queue
  const int item_begin = p.cta_begin[queue];
  const int item_end = p.cta_begin[queue + 1];
  unsigned long long *dbg = p.dbg_flag;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tm_q);
    prefetch_tensormap(&tm_k);
    prefetch_tensormap(&tm_v);
    mbar_init(bar(BAR_Q_FULL), 1);
    mbar_init(bar(BAR_Q_PEER), 1);
    mbar_init(bar(BAR_Q_EMPTY), 1);
    for (int s = 0; s < kSlots; ++s) {
      mbar_init(bar(BAR_KV_FULL + s), 1);
      mbar_init(bar(BAR_KV_PEER + s), 1);
      mbar_init(bar(BAR_KV_EMPTY + s), 1);
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar(BAR_S_FULL + b), 1);
      mbar_init(bar(BAR_P_LO + b), 16);   // all eight softmax warps of both CTAs
      mbar_init(bar(BAR_P_READY + b), 8); // the four upper-half warps of both CTAs
    }
    mbar_init(bar(BAR_PV_DONE), 1);
    mbar_init(bar(BAR_O_FINAL), 1);
    mbar_init(bar(BAR_O_FREE), 16);
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc2(tmem_ptr_smem, 512);
    tmem_relinquish2();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all(); // the peer's barriers are initialised (and its TMEM allocated) before anything reaches them
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  pdl_wait();
  pdl_launch_dependents();

  const int H = p.n_heads;
  const int P = 1 << p.page_log2;

  if (warp < 4) {
    setmaxnreg_dec<80>();
    if (warp == 0) {
      // ============================== TMA producer (both CTAs) ==============================
      uint32_t ring = 0;
      int n_item = 0;
      for (int k = item_begin; k < item_end; ++k, ++n_item) {
        const DevItem it = p.items[k];
        const ItemView v = uniform_view_of(it);
        const int head = uni(it.head), q_row0 = uni(it.q_row0), pt_off = uni(it.pt_off);
        mbar_wait(bar(BAR_Q_EMPTY), (uint32_t)((n_item & 1) ^ 1), 100, dbg);
        if (elect_one()) {
          mbar_expect_tx(bar(BAR_Q_FULL), kQTileBytes);
          for (int c = 0; c < 2; ++c)
            tma_load_2d(sQ + c * kQHalfBytes, &tm_q, bar(BAR_Q_FULL), head * 128 + c * 64, q_row0 + rank * kTileM);
        }
        __syncwarp();
        // this CTA's half of tile `j` of K (kv = 0: 64 of the keys, all of d) or V (kv = 1: all keys, 64 of the columns)
        auto load_half = [&](int j, int kv) {
          const int tile = v.tile_of(j);
          const int page = uni(__ldg(p.page_tables + pt_off + ((tile * kTileN) >> p.page_log2)));
          const int row = (page * H + head) * P + ((tile * kTileN) & (P - 1));
          const uint32_t slot = ring % kSlots;
          const uint32_t ph = (ring / kSlots) & 1u;
          mbar_wait(bar(BAR_KV_EMPTY + slot), ph ^ 1u, 110 + slot, dbg);
          if (elect_one()) {
            mbar_expect_tx(bar(BAR_KV_FULL + slot), kSlotBytes);
            const uint32_t dst = sKV + slot * kSlotBytes;
            if (kv == 0) {
              tma_load_2d(dst, &tm_k, bar(BAR_KV_FULL + slot), 0, row + 64 * rank);
              tma_load_2d(dst + kKHalfBytes, &tm_k, bar(BAR_KV_FULL + slot), 64, row + 64 * rank);
            } else {
              tma_load_2d(dst, &tm_v, bar(BAR_KV_FULL + slot), 64 * rank, row);
            }
          }
          __syncwarp();
          ++ring;
        };
        load_half(0, 0);
        if (v.T > 1) load_half(1, 0);
        for (int j = 0; j < v.T; ++j) {
          load_half(j, 1);
          if (j + 2 < v.T) load_half(j + 2, 0);
        }
      }
    } else if (warp == 1) {
      // masked key rows of this CTA's V half must be zero: P is 0 there, but 0 * NaN/Inf garbage would poison O
      auto zero_masked_v = [&](const ItemView &v, int j, uint32_t slot) {
        const int tile = v.tile_of(j);
        const int c_lo = max(0, v.lo_of(j) - tile * kTileN);
        const int c_hi = min(kTileN, v.hi_of(j) - tile * kTileN);
        if (c_lo > 0 || c_hi < kTileN) {
          const int n_zero = c_lo + (kTileN - c_hi);
          const uint32_t base = sKV + slot * kSlotBytes;
          for (int idx = lane; idx < n_zero * 8; idx += 32) {
            int r = idx >> 3;
            r = r < c_lo ? r : c_hi + (r - c_lo);
            const uint32_t addr = base + (uint32_t)r * 128u + (uint32_t)(idx & 7) * 16u;
            asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
          }
          fence_proxy_async_smem();
          fence_cluster(); // rare path (a ragged first / last key tile): the zeros are visible before the peer is told
          __syncwarp();
        }
      };
      if (rank == 1) {
        // ============================== relay (odd CTA): "my half has landed" ==============================
        const uint32_t q_peer = map_to_cta(bar(BAR_Q_PEER), 0);
        uint32_t ring = 0;
        int n_item = 0;
        for (int k = item_begin; k < item_end; ++k, ++n_item) {
          const DevItem it = p.items[k];
          const ItemView v = uniform_view_of(it);
          mbar_wait(bar(BAR_Q_FULL), (uint32_t)(n_item & 1), 400, dbg);
          if (elect_one()) mbar_arrive_cluster(q_peer);
          __syncwarp();
          auto relay = [&](int j, int kv) {
            const uint32_t slot = ring % kSlots, ph = (ring / kSlots) & 1u;
            mbar_wait(bar(BAR_KV_FULL + slot), ph, 410 + slot, dbg);
            if (kv == 1) zero_masked_v(v, j, slot);
            if (elect_one()) mbar_arrive_cluster(map_to_cta(bar(BAR_KV_PEER + slot), 0));
            __syncwarp();
            ++ring;
          };
          relay(0, 0);
          if (v.T > 1) relay(1, 0);
          for (int j = 0; j < v.T; ++j) {
            relay(j, 1);
            if (j + 2 < v.T) relay(j + 2, 0);
          }
        }
      } else {
        // ============================== MMA issuer (even CTA, for both) ==============================
        uint32_t ring = 0; // consumption index, same order as the producers' loads
        uint32_t cs = 0;   // Q K^T / P V steps issued so far (S buffer = step & 1, barrier parity = (step >> 1) & 1)
        uint32_t itn = 0;
        int n_item = 0;
        auto issue_qk = [&](uint32_t slot, uint32_t b) {
          const uint32_t b_base = sKV + slot * kSlotBytes;
          const uint32_t d = tmem_base + b * 128u;
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const uint32_t a_off = (uint32_t)(k >> 2) * kQHalfBytes + (uint32_t)(k & 3) * 32u;
            const uint32_t b_off = (uint32_t)(k >> 2) * kKHalfBytes + (uint32_t)(k & 3) * 32u;
            mma2_ss(d, make_smem_desc_sw128(sQ + a_off, 16, 1024), make_smem_desc_sw128(b_base + b_off, 16, 1024), kIdescQK,
                    k > 0 ? 1u : 0u);
          }
        };
        // P V over keys [64*half, 64*half + 64) of the tile (4 MMAs of K = 16); B = this CTA's 64 columns of V, MN-major
        auto issue_pv = [&](uint32_t slot, int half, uint32_t b, bool acc) {
          const uint32_t b_base = sKV + slot * kSlotBytes;
          const uint32_t d = tmem_base + 256u;
          const uint32_t a = tmem_base + b * 128u + (uint32_t)half * 64u; // P of half h: first 32 columns of its S half
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            const int k = half * 4 + kk;
            mma2_ts(d, a + (uint32_t)(kk * 8), make_smem_desc_sw128(b_base + (uint32_t)k * 2048u, kSlotBytes, 1024), kIdescPV,
                    (acc || k > 0) ? 1u : 0u);
          }
        };
        for (int k = item_begin; k < item_end; ++k, ++n_item) {
          const DevItem it = p.items[k];
          const ItemView v = uniform_view_of(it);
          mbar_wait(bar(BAR_Q_FULL), (uint32_t)(n_item & 1), 200, dbg);
          mbar_wait(bar(BAR_Q_PEER), (uint32_t)(n_item & 1), 201, dbg);
          // Q K_j^T into buffer (cs0 + j) & 1, consuming the next ring entry (a K slot)
          const uint32_t cs0 = cs;
          auto do_qk = [&](int j) {
            const uint32_t slot = ring % kSlots, ph = (ring / kSlots) & 1u;
            const uint32_t b = (cs0 + (uint32_t)j) & 1u;
            mbar_wait(bar(BAR_KV_FULL + slot), ph, 210 + slot, dbg);
            mbar_wait(bar(BAR_KV_PEER + slot), ph, 430 + slot, dbg);
            tc_fence_after();
            if (elect_one()) {
              issue_qk(slot, b);
              mma2_commit(bar(BAR_S_FULL + (int)b));
              mma2_commit(bar(BAR_KV_EMPTY + slot));
              if (j + 1 == v.T) mma2_commit(bar(BAR_Q_EMPTY));
            }
            __syncwarp();
            ++ring;
          };
          do_qk(0);
          if (v.T > 1) do_qk(1);
          for (int j = 0; j < v.T; ++j) {
            const uint32_t slot_v = ring % kSlots, ph_v = (ring / kSlots) & 1u;
            const uint32_t step = cs0 + (uint32_t)j;
            const uint32_t b = step & 1u, par = (step >> 1) & 1u;
            mbar_wait(bar(BAR_KV_FULL + slot_v), ph_v, 220 + slot_v, dbg);
            zero_masked_v(v, j, slot_v);
            mbar_wait(bar(BAR_KV_PEER + slot_v), ph_v, 440 + slot_v, dbg);
            SLACK_TRACE2(2, j, 0);
            mbar_wait(bar(BAR_P_LO + (int)b), par, 260, dbg);
            SLACK_TRACE2(2, j, 1);
            if (j == 0) mbar_wait(bar(BAR_O_FREE), (itn & 1u) ^ 1u, 240, dbg);
            tc_fence_after();
            if (elect_one()) issue_pv(slot_v, 0, b, j > 0);
            __syncwarp();
            mbar_wait(bar(BAR_P_READY + (int)b), par, 230, dbg);
            SLACK_TRACE2(2, j, 2);
            tc_fence_after();
            if (elect_one()) {
              issue_pv(slot_v, 1, b, true);
              mma2_commit(bar(BAR_PV_DONE));
              mma2_commit(bar(BAR_KV_EMPTY + slot_v));
              if (j + 1 == v.T) mma2_commit(bar(BAR_O_FINAL));
            }
            __syncwarp();
            ++ring;
            SLACK_TRACE2(2, j, 3);
            if (j + 2 < v.T) do_qk(j + 2); // into buffer b, free again once P_j V_j (just issued) has read P_j
          }
          cs = cs0 + (uint32_t)v.T;
          ++itn;
        }
      }
    }
  } else {
    // ============================== softmax + epilogue: 8 warps, two threads per query row ==============================
    setmaxnreg_inc<208>();
    const int h = (warp - 4) >> 2; // column half: keys [64h, 64h + 64) of every tile, columns [64h, 64h + 64) of O
    const int w4 = warp & 3;
    const int row = w4 * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(w4 * 32) << 16;
    const uint32_t tS0 = tmem_base + lane_addr + (uint32_t)(h * 64);
    const uint32_t tO = tmem_base + lane_addr + (uint32_t)(256 + h * 64);
    const uint32_t xch = smem_base + kOffXch + (uint32_t)(row * 4);    // + parity * 1024 + half * 512
    const uint32_t xch_l = smem_base + kOffXchL + (uint32_t)(row * 4); // + half * 512
    const int pair_bar = 1 + w4; // named barrier of the two warps that own these 32 rows
    const float sl2 = p.scale * kLog2e;
    // the issuer's barriers (in the even CTA) as shared::cluster addresses
    const uint32_t b_p_lo = map_to_cta(bar(BAR_P_LO), 0);
    const uint32_t b_p_ready = map_to_cta(bar(BAR_P_READY), 0);
    const uint32_t b_o_free = map_to_cta(bar(BAR_O_FREE), 0);
    uint32_t cnt = 0, itn = 0, xc = 0;
    auto exchange_max = [&](float mine) {
      const uint32_t base = xch + (xc & 1u) * 1024u;
      st_shared_f32(base + (uint32_t)h * 512u, mine);
      named_bar_sync(pair_bar, 64);
      ++xc;
      return ld_shared_f32(base + (uint32_t)(h ^ 1) * 512u);
    };
    for (int k = item_begin; k < item_end; ++k) {
      const DevItem it = p.items[k];
      const ItemView v = view_of(it);
      const int local_row = rank * kTileM + row;
      const bool valid = local_row < it.q_rows;
      float m = -INFINITY, l = 0.f;
      for (int j = 0; j < v.T; ++j) {
        const uint32_t b = cnt & 1u, par = (cnt >> 1) & 1u;
        const uint32_t tS = tS0 + b * 128u;
        [[maybe_unused]] const int trole = (w4 == 0) ? (rank * 3 + h) : -1;
        SLACK_TRACE2(trole, j, 0);
        mbar_wait(bar(BAR_S_FULL + (int)b), par, 300, dbg);
        tc_fence_after();
        SLACK_TRACE2(trole, j, 1);
#if defined(SLACK_WHATIF) && SLACK_WHATIF >= 3
        if (h == 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(b_p_lo + 8u * b);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster((h == 0 ? b_p_lo : b_p_ready) + 8u * b);
        ++cnt;
        continue;
#endif
        float s[64];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t r[32];
          tmem_ld32(tS + (uint32_t)(c * 32), r);
#pragma unroll
          for (int e = 0; e < 32; ++e) s[c * 32 + e] = __uint_as_float(r[e]);
        }
        tmem_wait_ld();
        SLACK_TRACE2(trole, j, 2);
        const int tile = v.tile_of(j);
        const int c_lo = max(0, v.lo_of(j) - tile * kTileN) - h * 64; // visible columns of this half: [c_lo, c_hi)
        const int c_hi = min(kTileN, v.hi_of(j) - tile * kTileN) - h * 64;
        if (c_lo > 0 || c_hi < 64) {
#pragma unroll
          for (int e = 0; e < 64; ++e) s[e] = (e >= c_lo && e < c_hi) ? s[e] : -INFINITY;
        }
        float mx;
        {
          float mxc[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) mxc[c] = max3(s[c * 16], s[c * 16 + 1], s[c * 16 + 2]);
#pragma unroll
          for (int e = 3; e + 1 < 16; e += 2) {
#pragma unroll
            for (int c = 0; c < 4; ++c) mxc[c] = max3(mxc[c], s[c * 16 + e], s[c * 16 + e + 1]);
          }
#pragma unroll
          for (int c = 0; c < 4; ++c) mxc[c] = fmaxf(mxc[c], s[c * 16 + 15]);
          const float mine = fmaxf(max3(mxc[0], mxc[1], mxc[2]), mxc[3]);
#if defined(SLACK_WHATIF) && SLACK_WHATIF >= 2
          mx = s[0];
#else
          mx = fmaxf(mine, exchange_max(mine));
#endif
        }
        SLACK_TRACE2(trole, j, 3);
        if (j == 0) {
          m = mx;
        } else {
          const bool need = (mx - m) * sl2 > kRescaleThreshold;
          if (__any_sync(0xffffffffu, need)) {
            // O must hold every earlier P V; the previous one may still be in flight (Q K_j^T was issued before it)
            mbar_wait(bar(BAR_PV_DONE), (cnt - 1u) & 1u, 320, dbg);
            tc_fence_after();
            const float alpha = need ? ex2((m - mx) * sl2) : 1.0f;
            m = need ? mx : m;
            l *= alpha;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              uint32_t r[32];
              tmem_ld32(tO + (uint32_t)(c * 32), r);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) r[e] = __float_as_uint(__uint_as_float(r[e]) * alpha);
              tmem_st32(tO + (uint32_t)(c * 32), r);
            }
            tmem_wait_st();
          }
        }
        if (h == 1) { // this half will not touch O again in this step
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(b_p_lo + 8u * b);
        }
        const uint64_t sl2_2 = pack2(sl2, sl2);
        const uint64_t negm_2 = pack2(-m * sl2, -m * sl2);
        uint64_t la0 = pack2(0.f, 0.f), la1 = la0, la2 = la0, la3 = la0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int e = 0; e < 16; ++e) {
            const uint64_t x2 = ffma2(pack2(s[c * 32 + 2 * e], s[c * 32 + 2 * e + 1]), sl2_2, negm_2);
            uint64_t p2;
#if defined(SLACK_WHATIF) && SLACK_WHATIF >= 1
            if (true) {
              p2 = x2;
            } else
#endif
            if ((e & 7) < kEmuOf8) {
              p2 = exp2_poly2(x2);
            } else {
              float x0, x1;
              unpack2(x2, x0, x1);
              p2 = pack2(ex2(x0), ex2(x1));
            }
            if ((e & 3) == 0) la0 = fadd2(la0, p2);
            else if ((e & 3) == 1) la1 = fadd2(la1, p2);
            else if ((e & 3) == 2) la2 = fadd2(la2, p2);
            else la3 = fadd2(la3, p2);
            float p0, p1;
            unpack2(p2, p0, p1);
            pk[e] = pack_bf16x2(p0, p1);
          }
          tmem_st16(tS + (uint32_t)(c * 16), pk);
        }
        {
          float a0, a1;
          unpack2(fadd2(fadd2(la0, la1), fadd2(la2, la3)), a0, a1);
          l += a0 + a1;
        }
        SLACK_TRACE2(trole, j, 4);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        SLACK_TRACE2(trole, j, 5);
        if (lane == 0) mbar_arrive_cluster((h == 0 ? b_p_lo : b_p_ready) + 8u * b);
        SLACK_TRACE2(trole, j, 6);
        ++cnt;
      }
      // ---------------- epilogue: O / l ----------------
      st_shared_f32(xch_l + (uint32_t)h * 512u, l);
      named_bar_sync(pair_bar, 64);
      l += ld_shared_f32(xch_l + (uint32_t)(h ^ 1) * 512u);
      mbar_wait(bar(BAR_O_FINAL), itn & 1u, 310, dbg);
      tc_fence_after();
      const float inv_l = 1.0f / l;
      const float lse_val = (m * sl2 + log2f(l)) * kLn2;
      if (it.partial_slot < 0) {
        __nv_bfloat16 *dst =
            reinterpret_cast<__nv_bfloat16 *>(p.out) + ((size_t)(it.q_row0 + local_row) * H + it.head) * 128 + h * 64;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t r[32];
          tmem_ld32(tO + (uint32_t)(c * 32), r);
          tmem_wait_ld();
          if (valid) {
#pragma unroll
            for (int e = 0; e < 32; e += 8) {
              uint4 o;
              o.x = pack_bf16x2(__uint_as_float(r[e + 0]) * inv_l, __uint_as_float(r[e + 1]) * inv_l);
              o.y = pack_bf16x2(__uint_as_float(r[e + 2]) * inv_l, __uint_as_float(r[e + 3]) * inv_l);
              o.z = pack_bf16x2(__uint_as_float(r[e + 4]) * inv_l, __uint_as_float(r[e + 5]) * inv_l);
              o.w = pack_bf16x2(__uint_as_float(r[e + 6]) * inv_l, __uint_as_float(r[e + 7]) * inv_l);
              *reinterpret_cast<uint4 *>(dst + c * 32 + e) = o;
            }
          }
        }
        if (valid && h == 0 && p.lse != nullptr) p.lse[(size_t)it.head * p.total_q + it.q_row0 + local_row] = lse_val;
      } else {
        float *dst = p.ws_o + ((size_t)it.partial_slot * kItemRows + local_row) * 128 + h * 64;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t r[32];
          tmem_ld32(tO + (uint32_t)(c * 32), r);
          tmem_wait_ld();
          if (valid) {
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
              float4 o;
              o.x = __uint_as_float(r[e + 0]) * inv_l;
              o.y = __uint_as_float(r[e + 1]) * inv_l;
              o.z = __uint_as_float(r[e + 2]) * inv_l;
              o.w = __uint_as_float(r[e + 3]) * inv_l;
              *reinterpret_cast<float4 *>(dst + c * 32 + e) = o;
            }
          }
        }
        if (valid && h == 0) p.ws_lse[(size_t)it.partial_slot * kItemRows + local_row] = lse_val;
      }
      // the row-sum exchange of the NEXT item cannot overwrite xch_l before both warps of the pair have read it: the
      // next write happens after the next item's steps, each of which passes the pair barrier
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(b_o_free);
      ++itn;
    }
  }

  // ---------------- teardown ----------------
  tc_fence_before();
  __syncthreads();
  cluster_sync_all(); // no CTA leaves (or frees TMEM) while the peer's MMAs, commits or arrivals may still reach it
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc2(tmem_base, 512);
  }
}

cudaError_t attn_tc2_configure() {
  return cudaFuncSetAttribute(attn_tc2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
}

// n_cta = 2 x the plan's queues; tm_k must be encoded with a 64-row box (each CTA loads half of a key tile's keys)
cudaError_t launch_attn_tc2(const TcParams &p, const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                            int n_cta, cudaStream_t st, int *n_launched) {
  cudaError_t e = launch_pdl(attn_tc2_kernel, dim3(n_cta), dim3(kThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  if (n_launched) *n_launched += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
