// attn_tc2.cu — A3 on a 2-CTA cluster: one 128-row query tile per SM, K/V tiles shared by TMA multicast.
//
// Same contract as attn_tc.cu (include/slack.h): every planned item (stream, head,
// <= 256 query rows, range of 128-key tiles) is computed as S = Q K^T -> online softmax -> P -> O += P V on tcgen05 /
// TMEM.  What differs is how the item's two 128-row query tiles are laid onto the machine:
//
//   * attn_tc.cu keeps both tiles in ONE CTA (TMEM: S0 S1 O0 O1 = 512 columns).  P_j has to overwrite S_j, so each
//     tile runs the serial chain softmax -> P V -> Q K^T -> softmax, and the two tiles' softmax warps share the SM's four
//     sub-partitions: the step time is two softmax legs, the tensor pipe idles a third of the time.
//   * here a CLUSTER of two CTAs (two SMs) takes the item, CTA rank r owning query tile r.  One tile per SM leaves TMEM
//     room for a DOUBLE-BUFFERED S (Sa Sb O = 384 columns): Q K_{j+1}^T is issued before P_j V_j, so the tensor pipe always
//     has the next S in flight while the softmax warps work, and the softmax of a tile has the SM to itself (eight warps:
//     two threads per row, 64 key columns each).  K/V tiles are still fetched from L2 once per 256 query rows: each CTA
//     loads HALF of every tile (64 keys) and the TMA multicasts it into both CTAs' shared memory.
//
// STATUS: experimental, selected only through slack_debug_set key 2 for plans made with sm_count <= SMs / 2, dense calls.
// It passes the same parity tests as attn_tc.cu (tests/test_gpu_cluster_kernel.py) but is 6 % SLOWER in SM cycles on
// BASELINE.json configs[4] (5.37 M vs 5.05 M cycles per launch, tensor pipe 60 % vs 62 % of elapsed): with the tensor
// pipe decoupled the step is bound by the softmax alone, and one tile's softmax on eight warps takes ~1750 cycles per
// 128-key step, no less than the ~1640 the two-tile kernel needs per tile-step; the SM's softmax instruction throughput,
// not the pipeline shape, is the limit.  Two variants measured on top of it did worse: two fully
// independent column streams with their own O accumulators and no per-step exchange (-12 %), and prefetching S of the
// next step into registers (S_{j+1} completes only ~1000 cycles into step j: -25 %).  The number of threads per query row
// was also varied on this pipeline, where the softmax never waits: 1 thread per row (4 softmax warps, 128 columns each)
// 6.08 M cycles, 2 per row (this file) 5.37 M, 4 per row (16 warps, 32 columns each, 128-thread barrier) 5.7 M.  One warp
// alone on a sub-partition needs ~1980 cycles per 128 x 128 tile step whether or not anything else runs beside it (it is
// latency-bound: a third of its time is fixed-latency dependency stalls), a sub-partition overlaps two such warps almost
// perfectly, and that is what the two-tile kernel already does.  Finally, a what-if build of this file WITHOUT the exponentials
// still needs 5.31 M cycles: the bound here is not the softmax arithmetic but (most likely) the shared-memory port: every
// SM ingests the whole K/V tile (64 KB per step) and the SS-mode MMAs read 98 KB of operands per step, 162 KB per 1024
// MMA cycles at 128 B/clk.  The remedy is cta_group::2 (each CTA stores and feeds half of every K/V tile).
//
// CTA = 384 threads: warp 0 TMA producer, warp 1 MMA issuer, warps 2-3 idle, warps 4-7 softmax of key columns 0..63,
// warps 8-11 of columns 64..127 (thread = query row = TMEM lane).  Both CTAs of a cluster walk the same planned queue
// (the plan is made for sm_count / 2 queues).  An item with a single query tile (<= 128 rows) leaves rank 1 computing
// rows that are never stored (it must keep loading and releasing its halves of the K/V tiles anyway).
//
// Ring protocol per K/V stage (32 KB, both CTAs use the same stage index for the same tile):
//   KV_EMPTY[s] (count 2): one arrival from EACH CTA's issuer (tcgen05.commit multicast to both CTAs) -> both producers
//                          may overwrite stage s in both CTAs
//   KV_FULL[s]  (count 1 + 32 KB): the local producer arms it; its own half and the peer's half complete the bytes
// Tiles are loaded in the order they are consumed: K_0, K_1, V_0, K_2, V_1, K_3, ... (Q K_{j+2}^T follows P_j V_j).
#include <cuda_bf16.h>

#include "kernels.h"
#include "ptx_sm100.cuh"

namespace slack {
using namespace ptx;

namespace {

constexpr int kStages = 5;
constexpr uint32_t kTileBytes = 32768;
constexpr uint32_t kHalfBytes = 16384;
constexpr int kThreads = 384;

constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffKV = kTileBytes;
constexpr uint32_t kOffBar = kOffKV + kStages * kTileBytes;

enum : int {
  BAR_Q_FULL = 0,
  BAR_Q_EMPTY = 1,
  BAR_KV_FULL = 2,
  BAR_KV_EMPTY = BAR_KV_FULL + kStages,
  BAR_S_FULL = BAR_KV_EMPTY + kStages, // [buffer 2]
  BAR_P_LO = BAR_S_FULL + 2,           // [2] P of keys 0..63 written AND the other half done touching O
  BAR_P_READY = BAR_P_LO + 2,          // [2] P of keys 64..127 written
  BAR_PV_DONE = BAR_P_READY + 2,       // one completion per P V (the rare O rescale waits on it)
  BAR_O_FINAL = BAR_PV_DONE + 1,
  BAR_O_FREE = BAR_O_FINAL + 1,
  NUM_BARS = BAR_O_FREE + 1
};
constexpr uint32_t kOffTmemPtr = kOffBar + NUM_BARS * 8;
constexpr uint32_t kOffXch = (kOffTmemPtr + 16 + 15) & ~15u; // row-max exchange [parity 2][half 2][128 rows] fp32
constexpr uint32_t kOffXchL = kOffXch + 2048;                 // row-sum exchange [half 2][128 rows] fp32
constexpr uint32_t kSmemUsed = kOffXchL + 1024;
constexpr uint32_t kSmemBytes = kSmemUsed + 1024; // slack for manual 1024-byte alignment

constexpr uint32_t kIdescQK = make_idesc_bf16(128, 128, 0, 0);
constexpr uint32_t kIdescPV = make_idesc_bf16(128, 128, 0, 1);

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr int kEmuOf8 = 2;
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

// ---- cluster-scope PTX used only here
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// 2-D tiled load delivered to the same shared-memory offset of every CTA in `mask`; completes bytes on the mbarrier at
// the same offset in each of them
__device__ __forceinline__ void tma_load_2d_mc(uint32_t smem_dst, const CUtensorMap *m, uint32_t bar, int32_t c0, int32_t c1,
                                               uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4}], [%2], %5;"
      ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(c0), "r"(c1), "h"(mask)
      : "memory");
}
// arrives (count 1) on the mbarrier at this offset in every CTA of `mask` once all tcgen05 ops issued before have completed
__device__ __forceinline__ void mma_commit_mc(uint32_t bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
               "h"(mask)
               : "memory");
}

} // namespace

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
attn_tc2_kernel(const TcParams p, const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                const __grid_constant__ CUtensorMap tm_v) {
  extern __shared__ uint8_t smem_raw[];
  // both CTAs of the cluster must use the SAME offsets (multicast writes to the same offset in the peer)
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base + kOffQ;
  const uint32_t sKV = smem_base + kOffKV;
  const uint32_t bars = smem_base + kOffBar;
  const uint32_t tmem_ptr_smem = smem_base + kOffTmemPtr;
  auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const int rank = (int)cluster_ctarank();       // query tile of every item this CTA owns
  const int queue = blockIdx.x >> 1;              // the cluster's planned queue
  const int item_begin = p.cta_begin[queue];
  const int item_end = p.cta_begin[queue + 1];
  unsigned long long *dbg = p.dbg_flag;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tm_q);
    prefetch_tensormap(&tm_k);
    prefetch_tensormap(&tm_v);
    mbar_init(bar(BAR_Q_FULL), 1);
    mbar_init(bar(BAR_Q_EMPTY), 1);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar(BAR_KV_FULL + s), 1);
      mbar_init(bar(BAR_KV_EMPTY + s), 2); // one release from each CTA of the cluster
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar(BAR_S_FULL + b), 1);
      mbar_init(bar(BAR_P_LO + b), 8);
      mbar_init(bar(BAR_P_READY + b), 4);
    }
    mbar_init(bar(BAR_PV_DONE), 1);
    mbar_init(bar(BAR_O_FINAL), 1);
    mbar_init(bar(BAR_O_FREE), 8);
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_ptr_smem, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all(); // the peer's barriers are initialised before anything is multicast to them
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));

  const int H = p.n_heads;
  const int P = 1 << p.page_log2;

  if (warp < 4) {
    setmaxnreg_dec<80>();
    if (warp == 0) {
      // ============================== TMA producer ==============================
      uint32_t ring = 0;
      int n_item = 0;
      for (int k = item_begin; k < item_end; ++k, ++n_item) {
        const DevItem it = p.items[k];
        const ItemView v = uniform_view_of(it);
        const int head = uni(it.head), q_row0 = uni(it.q_row0), pt_off = uni(it.pt_off);
        mbar_wait(bar(BAR_Q_EMPTY), (uint32_t)((n_item & 1) ^ 1), 100, dbg);
        if (elect_one()) {
          mbar_expect_tx(bar(BAR_Q_FULL), kTileBytes);
          for (int c = 0; c < 2; ++c)
            tma_load_2d(sQ + c * kHalfBytes, &tm_q, bar(BAR_Q_FULL), head * 128 + c * 64, q_row0 + rank * kTileM);
        }
        __syncwarp();
        // this CTA's half (64 keys) of tile `j` of K (kv = 0) or V (kv = 1), multicast to both CTAs
        auto load_half = [&](int j, int kv) {
          const int tile = v.tile_of(j);
          const int page = uni(__ldg(p.page_tables + pt_off + ((tile * kTileN) >> p.page_log2)));
          const int row = (page * H + head) * P + ((tile * kTileN) & (P - 1)) + rank * 64;
          const uint32_t stage = ring % kStages;
          const uint32_t ph = (ring / kStages) & 1u;
          mbar_wait(bar(BAR_KV_EMPTY + stage), ph ^ 1u, 110 + stage, dbg);
          if (elect_one()) {
            mbar_expect_tx(bar(BAR_KV_FULL + stage), kTileBytes); // my half and the peer's half
            const CUtensorMap *tm = kv == 0 ? &tm_k : &tm_v;
            const uint32_t dst = sKV + stage * kTileBytes + (uint32_t)rank * 8192u;
            tma_load_2d_mc(dst, tm, bar(BAR_KV_FULL + stage), 0, row, (uint16_t)3);
            tma_load_2d_mc(dst + kHalfBytes, tm, bar(BAR_KV_FULL + stage), 64, row, (uint16_t)3);
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
      // ============================== MMA issuer ==============================
      uint32_t ring = 0; // consumption index, same order as the producer's loads
      uint32_t cs = 0;   // Q K^T / P V steps issued so far (S buffer = step & 1, barrier parity = (step >> 1) & 1)
      uint32_t itn = 0;
      int n_item = 0;
      auto issue_qk = [&](uint32_t stage, uint32_t b) {
        const uint32_t a_base = sQ;
        const uint32_t b_base = sKV + stage * kTileBytes;
        const uint32_t d = tmem_base + b * 128u;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const uint32_t off = (uint32_t)(k >> 2) * kHalfBytes + (uint32_t)(k & 3) * 32u;
          mma_ss(d, make_smem_desc_sw128(a_base + off, 16, 1024), make_smem_desc_sw128(b_base + off, 16, 1024), kIdescQK,
                 k > 0 ? 1u : 0u);
        }
      };
      auto issue_pv = [&](uint32_t stage, int half, uint32_t b, bool acc) {
        const uint32_t b_base = sKV + stage * kTileBytes;
        const uint32_t d = tmem_base + 256u;
        const uint32_t a = tmem_base + b * 128u + (uint32_t)half * 64u; // P of half h: first 32 columns of its S half
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          const int k = half * 4 + kk;
          mma_ts(d, a + (uint32_t)(kk * 8), make_smem_desc_sw128(b_base + (uint32_t)k * 2048u, kHalfBytes, 1024), kIdescPV,
                 (acc || k > 0) ? 1u : 0u);
        }
      };
      for (int k = item_begin; k < item_end; ++k, ++n_item) {
        const DevItem it = p.items[k];
        const ItemView v = uniform_view_of(it);
        mbar_wait(bar(BAR_Q_FULL), (uint32_t)(n_item & 1), 200, dbg);
        // Q K_j^T into buffer (cs0 + j) & 1, consuming the next ring entry (a K tile)
        const uint32_t cs0 = cs;
        auto do_qk = [&](int j) {
          const uint32_t stage = ring % kStages, ph = (ring / kStages) & 1u;
          const uint32_t b = (cs0 + (uint32_t)j) & 1u;
          mbar_wait(bar(BAR_KV_FULL + stage), ph, 210 + stage, dbg);
          tc_fence_after();
          if (elect_one()) {
            issue_qk(stage, b);
            mma_commit(bar(BAR_S_FULL + (int)b));
            mma_commit_mc(bar(BAR_KV_EMPTY + stage), (uint16_t)3);
            if (j + 1 == v.T) mma_commit(bar(BAR_Q_EMPTY));
          }
          __syncwarp();
          ++ring;
        };
        do_qk(0);
        if (v.T > 1) do_qk(1);
        for (int j = 0; j < v.T; ++j) {
          const uint32_t stage_v = ring % kStages, ph_v = (ring / kStages) & 1u;
          const uint32_t step = cs0 + (uint32_t)j;
          const uint32_t b = step & 1u, par = (step >> 1) & 1u;
          mbar_wait(bar(BAR_KV_FULL + stage_v), ph_v, 220 + stage_v, dbg);
          {
            // masked key rows of V must be zero: P is 0 there, but 0 * NaN/Inf garbage would poison O
            const int tile = v.tile_of(j);
            const int c_lo = max(0, v.lo_of(j) - tile * kTileN);
            const int c_hi = min(kTileN, v.hi_of(j) - tile * kTileN);
            if (c_lo > 0 || c_hi < kTileN) {
              const int n_zero = c_lo + (kTileN - c_hi);
              const uint32_t base = sKV + stage_v * kTileBytes;
              for (int idx = lane; idx < n_zero * 16; idx += 32) {
                int r = idx >> 4;
                r = r < c_lo ? r : c_hi + (r - c_lo);
                const int w = idx & 15;
                const uint32_t addr = base + (uint32_t)(w >> 3) * kHalfBytes + (uint32_t)r * 128u + (uint32_t)(w & 7) * 16u;
                asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
              }
              fence_proxy_async_smem();
              __syncwarp();
            }
          }
          mbar_wait(bar(BAR_P_LO + (int)b), par, 260, dbg);
          if (j == 0) mbar_wait(bar(BAR_O_FREE), (itn & 1u) ^ 1u, 240, dbg);
          tc_fence_after();
          if (elect_one()) issue_pv(stage_v, 0, b, j > 0);
          __syncwarp();
          mbar_wait(bar(BAR_P_READY + (int)b), par, 230, dbg);
          tc_fence_after();
          if (elect_one()) {
            issue_pv(stage_v, 1, b, true);
            mma_commit(bar(BAR_PV_DONE));
            mma_commit_mc(bar(BAR_KV_EMPTY + stage_v), (uint16_t)3);
            if (j + 1 == v.T) mma_commit(bar(BAR_O_FINAL));
          }
          __syncwarp();
          ++ring;
          if (j + 2 < v.T) do_qk(j + 2); // into buffer b, free again once P_j V_j (just issued) has read P_j
        }
        cs = cs0 + (uint32_t)v.T;
        ++itn;
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
    const uint32_t xch = smem_base + kOffXch + (uint32_t)(row * 4);   // + parity * 1024 + half * 512
    const uint32_t xch_l = smem_base + kOffXchL + (uint32_t)(row * 4); // + half * 512
    const int pair_bar = 1 + w4; // named barrier of the two warps that own these 32 rows
    const float sl2 = p.scale * kLog2e;
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
        mbar_wait(bar(BAR_S_FULL + (int)b), par, 300, dbg);
        tc_fence_after();
        float s[64];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t r[32];
          tmem_ld32(tS + (uint32_t)(c * 32), r);
#pragma unroll
          for (int e = 0; e < 32; ++e) s[c * 32 + e] = __uint_as_float(r[e]);
        }
        tmem_wait_ld();
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
          mx = fmaxf(mine, exchange_max(mine));
        }
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
          if (lane == 0) mbar_arrive(bar(BAR_P_LO + (int)b));
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
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar((h == 0 ? BAR_P_LO : BAR_P_READY) + (int)b));
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
      // the pair's second row-sum exchange of the NEXT item must not overwrite xch_l before both have read it: the next
      // write happens after the next item's steps, each of which passes the pair barrier -> ordered
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(BAR_O_FREE));
      ++itn;
    }
  }

  // ---------------- teardown ----------------
  tc_fence_before();
  __syncthreads();
  cluster_sync_all(); // no CTA leaves while the peer may still multicast into it or arrive on its barriers
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

size_t attn_tc2_smem_bytes() { return kSmemBytes; }

cudaError_t attn_tc2_configure() {
  return cudaFuncSetAttribute(attn_tc2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
}

// tm_k / tm_v must be encoded with a 64-row box (each CTA loads half a key tile)
cudaError_t launch_attn_tc2(const TcParams &p, const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                            int n_clusters, cudaStream_t st, int *n_launched) {
  attn_tc2_kernel<<<2 * n_clusters, kThreads, kSmemBytes, st>>>(p, tm_q, tm_k, tm_v);
  if (n_launched) *n_launched += 1;
  return cudaGetLastError();
}

} // namespace slack
