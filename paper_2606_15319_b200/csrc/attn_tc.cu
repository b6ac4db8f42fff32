// attn_tc.cu — A3: ragged chunk attention on the 5th-gen tensor cores (tcgen05 + TMEM + TMA), bf16, head_dim 128 (or 64:
// the kD = 64 instantiations, same roles and barriers on half-sized tiles; the text below is written for 128).
//
// What it computes (include/slack.h; PAPER.md P:21, P:84 chunk attends to cached earlier chunks; P:86 rolling window;
// P:251 paged pool): for every planned item (stream, head, <=256 query rows, range of 128-key tiles)
//     S = Q K^T (fp32 in TMEM)  ->  online softmax (one thread per query row)  ->  P (bf16, TMEM)  ->  O += P V (TMEM)
// and, at the item's end, O / l written as bf16 (or as an fp32 partial + lse for split-KV items).
//
// CTA = 384 threads, persistent, one per SM, walking its planned queue:
//   warp 0        TMA producer: Q tiles once per item, then K_j, V_j through a ring of 32 KB stages
//   warp 1        MMA issuer (one lane issues tcgen05.mma); also owns TMEM alloc and zeroes masked V rows
//   warps 2-3     idle (keep warpgroup 0 whole for setmaxnreg)
//   warps 4-7     softmax + epilogue for query tile 0 (rows 0..127 of the item; thread = row = TMEM lane)
//   warps 8-11    same for query tile 1 (rows 128..255)
// The two query tiles ping-pong: while one tile's softmax runs on the ALU/MUFU pipes, the tensor pipe works on the
// other tile's P V and next Q K^T.  TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P_i is
// written over the first 64 columns of S_i (two bf16 per 32-bit column).
//
// Dual items (DevItem::dual; dense bf16 and FP8 instantiations of their own): two single-tile items (<= 128 query rows each: decode-like
// chunks, the 72-row tails of long chunks) of the same number of key steps share the CTA, one per query-tile slot, each
// with its OWN K/V tiles (ring entries K_a V_a K_b V_b per step): the idle slot of a single-tile item is filled, the key
// step costs what a two-tile step costs (3250 cycles) instead of 2 x 2755, and an HBM-bound batch keeps twice the
// bytes in flight per SM.  The other instantiations (block-sparse, head_dim 64) walk the two items one after the other.
//
// Block-sparse variant (kSparse, PAPER.md P:88 knob (2) "skips nonselected attention blocks with
// sparse masks"): an item visits only the key-tile steps listed for it by sparse_steps.cu (the device block mask changes
// per layer / denoising step, the host plan does not); every role walks that list instead of 0..T-1, an item with an
// empty list writes zeros (lse = -inf) and touches no barrier.
//
// FP8 variant (kFp8, PAPER.md P:88 knob (4); rule in include/slack.h slack_dtype / DESIGN.md A19):
// the pool holds e4m3 codes with one scale per (page, head, 128-slot block) = per key tile, Q arrives as e4m3 codes with one
// scale per (row, head) (quant.cu), both MMAs are tcgen05 kind::f8f6f4 (K = 32: 4 instructions per tile instead of 8) and
// P is rounded to e4m3 (4 codes per TMEM column).  With sq, sk_t, sv_t the scales of the row, of K tile t and of V tile t,
//     z = S * (scale log2e sq sk_t) + log2 sv_t,     P = 128 * 2^(z - m)  (m = running max of z, lazily rescaled),
//     O += P V8,   l += (sum_tile P) / (128 sv_t),   out = O / (128 l),   lse = (m + log2 l) ln 2
// i.e. the V scale rides inside P's exponent and the row sum is corrected once per tile: no per-element scale work.
//
// Shared memory layouts (all 128-byte swizzled, as TMA writes them and as the UMMA descriptors expect them):
//   Q tile / K tile: two 16 KB halves (d 0..63, d 64..127), each [128 rows][128 B]  -> K-major operands
//   V tile:          same bytes; read as the MN-major B operand of P V (N = d contiguous, K = keys)
//   FP8: every tile is ONE [128 rows][128 B] block of 16 KB (a row = the 128 codes of one token / query row)
#include <cuda_bf16.h>

#include "kernels.h"
#include "ptx_sm100.cuh"

namespace slack {
using namespace ptx;

namespace {

constexpr int kStages = 5;
constexpr uint32_t kTileBytes = 32768;
constexpr uint32_t kHalfBytes = 16384;
constexpr int kTcThreads = 384;

constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffKV = 2 * kTileBytes;
constexpr uint32_t kOffBar = kOffKV + kStages * kTileBytes;

enum : int {
  BAR_Q_FULL = 0,
  BAR_Q_EMPTY = 1,
  BAR_KV_FULL = 2,
  BAR_KV_EMPTY = BAR_KV_FULL + kStages,
  BAR_S_FULL = BAR_KV_EMPTY + kStages, // [2]
  BAR_P_READY = BAR_S_FULL + 2,        // [2] all of P written (keys 64..127 were the last)
  BAR_P_LO = BAR_P_READY + 2,          // [2] P of keys 0..63 written: the first half of P V may start
  BAR_O_FINAL = BAR_P_LO + 2,          // [2]
  BAR_O_FREE = BAR_O_FINAL + 2,        // [2]
  NUM_BARS = BAR_O_FREE + 2
};
constexpr uint32_t kOffTmemPtr = kOffBar + NUM_BARS * 8;
constexpr int kScaleRing = 16; // FP8: scale of ring entry r (a K or a V tile) at slot r % 16; the producer runs at most
                               // kStages entries ahead of the MMAs and the softmax at most 4 behind them
constexpr uint32_t kOffScale = kOffTmemPtr + 16;
constexpr uint32_t kSmemUsed = kOffScale + kScaleRing * 4;
constexpr uint32_t kSmemBytes = kSmemUsed + 1024; // slack for manual 1024-byte alignment

constexpr uint32_t kIdescQK = make_idesc_bf16(128, 128, 0, 0);
constexpr uint32_t kIdescQK8 = make_idesc_e4m3(128, 128, 0, 0);
constexpr uint32_t kIdescPV8 = make_idesc_e4m3(128, 128, 0, 1);
constexpr uint32_t kTileBytes8 = 16384;
constexpr float kRescaleThreshold8 = 1.0f; // FP8: P = 128 * 2^(z - m) must stay below e4m3's 448

// Register split of the 64K file (setmaxnreg): 4 warps x LOW + 8 softmax warps x HIGH must stay within the 12 x 168 = 2016
// the launch allocates (2048 exactly never gets its last increase granted: the bounded waits trap).  Measured on cfg5:
// 80 / 208: 1147 TFLOP/s, 72 / 216: 1169 (the softmax path wants ~210 registers: 44 instead of 88 bytes of spills),
// 64 / 216: 1169, 56 / 224: 1107 and 40 / 232: 1115 (producer / issuer starved), 88 / 208: 1148, 104 / 200: 1133.
// (The two idle warps cannot hand their share over: registers of warps that exit do not return to the pool.)
#ifndef SLACK_REG_LOW
#define SLACK_REG_LOW 72
#endif
#ifndef SLACK_REG_HIGH
#define SLACK_REG_HIGH 216
#endif
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
#ifndef SLACK_EMU_OF_8
#define SLACK_EMU_OF_8 2
#endif
constexpr int kEmuOf8 = SLACK_EMU_OF_8; // pairs out of every 8 whose exp2 runs on the FMA pipe instead of the MUFU
constexpr float kRescaleThreshold = 8.0f; // skip the O rescale while the row max grew by < 2^8 (in exp2 units)

// Key-tile steps of an item: ns sink tiles ("sink + local"; first piece of a row only) and then the window tiles
// [tb, te).  Step j visits tile_of(j); its visible positions are [lo_of(j), hi_of(j)).
struct ItemView {
  int tb, te, T, nq, ns, st0, s_lo, s_hi, w_lo, w_hi;
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
  v.nq = it.q_rows > kTileM ? 2 : 1;
  return v;
}
// the same view with every field broadcast from lane 0 (warp-uniform for the compiler)
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
  v.nq = uni(v.nq);
  return v;
}

// Epilogue stores of one warp: rows [row0, row0 + 32) of the item (those below q_rows are written), O / l as bf16 (final
// output; `base` = the item's first output row, `stride` elements between rows) or fp32 (split-KV partial).
// O leaves TMEM in the 16x256b fragment layout (a quad of lanes owns 8 consecutive columns of a row) and is transposed
// inside the quads, so that a store instruction writes 64-byte runs of 8 rows instead of 16 bytes of 32 rows: rows are
// 256 B .. 3 KB apart in memory, and 32 lines per store instruction kept the LSU busy for ~8000 cycles per item.
// Not inlined: the hot loop's register allocation must not see this code (8 bytes more of spills cost it 1.4 %).
template <int kD>
__device__ __noinline__ void store_o(uint32_t tO, float inv_l, int lane, int row0, int q_rows, bool final_out, void *base, size_t stride) {
  const int fg = lane >> 2, fc = lane & 3;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
#pragma unroll
    for (int cb = 0; cb < kD / 64; ++cb) {
      uint32_t r[32];
      tmem_ld_16x256b_x8(tO + ((uint32_t)(16 * half) << 16) + (uint32_t)(cb * 64), r);
      tmem_wait_ld();
#pragma unroll
      for (int rs = 0; rs < 2; ++rs) {
        const int wr = 16 * half + 8 * rs + fg; // row inside the warp's 32 (= the lane that owns it: its 1 / l)
        const float inv = __shfl_sync(0xffffffffu, inv_l, wr);
        const int lr = row0 + wr;
        const bool ok = lr < q_rows;
#pragma unroll
        for (int mm = 0; mm < 2; ++mm) {                // column groups 4 mm .. 4 mm + 3 of the 64-column block
          const int col = cb * 64 + 8 * (4 * mm + fc); // after the transpose: this lane's 8 columns
          if (final_out) {
            uint32_t a[4];
#pragma unroll
            for (int n = 0; n < 4; ++n)
              a[n] = pack_bf16x2(__uint_as_float(r[4 * (4 * mm + n) + 2 * rs]) * inv,
                                 __uint_as_float(r[4 * (4 * mm + n) + 2 * rs + 1]) * inv);
            quad_transpose4(a, fc);
            if (ok)
              *reinterpret_cast<uint4 *>(reinterpret_cast<__nv_bfloat16 *>(base) + (size_t)lr * stride + col) =
                  make_uint4(a[0], a[1], a[2], a[3]);
          } else {
            uint32_t lo[4], hi[4];
#pragma unroll
            for (int n = 0; n < 4; ++n) {
              lo[n] = __float_as_uint(__uint_as_float(r[4 * (4 * mm + n) + 2 * rs]) * inv);
              hi[n] = __float_as_uint(__uint_as_float(r[4 * (4 * mm + n) + 2 * rs + 1]) * inv);
            }
            quad_transpose4(lo, fc);
            quad_transpose4(hi, fc);
            if (ok) {
              uint4 *d = reinterpret_cast<uint4 *>(reinterpret_cast<float *>(base) + (size_t)lr * stride + col);
              d[0] = make_uint4(lo[0], hi[0], lo[1], hi[1]);
              d[1] = make_uint4(lo[2], hi[2], lo[3], hi[3]);
            }
          }
        }
      }
    }
  }
}

} // namespace

// kTrace (instantiated in -DSLACK_DIAGNOSTICS builds only): records clock64() time stamps of CTA 0's first item into p.dbg_t (slack_debug_set key 1):
// [role 0/1 = softmax tile 0/1, 2 = MMA issuer, 3 = per-warp arrivals][kv step < 64][8 slots], then per-CTA spans.  The production instantiation has no trace code.
#define SLACK_TRACE(role, step, slot)                                                                      \
  if constexpr (kTrace) {                                                                                  \
    if (p.dbg_t != nullptr && blockIdx.x == 0 && k == item_begin && (step) < 64 && (threadIdx.x & ((role) == 2 ? 31 : 127)) == 0)                    \
      p.dbg_t[((role) * 64 + (step)) * 8 + (slot)] = (uint32_t)clock64();                                  \
  }

template <bool kTrace, bool kSparse, bool kFp8, bool kDual = false, int kD = 128>
__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const TcParams p, const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
               const __grid_constant__ CUtensorMap tm_v) {
  // dual items (DevItem::dual) are served by a dense bf16 instantiation of their own, launched for plans that hold any:
  // carrying the extra paths costs the issuer warp registers (spills on its critical path: +4.6 % cycles per key step)
  constexpr bool kDualOk = kDual && !kSparse && kD == 128;
  // head_dim 64 (bf16 only): Q / K / V tiles are ONE 16 KB half ([128 rows][64 d]), Q K^T takes 4 MMAs of K = 16, P V has
  // N = 64 and O takes the first 64 columns of its TMEM slot; the softmax work per key tile is that of head_dim 128
  static_assert(kD == 128 || (kD == 64 && !kFp8 && !kDual), "head_dim 64 is served by the bf16 non-dual instantiations");
  constexpr uint32_t kTileBytesD = 128u * kD * 2u;
  constexpr uint32_t kIdescPVd = make_idesc_bf16(128, kD, 0, 1);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base + kOffQ;
  const uint32_t sKV = smem_base + kOffKV;
  const uint32_t bars = smem_base + kOffBar;
  const uint32_t tmem_ptr_smem = smem_base + kOffTmemPtr;
  const uint32_t sScale = smem_base + kOffScale;
  auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };

  // warp-uniform by construction, and provably so for the compiler (keeps the role branches and everything the
  // MMA issuer derives from them on the uniform datapath: UTCHMMA takes its descriptors from uniform registers)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const int item_begin = p.cta_begin[blockIdx.x];
  const int item_end = p.cta_begin[blockIdx.x + 1];
  unsigned long long *dbg = p.dbg_flag;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tm_q);
    prefetch_tensormap(&tm_k);
    prefetch_tensormap(&tm_v);
    mbar_init(bar(BAR_Q_FULL), 1);
    mbar_init(bar(BAR_Q_EMPTY), 1);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar(BAR_KV_FULL + s), 1);
      mbar_init(bar(BAR_KV_EMPTY + s), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar(BAR_S_FULL + i), 1);
      mbar_init(bar(BAR_P_READY + i), 4); // one arrival per softmax warp
      mbar_init(bar(BAR_P_LO + i), 4);
      mbar_init(bar(BAR_O_FINAL + i), 1);
      mbar_init(bar(BAR_O_FREE + i), 4);
    }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_ptr_smem, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  // PDL: everything above (barrier init, TMEM allocation, descriptor prefetch) overlapped the previous kernel's drain;
  // from here on the kernel reads memory its predecessors wrote (pool, Q, step lists) and writes Out / the workspace
  pdl_wait();
  pdl_launch_dependents();

  const int H = p.n_heads;
  const int P = 1 << p.page_log2;
  if constexpr (kTrace) { // per-CTA span: words [2048 + 4*cta .. +3] = {clock start, clock end, globaltimer start, end}
    if (threadIdx.x == 0 && p.dbg_t != nullptr) {
      unsigned long long gt;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
      p.dbg_t[2048 + 4 * blockIdx.x + 0] = (uint32_t)clock64();
      p.dbg_t[2048 + 4 * blockIdx.x + 2] = (uint32_t)gt;
    }
  }

  if (warp < 4) {
    setmaxnreg_dec<SLACK_REG_LOW>();
    if (warp == 0) {
      // ============================== TMA producer ==============================
      // The whole warp walks the loop (uniform control flow); one elected lane arms the barrier and issues the copies.
      uint32_t ring = 0;
      int n_item = 0; // items with at least one step (the others are skipped by every role)
      for (int k = item_begin; k < item_end; ++k) {
        const DevItem it = p.items[k];
        const ItemView v = uniform_view_of(it);
        const int Ts = kSparse ? uni(p.item_steps[k]) : v.T; // key-tile steps this item visits
        if (Ts == 0) continue;
        const uint16_t *steps = kSparse ? p.steps + uni(it.step_off) : nullptr;
        const int head = uni(it.head), q_row0 = uni(it.q_row0), pt_off = uni(it.pt_off);
        // dual item: the queue's next item rides in query-tile slot 1 with its own head / rows / page table / key tiles
        const bool dual = kDualOk && uni(it.dual) != 0;
        const DevItem itb = dual ? p.items[k + 1] : it;
        const ItemView vb = uniform_view_of(itb);
        const int head_b = uni(itb.head), q_row0_b = uni(itb.q_row0), pt_off_b = uni(itb.pt_off);
        const int nq = dual ? 2 : v.nq;
        mbar_wait(bar(BAR_Q_EMPTY), (uint32_t)((n_item & 1) ^ 1), 100, dbg);
        ++n_item;
        if (elect_one()) {
          if constexpr (kFp8) { // one [128 rows][128 codes] box per query tile
            mbar_expect_tx(bar(BAR_Q_FULL), (uint32_t)nq * kTileBytes8);
            for (int i = 0; i < nq; ++i) {
              const int h_i = (dual && i == 1) ? head_b : head;
              const int r_i = (dual && i == 1) ? q_row0_b : q_row0 + i * kTileM;
              tma_load_2d(sQ + i * kTileBytes, &tm_q, bar(BAR_Q_FULL), h_i * 128, r_i);
            }
          } else {
            mbar_expect_tx(bar(BAR_Q_FULL), (uint32_t)nq * kTileBytesD);
            for (int i = 0; i < nq; ++i) {
              const int h_i = (dual && i == 1) ? head_b : head;
              const int r_i = (dual && i == 1) ? q_row0_b : q_row0 + i * kTileM;
              for (int c = 0; c < kD / 64; ++c)
                tma_load_2d(sQ + i * kTileBytes + c * kHalfBytes, &tm_q, bar(BAR_Q_FULL), h_i * kD + c * 64, r_i);
            }
          }
        }
        __syncwarp();
        for (int j0 = 0; j0 < Ts; j0 += 32) { // 32 steps at a time: each lane looks up the pool row of one step's tile
          const int my_jj = j0 + lane;
          int my_row = 0, my_row_b = 0;
          [[maybe_unused]] float my_sk = 1.f, my_sv = 1.f, my_sk_b = 1.f, my_sv_b = 1.f;
          if (dual && my_jj < Ts) {
            const int tile_b = vb.tile_of(my_jj);
            const int page_b = __ldg(p.page_tables + pt_off_b + ((tile_b * kTileN) >> p.page_log2));
            my_row_b = (page_b * H + head_b) * P + ((tile_b * kTileN) & (P - 1));
            if constexpr (kFp8) {
              const size_t si = ((size_t)page_b * H + head_b) * (size_t)(P >> 7) + (size_t)(((tile_b * kTileN) & (P - 1)) >> 7);
              my_sk_b = __ldg(p.k_scale + si);
              my_sv_b = __ldg(p.v_scale + si);
            }
          }
          if (my_jj < Ts) {
            const int my_tile = v.tile_of(kSparse ? (int)__ldg(steps + my_jj) : my_jj);
            const int my_page = __ldg(p.page_tables + pt_off + ((my_tile * kTileN) >> p.page_log2));
            my_row = (my_page * H + head) * P + ((my_tile * kTileN) & (P - 1));
            if constexpr (kFp8) { // the tile's scales: one per (page, head, 128-slot block)
              const size_t si = ((size_t)my_page * H + head) * (size_t)(P >> 7) + (size_t)(((my_tile * kTileN) & (P - 1)) >> 7);
              my_sk = __ldg(p.k_scale + si);
              my_sv = __ldg(p.v_scale + si);
            }
          }
          const int cnt = min(32, Ts - j0);
          for (int j = 0; j < cnt; ++j) {
            const int row_a = __shfl_sync(0xffffffffu, my_row, j);
            const int row_b = dual ? __shfl_sync(0xffffffffu, my_row_b, j) : 0;
            [[maybe_unused]] float t_sk = 1.f, t_sv = 1.f;
            [[maybe_unused]] float t_sk_b = 1.f, t_sv_b = 1.f;
            if constexpr (kFp8) {
              t_sk = __shfl_sync(0xffffffffu, my_sk, j);
              t_sv = __shfl_sync(0xffffffffu, my_sv, j);
              if (dual) {
                t_sk_b = __shfl_sync(0xffffffffu, my_sk_b, j);
                t_sv_b = __shfl_sync(0xffffffffu, my_sv_b, j);
              }
            }
            for (int t = 0; t < (dual ? 2 : 1); ++t) { // dual: K_a V_a K_b V_b
            const int row = t == 0 ? row_a : row_b;
            if (t == 1) t_sk = t_sk_b, t_sv = t_sv_b;
#pragma unroll
            for (int kv = 0; kv < 2; ++kv) {
              const uint32_t stage = ring % kStages;
              const uint32_t ph = (ring / kStages) & 1u;
              mbar_wait(bar(BAR_KV_EMPTY + stage), ph ^ 1u, 110 + stage, dbg);
              if (elect_one()) {
                const CUtensorMap *tm = kv == 0 ? &tm_k : &tm_v;
                if constexpr (kFp8) {
                  st_shared_f32(sScale + (ring % kScaleRing) * 4u, kv == 0 ? t_sk : t_sv); // read by the softmax warps
                  mbar_expect_tx(bar(BAR_KV_FULL + stage), kTileBytes8);
                  tma_load_2d(sKV + stage * kTileBytes, tm, bar(BAR_KV_FULL + stage), 0, row);
                } else {
                  mbar_expect_tx(bar(BAR_KV_FULL + stage), kTileBytesD);
                  tma_load_2d(sKV + stage * kTileBytes, tm, bar(BAR_KV_FULL + stage), 0, row);
                  if constexpr (kD == 128) tma_load_2d(sKV + stage * kTileBytes + kHalfBytes, tm, bar(BAR_KV_FULL + stage), 64, row);
                }
              }
              __syncwarp();
              ++ring;
            }
            }
          }
        }
        if (dual) ++k; // the companion has been served
      }
    } else if (warp == 1) {
      // ============================== MMA issuer ==============================
      uint32_t ring = 0;
      // parities of the per-tile barriers, bit i = query tile i (kept in two scalars: indexed arrays would live in local
      // memory, on the issuer's critical path): steps seen (S_FULL / P_LO / P_READY) and items seen (O_FINAL / O_FREE)
      uint32_t cnt_par = 0, itn_par = 0;
      auto cnt_of = [&](int i) { return (cnt_par >> i) & 1u; };
      auto itn_of = [&](int i) { return (itn_par >> i) & 1u; };
      int n_item = 0;
      auto issue_qk = [&](int i, uint32_t stage) {
        const uint32_t a_base = sQ + i * kTileBytes;
        const uint32_t b_base = sKV + stage * kTileBytes;
        const uint32_t d = tmem_base + (uint32_t)(i * 128);
        if constexpr (kFp8) { // K = 32 codes = 32 bytes per instruction, the whole head_dim in one 128-byte row
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mma_ss_f8(d, make_smem_desc_sw128(a_base + (uint32_t)k * 32u, 16, 1024), make_smem_desc_sw128(b_base + (uint32_t)k * 32u, 16, 1024),
                      kIdescQK8, k > 0 ? 1u : 0u);
        } else {
#pragma unroll
          for (int k = 0; k < kD / 16; ++k) {
            const uint32_t off = (uint32_t)(k >> 2) * kHalfBytes + (uint32_t)(k & 3) * 32u;
            mma_ss(d, make_smem_desc_sw128(a_base + off, 16, 1024), make_smem_desc_sw128(b_base + off, 16, 1024), kIdescQK,
                   k > 0 ? 1u : 0u);
          }
        }
      };
      // P V over keys [64*half, 64*half + 64) of the tile (4 MMAs of K = 16)
      auto issue_pv = [&](int i, uint32_t stage, int half, bool acc) {
        const uint32_t b_base = sKV + stage * kTileBytes;
        const uint32_t d = tmem_base + (uint32_t)(256 + i * 128);
        const uint32_t a = tmem_base + (uint32_t)(i * 128);
        if constexpr (kFp8) { // 2 instructions of K = 32 keys (8 TMEM columns of P, 32 rows x 128 B of V) per half
#pragma unroll
          for (int kk = 0; kk < 2; ++kk) {
            const int k = half * 2 + kk;
            mma_ts_f8(d, a + (uint32_t)(k * 8), make_smem_desc_sw128(b_base + (uint32_t)k * 4096u, kHalfBytes, 1024), kIdescPV8,
                      (acc || k > 0) ? 1u : 0u);
          }
        } else {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            const int k = half * 4 + kk;
            mma_ts(d, a + (uint32_t)(k * 8), make_smem_desc_sw128(b_base + (uint32_t)k * 2048u, kHalfBytes, 1024), kIdescPVd,
                   (acc || k > 0) ? 1u : 0u);
          }
        }
      };
      for (int k = item_begin; k < item_end; ++k) {
        const DevItem it = p.items[k];
        const ItemView v = uniform_view_of(it);
        const int Ts = kSparse ? uni(p.item_steps[k]) : v.T;
        if (Ts == 0) continue;
        const uint16_t *steps = kSparse ? p.steps + uni(it.step_off) : nullptr;
        // dense step index of the item's jj-th visited step (block-sparse: read one step ahead of its use)
        auto step_at = [&](int jj) { return kSparse ? uni((int)__ldg(steps + min(jj, Ts - 1))) : jj; };
        int j_dense = step_at(0);
        const uint32_t r0 = ring;
        mbar_wait(bar(BAR_Q_FULL), (uint32_t)(n_item & 1), 200, dbg);
        ++n_item;
        // masked key rows of a V tile must be zero: P is 0 there, but 0 * NaN/Inf garbage would poison O
        auto zero_masked_v = [&](const ItemView &vv, int jd, uint32_t stage) {
          const int tile = vv.tile_of(jd);
          const int c_lo = max(0, vv.lo_of(jd) - tile * kTileN);
          const int c_hi = min(kTileN, vv.hi_of(jd) - tile * kTileN);
          if (c_lo > 0 || c_hi < kTileN) {
            const int n_zero = c_lo + (kTileN - c_hi);
            const uint32_t base = sKV + stage * kTileBytes;
            constexpr int kVecsD = kFp8 ? 8 : 16; // 16-byte vectors per key row
            for (int idx = lane; idx < n_zero * kVecsD; idx += 32) {
              int r = idx / kVecsD;
              r = r < c_lo ? r : c_hi + (r - c_lo);
              const int w = idx % kVecsD;
              const uint32_t addr = base + (uint32_t)(w >> 3) * kHalfBytes + (uint32_t)r * 128u + (uint32_t)(w & 7) * 16u;
              asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
            }
            fence_proxy_async_smem();
            __syncwarp();
          }
        };
        if (kDualOk && uni(it.dual) != 0) {
          // ---- dual item: tile slot i walks its own item (k + i) over its own ring entries K_i(j) = r0 + 4j + 2i, V_i(j) = K_i(j) + 1
          const DevItem itb = p.items[k + 1];
          const ItemView vb = uniform_view_of(itb);
          auto entry = [&](int i, int j, int kv, uint32_t &stage, uint32_t &ph) {
            const uint32_t r = r0 + 4u * (uint32_t)j + 2u * (uint32_t)i + (uint32_t)kv;
            stage = r % kStages;
            ph = (r / kStages) & 1u;
          };
          for (int i = 0; i < 2; ++i) {
            uint32_t stage, ph;
            entry(i, 0, 0, stage, ph);
            mbar_wait(bar(BAR_KV_FULL + stage), ph, 210 + stage, dbg);
            tc_fence_after();
            if (elect_one()) {
              issue_qk(i, stage);
              mma_commit(bar(BAR_S_FULL + i));
              mma_commit(bar(BAR_KV_EMPTY + stage));
              if (Ts == 1 && i == 1) mma_commit(bar(BAR_Q_EMPTY));
            }
            __syncwarp();
          }
          for (int j = 0; j < Ts; ++j) {
            const bool has_next = (j + 1) < Ts;
            for (int i = 0; i < 2; ++i) {
              uint32_t stage_v, ph_v, stage_k = 0, ph_k = 0;
              entry(i, j, 1, stage_v, ph_v);
              mbar_wait(bar(BAR_KV_FULL + stage_v), ph_v, 220 + stage_v, dbg);
              zero_masked_v(i == 0 ? v : vb, j, stage_v);
              mbar_wait(bar(BAR_P_LO + i), cnt_of(i), 260 + i, dbg);
              if (j == 0) mbar_wait(bar(BAR_O_FREE + i), itn_of(i) ^ 1u, 240 + i, dbg);
              tc_fence_after();
              if (elect_one()) issue_pv(i, stage_v, 0, j > 0);
              __syncwarp();
              mbar_wait(bar(BAR_P_READY + i), cnt_of(i), 230 + i, dbg);
              if (has_next) {
                entry(i, j + 1, 0, stage_k, ph_k);
                mbar_wait(bar(BAR_KV_FULL + stage_k), ph_k, 250 + stage_k, dbg);
              }
              tc_fence_after();
              if (elect_one()) {
                issue_pv(i, stage_v, 1, true);
                mma_commit(bar(BAR_KV_EMPTY + stage_v));
                if (has_next) {
                  issue_qk(i, stage_k);
                  mma_commit(bar(BAR_S_FULL + i));
                  mma_commit(bar(BAR_KV_EMPTY + stage_k));
                  if (i == 1 && j + 2 == Ts) mma_commit(bar(BAR_Q_EMPTY));
                } else {
                  mma_commit(bar(BAR_O_FINAL + i));
                }
              }
              __syncwarp();
              cnt_par ^= 1u << i;
              if (!has_next) itn_par ^= 1u << i;
            }
          }
          ring = r0 + 4u * (uint32_t)Ts;
          ++k; // the companion has been served
          continue;
        }
        {
          const uint32_t stage = r0 % kStages, ph = (r0 / kStages) & 1u;
          mbar_wait(bar(BAR_KV_FULL + stage), ph, 210 + stage, dbg);
          tc_fence_after();
          if (elect_one()) {
            for (int i = 0; i < v.nq; ++i) {
              issue_qk(i, stage);
              mma_commit(bar(BAR_S_FULL + i));
            }
            mma_commit(bar(BAR_KV_EMPTY + stage));
            if (Ts == 1) mma_commit(bar(BAR_Q_EMPTY));
          }
          __syncwarp();
        }
        for (int j = 0; j < Ts; ++j) {
          const int jd = j_dense;
          j_dense = step_at(j + 1);
          const uint32_t rv = r0 + 2u * (uint32_t)j + 1u;
          const uint32_t stage_v = rv % kStages, ph_v = (rv / kStages) & 1u;
          const bool has_next = (j + 1) < Ts;
          const uint32_t rk = rv + 1u;
          const uint32_t stage_k = rk % kStages, ph_k = (rk / kStages) & 1u;
          SLACK_TRACE(2, j, 0);
          mbar_wait(bar(BAR_KV_FULL + stage_v), ph_v, 220 + stage_v, dbg);
          SLACK_TRACE(2, j, 1);
          {
            // masked key rows of V must be zero: P is 0 there, but 0 * NaN/Inf garbage would poison O
            const int tile = v.tile_of(jd);
            const int c_lo = max(0, v.lo_of(jd) - tile * kTileN);
            const int c_hi = min(kTileN, v.hi_of(jd) - tile * kTileN);
            if (c_lo > 0 || c_hi < kTileN) {
              const int n_zero = c_lo + (kTileN - c_hi);
              const uint32_t base = sKV + stage_v * kTileBytes;
              constexpr int kVecs = kFp8 ? 8 : kD / 8; // 16-byte vectors per key row (FP8, head_dim 64: one 128-byte row; else two)
              for (int idx = lane; idx < n_zero * kVecs; idx += 32) {
                int r = idx / kVecs;
                r = r < c_lo ? r : c_hi + (r - c_lo);
                const int w = idx % kVecs;
                const uint32_t addr = base + (uint32_t)(w >> 3) * kHalfBytes + (uint32_t)r * 128u + (uint32_t)(w & 7) * 16u;
                asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
              }
              fence_proxy_async_smem();
              __syncwarp();
            }
          }
          tc_fence_after();
          for (int i = 0; i < v.nq; ++i) {
            mbar_wait(bar(BAR_P_LO + i), cnt_of(i), 260 + i, dbg);
            if (j == 0) mbar_wait(bar(BAR_O_FREE + i), itn_of(i) ^ 1u, 240 + i, dbg);
            tc_fence_after();
            SLACK_TRACE(2, j, 2 + 2 * i);
            if (elect_one()) issue_pv(i, stage_v, 0, j > 0);
            __syncwarp();
            mbar_wait(bar(BAR_P_READY + i), cnt_of(i), 230 + i, dbg);
            if (has_next && i == 0) mbar_wait(bar(BAR_KV_FULL + stage_k), ph_k, 250 + stage_k, dbg);
            tc_fence_after();
            if (elect_one()) {
              issue_pv(i, stage_v, 1, true);
              if (i == v.nq - 1) mma_commit(bar(BAR_KV_EMPTY + stage_v));
              if (has_next) {
                issue_qk(i, stage_k);
                mma_commit(bar(BAR_S_FULL + i));
                if (i == v.nq - 1) {
                  mma_commit(bar(BAR_KV_EMPTY + stage_k));
                  if (j + 2 == Ts) mma_commit(bar(BAR_Q_EMPTY));
                }
              } else {
                mma_commit(bar(BAR_O_FINAL + i));
              }
            }
            __syncwarp();
            SLACK_TRACE(2, j, 3 + 2 * i);
            cnt_par ^= 1u << i;
            if (!has_next) itn_par ^= 1u << i;
          }
        }
        ring = r0 + 2u * (uint32_t)Ts;
      }
    }
  } else {
    // ============================== softmax + epilogue warpgroups ==============================
    setmaxnreg_inc<SLACK_REG_HIGH>();
    const int i = warp >= 8 ? 1 : 0;
    const int w4 = warp & 3;
    const int row = w4 * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(w4 * 32) << 16;
    const uint32_t tS = tmem_base + lane_addr + (uint32_t)(i * 128);
    const uint32_t tO = tmem_base + lane_addr + (uint32_t)(256 + i * 128);
    const float sl2 = p.scale * kLog2e;
    uint32_t cnt = 0, itn = 0;
    [[maybe_unused]] uint32_t ring = 0; // FP8: ring entry of the item's first K tile (the producer's count; scale slots)
    bool first_item = true;
    int adv = 1;
    // The queue's records are read one item AHEAD (the loads of the next one are issued before the epilogue and land while
    // it runs): two dependent global loads at the top of every item cost the softmax warps ~4000 cycles per item.
    DevItem it0 = p.items[min(item_begin, max(item_end - 1, item_begin))];
    [[maybe_unused]] DevItem it1 = it0; // dual kernels: the record behind it0 (the companion of a dual item)
    if constexpr (kDualOk) it1 = p.items[min(item_begin + 1, max(item_end - 1, item_begin))];
    DevItem nx0 = it0;
    [[maybe_unused]] DevItem nx1 = it0;
    for (int k = item_begin; k < item_end; k += adv) {
      // dual item: tile slot 1 serves the queue's NEXT item (its own rows 0.., head, mask columns, output rows)
      const bool dual = kDualOk && it0.dual != 0;
      adv = dual ? 2 : 1;
      const DevItem it = (dual && i == 1) ? it1 : it0;
      auto load_next = [&]() {
        nx0 = p.items[min(k + adv, item_end - 1)];
        if constexpr (kDualOk) nx1 = p.items[min(k + adv + 1, item_end - 1)];
      };
      auto rotate = [&]() {
        it0 = nx0;
        if constexpr (kDualOk) it1 = nx1;
      };
      const ItemView v = view_of(it);
      const int row_base = dual ? 0 : i * kTileM; // this tile's first row inside ITS item
      [[maybe_unused]] const uint32_t r0 = ring;
      if constexpr (kFp8) ring += (dual ? 4u : 2u) * (uint32_t)v.T; // every role counts the tiles, also the one that skips the item
      if (!dual && i >= v.nq) {
        load_next();
        rotate();
        continue;
      }
      const int Ts = kSparse ? p.item_steps[k] : v.T;
      const uint16_t *steps = kSparse ? p.steps + it.step_off : nullptr;
      if (Ts == 0) { // block-sparse: no selected key tile in this item: out = 0, lse = -inf; no barrier is touched
        const int local_row = row_base + row;
        if (local_row < it.q_rows) {
          if (it.partial_slot < 0) {
            uint4 *dst = reinterpret_cast<uint4 *>(reinterpret_cast<__nv_bfloat16 *>(p.out) +
                                                   ((size_t)(it.q_row0 + local_row) * H + it.head) * kD);
#pragma unroll
            for (int e = 0; e < kD / 8; ++e) dst[e] = make_uint4(0u, 0u, 0u, 0u);
            if (p.lse != nullptr) p.lse[(size_t)it.head * p.total_q + it.q_row0 + local_row] = -INFINITY;
          } else {
            float4 *dst = reinterpret_cast<float4 *>(p.ws_o + ((size_t)it.partial_slot * kItemRows + local_row) * kD);
#pragma unroll
            for (int e = 0; e < kD / 4; ++e) dst[e] = make_float4(0.f, 0.f, 0.f, 0.f);
            p.ws_lse[(size_t)it.partial_slot * kItemRows + local_row] = -INFINITY;
          }
        }
        load_next();
        rotate();
        continue;
      }
      float m = -INFINITY, l = 0.f;
      // FP8: scale of this thread's query row (rows past the end of Q hold garbage that is never stored)
      [[maybe_unused]] float q_sc = 1.f;
      if constexpr (kFp8) q_sc = __ldg(p.q_scale + (size_t)it.head * p.total_q + min(it.q_row0 + row_base + row, p.total_q - 1));
      int j_dense = kSparse ? (int)__ldg(steps) : 0;
      for (int j = 0; j < Ts; ++j) {
        const int jd = j_dense; // dense step index (block-sparse: the next one is fetched a step ahead)
        j_dense = kSparse ? (int)__ldg(steps + min(j + 1, Ts - 1)) : j + 1;
        SLACK_TRACE(i, j, 0);
        mbar_wait(bar(BAR_S_FULL + i), cnt & 1u, 300 + i, dbg);
        tc_fence_after();
        SLACK_TRACE(i, j, 1);
        float s[128];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t r[32];
          tmem_ld32(tS + (uint32_t)(c * 32), r);
#pragma unroll
          for (int e = 0; e < 32; ++e) s[c * 32 + e] = __uint_as_float(r[e]);
        }
        tmem_wait_ld();
        SLACK_TRACE(i, j, 2);
        const int tile = v.tile_of(jd);
        const int c_lo = max(0, v.lo_of(jd) - tile * kTileN);
        const int c_hi = min(kTileN, v.hi_of(jd) - tile * kTileN);
        if (c_lo > 0 || c_hi < kTileN) {
#pragma unroll
          for (int e = 0; e < 128; ++e) s[e] = (e >= c_lo && e < c_hi) ? s[e] : -INFINITY;
        }
        if constexpr (kTrace) {
          if (p.dbg_s != nullptr && blockIdx.x == 0 && first_item && j == 0) {
#pragma unroll
            for (int e = 0; e < 128; ++e) p.dbg_s[(i * 128 + row) * 128 + e] = s[e];
          }
        }
        // Row max of the tile: four independent FMNMX3 chains.  On the first tile of an item it is needed before any
        // exponential; later it is evaluated in the same instruction stream as the first 64 columns' exponentials
        // (which use the running max), and only a growth beyond the threshold forces those 64 columns to be redone.
        auto row_max = [&]() {
          float mxc[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) mxc[c] = max3(s[c * 32], s[c * 32 + 1], s[c * 32 + 2]);
#pragma unroll
          for (int e = 3; e + 1 < 32; e += 2) {
#pragma unroll
            for (int c = 0; c < 4; ++c) mxc[c] = max3(mxc[c], s[c * 32 + e], s[c * 32 + e + 1]);
          }
#pragma unroll
          for (int c = 0; c < 4; ++c) mxc[c] = fmaxf(mxc[c], s[c * 32 + 31]);
          return fmaxf(max3(mxc[0], mxc[1], mxc[2]), mxc[3]);
        };
        // logit -> exponent: z = s * cz + az.  bf16: cz = scale log2e, az = 0 and m is kept in units of s (z = s cz).
        // FP8: cz = scale log2e sq sk_t, az = log2 sv_t (the V scale rides inside P), m is kept in units of z, and P is
        // scaled by 2^7 so that its e4m3 codes use the range up to 128 (x 2 before a lazy rescale) of the format's 448.
        [[maybe_unused]] float cz = sl2, az = 0.f, l_fix = 1.f;
        if constexpr (kFp8) {
          // ring entry of this tile slot's K tile at step j (dual items: K_a V_a K_b V_b per step)
          const uint32_t rk = dual ? r0 + 4u * (uint32_t)j + 2u * (uint32_t)i : r0 + 2u * (uint32_t)j;
          const float t_sk = ld_shared_f32(sScale + (rk % kScaleRing) * 4u);
          const float t_sv = ld_shared_f32(sScale + ((rk + 1u) % kScaleRing) * 4u);
          cz = sl2 * q_sc * t_sk;
          az = log2f(t_sv);
          l_fix = 0.0078125f / t_sv; // this tile's P sums, taken in units of 128 sv_t, back to plain probabilities
        }
        auto to_m = [&](float mx_s) { // row max of s -> units of m
          if constexpr (kFp8) return fmaf(mx_s, cz, az);
          else return mx_s;
        };
        auto neg_m = [&]() { // addend of the exponent
          if constexpr (kFp8) return az - m + 7.0f;
          else return -m * sl2;
        };
        constexpr float kThr = kFp8 ? kRescaleThreshold8 : kRescaleThreshold;
        if (j == 0) m = to_m(row_max());
        SLACK_TRACE(i, j, 3);
        // P = 2^(s*cz + addend) on packed pairs: FFMA2 for the argument, then either 2 MUFU.EX2 or (kEmuOf8 pairs out
        // of every 8) the FMA-pipe polynomial; FADD2 row sums; one F2FP per pair (FP8: per four).
        const uint64_t sl2_2 = kFp8 ? pack2(cz, cz) : pack2(sl2, sl2);
        uint64_t negm_2 = pack2(neg_m(), neg_m());
        uint64_t la0 = pack2(0.f, 0.f), la1 = la0;
        auto exp_chunk = [&](int c) { // 32 columns -> 16 packed bf16x2 (FP8: 8 packed e4m3x4) columns of P
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
            if (e & 1) la1 = fadd2(la1, p2); else la0 = fadd2(la0, p2);
            float p0, p1;
            unpack2(p2, p0, p1);
            if constexpr (kFp8) { // two pairs -> one column of four e4m3 codes
              if (e & 1) pk[e >> 1] = pack_e4m3x4(__uint_as_float(pk[e >> 1]), __uint_as_float(pk[8 + (e >> 1)]), p0, p1);
              else pk[e >> 1] = __float_as_uint(p0), pk[8 + (e >> 1)] = __float_as_uint(p1);
            } else {
              pk[e] = pack_bf16x2(p0, p1);
            }
          }
          if constexpr (kFp8) {
            uint32_t p8[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) p8[e] = pk[e];
            tmem_st8(tS + (uint32_t)(c * 8), p8);
          } else {
            tmem_st16(tS + (uint32_t)(c * 16), pk);
          }
        };
        // the row sums collected since the last call, into l (FP8: in this tile's units of 128 sv_t)
        auto flush_sums = [&]() {
          float a0, a1;
          unpack2(fadd2(la0, la1), a0, a1);
          if constexpr (kFp8) l = fmaf(a0 + a1, l_fix, l);
          else l += a0 + a1;
        };
        {
          const float mx = to_m(row_max()); // independent of the two chunks below: the scheduler interleaves them
          exp_chunk(0);
          exp_chunk(1);
          float grow;
          if constexpr (kFp8) grow = mx - m;
          else grow = (mx - m) * sl2;
          const bool need = grow > kThr; // never on the first tile (m == mx)
          if (__any_sync(0xffffffffu, need)) {
            // PV of the previous key tile has completed (its commit precedes S_FULL in the in-order tensor pipe)
            const float alpha = need ? ex2(-grow) : 1.0f;
            m = need ? mx : m;
            l *= alpha;
#pragma unroll
            for (int c = 0; c < kD / 32; ++c) {
              uint32_t r[32];
              tmem_ld32(tO + (uint32_t)(c * 32), r);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) r[e] = __float_as_uint(__uint_as_float(r[e]) * alpha);
              tmem_st32(tO + (uint32_t)(c * 32), r);
            }
            negm_2 = pack2(neg_m(), neg_m());
            la0 = la1 = pack2(0.f, 0.f);
            exp_chunk(0);
            exp_chunk(1);
          }
        }
        SLACK_TRACE(i, j, 4);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_LO + i)); // P V over keys 0..63 may start
        exp_chunk(2);
        exp_chunk(3);
        flush_sums();
        SLACK_TRACE(i, j, 5);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_READY + i));
        SLACK_TRACE(i, j, 6);
        if constexpr (kTrace) { // per-warp arrival times (rows 3.. : [3][j][warp - 4])
          if (p.dbg_t != nullptr && blockIdx.x == 0 && k == item_begin && j < 64 && lane == 0) p.dbg_t[(3 * 64 + j) * 8 + (warp - 4)] = (uint32_t)clock64();
        }
        ++cnt;
      }
      // ---------------- epilogue: O / l ----------------
      load_next();
      mbar_wait(bar(BAR_O_FINAL + i), itn & 1u, 310 + i, dbg);
      tc_fence_after();
      const float inv_l = kFp8 ? 0.0078125f / l : 1.0f / l; // FP8: O was accumulated from P = 128 * probabilities
      const int local_row = row_base + row;
      const bool valid = local_row < it.q_rows;
      const float lse_val = ((kFp8 ? m : m * sl2) + log2f(l)) * kLn2;
      store_o<kD>(tO, inv_l, lane, row_base + w4 * 32, it.q_rows, it.partial_slot < 0,
                  it.partial_slot < 0
                      ? static_cast<void *>(reinterpret_cast<__nv_bfloat16 *>(p.out) + ((size_t)it.q_row0 * H + it.head) * kD)
                      : static_cast<void *>(p.ws_o + (size_t)it.partial_slot * kItemRows * kD),
                  it.partial_slot < 0 ? (size_t)H * kD : (size_t)kD);
      if (valid) {
        if (it.partial_slot >= 0) p.ws_lse[(size_t)it.partial_slot * kItemRows + local_row] = lse_val;
        else if (p.lse != nullptr) p.lse[(size_t)it.head * p.total_q + it.q_row0 + local_row] = lse_val;
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(BAR_O_FREE + i));
      rotate();
      ++itn;
      first_item = false;
    }
  }

  // ---------------- teardown ----------------
  tc_fence_before();
  __syncthreads();
  if constexpr (kTrace) {
    if (threadIdx.x == 0 && p.dbg_t != nullptr) {
      unsigned long long gt;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
      p.dbg_t[2048 + 4 * blockIdx.x + 1] = (uint32_t)clock64();
      p.dbg_t[2048 + 4 * blockIdx.x + 3] = (uint32_t)gt;
    }
  }
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

size_t attn_tc_smem_bytes() { return kSmemBytes; }

cudaError_t attn_tc_configure() {
  cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, false, false, false, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<false, true, false, false, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
#ifdef SLACK_DIAGNOSTICS
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attn_tc_kernel<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
#endif
  return e;
}

// p.q_scale != null selects the FP8 instantiation (tm_q / tm_k / tm_v are then byte maps with [128 x 128 B] boxes);
// p.steps != null the block-sparse one; p.has_dual the one that serves dual items (the others walk them one by one)
cudaError_t launch_attn_tc(const TcParams &p, const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                           int n_cta, cudaStream_t st, int *n_launched) {
  cudaError_t e;
  if (p.head_dim == 64) {
    if (p.q_scale != nullptr) return cudaErrorInvalidValue; // FP8 pools: head_dim 128 only (the planner refuses the rest)
    if (p.steps != nullptr)
      e = launch_pdl(attn_tc_kernel<false, true, false, false, 64>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
    else
      e = launch_pdl(attn_tc_kernel<false, false, false, false, 64>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  } else if (p.has_dual && p.q_scale == nullptr && p.steps == nullptr)
    e = launch_pdl(attn_tc_kernel<false, false, false, true>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  else if (p.q_scale != nullptr && p.has_dual)
    e = launch_pdl(attn_tc_kernel<false, false, true, true>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  else if (p.q_scale != nullptr)
    e = launch_pdl(attn_tc_kernel<false, false, true>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  else if (p.steps != nullptr)
    e = launch_pdl(attn_tc_kernel<false, true, false>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
#ifdef SLACK_DIAGNOSTICS
  else if (p.dbg_t != nullptr || p.dbg_s != nullptr)
    e = launch_pdl(attn_tc_kernel<true, false, false>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
#endif
  else
    e = launch_pdl(attn_tc_kernel<false, false, false>, dim3(n_cta), dim3(kTcThreads), kSmemBytes, st, p, tm_q, tm_k, tm_v);
  if (n_launched) *n_launched += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
