// smallm_swiglu_kernel.cuh -- decode-sized batches (M <= 128): weight streaming is the whole
// cost (bytes ~ 4*K*N, AI ~ M FLOP/B), so the kernel is built around HBM, not the tensor pipe.
//
//  * swap-AB: the 128-row UMMA operand is a W tile (128 output columns n, MN-major as W is
//    [K,N] row-major), the narrow UMMA-N operand is A (MP = 16/32/64/128 padded tokens,
//    K-major).  Accumulators are Gate^T and Up^T: TMEM lane = n, column = m.  All 128
//    epilogue threads have work even at M = 1.
//  * split-K over a thread-block cluster: the S CTAs of a cluster share one 128-column tile
//    and each streams 1/S of K, so every SM streams equal bytes whatever N/128 is.
//    SiLU is non-linear, so partial Gate/Up sums are reduced BEFORE the activation: each CTA
//    parks its fp32 partials in its own shared memory, and after a cluster barrier CTA r sums
//    rows m = r, r+S, ... over all peers through distributed shared memory in rank order
//    (deterministic; the loads of two rows x 2S peers are in flight together), applies
//    SiLU-multiply and stores bf16, 8 bytes per thread, 256 contiguous bytes per warp.  No
//    global workspace, Gate/Up never reach HBM (BASELINE.json north_star "Small M").
//  * fixed costs matter at these sizes (a call is 3-15 us): the producer thread initialises
//    its barriers and issues the first ring of TMA loads BEFORE the CTA-wide setup barrier
//    (TMEM allocation overlaps the HBM latency of the first loads), and warp 0 issues L2
//    prefetches for the CTA's weight blocks before griddepcontrol.wait, so under programmatic
//    dependent launch the weights start moving while the previous kernel drains.  A prefetch
//    is a hint: it cannot observe or produce stale data (L2 is the point of coherence).
//  * prepacked weights (kWeightsPacked, swiglu_pack_weights): one 3-D TMA box per stage brings
//    the four slabs g0 u0 g1 u1 of the tile (32 KB) instead of four 2-D boxes, and -- because a
//    packed buffer is a constant by contract (include/swiglu_mlp.h) -- the REAL weight loads of
//    the first ring go out before griddepcontrol.wait; only the activation tile waits for the
//    previous kernel.
#pragma once
#include <cuda.h>

#include "gemm_swiglu_kernel.cuh"

namespace swiglu {

constexpr int kSmallMMax = 128;
constexpr int kSmallThreads = 192;  // warp 0 TMA, warp 1 MMA, warps 2-5 epilogue
constexpr int kSmallPrefetchMax = 32;     // k-blocks per CTA prefetched to L2 (one per lane)

// kDeep: one CTA per SM with a six-stage ring (up to 204 KB of weights in flight per CTA) instead
// of two co-resident CTAs with three stages each: half the CTAs (and clusters) to launch for the
// same bytes in flight, used when n-tiles x S fits one CTA per SM (MP <= 32 only).
// kStack: a 64-column tile whose W1 slab and W2 slab are STACKED into one 128-row UMMA operand
// (rows 0-63 = 64 columns of W1, rows 64-127 = the same 64 columns of W2): one MMA per k-step,
// Gate^T in TMEM lanes 0-63 and Up^T in lanes 64-127 of the same MP columns.  Twice the tiles
// of the 128-column form, so shapes with N/128 < #SMs (0.5B, 1.5B) fill the GPU WITHOUT a
// cluster split of K: no cluster launch (an empty cluster-of-4 launch alone is 3.6 us in a
// dependent chain against 1.7 us without clusters, profiles/r02_decode_study.md), no DSMEM
// reduction, no cluster barriers.  One CTA per SM with a deep ring of 18 KB stages.
template <int MP, bool kDeep = false, bool kStack = false>
struct SmallCfg {
  static_assert(!kDeep || MP <= 32, "deep ring: MP <= 32");
  static_assert(!kStack || (MP <= 32 && !kDeep), "stacked 64-column tile: MP <= 32, always a deep ring");
  static constexpr int kTileN = kStack ? 64 : 128;  // output columns per tile
  static constexpr int kCtasPerSm = kDeep ? 1 : ((MP <= 64) ? 2 : 1);
  static constexpr int kStages = kStack ? 5 : kDeep ? 6 : ((MP <= 32) ? 3 : (MP == 64 ? 2 : 4));
  static constexpr int kWBytes = kTileN * BK * 2;  // one W tile: 128 (64) n x 64 k = 16 (8) KB
  static constexpr int kABytes = MP * BK * 2;   // MP tokens x 64 k
  static constexpr int kStageBytes = 2 * kWBytes + kABytes;
  static constexpr int kPartialBytes = 2 * MP * kTileN * 4;  // fp32 Gate^T|Up^T, aliases the ring
  static constexpr int kTmemCols = kStack ? 32 : ((2 * MP < 32) ? 32 : 2 * MP);
  static constexpr int kSmemBytes = kStages * kStageBytes + 256 + 1024;
  static_assert(kPartialBytes <= kStages * kStageBytes, "partials must fit in the ring");
};

struct SmallParams {
  int M, N, K;
  int ksplit;         // cluster size S
  int prefetch_blocks;  // leading k-blocks of each CTA's weight stream to prefetch into L2
  int packed_pre;       // kWeightsPacked: ring stages whose weight loads go out before griddepcontrol.wait
  int probe;          // launch-floor probe (swiglu_launch_floor_probe): 1 = prologue and teardown
                      // only (no loads, MMAs, reduction or stores); 0 = the real kernel
  long long ldy;      // = N
  uint16_t* U;        // kStoreGU only: bf16 Up output (Gate goes to the Y argument)
  unsigned long long* clk;  // optional {SM cycles, globaltimer ns} of CTA 0 (swiglu_set_clock_probe)
  float scale_gate, scale_up;  // kOperandsFp8: Gate / Up dequantisation scales (else unused)
#ifdef SWIGLU_TRACE
  unsigned long long* trace;  // [grid][16] globaltimer stamps (debug builds only)
#endif
};

__device__ __forceinline__ float4 ld_dsmem_v4(uint32_t cluster_addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "r"(cluster_addr)
               : "memory");
  return v;
}

// kStoreGU = true: the merged Gate|Up GEMM of the UNFUSED comparison path at decode sizes (a7):
//   the reduced fp32 Gate and Up are each rounded to bf16 and written to HBM (Y argument = Gate,
//   p.U = Up) instead of going through the activation -- one launch for both projections, the
//   "merged gate_up_proj" serving stacks run before their silu_and_mul kernel.
template <int MP, int kAct = kActSilu, int kWMode = kWeightsKN, bool kStoreGU = false,
          bool kDeep = false, bool kStack = false>
__global__ void __launch_bounds__(kSmallThreads, SmallCfg<MP, kDeep, kStack>::kCtasPerSm)
smallm_swiglu_kernel(const __grid_constant__ CUtensorMap tmap_a,
                     const __grid_constant__ CUtensorMap tmap_w1,
                     const __grid_constant__ CUtensorMap tmap_w2, uint16_t* __restrict__ Y,
                     const SmallParams p) {
  using Cfg = SmallCfg<MP, kDeep, kStack>;
  constexpr int kStages = Cfg::kStages;
  constexpr int kTileN = Cfg::kTileN;
  constexpr bool kF8 = (kWMode == kOperandsFp8);   // E4M3 A and [N,K] weights (gemm kernel header)
  constexpr bool kWK = (kWMode == kWeightsNK) || kF8;
  constexpr bool kPacked = (kWMode == kWeightsPacked);
  constexpr int kBKe = kF8 ? 128 : BK;              // elements of k per stage (128-byte rows)
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + kStages * Cfg::kStageBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
  const uint32_t acc_full_bar = bar_base + 8u * (2 * kStages);
  const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 1);
  // stage layout, unpacked: [W1 c0 | W1 c1 | W2 c0 | W2 c1 | A]; packed: [g0 | u0 | g1 | u1 | A]
  auto smem_w = [&](int s) { return smem_base + s * Cfg::kStageBytes; };
  auto smem_act = [&](int s) { return smem_base + s * Cfg::kStageBytes + 2 * Cfg::kWBytes; };

  const uint32_t warp = threadIdx.x >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  const int S = p.ksplit;
  const uint32_t rank = (S > 1) ? cluster_ctarank() : 0u;
  const int n_tile = blockIdx.x / S;
  const int n_base = n_tile * kTileN;
  const int k_blocks = (p.K + kBKe - 1) / kBKe;
  const int kb_begin = (int)(((long long)k_blocks * rank) / S);
  const int kb_end = (int)(((long long)k_blocks * (rank + 1)) / S);

  // Weights of one k-block into ring slot s (completes on full_bar(s)).  Read exactly once per
  // call: evict-first, so they do not push A out of L2.
  auto issue_w = [&](int kb, int s) {
    const uint32_t fb = full_bar(s);
    const int k0 = kb * kBKe;
    if constexpr (kPacked) {
      // g0 u0 g1 u1: 32 KB (stacked 64-column tile: its g u pair, 16 KB)
      tma_load_3d(smem_w(s), &tmap_w1, fb, 0, k0, n_tile * (kTileN / 32), kEvictFirst);
    } else if constexpr (kStack) {
      tma_load_2d(smem_w(s), &tmap_w1, fb, kWK ? k0 : n_base, kWK ? n_base : k0, kEvictFirst);
      tma_load_2d(smem_w(s) + 8192, &tmap_w2, fb, kWK ? k0 : n_base, kWK ? n_base : k0, kEvictFirst);
    } else {
      // one 64-column x 64-k slab per load; inner tensor-map dimension is N ([K,N]) or K ([N,K])
      auto load_w = [&](uint32_t dst, const CUtensorMap* tm, int n) {
        tma_load_2d(dst, tm, fb, kWK ? k0 : n, kWK ? n : k0, kEvictFirst);
      };
      load_w(smem_w(s), &tmap_w1, n_base);
      load_w(smem_w(s) + 8192, &tmap_w1, n_base + 64);
      load_w(smem_w(s) + 16384, &tmap_w2, n_base);
      load_w(smem_w(s) + 24576, &tmap_w2, n_base + 64);
    }
  };
  auto issue_a = [&](int kb, int s) {
    tma_load_2d(smem_act(s), &tmap_a, full_bar(s), kb * kBKe, 0, kEvictLast);
  };

  if (threadIdx.x == 0) SWIGLU_TRACE_POINT(0);
  const bool clk_probe = p.clk != nullptr && blockIdx.x == 0 && threadIdx.x == 0;
  long long clk_c0 = 0;
  uint64_t clk_t0 = 0;
  if (clk_probe) { clk_c0 = clock64(); clk_t0 = globaltimer_ns(); }
  const bool live = p.probe == 0;
  // ------------------------------------------------------------------ setup
  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tmap_w1);
      if (!kPacked) prefetch_tensormap(&tmap_w2);
      prefetch_tensormap(&tmap_a);
      for (int s = 0; s < kStages; ++s) {
        mbar_init(full_bar(s), 1);
        mbar_init(empty_bar(s), 1);
      }
      mbar_init(acc_full_bar, 1);
      fence_mbar_init();
      fence_proxy_async_all();
    }
    if constexpr (kPacked) {
      // Packed weights are constants (header contract): their loads need not wait for the
      // previous kernel.  Fill the ring's weight half now; the A half follows the dependency.
      const int pre = min(kStages, p.packed_pre);  // ring stages whose weights go out before the wait
      if (lane == 0 && live) {
        for (int i = 0; i < pre && kb_begin + i < kb_end; ++i) {
          mbar_arrive_expect_tx(full_bar(i), Cfg::kStageBytes);
          issue_w(kb_begin + i, i);
        }
      }
      // the next blocks of the CTA's weight stream: L2 prefetch, one k-block per lane
      const int kb = kb_begin + pre + (int)lane;
      if (live && (int)lane < p.prefetch_blocks && kb < kb_end)
        tma_prefetch_l2_3d(&tmap_w1, 0, kb * kBKe, n_tile * (kTileN / 32));
      if (lane == 0 && live) {
        pdl_wait_prior_grid();  // A may be the previous kernel's output
        SWIGLU_TRACE_POINT(2);
        for (int i = 0; i < kStages && kb_begin + i < kb_end; ++i) {
          if (i >= pre) {
            mbar_arrive_expect_tx(full_bar(i), Cfg::kStageBytes);
            issue_w(kb_begin + i, i);
          }
          issue_a(kb_begin + i, i);
        }
      }
    } else {
      // L2 prefetch of this CTA's weight stream (hint; legal before griddepcontrol.wait)
      const int kb = kb_begin + (int)lane;
      if (live && (int)lane < p.prefetch_blocks && kb < kb_end) {
        const int k0 = kb * kBKe;
        tma_prefetch_l2_2d(&tmap_w1, kWK ? k0 : n_base, kWK ? n_base : k0);
        if (!kStack) tma_prefetch_l2_2d(&tmap_w1, kWK ? k0 : n_base + 64, kWK ? n_base + 64 : k0);
        tma_prefetch_l2_2d(&tmap_w2, kWK ? k0 : n_base, kWK ? n_base : k0);
        if (!kStack) tma_prefetch_l2_2d(&tmap_w2, kWK ? k0 : n_base + 64, kWK ? n_base + 64 : k0);
      }
      if (lane == 0 && live) {
        // W or A may be the previous kernel's output: real loads only after the grid dependency
        pdl_wait_prior_grid();
        SWIGLU_TRACE_POINT(2);
        for (int i = 0; i < kStages && kb_begin + i < kb_end; ++i) {
          mbar_arrive_expect_tx(full_bar(i), Cfg::kStageBytes);
          issue_w(kb_begin + i, i);
          issue_a(kb_begin + i, i);
        }
      }
    }
  } else if (warp == 1) {
    tmem_alloc<1>(tmem_slot, Cfg::kTmemCols);
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_launch_dependents();
  if (threadIdx.x == 0) SWIGLU_TRACE_POINT(1);

  if (live) {
    if (warp == 0 && lane == 0) {
      // ================================================================ TMA producer (rest)
      int s = 0;
      uint32_t ph = 1;  // the first kStages blocks went out above; now on the ring's second lap
      for (int kb = kb_begin + kStages; kb < kb_end; ++kb) {
        mbar_wait(empty_bar(s), ph ^ 1u);
        mbar_arrive_expect_tx(full_bar(s), Cfg::kStageBytes);
        issue_w(kb, s);
        issue_a(kb, s);
        if (++s == kStages) { s = 0; ph ^= 1u; }
      }
    } else if (warp == 1 && lane == 0) {
      // ================================================================ MMA issuer
      constexpr uint32_t idesc = kF8 ? idesc_e4m3_f32(128, MP)
                                     : idesc_bf16_f32(128, MP, /*a_mn=*/!kWK, /*b_mn=*/false);
      int s = 0;
      uint32_t ph = 0;
      for (int kb = kb_begin; kb < kb_end; ++kb) {
        mbar_wait(full_bar(s), ph);
        if (kb == kb_begin) SWIGLU_TRACE_POINT(3);
        tcgen05_fence_after();
        const uint32_t sw = smem_w(s);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k) {
          const uint32_t acc = (kb > kb_begin || k > 0) ? 1u : 0u;
          // W tiles as the 128-row "A" operand.  [K,N] weights: MN-major, 16 k rows = 2 KB per
          // step, the two 64-column atoms 8 KB apart (Gate at +0, Up at +16 KB).  Packed: the
          // atoms g0, g1 are 16 KB apart (u0 sits between them), Up starts at +8 KB.
          // [N,K] weights: K-major, +32 B per step, the two 64-row slabs are contiguous.
          if constexpr (kStack) {
            // stacked operand: rows 0-63 = the W1 slab, rows 64-127 = the W2 slab 8 KB behind it
            // (MN-major: the second 64-element atom; K-major: the next 64 rows)
            const uint64_t wd = kWK ? smem_desc_sw128(sw + k * (UMMA_K * 2), 16, 1024)
                                    : smem_desc_sw128(sw + k * (UMMA_K * 128), 8192, 1024);
            const uint64_t ad = smem_desc_sw128(smem_act(s) + k * (UMMA_K * 2), 16, 1024);
            if constexpr (kF8) umma_f8<1>(tmem_base, wd, ad, idesc, acc);
            else umma_bf16<1>(tmem_base, wd, ad, idesc, acc);  // lanes 0-63 Gate^T, 64-127 Up^T
            continue;
          }
          uint64_t w1d, w2d;
          if constexpr (kWK) {
            w1d = smem_desc_sw128(sw + k * (UMMA_K * 2), 16, 1024);
            w2d = smem_desc_sw128(sw + 16384 + k * (UMMA_K * 2), 16, 1024);
          } else if constexpr (kPacked) {
            w1d = smem_desc_sw128(sw + k * (UMMA_K * 128), 16384, 1024);
            w2d = smem_desc_sw128(sw + 8192 + k * (UMMA_K * 128), 16384, 1024);
          } else {
            w1d = smem_desc_sw128(sw + k * (UMMA_K * 128), 8192, 1024);
            w2d = smem_desc_sw128(sw + 16384 + k * (UMMA_K * 128), 8192, 1024);
          }
          // activations: K-major "B" operand, +32 B per step inside the swizzle row
          const uint64_t ad = smem_desc_sw128(smem_act(s) + k * (UMMA_K * 2), 16, 1024);
          if constexpr (kF8) {
            umma_f8<1>(tmem_base, w1d, ad, idesc, acc);
            umma_f8<1>(tmem_base + MP, w2d, ad, idesc, acc);
          } else {
            umma_bf16<1>(tmem_base, w1d, ad, idesc, acc);       // Gate^T -> columns [0, MP)
            umma_bf16<1>(tmem_base + MP, w2d, ad, idesc, acc);  // Up^T   -> columns [MP, 2MP)
          }
        }
        umma_commit<1>(empty_bar(s));
        if (++s == kStages) { s = 0; ph ^= 1u; }
      }
      umma_commit<1>(acc_full_bar);
      SWIGLU_TRACE_POINT(4);
    }

    // ================================================================ epilogue
    // 1. park this CTA's partial Gate^T / Up^T (fp32 [2][MP][128], n contiguous) in the drained ring
    const uint32_t part = smem_base;
    if (warp >= 2) {
      const uint32_t q = warp & 3u;
      const uint32_t nl = q * 32u + lane;  // local output column = TMEM lane
      const bool have = kb_end > kb_begin;
      if (have) {
        mbar_wait(acc_full_bar, 0);
        tcgen05_fence_after();
      }
      if (threadIdx.x == 64) SWIGLU_TRACE_POINT(5);
      const uint32_t tacc = tmem_base + ((q * 32u) << 16);
#pragma unroll
      for (int c = 0; c < MP / 16; ++c) {
        if (c * 16 >= p.M) break;  // rows >= M are never read back
        uint32_t g[16], u[16];
        if constexpr (kStack) {
          // lanes 0-63 hold Gate^T, lanes 64-127 Up^T of columns n = nl % 64
          if (have) {
            tmem_ld_32x32b_x16(tacc + c * 16, g);
            tmem_ld_wait();
          } else {
#pragma unroll
            for (int j = 0; j < 16; ++j) g[j] = 0u;
          }
          const uint32_t row0 = (q >> 1) * MP + c * 16, col = nl & 63u;
#pragma unroll
          for (int j = 0; j < 16; ++j)
            asm volatile("st.shared.b32 [%0], %1;" ::"r"(part + ((row0 + j) * 64u + col) * 4u), "r"(g[j])
                         : "memory");
          continue;
        }
        if (have) {
          tmem_ld_32x32b_x16(tacc + c * 16, g);
          tmem_ld_32x32b_x16(tacc + MP + c * 16, u);
          tmem_ld_wait();
        } else {
#pragma unroll
          for (int j = 0; j < 16; ++j) g[j] = u[j] = 0u;  // this rank got no k-blocks
        }
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int m = c * 16 + j;
          asm volatile("st.shared.b32 [%0], %1;" ::"r"(part + (uint32_t)(m * 128 + nl) * 4u),
                       "r"(g[j]) : "memory");
          asm volatile("st.shared.b32 [%0], %1;" ::"r"(part + (uint32_t)((MP + m) * 128 + nl) * 4u),
                       "r"(u[j]) : "memory");
        }
      }
      tcgen05_fence_before();
    }
    // 2. all partials of the cluster are in place
    if (S > 1) {
      __syncwarp();
      cluster_sync();
    } else {
      __syncthreads();
    }
    if (threadIdx.x == 64) SWIGLU_TRACE_POINT(6);
    // 3. rank r reduces rows m = r, r+S, ... over all peers (fixed rank order), SiLU-mul, store.
    //    Two rows per pass, so that 4S remote float4 loads share one DSMEM round trip.
    if (warp >= 2) {
      pdl_wait_prior_grid();  // Y may still be being written by the previous kernel in the stream
      const uint32_t et = threadIdx.x - 64u;
      constexpr uint32_t kColThreads = kTileN / 4, kRowSlots = 128 / kColThreads;
      const uint32_t c4 = (et % kColThreads) * 4u;  // 4 consecutive output columns per thread
      const uint32_t sub = et / kColThreads;        // 4 (stacked tile: 8) row slots
      const int n = n_base + (int)c4;
      uint32_t peer[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) peer[r] = (r < S) ? mapa_shared(part, (uint32_t)r) : 0u;
      auto finish_row = [&](int m, float4 gs, float4 us) {
        if constexpr (kF8) {  // dequantise: one scale per projection
          gs.x *= p.scale_gate; gs.y *= p.scale_gate; gs.z *= p.scale_gate; gs.w *= p.scale_gate;
          us.x *= p.scale_up; us.y *= p.scale_up; us.z *= p.scale_up; us.w *= p.scale_up;
        }
        if (n < p.N) {  // N % 8 == 0 and n % 4 == 0: the 4 columns are in range together
          if constexpr (kStoreGU) {
            *reinterpret_cast<uint2*>(Y + (long long)m * p.ldy + n) =
                make_uint2(pack_bf16x2_rn(gs.x, gs.y), pack_bf16x2_rn(gs.z, gs.w));
            *reinterpret_cast<uint2*>(p.U + (long long)m * p.ldy + n) =
                make_uint2(pack_bf16x2_rn(us.x, us.y), pack_bf16x2_rn(us.z, us.w));
          } else {
            const uint32_t lo = pack_bf16x2_rn(glu_mul<kAct>(gs.x, us.x), glu_mul<kAct>(gs.y, us.y));
            const uint32_t hi = pack_bf16x2_rn(glu_mul<kAct>(gs.z, us.z), glu_mul<kAct>(gs.w, us.w));
            *reinterpret_cast<uint2*>(Y + (long long)m * p.ldy + n) = make_uint2(lo, hi);
          }
        }
      };
      auto add4 = [](float4& a, const float4& b) { a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; };
      for (int m0 = (int)rank + S * (int)sub; m0 < p.M; m0 += 2 * (int)kRowSlots * S) {
        const int m1 = m0 + (int)kRowSlots * S;
        const bool two = m1 < p.M;
        float4 g0[8], u0[8], g1[8], u1[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          if (r < S) {
            g0[r] = ld_dsmem_v4(peer[r] + (uint32_t)(m0 * kTileN + (int)c4) * 4u);
            u0[r] = ld_dsmem_v4(peer[r] + (uint32_t)((MP + m0) * kTileN + (int)c4) * 4u);
            if (two) {
              g1[r] = ld_dsmem_v4(peer[r] + (uint32_t)(m1 * kTileN + (int)c4) * 4u);
              u1[r] = ld_dsmem_v4(peer[r] + (uint32_t)((MP + m1) * kTileN + (int)c4) * 4u);
            }
          }
        }
        float4 gs = g0[0], us = u0[0];
#pragma unroll
        for (int r = 1; r < 8; ++r)
          if (r < S) { add4(gs, g0[r]); add4(us, u0[r]); }
        finish_row(m0, gs, us);
        if (two) {
          gs = g1[0]; us = u1[0];
#pragma unroll
          for (int r = 1; r < 8; ++r)
            if (r < S) { add4(gs, g1[r]); add4(us, u1[r]); }
          finish_row(m1, gs, us);
        }
      }
    }
    if (threadIdx.x == 64) SWIGLU_TRACE_POINT(7);
    if (S > 1) {
      // peers may still be reading this CTA's partials: wait for all of them.  Nothing is
      // published here (Y needs no ordering inside the cluster), so the arrival is relaxed: a
      // release would first wait for this thread's Y stores to reach L2.
      __syncwarp();
      cluster_arrive_relaxed();
      cluster_wait_acquire();
    } else {
      __syncthreads();
    }
  } else {
    // launch-floor probe: same grid, cluster, shared memory, barriers and TMEM, nothing else;
    // still ordered after the previous kernel like the real one
    pdl_wait_prior_grid();
    __syncthreads();
  }
  if (warp == 1) {
    tcgen05_fence_after();
    tmem_dealloc<1>(tmem_base, Cfg::kTmemCols);
  }
  if (threadIdx.x == 0) SWIGLU_TRACE_POINT(8);
  if (clk_probe) {
    p.clk[0] = (unsigned long long)(clock64() - clk_c0);
    p.clk[1] = globaltimer_ns() - clk_t0;
  }
}

// ---------------------------------------------------------------------------------------
// One-time weight prepack (Kernel-2's "one-time preprocessing
// step" that interleaves W1 and W2; here at 64-column slab granularity, the unit a 128-byte
// swizzled TMA box and a UMMA operand atom share).
//   Wp[t][s][k][c], t = n-tile of 128 columns, s in {g0,u0,g1,u1}, k < Kp, c < 64:
//     = W{1 if s even else 2}[k][128 t + 64 (s >> 1) + c]      (0 beyond column N or row K)
//   Kp = K + 8 or 16 padding rows per slab (an odd number of KiB between slabs: address spread).
// Index work only: each output element is a copy of one input element.
// ---------------------------------------------------------------------------------------
template <bool kWK>
__global__ void __launch_bounds__(256)
pack_weights_kernel(const uint16_t* __restrict__ W1, const uint16_t* __restrict__ W2,
                    uint16_t* __restrict__ Wp, int N, int K, int Kp, long long total_vec) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < total_vec; v += stride) {
    // v indexes 8-element (16-byte) groups of Wp: [slab][k][c8], c8 < 8
    const int c8 = (int)(v & 7);
    const long long row = v >> 3;
    const int k = (int)(row % Kp);
    const long long slab = row / Kp;
    const int s = (int)(slab & 3);
    const int n = (int)(slab >> 2) * 128 + (s >> 1) * 64 + c8 * 8;
    const uint16_t* W = (s & 1) ? W2 : W1;
    uint4 out = make_uint4(0u, 0u, 0u, 0u);
    if (n < N && k < K) {  // N % 8 == 0: the 8 columns are in range together
      if constexpr (!kWK) {
        out = __ldg(reinterpret_cast<const uint4*>(W + (long long)k * N + n));
      } else {
        uint16_t e[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) e[j] = __ldg(W + (long long)(n + j) * K + k);
        out = make_uint4(e[0] | (uint32_t)e[1] << 16, e[2] | (uint32_t)e[3] << 16,
                         e[4] | (uint32_t)e[5] << 16, e[6] | (uint32_t)e[7] << 16);
      }
    }
    reinterpret_cast<uint4*>(Wp)[v] = out;
  }
}

}  // namespace swiglu
