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
//    (deterministic; all 2S loads of a row are in flight together), applies SiLU-multiply and
//    stores bf16, 8 bytes per thread, 256 contiguous bytes per warp.  No global workspace,
//    Gate/Up never reach HBM (BASELINE.json north_star "Small M").
//  * fixed costs matter at these sizes (a call is 3-15 us): the producer thread initialises
//    its barriers and issues the first ring of TMA loads BEFORE the CTA-wide setup barrier
//    (TMEM allocation overlaps the HBM latency of the first loads), and warp 0 issues L2
//    prefetches for the CTA's weight blocks before griddepcontrol.wait, so under programmatic
//    dependent launch the weights start moving while the previous kernel drains.  A prefetch
//    is a hint: it cannot observe or produce stale data (L2 is the point of coherence).
#pragma once
#include <cuda.h>

#include "gemm_swiglu_kernel.cuh"

namespace swiglu {

constexpr int kSmallMMax = 128;
constexpr int kSmallThreads = 192;  // warp 0 TMA, warp 1 MMA, warps 2-5 epilogue
constexpr int kSmallPrefetchMax = 32;     // k-blocks per CTA prefetched to L2 (one per lane)

template <int MP>
struct SmallCfg {
  static constexpr int kCtasPerSm = (MP <= 64) ? 2 : 1;
  static constexpr int kStages = (MP <= 32) ? 3 : (MP == 64 ? 2 : 4);
  static constexpr int kWBytes = 128 * BK * 2;  // one W tile: 128 n x 64 k = 16 KB
  static constexpr int kABytes = MP * BK * 2;   // MP tokens x 64 k
  static constexpr int kStageBytes = 2 * kWBytes + kABytes;
  static constexpr int kPartialBytes = 2 * MP * 128 * 4;  // fp32 Gate^T|Up^T, aliases the ring
  static constexpr int kTmemCols = (2 * MP < 32) ? 32 : 2 * MP;
  static constexpr int kSmemBytes = kStages * kStageBytes + 256 + 1024;
  static_assert(kPartialBytes <= kStages * kStageBytes, "partials must fit in the ring");
};

struct SmallParams {
  int M, N, K;
  int ksplit;         // cluster size S
  int prefetch_blocks;  // leading k-blocks of each CTA's weight stream to prefetch into L2
  long long ldy;      // = N
  uint16_t* U;        // kStoreGU only: bf16 Up output (Gate goes to the Y argument)
  unsigned long long* clk;  // optional {SM cycles, globaltimer ns} of CTA 0 (swiglu_set_clock_probe)
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
template <int MP, int kAct = kActSilu, bool kWK = false, bool kStoreGU = false>
__global__ void __launch_bounds__(kSmallThreads, SmallCfg<MP>::kCtasPerSm)
smallm_swiglu_kernel(const __grid_constant__ CUtensorMap tmap_a,
                     const __grid_constant__ CUtensorMap tmap_w1,
                     const __grid_constant__ CUtensorMap tmap_w2, uint16_t* __restrict__ Y,
                     const SmallParams p) {
  using Cfg = SmallCfg<MP>;
  constexpr int kStages = Cfg::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + kStages * Cfg::kStageBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
  const uint32_t acc_full_bar = bar_base + 8u * (2 * kStages);
  const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 1);
  auto smem_w1 = [&](int s) { return smem_base + s * Cfg::kStageBytes; };
  auto smem_w2 = [&](int s) { return smem_base + s * Cfg::kStageBytes + Cfg::kWBytes; };
  auto smem_act = [&](int s) { return smem_base + s * Cfg::kStageBytes + 2 * Cfg::kWBytes; };

  const uint32_t warp = threadIdx.x >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  const int S = p.ksplit;
  const uint32_t rank = (S > 1) ? cluster_ctarank() : 0u;
  const int n_tile = blockIdx.x / S;
  const int n_base = n_tile * 128;
  const int k_blocks = (p.K + BK - 1) / BK;
  const int kb_begin = (int)(((long long)k_blocks * rank) / S);
  const int kb_end = (int)(((long long)k_blocks * (rank + 1)) / S);

  auto issue_stage = [&](int kb, int s) {
    const uint32_t fb = full_bar(s);
    mbar_arrive_expect_tx(fb, Cfg::kStageBytes);
    const int k0 = kb * BK;
    // weights are read exactly once per call: do not let them push A out of L2
    // one 64-column x 64-k slab per load; inner tensor-map dimension is N ([K,N]) or K ([N,K])
    auto load_w = [&](uint32_t dst, const CUtensorMap* tm, int n) {
      tma_load_2d(dst, tm, fb, kWK ? k0 : n, kWK ? n : k0, kEvictFirst);
    };
    load_w(smem_w1(s), &tmap_w1, n_base);
    load_w(smem_w1(s) + 8192, &tmap_w1, n_base + 64);
    load_w(smem_w2(s), &tmap_w2, n_base);
    load_w(smem_w2(s) + 8192, &tmap_w2, n_base + 64);
    tma_load_2d(smem_act(s), &tmap_a, fb, k0, 0, kEvictLast);
  };

  if (threadIdx.x == 0) SWIGLU_TRACE_POINT(0);
  const bool clk_probe = p.clk != nullptr && blockIdx.x == 0 && threadIdx.x == 0;
  long long clk_c0 = 0;
  uint64_t clk_t0 = 0;
  if (clk_probe) { clk_c0 = clock64(); clk_t0 = globaltimer_ns(); }
  // ------------------------------------------------------------------ setup
  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tmap_w1);
      prefetch_tensormap(&tmap_w2);
      prefetch_tensormap(&tmap_a);
      for (int s = 0; s < kStages; ++s) {
        mbar_init(full_bar(s), 1);
        mbar_init(empty_bar(s), 1);
      }
      mbar_init(acc_full_bar, 1);
      fence_mbar_init();
      fence_proxy_async_all();
    }
    // L2 prefetch of this CTA's weight stream (hint; legal before griddepcontrol.wait)
    const int kb = kb_begin + (int)lane;
    if ((int)lane < p.prefetch_blocks && kb < kb_end) {
      const int k0 = kb * BK;
      tma_prefetch_l2_2d(&tmap_w1, kWK ? k0 : n_base, kWK ? n_base : k0);
      tma_prefetch_l2_2d(&tmap_w1, kWK ? k0 : n_base + 64, kWK ? n_base + 64 : k0);
      tma_prefetch_l2_2d(&tmap_w2, kWK ? k0 : n_base, kWK ? n_base : k0);
      tma_prefetch_l2_2d(&tmap_w2, kWK ? k0 : n_base + 64, kWK ? n_base + 64 : k0);
    }
    if (lane == 0) {
      // A may be the previous kernel's output: real loads only after the grid dependency
      pdl_wait_prior_grid();
      SWIGLU_TRACE_POINT(2);
      for (int i = 0; i < kStages && kb_begin + i < kb_end; ++i) issue_stage(kb_begin + i, i);
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

  if (warp == 0 && lane == 0) {
    // ================================================================ TMA producer (rest)
    int s = 0;
    uint32_t ph = 1;  // the first kStages blocks went out above; now on the ring's second lap
    for (int kb = kb_begin + kStages; kb < kb_end; ++kb) {
      mbar_wait(empty_bar(s), ph ^ 1u);
      issue_stage(kb, s);
      if (++s == kStages) { s = 0; ph ^= 1u; }
    }
  } else if (warp == 1 && lane == 0) {
    // ================================================================ MMA issuer
    constexpr uint32_t idesc = idesc_bf16_f32(128, MP, /*a_mn=*/!kWK, /*b_mn=*/false);
    int s = 0;
    uint32_t ph = 0;
    for (int kb = kb_begin; kb < kb_end; ++kb) {
      mbar_wait(full_bar(s), ph);
      if (kb == kb_begin) SWIGLU_TRACE_POINT(3);
      tcgen05_fence_after();
#pragma unroll
      for (int k = 0; k < BK / UMMA_K; ++k) {
        const uint32_t acc = (kb > kb_begin || k > 0) ? 1u : 0u;
        // W tiles: MN-major "A" operand, 16 k rows = 2 KB per step, 64-column atoms 8 KB apart
        // ([N,K] weights: K-major, +32 B per step, the two 64-row slabs are contiguous)
        const uint64_t w1d = kWK ? smem_desc_sw128(smem_w1(s) + k * (UMMA_K * 2), 16, 1024)
                                 : smem_desc_sw128(smem_w1(s) + k * (UMMA_K * 128), 8192, 1024);
        const uint64_t w2d = kWK ? smem_desc_sw128(smem_w2(s) + k * (UMMA_K * 2), 16, 1024)
                                 : smem_desc_sw128(smem_w2(s) + k * (UMMA_K * 128), 8192, 1024);
        // activations: K-major "B" operand, +32 B per step inside the swizzle row
        const uint64_t ad = smem_desc_sw128(smem_act(s) + k * (UMMA_K * 2), 16, 1024);
        umma_bf16<1>(tmem_base, w1d, ad, idesc, acc);       // Gate^T -> columns [0, MP)
        umma_bf16<1>(tmem_base + MP, w2d, ad, idesc, acc);  // Up^T   -> columns [MP, 2MP)
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
  // 3. rank r reduces rows m = r, r+S, ... over all peers (fixed rank order), SiLU-mul, store
  if (warp >= 2) {
    pdl_wait_prior_grid();  // Y may still be being written by the previous kernel in the stream
    const uint32_t et = threadIdx.x - 64u;
    const uint32_t c4 = (et & 31u) * 4u;  // 4 consecutive output columns per thread
    const uint32_t sub = et >> 5;         // 4 rows in flight per pass
    const int n = n_base + (int)c4;
    uint32_t peer[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) peer[r] = (r < S) ? mapa_shared(part, (uint32_t)r) : 0u;
    for (int m = (int)rank + S * (int)sub; m < p.M; m += 4 * S) {
      const uint32_t goff = (uint32_t)(m * 128 + (int)c4) * 4u;
      const uint32_t uoff = (uint32_t)((MP + m) * 128 + (int)c4) * 4u;
      float4 g[8], u[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        if (r < S) {
          g[r] = ld_dsmem_v4(peer[r] + goff);
          u[r] = ld_dsmem_v4(peer[r] + uoff);
        }
      }
      float4 gs = g[0], us = u[0];
#pragma unroll
      for (int r = 1; r < 8; ++r) {
        if (r < S) {
          gs.x += g[r].x; gs.y += g[r].y; gs.z += g[r].z; gs.w += g[r].w;
          us.x += u[r].x; us.y += u[r].y; us.z += u[r].z; us.w += u[r].w;
        }
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
    }
  }
  if (threadIdx.x == 64) SWIGLU_TRACE_POINT(7);
  if (S > 1) {
    __syncwarp();
    cluster_sync();  // peers may still be reading this CTA's partials
  } else {
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

}  // namespace swiglu
