// smallm_swiglu_kernel.cuh -- decode-sized batches (M <= 64): weight streaming is the whole
// cost (bytes ~ 4*K*N, AI ~ M FLOP/B), so the kernel is built around HBM, not the tensor pipe.
//
//  * swap-AB: the 128-row UMMA operand is a W tile (128 output columns n, MN-major as W is
//    [K,N] row-major), the narrow UMMA-N operand is A (MP = 16/32/64 padded tokens, K-major).
//    Accumulators are Gate^T and Up^T: TMEM lane = n, column = m.  All 128 epilogue threads
//    have work even at M = 1.
//  * split-K over a thread-block cluster: the S CTAs of a cluster share one 128-column tile
//    and each streams 1/S of K, so ~150-300 CTAs stream equal bytes whatever N/128 is.
//    SiLU is non-linear, so partial Gate/Up sums are reduced BEFORE the activation: each CTA
//    parks its fp32 partials in its own shared memory, and after a cluster barrier CTA r sums
//    rows m = r, r+S, ... over all peers through distributed shared memory in rank order
//    (deterministic), applies SiLU-multiply and stores bf16.  No global workspace, Gate/Up
//    never reach HBM (BASELINE.json north_star "Small M").
//  * two CTAs per SM, 3-stage TMA ring each (~200 KB of loads in flight per SM).
#pragma once
#include <cuda.h>

#include "gemm_swiglu_kernel.cuh"

namespace swiglu {

constexpr int kSmallMMax = 64;
constexpr int kSmallThreads = 192;  // warp 0 TMA, warp 1 MMA, warps 2-5 epilogue

template <int MP>
struct SmallCfg {
  static constexpr int kStages = (MP <= 32) ? 3 : 2;
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
  long long ldy;      // = N
};

__device__ __forceinline__ float ld_dsmem_f32(uint32_t cluster_addr) {
  float v;
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(cluster_addr) : "memory");
  return v;
}

template <int MP>
__global__ void __launch_bounds__(kSmallThreads, 2)
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

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmap_a);
    prefetch_tensormap(&tmap_w1);
    prefetch_tensormap(&tmap_w2);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    mbar_init(acc_full_bar, 1);
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc<1>(tmem_slot, Cfg::kTmemCols);
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  pdl_wait_prior_grid();
  pdl_launch_dependents();

  if (warp == 0 && lane == 0) {
    // ================================================================ TMA producer
    int s = 0;
    uint32_t ph = 0;
    for (int kb = kb_begin; kb < kb_end; ++kb) {
      mbar_wait(empty_bar(s), ph ^ 1u);
      const uint32_t fb = full_bar(s);
      mbar_arrive_expect_tx(fb, Cfg::kStageBytes);
      const int k0 = kb * BK;
      // weights are read exactly once per call: do not let them push A out of L2
      tma_load_2d(smem_w1(s), &tmap_w1, fb, n_base, k0, kEvictFirst);
      tma_load_2d(smem_w1(s) + 8192, &tmap_w1, fb, n_base + 64, k0, kEvictFirst);
      tma_load_2d(smem_w2(s), &tmap_w2, fb, n_base, k0, kEvictFirst);
      tma_load_2d(smem_w2(s) + 8192, &tmap_w2, fb, n_base + 64, k0, kEvictFirst);
      tma_load_2d(smem_act(s), &tmap_a, fb, k0, 0, kEvictLast);
      if (++s == kStages) { s = 0; ph ^= 1u; }
    }
  } else if (warp == 1 && lane == 0) {
    // ================================================================ MMA issuer
    constexpr uint32_t idesc = idesc_bf16_f32(128, MP, /*a_mn=*/true, /*b_mn=*/false);
    int s = 0;
    uint32_t ph = 0;
    for (int kb = kb_begin; kb < kb_end; ++kb) {
      mbar_wait(full_bar(s), ph);
      tcgen05_fence_after();
#pragma unroll
      for (int k = 0; k < BK / UMMA_K; ++k) {
        const uint32_t acc = (kb > kb_begin || k > 0) ? 1u : 0u;
        // W tiles: MN-major "A" operand, 16 k rows = 2 KB per step, 64-column atoms 8 KB apart
        const uint64_t w1d = smem_desc_sw128(smem_w1(s) + k * (UMMA_K * 128), 8192, 1024);
        const uint64_t w2d = smem_desc_sw128(smem_w2(s) + k * (UMMA_K * 128), 8192, 1024);
        // activations: K-major "B" operand, +32 B per step inside the swizzle row
        const uint64_t ad = smem_desc_sw128(smem_act(s) + k * (UMMA_K * 2), 16, 1024);
        umma_bf16<1>(tmem_base, w1d, ad, idesc, acc);       // Gate^T -> columns [0, MP)
        umma_bf16<1>(tmem_base + MP, w2d, ad, idesc, acc);  // Up^T   -> columns [MP, 2MP)
      }
      umma_commit<1>(empty_bar(s));
      if (++s == kStages) { s = 0; ph ^= 1u; }
    }
    umma_commit<1>(acc_full_bar);
  }

  // ================================================================ epilogue
  const uint32_t q = warp & 3u;
  const uint32_t nl = q * 32u + lane;  // local output column = TMEM lane
  const int n = n_base + (int)nl;
  const uint32_t part = smem_base;     // fp32 [2][MP][128], aliases the (drained) ring
  if (warp >= 2) {
    if (kb_end > kb_begin) {
      mbar_wait(acc_full_bar, 0);
      tcgen05_fence_after();
    }
    const uint32_t tacc = tmem_base + ((q * 32u) << 16);
#pragma unroll
    for (int c = 0; c < MP / 16; ++c) {
      uint32_t g[16], u[16];
      if (kb_end > kb_begin) {
        tmem_ld_32x32b_x16(tacc + c * 16, g);
        tmem_ld_32x32b_x16(tacc + MP + c * 16, u);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) g[j] = u[j] = 0u;  // this rank got no k-blocks
      }
      if (S == 1) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int m = c * 16 + j;
          if (m < p.M && n < p.N) {
            const float y = silu_mul(__uint_as_float(g[j]), __uint_as_float(u[j]));
            Y[(long long)m * p.ldy + n] = (uint16_t)(pack_bf16x2_rn(y, 0.f) & 0xFFFFu);
          }
        }
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int m = c * 16 + j;
          asm volatile("st.shared.b32 [%0], %1;" ::"r"(part + (uint32_t)(m * 128 + nl) * 4u),
                       "r"(g[j]) : "memory");
          asm volatile("st.shared.b32 [%0], %1;" ::"r"(part + (uint32_t)((MP + m) * 128 + nl) * 4u),
                       "r"(u[j]) : "memory");
        }
      }
    }
  }
  __syncwarp();
  if (S > 1) {
    cluster_sync();  // every CTA's partials are in its shared memory
    if (warp >= 2) {
      for (int m = (int)rank; m < p.M; m += S) {
        float gs = 0.f, us = 0.f;
        for (int r = 0; r < S; ++r) {  // fixed rank order: run-to-run deterministic
          gs += ld_dsmem_f32(mapa_shared(part + (uint32_t)(m * 128 + nl) * 4u, r));
          us += ld_dsmem_f32(mapa_shared(part + (uint32_t)((MP + m) * 128 + nl) * 4u, r));
        }
        if (n < p.N)
          Y[(long long)m * p.ldy + n] = (uint16_t)(pack_bf16x2_rn(silu_mul(gs, us), 0.f) & 0xFFFFu);
      }
    }
    __syncwarp();
    cluster_sync();  // peers may still be reading this CTA's partials
  }
  tcgen05_fence_before();
  __syncthreads();
  if (warp == 1) {
    tcgen05_fence_after();
    tmem_dealloc<1>(tmem_base, Cfg::kTmemCols);
  }
}

}  // namespace swiglu
