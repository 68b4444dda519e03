// gemm_swiglu_kernel.cuh -- the large-M kernel: persistent, warp-specialised, TMA ->
// smem ring -> tcgen05.mma -> TMEM (double-buffered) -> epilogue -> TMA store.
//
// kFused = true : Y[m, n] = bf16( SiLU(A.W1)[m,n] * (A.W2)[m,n] )      (Eq. 1-3)
//   One UMMA of N = 256 per k-step covers the W1 tile (TMEM columns [0,128) = Gate) and the
//   W2 tile (columns [128,256) = Up) of the same 128 output columns: the tile-level form of
//   the paper's Kernel-2 "[M,2N]" pairing with no interleaved
//   weight copy, and of Kernel-1's "both accumulators in one threadblock" (lines 130-139)
//   with A streamed once instead of twice.  SiLU-multiply of tile i runs in the epilogue
//   warps while the MMA warp accumulates tile i+1 into the other TMEM stage -- the sm_100
//   counterpart of the paper's Swish-under-loads / SwiGLU-under-stores overlaps (lines 128,
//   165).
// kFused = false: C[m, n] = bf16( (A.W)[m,n] ), a plain GEMM with 256-column tiles; used
//   twice (Gate, Up) by the unfused comparison path.
//
// kCtaGroup = 1: one CTA per 128-row tile.  kCtaGroup = 2: a CTA pair (cluster 2x1) shares one
//   256-row tile; each CTA loads its 128 rows of A and HALF of the B columns (fused: rank 0
//   loads the W1 tile, rank 1 the W2 tile), the leader issues cta_group::2 MMAs.
#pragma once
#include <cuda.h>

#include "sm100_ptx.cuh"

namespace swiglu {

using namespace sm100;

constexpr int BM = 128;      // rows of A / Y per CTA
constexpr int BK = 64;       // k per pipeline stage: 64 bf16 = one 128-byte swizzle row
constexpr int UMMA_K = 16;   // k per tcgen05.mma (kind::f16)
// Eight epilogue warps: two per TMEM lane quarter (a warp may only read lanes 32*(warp%4)..+31).
// Of every 64-column output chunk, warps 2-5 take columns [0,32) and warps 6-9 columns [32,64):
// two warps per SM sub-partition hide each other's TMEM-load / MUFU latencies, which halves the
// drain time of a tile (3.6 -> 1.8 us per 128x128 tile) wherever it is exposed: one tile per CTA
// near the ridge, the last tile of every call, FP8 at small K.
constexpr int kEpiWarps = 8;
constexpr int kGemmThreads = 64 + 32 * kEpiWarps;  // warp 0 TMA, warp 1 MMA, warps 2-9 epilogue
constexpr int kOutBufBytes = BM * 64 * 2;          // one 64-column bf16 output chunk (16 KB)
constexpr int kQuarterBufBytes = 32 * 64 * 2;      // ... of which each TMEM lane quarter stages 32 rows (4 KB)

// kUmmaN = accumulator columns per tile: 256 (fused: Gate 128 | Up 128; unfused: 256 plain
// columns) or, for the narrow fused tile used when N/128 tiles cannot fill the GPU,
// 128 (Gate 64 | Up 64).
template <int kCtaGroup, int kUmmaN = 256, int kMB = 1>
struct GemmCfg {
  static constexpr int kBColsPerCta = kUmmaN / kCtaGroup;
  static constexpr int kABytes = kMB * BM * BK * 2;      // 16 KB per 128-row block of A
  static constexpr int kBBytes = kBColsPerCta * BK * 2;  // 32 KB (1-CTA) / 16 KB (2-CTA, narrow)
  static constexpr int kStageBytes = kABytes + kBBytes;
  static constexpr int kStages = (kStageBytes >= 48 * 1024) ? 4 : 6;
  static constexpr int kTmemCols = 2 * kUmmaN;           // 2 accumulator stages (kMB = 2: 2 row blocks)
  static constexpr int kBarBytes = 1024;
  // +1024: slack to align the dynamic smem base to 1024 B (128-byte swizzle atoms)
  static constexpr int kSmemBytes = kStages * kStageBytes + 2 * kOutBufBytes + kBarBytes + 1024;
};

struct GemmParams {
  int M, N, K;
  int m_tiles;   // ceil(M / (128*kCtaGroup))
  int n_tiles;   // ceil(N / (fused ? 128 : 256))
  int group_m;   // m-tiles per L2 raster group
  int wide_tiles;   // tiles [0, wide_tiles) are whole (full width, all of K); the rest -- the last
                    // partial wave -- are cut into units: tail_ksplit K-ranges each (tail_ksplit
                    // >= 2), or two 64-column half tiles (tail_ksplit == 0)
  int total_tiles;  // schedule slots: wide_tiles + units of the cut tiles
  int tail_ksplit;  // s: K-ranges per tile of the last wave (0 = no K split)
  int skew;         // kMB = 2: k-blocks row block 0 runs ahead of block 1 at tile boundaries
  int tail_div;     // kMB = 2: units per super tile of the last partial wave (1, 2 or 4)
  float* split_ws;  // [tail tile][CTA of the group][s][256 columns / 4][128 rows] float4 partials
  int* split_ctr;   // [tail tile][CTA of the group] arrival counters, zero between launches
  int early_issue;      // 1: fill the ring before the CTA-wide setup barrier (small grids)
  int early_prefetch;   // ... after an L2 prefetch of this many weight k-blocks ahead of griddepcontrol.wait
  unsigned long long w_policy, a_policy;  // L2 eviction-priority hints of the weight / A loads
  unsigned long long y_policy;            // ... and of the Y stores
  unsigned long long* clk;  // optional {SM cycles, globaltimer ns} of CTA 0 (swiglu_set_clock_probe)
  float scale_gate, scale_up;  // kOperandsFp8: Gate / Up dequantisation scales (else unused)
#ifdef SWIGLU_TRACE
  unsigned long long* trace;  // [grid][kGemmTraceStride] globaltimer stamps (debug builds only)
#endif
};

// Debug-build timeline stamps (compiled out unless -DSWIGLU_TRACE): slot i of this CTA.
// Per tile (8 slots): MMA thread 0-2 (+5, 6 in the super-tile kernel), epilogue 3, 4 (7: second
// region); in the 256-row kernels slots 5-7 time chunk SWIGLU_TRACE_H of the epilogue (after the
// first barrier / the TMEM loads / the second barrier).
#ifndef SWIGLU_TRACE_H
#define SWIGLU_TRACE_H 0
#endif
constexpr int kGemmTraceStride = 8 + 8 * 32;
#ifdef SWIGLU_TRACE
#define SWIGLU_TRACE_POINT(i)                                                         \
  do {                                                                                \
    if (p.trace) p.trace[(size_t)blockIdx.x * 16 + (i)] = globaltimer_ns();           \
  } while (0)
#define SWIGLU_GEMM_TRACE(i)                                                          \
  do {                                                                                \
    if (p.trace && (i) < kGemmTraceStride)                                            \
      p.trace[(size_t)blockIdx.x * kGemmTraceStride + (i)] = globaltimer_ns();        \
  } while (0)
#else
#define SWIGLU_TRACE_POINT(i) do { } while (0)
#define SWIGLU_GEMM_TRACE(i) do { } while (0)
#endif

// Tile order: groups of `group_m` row-tiles x all column-tiles, row-tile fastest inside a
// group, so the CTAs running at one time share a slab of A that stays in L2 and stream W.
__device__ __forceinline__ void decode_tile(const GemmParams& p, int t, int& tm, int& tn) {
  const int per_group = p.group_m * p.n_tiles;
  const int g = t / per_group;
  const int r = t - g * per_group;
  const int m0 = g * p.group_m;
  const int gm = min(p.group_m, p.m_tiles - m0);
  tn = r / gm;
  tm = m0 + (r - tn * gm);
}

// 1 / x for 1 <= x <= 2^126 on the FMA pipe: exponent-flip seed (|error| <= 5 %) and two Newton
// steps, relative error <= 7e-6 (fp32 arithmetic; the bf16 result keeps 8 bits).  The epilogue of
// a tile is MUFU-bound (16 lanes per clock per SM against 128 FMA lanes): taking the reciprocal off
// the MUFU pipe halves its MUFU work.
__device__ __forceinline__ float rcp_ge1_fma(float x) {
  float r = __int_as_float(0x7EF31000 - __float_as_int(x));
  r = r * fmaf(-x, r, 2.0f);
  return r * fmaf(-x, r, 2.0f);
}
// sigma(z) * p = p / (1 + 2^(-z*log2 e)), one MUFU (ex2).  The exponent is capped at 126 so that
// 1 + e stays finite for any z (the result is then ~1e-38 * p: zero for every purpose here).
__device__ __forceinline__ float sigmoid_mul(float z, float p) {
  float e;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(fminf(z * -1.4426950408889634f, 126.0f)));
  return p * rcp_ge1_fma(1.0f + e);
}
__device__ __forceinline__ float silu_mul(float g, float u) {
  // SiLU(g)*u = g*u / (1 + 2^(-g*log2 e)); fp32 throughout.
  return sigmoid_mul(g, g * u);
}

// Tile t of the schedule -> (row tile, first output column, width in output columns).
// The last partial wave of a fused 128-column schedule may be cut into 64-column half tiles
// (two consecutive schedule slots per wide tile), so that it occupies all SMs for half a
// tile time instead of half the SMs for a whole one (a1: wave quantisation).
template <int kOutCols>
__device__ __forceinline__ void decode_tile_w(const GemmParams& p, int t, int& tm, int& n_base,
                                              int& w) {
  int tn;
  if (t < p.wide_tiles) {
    decode_tile(p, t, tm, tn);
    n_base = tn * kOutCols;
    w = kOutCols;
  } else {
    const int j = t - p.wide_tiles;
    decode_tile(p, p.wide_tiles + (j >> 1), tm, tn);
    n_base = tn * kOutCols + (j & 1) * 64;
    w = 64;
  }
}

// One schedule slot: which tile, which columns, which k-blocks.  tail >= 0: a K-range unit of
// tail tile `tail` (rank `krank` of p.tail_ksplit), whose fp32 partial accumulators are combined
// through p.split_ws by the last unit of that tile to arrive (a1: the stream-K treatment of the
// last partial wave -- idle CTA groups take K-ranges of the tail tiles
// discuss the wave quantisation this removes).
struct TileUnit {
  int tm, n_base, w, kb0, kb1, tail, krank;
  int mb0, nmb;  // kMB = 2: first 256-row block of the super tile this unit covers, and how many
};
template <int kOutCols, int kMB = 1>
__device__ __forceinline__ TileUnit decode_unit(const GemmParams& p, int t, int k_blocks) {
  TileUnit u;
  u.kb0 = 0; u.kb1 = k_blocks; u.tail = -1; u.krank = 0; u.mb0 = 0; u.nmb = 1;
  if constexpr (kMB == 2) {
    // Super tiles (two row blocks); the last partial wave is cut into p.tail_div units per
    // tile: 2 = its two row blocks, 4 = row blocks x 64-column halves, each run by one CTA pair
    // with a single accumulator region.  A super tile whose second block lies beyond M (ragged
    // M) is run as one block.
    int tn;
    if (t < p.wide_tiles) {
      decode_tile(p, t, u.tm, tn);
      u.n_base = tn * kOutCols;
      u.w = kOutCols;
      u.nmb = ((u.tm * 4 + 2) * BM < p.M) ? 2 : 1;
    } else {
      const int j = t - p.wide_tiles;
      const int tile = j / p.tail_div, sub = j - tile * p.tail_div;
      decode_tile(p, p.wide_tiles + tile, u.tm, tn);
      u.mb0 = sub & 1;
      u.w = (p.tail_div == 4) ? 64 : kOutCols;
      u.n_base = tn * kOutCols + ((p.tail_div == 4) ? (sub >> 1) * 64 : 0);
    }
    return u;
  }
  if (t >= p.wide_tiles && p.tail_ksplit >= 2) {
    const int idx = t - p.wide_tiles;
    u.tail = idx / p.tail_ksplit;
    u.krank = idx - u.tail * p.tail_ksplit;
    int tn;
    decode_tile(p, p.wide_tiles + u.tail, u.tm, tn);
    u.n_base = tn * kOutCols;
    u.w = kOutCols;
    u.kb0 = (int)(((long long)k_blocks * u.krank) / p.tail_ksplit);
    u.kb1 = (int)(((long long)k_blocks * (u.krank + 1)) / p.tail_ksplit);
  } else {
    decode_tile_w<kOutCols>(p, t, u.tm, u.n_base, u.w);
  }
  return u;
}

// Gate activations of the GLU family (include/swiglu_mlp.h swiglu_activation; PAPER.md line 56
// and line 392 item 4).  All in fp32 on the fp32 accumulators, like SiLU (line 370).
enum : int { kActSilu = 0, kActGelu = 1, kActGeluTanh = 2, kActRelu = 3, kNumActs = 4 };

template <int kAct>
__device__ __forceinline__ float glu_mul(float g, float u) {
  if constexpr (kAct == kActSilu) {
    return silu_mul(g, u);
  } else if constexpr (kAct == kActGeluTanh) {
    // 0.5 g (1 + tanh(c (g + 0.044715 g^3))) = g * sigma(2c (g + 0.044715 g^3)): the SiLU
    // form with a cubic argument -- no cancellation in the negative tail.
    const float z = g * fmaf(0.07135481627f, g * g, 1.5957691216f);  // 2c*0.044715, 2c
    return sigmoid_mul(z, g * u);
  } else if constexpr (kAct == kActGelu) {
    // g * Phi(g), Phi(g) = erfc(-g / sqrt 2) / 2.  erfc(t), t >= 0, from Abramowitz & Stegun
    // 7.1.26: (a1 k + ... + a5 k^5) exp(-t^2), k = 1 / (1 + 0.3275911 t), |error| <= 1.5e-7 --
    // fp32-epsilon level where Phi ~ 1, and |g u| * 1.5e-7 is far below the 2e-3 absolute
    // floor of the tolerance in the tail.  2 MUFU + ~10 FMA per element (libm erfcf is ~5x that
    // and does not hide under the next tile's MMAs).
    const float t = fabsf(g) * 0.70710678118654752f;
    float k, e;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(k) : "f"(fmaf(0.3275911f, t, 1.0f)));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(t * t * -1.4426950408889634f));
    float q = fmaf(1.061405429f, k, -1.453152027f);
    q = fmaf(q, k, 1.421413741f);
    q = fmaf(q, k, -0.284496736f);
    q = fmaf(q, k, 0.254829592f);
    q = 0.5f * (q * k) * e;                       // Phi(-|g|)
    const float phi = (g < 0.0f) ? q : 1.0f - q;  // Phi(g)
    return (g * u) * phi;
  } else {
    return fmaxf(g, 0.0f) * u;
  }
}

// Weight source (kWMode):
//   kWeightsKN: [K,N] row-major (N contiguous; the paper's layout) -- an
//     MN-major UMMA "B" operand.
//   kWeightsNK: [N,K] row-major (K contiguous, the nn.Linear layout serving stacks store, lines
//     72-74) -- a K-major operand.
//   Either way a 64-column slab of a weight tile is one 8 KB TMA box (64 x 64 bf16, 128-byte
//   swizzle) and the slabs W1[0:64) W1[64:128) W2[0:64) W2[64:128) sit 8 KB apart in smem.
//   kWeightsPacked: the tile-interleaved W_fused of swiglu_pack_weights (the sm_100 form of the
//     paper's Kernel-2 one-time interleave, lines 159, 167-169): slab-major
//     [n-tile][g0,u0,g1,u1][K][64], so ONE 3-D TMA box per stage fetches Gate|Up slabs
//     (tmap_b1: the multi-slab box; tmap_b2: a single-slab box for 2-CTA / 1-CTA half tiles).
//     MN-major like KN; accumulator columns come out as g0 u0 g1 u1.
//   kOperandsFp8: A [M,K] AND both weight matrices [N,K] are OCP FP8 E4M3 bytes (PAPER.md lines
//     382, 392 item 2): K-major operands, a k-block is 128 elements (the
//     same 128-byte rows, so every shared-memory size and descriptor stride is unchanged),
//     tcgen05.mma kind::f8f6f4 with 32 k per instruction, and the per-projection dequantisation
//     scales multiply the fp32 accumulators in the epilogue before the activation.
enum : int { kWeightsKN = 0, kWeightsNK = 1, kWeightsPacked = 2, kOperandsFp8 = 3 };

// kPairs = 2 (with kCtaGroup = 2): a cluster of FOUR CTAs = two CTA pairs working on two
//   vertically adjacent 256-row tiles of the SAME 128 output columns.  Both pairs need the same
//   W1|W2 tile: each CTA TMA-loads ONE 64-column slab of its matrix and MULTICASTS it to its
//   counterpart in the other pair, so every weight byte crosses L2 -> SM once per 512 rows
//   instead of once per 256 (a quarter less L2 -> SM traffic per FLOP, and the two pairs stay
//   in lock-step, which roughly halves the DRAM re-reads at the 72B shape:
//   profiles/r02_ncu_summary.md).  Smem-slot reuse is then gated on BOTH pairs' MMAs: the
//   tcgen05.commit that frees a stage arrives on all four CTAs' empty barriers.
//
// kMB = 2 (with kCtaGroup = 2, one pair per cluster): a 512-row x 128-column SUPER TILE per CTA
//   pair.  Each CTA stages TWO 128-row blocks of A per k-block (rows +0 and +256 of the tile) next
//   to its half of the W1|W2 tile, and the leader issues two M = 256 MMAs per k-step that share the
//   weight operand: accumulator region 0 (TMEM columns [0,256)) = rows [0,256) of the tile, region
//   1 (columns [256,512)) = rows [256,512).  Per FLOP a quarter less L2 -> SM traffic than the
//   256-row pair tile (96 KB instead of 128 KB per 512x128x64 block), on every SM and with no
//   cluster wider than the pair.  All of TMEM then belongs to ONE tile, so the epilogue is hidden
//   by SKEWING the row blocks at tile boundaries instead of by a second accumulator stage: the
//   last L k-blocks of a tile run "block 0 first" (region 0 is complete L k-blocks early and
//   drains under block 1's last MMAs) and the first L k-blocks of the next tile likewise (block
//   0's MMAs run while region 1 still drains).  L <= ring depth; in between the blocks interleave
//   so that the ring keeps its full prefetch depth.
template <int kCtaGroup, bool kFused, int kBN = 128, int kAct = kActSilu, int kWMode = kWeightsKN,
          int kPairs = 1, int kMB = 1>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_swiglu_kernel(const __grid_constant__ CUtensorMap tmap_a,
                   const __grid_constant__ CUtensorMap tmap_b1,
                   const __grid_constant__ CUtensorMap tmap_b2,
                   const __grid_constant__ CUtensorMap tmap_y, const GemmParams p) {
  static_assert(kBN == 128 || (kBN == 64 && kFused && kCtaGroup == 1), "narrow tile: fused 1-CTA");
  static_assert(kWMode != kWeightsPacked || kFused, "packed weights: fused path only");
  static_assert(kPairs == 1 || (kPairs == 2 && kCtaGroup == 2 && kFused && kBN == 128),
                "two pairs per cluster: fused 2-CTA 128-column tiles only");
  static_assert(kMB == 1 || (kMB == 2 && kCtaGroup == 2 && kBN == 128 && kPairs == 1),
                "two row blocks per CTA: 2-CTA tiles of 256 accumulator columns, one pair per cluster");
  constexpr int kClusterCtas = kCtaGroup * kPairs;
  static_assert(kWMode != kOperandsFp8 || kFused, "FP8 operands: fused path only");
  constexpr bool kF8 = (kWMode == kOperandsFp8);
  constexpr bool kWK = (kWMode == kWeightsNK) || kF8;
  constexpr bool kPacked = (kWMode == kWeightsPacked);
  constexpr int kBKe = kF8 ? 128 : BK;            // elements of k per stage (128-byte rows)
  constexpr int UMMA_N = kFused ? 2 * kBN : 256;  // accumulator columns per tile
  using Cfg = GemmCfg<kCtaGroup, UMMA_N, kMB>;
  constexpr int kStages = Cfg::kStages;
  constexpr int kTmemCols = Cfg::kTmemCols;
  constexpr int kOutCols = kFused ? kBN : 256;  // output columns per tile
  constexpr int kChunks = kOutCols / 64;        // 64-column epilogue chunks per tile

  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t smem_out = smem_base + kStages * Cfg::kStageBytes;
  const uint32_t bar_base = smem_out + 2 * kOutBufBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
  auto acc_full_bar = [&](int a) { return bar_base + 8u * (2 * kStages + a); };
  auto acc_empty_bar = [&](int a) { return bar_base + 8u * (2 * kStages + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 4);
  auto smem_a = [&](int s) { return smem_base + s * Cfg::kStageBytes; };
  auto smem_b = [&](int s) { return smem_base + s * Cfg::kStageBytes + Cfg::kABytes; };

  const uint32_t warp = threadIdx.x >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t crank = (kCtaGroup == 2) ? cluster_ctarank() : 0u;  // rank in the cluster
  const uint32_t rank = crank & 1u;                // rank in the CTA pair (0 = leader)
  const uint32_t pair = (kPairs == 2) ? crank >> 1 : 0u;
  const uint16_t pair_mask = (uint16_t)(0x3u << (2u * pair));        // this pair's two CTAs
  const uint16_t all_mask = (uint16_t)((1u << kClusterCtas) - 1u);   // every CTA of the cluster
  const int num_groups = gridDim.x / kClusterCtas;  // clusters (or lone CTAs) sharing the tile list
  const int group_id = blockIdx.x / kClusterCtas;
  const int total_tiles = p.total_tiles;
  const int k_blocks = (p.K + kBKe - 1) / kBKe;

  // (host: a single row of tiles reads every weight byte exactly once -> evict-first)
  const uint64_t w_policy = p.w_policy, a_policy = p.a_policy;
  // One k-block of A and B into ring slot s (no waiting here: the caller owns the ring state).
  // w = output columns of the tile (kOutCols, or 64 for a half tile of the last wave).
  auto issue_loads = [&](int s, int kb, int m_base, int n_base, int w, int nmb = kMB) {
    const bool half = kFused && kBN == 128 && w == 64;
    if (rank == 0) {
      const uint32_t b_bytes = half ? Cfg::kBBytes / 2 : Cfg::kBBytes;
      const uint32_t a_bytes = (kMB == 2 && nmb == 1) ? Cfg::kABytes / 2 : Cfg::kABytes;
      mbar_arrive_expect_tx(full_bar(s), (a_bytes + b_bytes) * kCtaGroup);
    }
    const int k0 = kb * kBKe;
    const uint32_t sa = smem_a(s), sb = smem_b(s), fb = full_bar(s);
    // one 64-column x 64-k weight slab; the tensor map's inner dimension is N ([K,N]) or K ([N,K])
    auto load_w = [&](uint32_t dst, const CUtensorMap* tm, int n) {
      if constexpr (kCtaGroup == 1) tma_load_2d(dst, tm, fb, kWK ? k0 : n, kWK ? n : k0, w_policy);
      else tma_load_2d_pair(dst, tm, fb, kWK ? k0 : n, kWK ? n : k0, w_policy);
    };
    if constexpr (kPacked) {
      // slab index of (n_base, Gate): tiles of 128 columns hold 4 slabs g0 u0 g1 u1
      const int slab = (n_base >> 7) * 4 + ((n_base >> 6) & 1) * 2;
      if constexpr (kCtaGroup == 1) {
        tma_load_2d(sa, &tmap_a, fb, k0, m_base, a_policy);
        if (half) {  // g_h | u_h as two single-slab boxes
          tma_load_3d(sb, &tmap_b2, fb, 0, k0, slab, w_policy);
          tma_load_3d(sb + 8192, &tmap_b2, fb, 0, k0, slab + 1, w_policy);
        } else {     // one box: 4 slabs (128-column tile) or 2 slabs (64-column tile)
          tma_load_3d(sb, &tmap_b1, fb, 0, k0, slab, w_policy);
        }
      } else {
        tma_load_2d_pair(sa, &tmap_a, fb, k0, m_base, a_policy);
        if (kMB == 2 && nmb == 2) tma_load_2d_pair(sa + BM * BK * 2, &tmap_a, fb, k0, m_base + 2 * BM, a_policy);
        if constexpr (kPairs == 2) {
          // this CTA needs slabs {2 rank, 2 rank + 1}; it fetches slab 2 rank + pair for itself
          // and its counterpart in the other pair
          tma_load_3d_pair_mc(sb + 8192u * pair, &tmap_b2, fb, 0, k0, slab + 2 * (int)rank + (int)pair,
                              (uint16_t)(0x5u << rank), w_policy);
        } else if (half) {
          tma_load_3d_pair(sb, &tmap_b2, fb, 0, k0, slab + (int)rank, w_policy);
        } else {
          tma_load_3d_pair(sb, &tmap_b1, fb, 0, k0, slab + 2 * (int)rank, w_policy);
        }
      }
    } else if constexpr (kCtaGroup == 1) {
      tma_load_2d(sa, &tmap_a, fb, k0, m_base, a_policy);
      if constexpr (kFused) {
        if (kBN == 64 || half) {  // W1 slab | W2 slab
          load_w(sb, &tmap_b1, n_base);
          load_w(sb + 8192, &tmap_b2, n_base);
        } else {                  // W1 slabs 0,1 | W2 slabs 0,1
          load_w(sb, &tmap_b1, n_base);
          load_w(sb + 8192, &tmap_b1, n_base + 64);
          load_w(sb + 16384, &tmap_b2, n_base);
          load_w(sb + 24576, &tmap_b2, n_base + 64);
        }
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) load_w(sb + j * 8192, &tmap_b1, n_base + j * 64);
      }
    } else {
      tma_load_2d_pair(sa, &tmap_a, fb, k0, m_base, a_policy);
      if (kMB == 2 && nmb == 2) tma_load_2d_pair(sa + BM * BK * 2, &tmap_a, fb, k0, m_base + 2 * BM, a_policy);
      if constexpr (kFused) {
        const CUtensorMap* tb = (rank == 0) ? &tmap_b1 : &tmap_b2;
        if constexpr (kPairs == 2) {
          // one 64-column slab of this CTA's matrix, for itself and its counterpart
          const int n = n_base + 64 * (int)pair;
          tma_load_2d_pair_mc(sb + 8192u * pair, tb, fb, kWK ? k0 : n, kWK ? n : k0,
                              (uint16_t)(0x5u << rank), w_policy);
        } else {
          load_w(sb, tb, n_base);
          if (!half) load_w(sb + 8192, tb, n_base + 64);
        }
      } else {
        const int nb = n_base + (int)rank * 128;
        load_w(sb, &tmap_b1, nb);
        load_w(sb + 8192, &tmap_b1, nb + 64);
      }
    }
  };
  int pre = 0;  // k-blocks of this CTA's first tile issued before the setup barrier

  // ------------------------------------------------------------------ one-time setup
  if (threadIdx.x == 0) SWIGLU_GEMM_TRACE(0);
  const bool clk_probe = p.clk != nullptr && blockIdx.x == 0 && threadIdx.x == 0;
  long long clk_c0 = 0;
  uint64_t clk_t0 = 0;
  if (clk_probe) { clk_c0 = clock64(); clk_t0 = globaltimer_ns(); }
  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tmap_a);
      prefetch_tensormap(&tmap_b1);
      if (kFused) prefetch_tensormap(&tmap_b2);
      prefetch_tensormap(&tmap_y);
      for (int s = 0; s < kStages; ++s) {
        mbar_init(full_bar(s), 1);
        mbar_init(empty_bar(s), kPairs);  // one commit per pair that reads (or fills) the slot
      }
      for (int a = 0; a < 2; ++a) {
        mbar_init(acc_full_bar(a), 1);
        mbar_init(acc_empty_bar(a), kEpiWarps * kCtaGroup);
      }
      fence_mbar_init();
      fence_proxy_async_all();
    }
    if constexpr (kCtaGroup == 1 && kFused) {
      if (lane == 0) {
        // The producer needs only the barriers it has just initialised: fill the ring before
        // the CTA-wide setup barrier so TMEM allocation overlaps the first loads' latency.
        if (p.early_issue && group_id < total_tiles) {  // (host: never with a K-split tail)
          int tm, n_base, w;
          decode_tile_w<kOutCols>(p, group_id, tm, n_base, w);
          if constexpr (kWMode == kWeightsKN) {
            // L2 prefetch (a hint) of the first few weight k-blocks ahead of the grid dependency,
            // as in the decode kernel: covers the start-up latency behind griddepcontrol.wait
            for (int kb = 0; kb < p.early_prefetch && kb < k_blocks; ++kb) {
              tma_prefetch_l2_2d(&tmap_b1, n_base, kb * BK);
              tma_prefetch_l2_2d(&tmap_b2, n_base, kb * BK);
              if (w == 128) {
                tma_prefetch_l2_2d(&tmap_b1, n_base + 64, kb * BK);
                tma_prefetch_l2_2d(&tmap_b2, n_base + 64, kb * BK);
              }
            }
          }
          pdl_wait_prior_grid();
          for (; pre < kStages && pre < k_blocks; ++pre)
            issue_loads(pre, pre, tm * BM, n_base, w);  // fresh ring: nothing to wait for
        }
      }
    }
  }
  if (warp == 1) tmem_alloc<kCtaGroup>(tmem_slot, kTmemCols);
  tcgen05_fence_before();
  if (kCtaGroup == 2) cluster_sync(); else __syncthreads();
  tcgen05_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // PDL: everything above overlapped the previous kernel's tail; its output (and, for the
  // unfused path, the Gate/Up it wrote) must be complete before we touch global memory.
  pdl_wait_prior_grid();
  pdl_launch_dependents();  // the next kernel may start its own prologue as SMs free up
  if (threadIdx.x == 0) SWIGLU_GEMM_TRACE(1);

  if (warp == 0 && lane == 0) {
    // ================================================================ TMA producer
    int s = (pre == kStages) ? 0 : pre;
    uint32_t ph = (pre == kStages) ? 1u : 0u;
    for (int t = group_id; t < total_tiles; t += num_groups) {
      const TileUnit u = decode_unit<kOutCols, kMB>(p, t, k_blocks);
      const int m_base = ((u.tm * kPairs * kMB + (int)pair + u.mb0) * kCtaGroup + (int)rank) * BM;
      for (int kb = (t == group_id) ? u.kb0 + pre : u.kb0; kb < u.kb1; ++kb) {
        mbar_wait(empty_bar(s), ph ^ 1u);
        issue_loads(s, kb, m_base, u.n_base, u.w, u.nmb);
        if (++s == kStages) { s = 0; ph ^= 1u; }
      }
    }
  } else if (warp == 1 && lane == 0 && rank == 0) {
    // ================================================================ MMA issuer
    constexpr uint32_t idesc_full =
        kF8 ? idesc_e4m3_f32(BM * kCtaGroup, UMMA_N)
            : idesc_bf16_f32(BM * kCtaGroup, UMMA_N, /*a_mn=*/false, /*b_mn=*/!kWK);
    constexpr uint32_t idesc_half = kF8 ? idesc_e4m3_f32(BM * kCtaGroup, 128)
                                        : idesc_bf16_f32(BM * kCtaGroup, 128, false, !kWK);
    if constexpr (kMB == 2) {
      // Two row blocks per tile sharing every weight stage; block 0 runs ahead of block 1 by up
      // to L k-blocks at the head and at the tail of a tile (see the kernel comment).  s0 / s1:
      // ring slots of the next k-block of block 0 / block 1; a slot is waited for once (block 0
      // always touches it first) and freed by the commit after block 1's MMAs.
      int s0 = 0, s1 = 0;
      uint32_t ph0 = 0;
      uint32_t it0 = 0, it1 = 0;  // uses of accumulator region 0 / 1 so far (barrier phases)
      const int L = min(max(p.skew, 1), kStages);
      [[maybe_unused]] int it = -1;  // tile counter of the debug-build timeline stamps
      for (int t = group_id; t < total_tiles; t += num_groups) {
        ++it;
        const TileUnit u = decode_unit<kOutCols, kMB>(p, t, k_blocks);
        const int n = u.kb1 - u.kb0;
        const uint32_t idesc = (u.w == 64) ? idesc_half : idesc_full;
        auto mma_block = [&](int b, int s, bool first) {
          const uint32_t sa = smem_a(s) + b * (BM * BK * 2), sb = smem_b(s);
          const uint32_t d_tmem = tmem_base + b * UMMA_N;
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k) {
            const uint64_t adesc = smem_desc_sw128(sa + k * (UMMA_K * 2), 16, 1024);
            const uint64_t bdesc = kWK ? smem_desc_sw128(sb + k * (UMMA_K * 2), 16, 1024)
                                       : smem_desc_sw128(sb + k * (UMMA_K * 128), 8192, 1024);
            if constexpr (kF8) umma_f8<kCtaGroup>(d_tmem, adesc, bdesc, idesc, (!first || k > 0) ? 1u : 0u);
            else umma_bf16<kCtaGroup>(d_tmem, adesc, bdesc, idesc, (!first || k > 0) ? 1u : 0u);
          }
        };
        if (u.nmb == 1) {
          // one row block (a unit of the cut last wave, or a ragged last row tile): region 0 only
          mbar_wait(acc_empty_bar(0), (it0 & 1u) ^ 1u);
          tcgen05_fence_after();
          for (int i = 0; i < n; ++i) {
            mbar_wait(full_bar(s0), ph0);
            tcgen05_fence_after();
            mma_block(0, s0, i == 0);
            umma_commit<kCtaGroup>(empty_bar(s0), all_mask);
            if (++s0 == kStages) { s0 = 0; ph0 ^= 1u; }
          }
          s1 = s0;
          umma_commit<kCtaGroup>(acc_full_bar(0), pair_mask);
          ++it0;
          continue;
        }
        const uint32_t aph0 = it0 & 1u, aph1 = it1 & 1u;
        ++it0; ++it1;
        const int H = min(L, n), T = min(L, n - H);
        int i0 = 0, i1 = 0;
        auto do0 = [&]() {
          mbar_wait(full_bar(s0), ph0);
          tcgen05_fence_after();
          mma_block(0, s0, i0 == 0);
          ++i0;
          if (++s0 == kStages) { s0 = 0; ph0 ^= 1u; }
        };
        auto do1 = [&]() {
          mma_block(1, s1, i1 == 0);
          umma_commit<kCtaGroup>(empty_bar(s1), all_mask);  // both blocks have read the stage
          ++i1;
          if (++s1 == kStages) s1 = 0;
        };
        mbar_wait(acc_empty_bar(0), aph0 ^ 1u);  // region 0 drained
        SWIGLU_GEMM_TRACE(8 + it * 8 + 0);
        tcgen05_fence_after();
        for (int i = 0; i < H; ++i) do0();
        SWIGLU_GEMM_TRACE(8 + it * 8 + 1);
        if (T == 0) umma_commit<kCtaGroup>(acc_full_bar(0), pair_mask);  // the whole K range fitted the head
        mbar_wait(acc_empty_bar(1), aph1 ^ 1u);  // region 1 drained
        SWIGLU_GEMM_TRACE(8 + it * 8 + 2);
        tcgen05_fence_after();
        for (int i = 0; i < H; ++i) do1();
        for (int i = n - H - T; i > 0; --i) { do0(); do1(); }
        if (T > 0) {
          for (int i = 0; i < T; ++i) do0();
          umma_commit<kCtaGroup>(acc_full_bar(0), pair_mask);  // region 0 complete: drains under block 1's tail
          SWIGLU_GEMM_TRACE(8 + it * 8 + 5);
          for (int i = 0; i < T; ++i) do1();
        }
        umma_commit<kCtaGroup>(acc_full_bar(1), pair_mask);
        SWIGLU_GEMM_TRACE(8 + it * 8 + 6);
      }
    } else {
    int s = 0;
    uint32_t ph = 0;
    int it = 0;
    for (int t = group_id; t < total_tiles; t += num_groups, ++it) {
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1u;
      mbar_wait(acc_empty_bar(as), aph ^ 1u);  // epilogue has drained this TMEM stage
      SWIGLU_GEMM_TRACE(8 + it * 8 + 0);
      tcgen05_fence_after();
      const uint32_t d_tmem = tmem_base + as * UMMA_N;
      // half tiles of the last wave (Gate 64 | Up 64) use an N = 128 instruction
      const TileUnit u = decode_unit<kOutCols>(p, t, k_blocks);
      const uint32_t idesc = (kFused && kBN == 128 && u.w == 64) ? idesc_half : idesc_full;
      for (int kb = u.kb0; kb < u.kb1; ++kb) {
        mbar_wait(full_bar(s), ph);
        if (kb == u.kb0) SWIGLU_GEMM_TRACE(8 + it * 8 + 1);
        tcgen05_fence_after();
        const uint32_t sa = smem_a(s), sb = smem_b(s);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k) {
          // A: K-major, +32 B per 16-k step inside the 128-byte swizzle row.
          const uint64_t adesc = smem_desc_sw128(sa + k * (UMMA_K * 2), 16, 1024);
          // B, [K,N] weights: MN-major, 16 k rows = 2 KB per step, 64-column slabs 8 KB apart.
          // B, [N,K] weights: K-major like A (slabs of 64 n-rows are 8 KB = 8 groups of 8 rows).
          const uint64_t bdesc = kWK ? smem_desc_sw128(sb + k * (UMMA_K * 2), 16, 1024)
                                     : smem_desc_sw128(sb + k * (UMMA_K * 128), 8192, 1024);
          if constexpr (kF8) umma_f8<kCtaGroup>(d_tmem, adesc, bdesc, idesc, (kb > u.kb0 || k > 0) ? 1u : 0u);
          else umma_bf16<kCtaGroup>(d_tmem, adesc, bdesc, idesc, (kb > u.kb0 || k > 0) ? 1u : 0u);
        }
        umma_commit<kCtaGroup>(empty_bar(s), all_mask);  // smem stage free once these MMAs retire
        if (++s == kStages) { s = 0; ph ^= 1u; }
      }
      umma_commit<kCtaGroup>(acc_full_bar(as), pair_mask);  // accumulator complete -> epilogue
      SWIGLU_GEMM_TRACE(8 + it * 8 + 2);
    }
    }
  } else if (warp >= 2) {
    // ================================================================ epilogue
    const uint32_t q = warp & 3u;  // TMEM lane quarter this warp may read
    const uint32_t row = q * 32u + lane;
    const uint32_t eg = (warp - 2u) >> 2;  // 0: columns [0,32) of each 64-column chunk, 1: [32,64)
    const bool issuer = (threadIdx.x == 64);         // K-split ticket, debug stamps
    const bool q_issuer = (eg == 0u && lane == 0u);  // TMA stores of this lane quarter
    const uint32_t leader_acc_empty0 =
        (kCtaGroup == 2) ? mapa_shared(acc_empty_bar(0), crank & ~1u) : 0u;  // the pair leader's
    int it = 0;
    uint32_t reg_phase = 0;  // kMB = 2: bit r = barrier phase of accumulator region r
    uint32_t chunk_ctr = 0;
    const uint32_t ticket_slot = tmem_slot + 4u;
    for (int t = group_id; t < total_tiles; t += num_groups, ++it) {
      const TileUnit tu = decode_unit<kOutCols, kMB>(p, t, k_blocks);
      const int n_base = tu.n_base, w = tu.w;
      // does the MMA thread wait for this tile's accumulator region(s) again?  (kMB = 1: stage
      // it & 1 is reused two tiles later; kMB = 2: by the next tile)
      const bool hand_back = t + (kMB == 2 ? 1 : 2) * num_groups < total_tiles;
      const int chunks = kFused ? w / 64 : kChunks;  // 64-column chunks in this tile
#pragma unroll 1
      for (int mb = 0; mb < tu.nmb; ++mb) {  // accumulator regions of the tile (kMB = 2: row blocks)
      const int m_base = ((tu.tm * kPairs * kMB + (int)pair + tu.mb0 + mb) * kCtaGroup + (int)rank) * BM;
      const int as = (kMB == 2) ? mb : (it & 1);
      const uint32_t aph = (kMB == 2) ? ((reg_phase >> mb) & 1u) : ((it >> 1) & 1u);
      reg_phase ^= 1u << mb;
      mbar_wait(acc_full_bar(as), aph);
      if (issuer) SWIGLU_GEMM_TRACE(8 + it * 8 + (mb == 0 ? 3 : 7));
      tcgen05_fence_after();
      const uint32_t tacc = tmem_base + ((q * 32u) << 16) + as * UMMA_N;
      // K-range unit of a tail tile: park the fp32 partial accumulators in the workspace
      // ([column/4][row] float4: a warp writes 512 contiguous bytes), then the LAST unit of the
      // tile to arrive sums all partials in k-range order (fixed order: bitwise deterministic
      // whoever is last) and runs the normal activation / store epilogue on the sums.
      const float4* split_src = nullptr;
      if constexpr (kFused && kBN == 128) {
        if (tu.tail >= 0) {
          const int S = p.tail_ksplit;
          const size_t slot = (size_t)tu.tail * kCtaGroup + rank;
          float4* part = reinterpret_cast<float4*>(p.split_ws) + (slot * S + tu.krank) * (size_t)(64 * BM);
#pragma unroll 1
          for (int cc = (int)eg; cc < UMMA_N / 32; cc += 2) {
            uint32_t v[32];
            tmem_ld_32x32b_x32(tacc + cc * 32, v);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 8; ++j)
              part[(size_t)(cc * 8 + j) * BM + row] =
                  make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                              __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
          }
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0 && hand_back) {  // TMEM stage drained (relaxed: see the hand-back in the chunk loop)
            if constexpr (kCtaGroup == 2) mbar_arrive_relaxed_cluster(leader_acc_empty0 + 8u * as);
            else mbar_arrive_relaxed(acc_empty_bar(as));
          }
          __threadfence();  // partials visible device-wide before the arrival is counted
          named_bar_sync(1, kEpiWarps * 32);
          if (issuer) {
            const int ticket = atomicAdd(p.split_ctr + slot, 1);
            if (ticket == S - 1) p.split_ctr[slot] = 0;  // all S arrived: clean for the next launch
            __threadfence();
            asm volatile("st.shared.b32 [%0], %1;" ::"r"(ticket_slot), "r"(ticket) : "memory");
          }
          named_bar_sync(1, kEpiWarps * 32);
          int ticket;
          asm volatile("ld.shared.b32 %0, [%1];" : "=r"(ticket) : "r"(ticket_slot) : "memory");
          if (ticket != S - 1) continue;  // a later unit will finish this tile
          split_src = reinterpret_cast<const float4*>(p.split_ws) + slot * S * (size_t)(64 * BM);
        }
      }
#pragma unroll 1
      for (int h = 0; h < chunks; ++h, ++chunk_ctr) {
        // Each TMEM lane quarter is its own store pipeline: the two warps of quarter q (columns
        // [0,32) and [32,64) of the chunk) share a double-buffered 32-row x 128-byte staging area,
        // synchronise with each other only (named barrier 2 + q, 64 threads) and one of them issues
        // the 64-column x 32-row TMA store.  The four quarters drift freely, so one quarter's TMEM
        // loads and MUFU work overlap another's barrier and store issue.
        const uint32_t obuf = smem_out + q * (2u * kQuarterBufBytes) + (chunk_ctr & 1u) * kQuarterBufBytes;
        // the TMA store that last read this buffer (2 chunks ago) must have finished reading
        if (q_issuer) tma_store_wait_read<1>();
        named_bar_sync(2u + q, 64);
        if (issuer && kMB == 1 && h == SWIGLU_TRACE_H) SWIGLU_GEMM_TRACE(8 + it * 8 + 5);
        {
          const int c = (int)eg;  // this warp's half of the chunk
          uint32_t packed[16];
          if constexpr (kFused) {
            uint32_t g[32], u[32];
            // accumulator columns: [Gate w | Up w], or g0 u0 g1 u1 for packed weights
            const uint32_t gcol = kPacked ? h * 128 + c * 32 : h * 64 + c * 32;
            const uint32_t ucol = kPacked ? gcol + 64 : gcol + w;
            if (kBN == 128 && split_src != nullptr) {
              // sums of the K-range partials, k-range 0 first
              float gs[32], us[32];
#pragma unroll
              for (int j = 0; j < 32; ++j) gs[j] = us[j] = 0.0f;
#pragma unroll 1
              for (int r = 0; r < p.tail_ksplit; ++r) {
                const float4* pr = split_src + (size_t)r * (64 * BM) + row;
                float4 a[8], b[8];  // 16 loads in flight per thread, then the adds in k-range order
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  a[j] = __ldcg(pr + (size_t)(gcol / 4 + j) * BM);
                  b[j] = __ldcg(pr + (size_t)(ucol / 4 + j) * BM);
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  gs[4 * j] += a[j].x; gs[4 * j + 1] += a[j].y; gs[4 * j + 2] += a[j].z; gs[4 * j + 3] += a[j].w;
                  us[4 * j] += b[j].x; us[4 * j + 1] += b[j].y; us[4 * j + 2] += b[j].z; us[4 * j + 3] += b[j].w;
                }
              }
#pragma unroll
              for (int j = 0; j < 32; ++j) { g[j] = __float_as_uint(gs[j]); u[j] = __float_as_uint(us[j]); }
            } else {
              tmem_ld_32x32b_x32(tacc + gcol, g);
              tmem_ld_32x32b_x32(tacc + ucol, u);
              tmem_ld_wait();
              if (issuer && kMB == 1 && h == SWIGLU_TRACE_H) SWIGLU_GEMM_TRACE(8 + it * 8 + 6);
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              float g0 = __uint_as_float(g[2 * j]), u0 = __uint_as_float(u[2 * j]);
              float g1 = __uint_as_float(g[2 * j + 1]), u1 = __uint_as_float(u[2 * j + 1]);
              if constexpr (kF8) {  // dequantise: one scale per projection
                g0 *= p.scale_gate; g1 *= p.scale_gate;
                u0 *= p.scale_up; u1 *= p.scale_up;
              }
              packed[j] = pack_bf16x2_rn(glu_mul<kAct>(g0, u0), glu_mul<kAct>(g1, u1));
            }
          } else {
            uint32_t v[32];
            tmem_ld_32x32b_x32(tacc + h * 64 + c * 32, v);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 16; ++j)
              packed[j] = pack_bf16x2_rn(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
          }
          if (h == chunks - 1 && split_src == nullptr) {
            // last TMEM read of this tile is done: hand the accumulator stage back to the MMA
            tcgen05_fence_before();
            __syncwarp();
            if (lane == 0 && hand_back) {
              // RELAXED arrive: the only thing the MMA thread needs from this warp is that its
              // TMEM reads are over, and tcgen05.wait::ld above has already retired them into
              // registers; there is no memory to publish.  (A release at cluster scope here cost
              // 1.2 us per hand-back -- it drains this thread's earlier stores first: measured
              // 3.4 -> 2.2 us per 128x128 tile epilogue.)  Not sent at all when the
              // MMA thread will not reuse the region (hand_back): no remote arrival may still be
              // in flight towards the pair leader's shared memory when that CTA exits.
              if constexpr (kCtaGroup == 2) mbar_arrive_relaxed_cluster(leader_acc_empty0 + 8u * as);
              else mbar_arrive_relaxed(acc_empty_bar(as));
            }
          }
          // 128-byte swizzled staging: row r, 16-byte chunk j -> chunk (j ^ (r & 7))
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t chunk = (uint32_t)(c * 4 + j) ^ (row & 7u);
            st_shared_v4(obuf + lane * 128u + chunk * 16u, packed[4 * j], packed[4 * j + 1],
                         packed[4 * j + 2], packed[4 * j + 3]);
          }
        }
        fence_proxy_async_smem();
        named_bar_sync(2u + q, 64);
        if (issuer && kMB == 1 && h == SWIGLU_TRACE_H) SWIGLU_GEMM_TRACE(8 + it * 8 + 7);
        if (q_issuer) {
          tma_store_2d_hint(&tmap_y, obuf, n_base + h * 64, m_base + (int)(q * 32u), p.y_policy);  // OOB rows/cols are clipped
          tma_store_commit();
        }
      }
      }
      if (issuer) SWIGLU_GEMM_TRACE(8 + it * 8 + 4);
    }
    // shared memory may go once the last stores have READ it; their global writes complete with
    // the grid (and before any dependent grid passes griddepcontrol.wait)
    if (q_issuer) tma_store_wait_read<0>();
  }

  // ------------------------------------------------------------------ teardown
  __syncwarp();
  tcgen05_fence_before();
  // (relaxed arrival: the barrier only says "this CTA no longer touches its peers' shared memory,
  // barriers or TMEM"; there is nothing to publish, so no release that drains the stores first)
  if (kCtaGroup == 2) { cluster_arrive_relaxed(); cluster_wait_acquire(); } else __syncthreads();
  if (warp == 1) {
    tcgen05_fence_after();
    tmem_dealloc<kCtaGroup>(tmem_base, kTmemCols);
  }
  if (threadIdx.x == 0) SWIGLU_GEMM_TRACE(2);
  if (clk_probe) {
    p.clk[0] = (unsigned long long)(clock64() - clk_c0);
    p.clk[1] = globaltimer_ns() - clk_t0;
  }
}

// ---------------------------------------------------------------------------------------
// Elementwise stage of the unfused path: Y = bf16( SiLU(float(G)) * float(U) )
// (read Gate, read Up, write Y).  16-byte vector accesses.
// ---------------------------------------------------------------------------------------
template <int kAct>
__global__ void __launch_bounds__(256)
silu_mul_kernel(const uint4* __restrict__ G, const uint4* __restrict__ U, uint4* __restrict__ Y,
                int64_t n_vec) {
  pdl_wait_prior_grid();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) {
    const uint4 g = __ldg(G + i), u = __ldg(U + i);
    const uint32_t gw[4] = {g.x, g.y, g.z, g.w}, uw[4] = {u.x, u.y, u.z, u.w};
    uint32_t yw[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float g0 = __uint_as_float(gw[j] << 16), g1 = __uint_as_float(gw[j] & 0xFFFF0000u);
      const float u0 = __uint_as_float(uw[j] << 16), u1 = __uint_as_float(uw[j] & 0xFFFF0000u);
      yw[j] = pack_bf16x2_rn(glu_mul<kAct>(g0, u0), glu_mul<kAct>(g1, u1));
    }
    Y[i] = make_uint4(yw[0], yw[1], yw[2], yw[3]);
  }
  pdl_launch_dependents();
}

}  // namespace swiglu
