// swiglu_api.cu -- the C ABI of include/swiglu_mlp.h: validation, variant table, tensor
// maps, workspace, launches.  Host logic only; the kernels are in the .cuh files.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <atomic>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/swiglu_mlp.h"
#include "gemm_swiglu_kernel.cuh"
#include "smallm_swiglu_kernel.cuh"

// Scratch of swiglu_mlp_unfused_static (include/swiglu_mlp.h): bf16 Gate | Up of one call.  In HOST
// code this name is only a stand-in for the symbol, not a device address: the address is taken
// once per device with cudaGetSymbolAddress (static_scratch_address below) and passed to the kernels.
static __device__ __align__(256) unsigned char g_static_scratch[SWIGLU_STATIC_SCRATCH_BYTES];

namespace {

using swiglu::kWeightsKN;
using swiglu::kWeightsNK;
using swiglu::kWeightsPacked;
using swiglu::kOperandsFp8;

// ------------------------------------------------------------------ error bookkeeping
thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}
int fail_cuda(cudaError_t e, const char* what) {
  return fail(SWIGLU_ERR_CUDA, "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
}
#define CUDA_TRY(expr)                                   \
  do {                                                   \
    cudaError_t _e = (expr);                             \
    if (_e != cudaSuccess) return fail_cuda(_e, #expr);  \
  } while (0)

#ifdef SWIGLU_TRACE
unsigned long long* g_trace = nullptr;  // debug builds: device buffer for globaltimer stamps
#endif
// swiglu_set_clock_probe: device buffer of two uint64 that CTA 0 of every GEMM-class launch
// fills with {SM cycles, nanoseconds} from entry to exit (measurement aid: the SM clock the
// kernel actually ran at = cycles / ns).  NULL = off.
std::atomic<unsigned long long*> g_clk{nullptr};

// ------------------------------------------------------------------ variant tables
enum FusedVariant {
  kFused1Cta = 0,     // 128x128 (Gate|Up) tile per CTA
  kFused2Cta = 1,     // 256x128 tile per CTA pair, cta_group::2
  kFusedSmallM = 2,   // swap-AB, split-K over a cluster, for M <= 128
  kFused1CtaN64 = 3,  // 128x64 (Gate|Up) tile per CTA: twice the tiles when N/128 < #SMs
  kFused2Cta4 = 4,    // cluster of 4 = two CTA pairs on a 512x128 super-tile, W tile multicast
  kFused2CtaMB2 = 5,  // 512x128 super-tile per CTA pair: two row blocks share each weight stage
  kNumFused = 6
};
enum UnfusedVariant {
  kUnfused1Cta = 0,    // GEMM 128x256 tiles x2 + elementwise
  kUnfused2Cta = 1,    // GEMM 256x256 pair tiles x2 + elementwise
  kUnfusedSmallM = 2,  // M <= 128: ONE merged Gate|Up swap-AB split-K GEMM + elementwise
  kUnfused2CtaMB2 = 3, // GEMM 512x256 super tiles (two row blocks per CTA) x2 + elementwise
  kNumUnfused = 4
};
const char* const kFusedNames[kNumFused] = {"fused_1cta_128x128", "fused_2cta_256x128",
                                            "fused_smallm_swapab_splitk", "fused_1cta_128x64",
                                            "fused_2cta_x2_512x128_wmcast",
                                            "fused_2cta_512x128_2rowblocks"};
const char* const kUnfusedNames[kNumUnfused] = {"unfused_1cta_gemm128x256+silu_mul",
                                                "unfused_2cta_gemm256x256+silu_mul",
                                                "unfused_smallm_gateup_gemm+silu_mul",
                                                "unfused_2cta_gemm512x256+silu_mul"};

int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  return (v && *v) ? atoi(v) : dflt;
}

// Experiment / A-B overrides.  Read from the environment ONCE, at the
// first call into the library (and again only on swiglu_reload_env()): the hot path does no
// getenv.  All default to "off" / "automatic".
struct Env {
  int variant = -1, unfused_variant = -1, ksplit = 0, group_m = 0, host_chunks = 8, tail_ksplit = 0;
  int skew = 4;  // super-tile kernel: k-blocks row block 0 leads block 1 at tile boundaries
  bool no_pdl = false, no_prefetch = false, no_early = false, no_tail_split = false,
       no_tail_ksplit = false, no_w_evict_first = false, no_tmap_cache = false;
  int smallm_deep = -1;  // -1 automatic, 0 never, 1 whenever it fits
  int smallm_stack = -1;  // stacked 64-column decode tile: -1 automatic, 0 never, 1 whenever instantiated
  int w_policy = -1, a_policy = -1, y_policy = -1;  // large-M kernel L2 hints: -1 automatic, 0 normal, 1 first, 2 last
};
Env g_env;
std::once_flag g_env_once;
void load_env() {
  Env e;
  e.variant = env_int("SWIGLU_VARIANT", -1);
  e.unfused_variant = env_int("SWIGLU_UNFUSED_VARIANT", -1);
  e.ksplit = env_int("SWIGLU_KSPLIT", 0);
  e.group_m = env_int("SWIGLU_GROUP_M", 0);
  e.tail_ksplit = env_int("SWIGLU_TAIL_KSPLIT", 0);
  if (e.tail_ksplit > 8) e.tail_ksplit = 8;
  e.host_chunks = env_int("SWIGLU_HOST_CHUNKS", 8);
  if (e.host_chunks <= 0) e.host_chunks = 8;
  e.no_pdl = env_int("SWIGLU_NO_PDL", 0) != 0;
  e.no_prefetch = env_int("SWIGLU_NO_PREFETCH", 0) != 0;
  e.no_early = env_int("SWIGLU_NO_EARLY", 0) != 0;
  e.no_tail_split = env_int("SWIGLU_NO_TAIL_SPLIT", 0) != 0;
  e.no_tail_ksplit = env_int("SWIGLU_NO_TAIL_KSPLIT", 0) != 0;
  e.no_w_evict_first = env_int("SWIGLU_NO_W_EVICT_FIRST", 0) != 0;
  e.no_tmap_cache = env_int("SWIGLU_NO_TMAP_CACHE", 0) != 0;
  e.smallm_deep = env_int("SWIGLU_SMALLM_DEEP", -1);
  e.skew = env_int("SWIGLU_SKEW", 4);
  e.smallm_stack = env_int("SWIGLU_SMALLM_STACK", -1);
  e.w_policy = env_int("SWIGLU_W_POLICY", -1);
  e.a_policy = env_int("SWIGLU_A_POLICY", -1);
  e.y_policy = env_int("SWIGLU_Y_POLICY", -1);
  g_env = e;
}
const Env& env() {
  std::call_once(g_env_once, load_env);
  return g_env;
}

struct TailPlan { int64_t wide, total; int ksplit; };
TailPlan plan_tail(int64_t tiles, int G, int64_t k_blocks, bool fused128, bool have_ws);
int super_tail_div(int64_t tiles, int G, int max_div = 4);
int64_t super_tail_cost4(int64_t rem, int G, int div);

// Wave efficiency (ideal waves / scheduled waves, in tile times) of the two pair kernels on
// `pairs` CTA pairs: the 256-row kernel with its last-wave plan, the 512-row super-tile kernel
// with its cut last wave.
double wave_eff_pair(int64_t M, int64_t N, int64_t K, int pairs) {
  const int64_t tiles = ((M + 255) / 256) * ((N + 127) / 128);
  const TailPlan t = plan_tail(tiles, pairs, (K + 63) / 64, true, true);
  const int64_t rem = tiles % pairs;
  double waves = (double)(tiles / pairs);
  if (rem) waves += t.ksplit >= 2 ? 1.0 / t.ksplit + 0.1 : (t.total > tiles ? 0.5 : 1.0);
  return (double)tiles / pairs / waves;
}
double wave_eff_super(int64_t M, int64_t N, int pairs, int cols = 128) {
  const int64_t n_tiles = (N + cols - 1) / cols;
  const int64_t tiles = ((M + 511) / 512) * n_tiles;
  const int64_t rem = tiles % pairs;
  double waves = (double)(tiles / pairs);
  if (rem) waves += super_tail_cost4(rem, pairs, super_tail_div(tiles, pairs, cols == 128 ? 4 : 2)) / 4.0;
  // a ragged last row tile with one block costs half a tile
  const double work = (double)((M + 255) / 256) * n_tiles / 2.0;
  return work / pairs / waves;
}

// Three or five 128-row tiles (256 < M <= 384, 512 < M <= 640): the pair kernels pad M to a
// multiple of 256 and would compute a quarter / a sixth more rows than the 1-CTA kernel, which
// outweighs its heavier L2 traffic (profiles/r02b_variant_sweep_odd_m.md: M = 384 / 640 -- 0.5B
// 13.8 -> 9.9 / 15.3 -> 14.4 us, 7B 106 -> 90 / 162 -> 145, 72B 380 -> 325 / 580 -> 497; ties at 1.5B;
// from seven row tiles on the two are within noise or the pair kernels win).
bool odd_row_tiles(int64_t M) {
  const int64_t r = (M + 127) / 128;
  return r == 3 || r == 5;
}

// Measured dispatch (table regenerated from bench sweeps).
int select_fused(int64_t M, int64_t N, int64_t K) {
  const int forced = env().variant;
  if (forced >= 0 && forced < kNumFused) {
    if (forced != kFusedSmallM || M <= swiglu::kSmallMMax) return forced;
  }
  // Measured (profiles/r01_variant_sweep.md).  All of M <= 128 is HBM-bound; what matters is
  // how many SMs stream weights and what the reduction costs:
  //  * M <= 32: swap-AB split-K kernel (cluster DSMEM reduction is cheap for few rows);
  //  * 32 < M <= 128: if N/128 tiles cannot fill ~3/4 of the 148 SMs, 64-column tiles (twice
  //    the CTAs, no reduction); otherwise the split-K kernel up to M = 64 and the 128x128
  //    1-CTA kernel above it;
  //  * M > 128: the 2-CTA pair kernel.
  const int64_t n_tiles = (N + 127) / 128;
  const bool few_tiles = n_tiles * 4 <= 148 * 3;
  if (M <= 32) return kFusedSmallM;
  if (M <= 64) return few_tiles ? kFused1CtaN64 : kFusedSmallM;
  if (M <= 128) return few_tiles ? kFused1CtaN64 : kFused1Cta;
  // M > 128: a CTA-pair kernel.  The 512-row super tile moves a quarter less data per FLOP: these
  // calls are power-bound under load and L2->SM-bound at high clocks (
  // profiles/r02b_variant_sweep_super_tile.md: +1-9 % in short bursts, +3-7 % sustained, at
  // every K from 896 up once the accumulator hand-back stopped costing 1.2 us per region) --
  // wherever the 512-row granularity does not cost more in wave quantisation than it gains.
  if (odd_row_tiles(M)) return kFused1Cta;
  if (M > 512 && K >= 768 && wave_eff_super(M, N, 74) >= wave_eff_pair(M, N, K, 74) - 0.03)
    return kFused2CtaMB2;
  return kFused2Cta;
}
int select_unfused(int64_t M, int64_t N, int64_t K) {
  const int forced = env().unfused_variant;
  if (forced >= 0 && forced < kNumUnfused && (forced != kUnfusedSmallM || M <= swiglu::kSmallMMax))
    return forced;
  // Decode sizes: the same swap-AB split-K streaming kernel as the fused path, writing bf16
  // Gate and Up -- so that fused vs unfused compares fusion, not tile shapes.
  if (M <= 128) return kUnfusedSmallM;
  // Large M: the same super-tile rule as the fused path (same mainloop, same power argument).
  if (M > 512 && K >= 768) {
    const int64_t tiles = ((M + 255) / 256) * ((N + 255) / 256), rem = tiles % 74;
    const double eff_pair = (double)tiles / 74 / (double)(tiles / 74 + (rem ? 1 : 0));
    if (wave_eff_super(M, N, 74, 256) >= eff_pair - 0.03) return kUnfused2CtaMB2;
  }
  return kUnfused2Cta;
}

// ------------------------------------------------------------------ validation (no CUDA)
bool overlaps(const void* a, int64_t abytes, const void* b, int64_t bbytes) {
  const uintptr_t a0 = (uintptr_t)a, a1 = a0 + (uintptr_t)abytes;
  const uintptr_t b0 = (uintptr_t)b, b1 = b0 + (uintptr_t)bbytes;
  return a0 < b1 && b0 < a1;
}
bool mul_overflows(int64_t a, int64_t b, int64_t limit) { return a != 0 && b > limit / a; }

int validate(const void* A, const void* W1, const void* W2, const void* Y, int64_t M, int64_t N,
             int64_t K) {
  if (M < 0 || N <= 0 || K <= 0)
    return fail(SWIGLU_ERR_BAD_SHAPE, "bad shape M=%lld N=%lld K=%lld (need M>=0, N>0, K>0)",
                (long long)M, (long long)N, (long long)K);
  const int64_t lim = INT64_MAX / 4;
  if (mul_overflows(M, K, lim) || mul_overflows(K, N, lim) || mul_overflows(M, N, lim) ||
      M > INT32_MAX - 256 || N > INT32_MAX - 256 || K > INT32_MAX - 256)
    return fail(SWIGLU_ERR_BAD_SHAPE, "shape too large M=%lld N=%lld K=%lld", (long long)M,
                (long long)N, (long long)K);
  if ((K % 8) != 0 || (N % 8) != 0)
    return fail(SWIGLU_ERR_UNSUPPORTED,
                "K=%lld and N=%lld must be multiples of 8 (16-byte row pitch for TMA)",
                (long long)K, (long long)N);
  if (M == 0) return SWIGLU_OK;
  if (!A || !W1 || !W2 || !Y) return fail(SWIGLU_ERR_NULL_POINTER, "A, W1, W2 or Y is NULL");
  if (((uintptr_t)A | (uintptr_t)W1 | (uintptr_t)W2 | (uintptr_t)Y) & 15u)
    return fail(SWIGLU_ERR_MISALIGNED, "A, W1, W2 and Y must be 16-byte aligned");
  const int64_t ab = M * K * 2, wb = K * N * 2, yb = M * N * 2;
  if (overlaps(Y, yb, A, ab) || overlaps(Y, yb, W1, wb) || overlaps(Y, yb, W2, wb))
    return fail(SWIGLU_ERR_ALIASING, "Y overlaps an input");
  return SWIGLU_OK;
}

// ------------------------------------------------------------------ device state
struct DeviceState {
  bool ready = false;
  int device = -1;
  int sm_count = 0;
  int cc_major = 0;
  // Library-owned buffers are PER STREAM: two calls on different streams may run at the same
  // time and must not share Gate/Up workspace or staging memory.
  struct Buf { void* ptr = nullptr; size_t bytes = 0; };
  std::map<cudaStream_t, Buf> workspace;     // unfused path: bf16 Gate | Up
  std::map<cudaStream_t, Buf> host_scratch;  // swiglu_mlp_host: device copies of A, W1, W2, Y
  std::map<cudaStream_t, Buf> split_ws;      // fused large-M: K-split partials of the last wave
  // swiglu_mlp_host_batched: copy streams and events of its H2D / compute / D2H pipeline;
  // host_mu admits one such pipeline per device at a time
  std::mutex host_mu;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_a = nullptr, ev_in[2] = {nullptr, nullptr}, ev_cmp[2] = {nullptr, nullptr},
              ev_out[2] = {nullptr, nullptr};
};
std::mutex g_mu;
DeviceState g_dev[64];

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

// Opt every fused kernel of activation kAct in to its dynamic shared-memory size.
template <int kAct, int kWK>
int set_smem_attrs() {
  using namespace swiglu;
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<1, true, 128, kAct, kWK>, attr, GemmCfg<1>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<1, true, 64, kAct, kWK>, attr, GemmCfg<1, 128>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<2, true, 128, kAct, kWK>, attr, GemmCfg<2>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<2, true, 128, kAct, kWK, 2>, attr, GemmCfg<2>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<2, true, 128, kAct, kWK, 1, 2>, attr, GemmCfg<2, 256, 2>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<16, kAct, kWK>, attr, SmallCfg<16>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<32, kAct, kWK>, attr, SmallCfg<32>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<64, kAct, kWK>, attr, SmallCfg<64>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<128, kAct, kWK>, attr, SmallCfg<128>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<16, kAct, kWK, false, false, true>, attr, SmallCfg<16, false, true>::kSmemBytes));
  CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<32, kAct, kWK, false, false, true>, attr, SmallCfg<32, false, true>::kSmemBytes));
  if constexpr (kWK == kWeightsKN || kWK == kWeightsPacked) {
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<16, kAct, kWK, false, true>, attr, SmallCfg<16, true>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<32, kAct, kWK, false, true>, attr, SmallCfg<32, true>::kSmemBytes));
  }
  if constexpr (kAct == kActSilu && kWK != kWeightsPacked && kWK != kOperandsFp8) {  // plain GEMMs: no activation
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<16, kActSilu, kWK, true, false, true>, attr, SmallCfg<16, false, true>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<32, kActSilu, kWK, true, false, true>, attr, SmallCfg<32, false, true>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<16, kActSilu, kWK, true>, attr, SmallCfg<16>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<32, kActSilu, kWK, true>, attr, SmallCfg<32>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<64, kActSilu, kWK, true>, attr, SmallCfg<64>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(smallm_swiglu_kernel<128, kActSilu, kWK, true>, attr, SmallCfg<128>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<1, false, 128, kActSilu, kWK>, attr, GemmCfg<1>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<2, false, 128, kActSilu, kWK>, attr, GemmCfg<2>::kSmemBytes));
    CUDA_TRY(cudaFuncSetAttribute(gemm_swiglu_kernel<2, false, 128, kActSilu, kWK, 1, 2>, attr, GemmCfg<2, 256, 2>::kSmemBytes));
  }
  return SWIGLU_OK;
}

int get_device_state(DeviceState** out) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(SWIGLU_ERR_CUDA, "device index %d out of range", dev);
  std::lock_guard<std::mutex> lk(g_mu);
  DeviceState& d = g_dev[dev];
  if (!d.ready) {
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    d.device = dev;
    d.sm_count = prop.multiProcessorCount;
    d.cc_major = prop.major;
    if (prop.major != 10)
      return fail(SWIGLU_ERR_ARCH, "device %d is sm_%d%d; this library is sm_100a only", dev,
                  prop.major, prop.minor);
    if (!g_encode) {
      void* fn = nullptr;
      cudaDriverEntryPointQueryResult qres;
      CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
      if (!fn || qres != cudaDriverEntryPointSuccess)
        return fail(SWIGLU_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
      g_encode = (EncodeTiledFn)fn;
    }
    using namespace swiglu;
    int rc;
    if ((rc = set_smem_attrs<kActSilu, kWeightsKN>()) || (rc = set_smem_attrs<kActGelu, kWeightsKN>()) ||
        (rc = set_smem_attrs<kActGeluTanh, kWeightsKN>()) || (rc = set_smem_attrs<kActRelu, kWeightsKN>()) ||
        (rc = set_smem_attrs<kActSilu, kWeightsNK>()) || (rc = set_smem_attrs<kActGelu, kWeightsNK>()) ||
        (rc = set_smem_attrs<kActGeluTanh, kWeightsNK>()) || (rc = set_smem_attrs<kActRelu, kWeightsNK>()) ||
        (rc = set_smem_attrs<kActSilu, kWeightsPacked>()) || (rc = set_smem_attrs<kActGelu, kWeightsPacked>()) ||
        (rc = set_smem_attrs<kActGeluTanh, kWeightsPacked>()) || (rc = set_smem_attrs<kActRelu, kWeightsPacked>()) ||
        (rc = set_smem_attrs<kActSilu, kOperandsFp8>()))
      return rc;
    d.ready = true;
  }
  *out = &d;
  return SWIGLU_OK;
}

// Tensor-map cache (a0: "build or fetch cached CUtensorMaps").  A map is a pure function of
// (base, dims, box): a cached copy can never be stale, whatever happened to the
// allocation in between.  Thread-local (the hot path takes no lock), 64 sets x 4 ways, LRU.
struct TmapKey {
  const void* base; int64_t d0, d1, d2; uint32_t b0, b1, b2; uint32_t esize;  // 2 = bf16, 1 = fp8
  int64_t pitch1;  // rows between consecutive d2 slices (>= d1; 0 = dense)
  bool operator==(const TmapKey& o) const {
    return base == o.base && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b0 == o.b0 && b1 == o.b1 &&
           b2 == o.b2 && esize == o.esize && pitch1 == o.pitch1;
  }
};
struct TmapSlot { bool used = false; uint64_t tick = 0; TmapKey key; CUtensorMap map; };
constexpr int kTmapSlots = 256;
constexpr int kTmapWays = 4;
thread_local TmapSlot t_tmaps[kTmapSlots];
thread_local uint64_t t_tmap_tick = 0;
thread_local uint64_t t_tmap_hits = 0, t_tmap_misses = 0;

// bf16 (or 1-byte) tensor, dense row-major, dims innermost first (d2 == 0: 2-D), box b0 x b1
// [x b2], 128-byte swizzle (b0 * esize must be 128 bytes), out-of-bounds reads give zeros.
int encode_tmap(CUtensorMap* out, const TmapKey& k) {
  const cuuint32_t rank = k.d2 ? 3 : 2;
  const cuuint64_t dims[3] = {(cuuint64_t)k.d0, (cuuint64_t)k.d1, (cuuint64_t)k.d2};
  const cuuint64_t strides[2] = {(cuuint64_t)k.d0 * k.esize,
                                 (cuuint64_t)k.d0 * k.esize * (cuuint64_t)(k.pitch1 ? k.pitch1 : k.d1)};
  const cuuint32_t box[3] = {k.b0, k.b1, k.b2};
  const cuuint32_t elem[3] = {1, 1, 1};
  const CUresult r =
      g_encode(out, k.esize == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
               rank, const_cast<void*>(k.base), dims,
               strides, box, elem, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS)
    return fail(SWIGLU_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) dims=%lld x %lld x %lld",
                (int)r, (long long)k.d0, (long long)k.d1, (long long)k.d2);
  return SWIGLU_OK;
}

int cached_tmap(CUtensorMap* out, const TmapKey& key) {
  if (env().no_tmap_cache) return encode_tmap(out, key);
  uint64_t h = (uint64_t)(uintptr_t)key.base * 0x9E3779B97F4A7C15ull;
  h ^= ((uint64_t)key.d0 * 0xC2B2AE3D27D4EB4Full) ^ ((uint64_t)key.d1 * 0x165667B19E3779F9ull) ^
       ((uint64_t)key.d2 * 0x27D4EB2F165667C5ull) ^ ((uint64_t)key.b1 << 7) ^ ((uint64_t)key.b2 << 17) ^
       ((uint64_t)key.esize << 27) ^ ((uint64_t)key.pitch1 << 31);
  // four-way set associative with least-recently-used replacement (t_tmap_tick stamps every use):
  // the handful of live maps of one call -- A, W1, W2, Y -- cannot evict each other on every call
  // when their hashes collide, as they would in a direct-mapped table
  const uint32_t set = (uint32_t)(h >> 40) & (kTmapSlots / kTmapWays - 1);
  TmapSlot* ways = t_tmaps + (size_t)set * kTmapWays;
  ++t_tmap_tick;
  for (int w = 0; w < kTmapWays; ++w) {
    if (ways[w].used && ways[w].key == key) {
      ++t_tmap_hits;
      ways[w].tick = t_tmap_tick;
      *out = ways[w].map;
      return SWIGLU_OK;
    }
  }
  ++t_tmap_misses;
  const int rc = encode_tmap(out, key);
  if (rc) return rc;
  int victim = 0;
  for (int w = 0; w < kTmapWays; ++w) {
    if (!ways[w].used) { victim = w; break; }
    if (ways[w].tick < ways[victim].tick) victim = w;
  }
  ways[victim].used = true;
  ways[victim].key = key;
  ways[victim].map = *out;
  ways[victim].tick = t_tmap_tick;
  return SWIGLU_OK;
}

// 2-D tensor [outer, inner] (inner contiguous), box = box_outer x box_inner.
int make_tmap(CUtensorMap* out, const void* base, int64_t inner, int64_t outer,
              uint32_t box_inner, uint32_t box_outer) {
  return cached_tmap(out, TmapKey{base, inner, outer, 0, box_inner, box_outer, 0, 2, 0});
}
// FP8 (1-byte) 2-D tensor [outer, inner]: a box row is 128 elements = 128 bytes.
int make_tmap_u8(CUtensorMap* out, const void* base, int64_t inner, int64_t outer,
                 uint32_t box_outer) {
  return cached_tmap(out, TmapKey{base, inner, outer, 0, 128, box_outer, 0, 1, 0});
}
// Rows per slab of the prepacked buffer: K plus 8 or 16 padding rows, chosen so that the slab
// pitch (rows x 128 B) is an ODD number of KiB.  With a power-of-two-ish pitch (K = 5120: 640 KiB)
// the CTAs of a decode call -- all at the same k, one slab pitch apart -- walk addresses that
// collide in the L2 / HBM channel hash (32B decode: 94 us packed vs 84 us plain before the pad).
inline int64_t packed_rows(int64_t K) { return K + ((((K + 7) / 8) % 2 == 0) ? 8 : 16); }
// Prepacked weights Wp[slab][packed_rows(K)][64]: {64, K, slabs}, box = 64 x 64 x box_slabs.
int make_tmap_packed(CUtensorMap* out, const void* base, int64_t K, int64_t slabs,
                     uint32_t box_slabs) {
  return cached_tmap(out, TmapKey{base, 64, K, slabs, 64, 64, box_slabs, 2, packed_rows(K)});
}
inline int64_t packed_slabs(int64_t N) { return 4 * ((N + 127) / 128); }

bool pdl_enabled() { return !env().no_pdl; }

// ------------------------------------------------------------------ last-wave plan (a1)
// The last partial wave of a 128-column fused schedule (rem tiles on G CTA groups):
//  * K split ("stream-K tail"): each tail tile is cut into s K-ranges run by otherwise idle
//    groups; partial fp32 accumulators meet in a global workspace and the last range to arrive
//    finishes the tile.  The finisher alone moves s x 128 KB per CTA through L2 (measured
//    ~2 us per partial, profiles/r02_tail_ksplit.md), so the split pays only when half tiles
//    would leave most of the machine idle (4 rem <= G) and every range keeps >= 16 k-blocks of
//    mainloop: the big-K shapes near the ridge (72B at M = 256, 512).  s <= 4.
//  * else, if at most half of the groups would be busy: two 64-column half tiles per tile.
constexpr int kSplitMaxS = 4;
constexpr int kSplitMinKBlocks = 16;
constexpr size_t kSplitCtrBytes = 4096;                      // counters: one int per (tile, CTA)
constexpr size_t kSplitPartialBytes = 256 * 128 * 4;         // one CTA's fp32 accumulators
constexpr size_t kSplitWsBytes = kSplitCtrBytes + 160 * kSplitPartialBytes;  // up to 160 SMs
// Super-tile kernel: units per tile of the last partial wave (1 = whole tiles, 2 = row blocks,
// 4 = row blocks x 64-column halves): the coarsest cut that minimises the time of the tail,
// ceil(rem * div / G) / div tile times.
int64_t super_tail_cost4(int64_t rem, int G, int div) { return (rem * div + G - 1) / G * (4 / div); }
int super_tail_div(int64_t tiles, int G, int max_div) {
  const int64_t rem = tiles % G;
  if (rem == 0 || env().no_tail_split) return 1;
  if (env().tail_ksplit == 2 || env().tail_ksplit == max_div) return env().tail_ksplit;  // experiments
  int best = 1;
  for (int div = 2; div <= max_div; div *= 2)
    if (super_tail_cost4(rem, G, div) < super_tail_cost4(rem, G, best)) best = div;
  return best;
}
TailPlan plan_tail(int64_t tiles, int G, int64_t k_blocks, bool fused128, bool have_ws) {
  TailPlan t{tiles, tiles, 0};
  const int64_t rem = tiles % G;
  if (!fused128 || rem == 0 || env().no_tail_split) return t;
  int s = (int)(G / rem);
  if (s > kSplitMaxS) s = kSplitMaxS;
  if (env().tail_ksplit > 0) s = env().tail_ksplit;   // experiments: force s (if it fits)
  while (s >= 2 && (rem * s > G || k_blocks / s < (env().tail_ksplit > 0 ? 1 : kSplitMinKBlocks))) --s;
  const bool sparse_tail = 4 * rem <= G || env().tail_ksplit > 0;
  if (have_ws && s >= 2 && sparse_tail && !env().no_tail_ksplit) {
    t.wide = tiles - rem;
    t.ksplit = s;
    t.total = t.wide + rem * s;
  } else if (tiles > G && 2 * rem <= G) {
    t.wide = tiles - rem;
    t.total = tiles + rem;
  }
  return t;
}

// ------------------------------------------------------------------ launches
template <int kCtaGroup, bool kFused, int kBN = 128, int kAct = swiglu::kActSilu, int kWMode = 0,
          int kPairs = 1, int kMB = 1>
int launch_gemm(const DeviceState& d, const void* A, const void* B1, const void* B2, void* Yout,
                int64_t M, int64_t N, int64_t K, cudaStream_t stream, void* split_ws = nullptr,
                float scale_gate = 1.0f, float scale_up = 1.0f) {
  using namespace swiglu;
  CUtensorMap ta, tb1, tb2, ty;
  int rc;
  constexpr bool kWK = (kWMode == kWeightsNK);
  constexpr int kBKe = (kWMode == kOperandsFp8) ? 128 : BK;   // k elements per stage
  if constexpr (kWMode == kOperandsFp8) {
    if ((rc = make_tmap_u8(&ta, A, K, M, 128))) return rc;
    if ((rc = make_tmap_u8(&tb1, B1, K, N, 64))) return rc;    // [N,K] E4M3: 64 n-rows x 128 k
    if ((rc = make_tmap_u8(&tb2, B2, K, N, 64))) return rc;
  } else if ((rc = make_tmap(&ta, A, K, M, 64, 128))) {
    return rc;
  }
  if constexpr (kWMode == kOperandsFp8) {
  } else if constexpr (kWMode == kWeightsPacked) {
    // B1 = Wp: one box per stage -- 4 slabs (1-CTA, 128 columns) or 2 (64-column tile; each
    // CTA of a pair); single-slab boxes for the half tiles of the last wave and for the
    // multicast loads of the two-pair cluster
    const uint32_t box = (kCtaGroup == 1 && kBN == 128) ? 4 : 2;
    if ((rc = make_tmap_packed(&tb1, B1, K, packed_slabs(N), box))) return rc;
    if ((rc = make_tmap_packed(&tb2, B1, K, packed_slabs(N), 1))) return rc;
  } else {
    // weights: [K,N] (inner N) or [N,K] (inner K); a box is always one 64 x 64 slab
    if ((rc = make_tmap(&tb1, B1, kWK ? K : N, kWK ? N : K, 64, 64))) return rc;
    if ((rc = make_tmap(&tb2, kFused ? B2 : B1, kWK ? K : N, kWK ? N : K, 64, 64))) return rc;
  }
  if ((rc = make_tmap(&ty, Yout, N, M, 64, 32))) return rc;   // one store per TMEM lane quarter
  using Cfg = GemmCfg<kCtaGroup, kFused ? 2 * kBN : 256, kMB>;
  GemmParams p;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  const int rows_per_tile = BM * kCtaGroup * kPairs * kMB;
  const int out_cols = kFused ? kBN : 256;
  p.m_tiles = (int)((M + rows_per_tile - 1) / rows_per_tile);
  p.n_tiles = (int)((N + out_cols - 1) / out_cols);
  // L2 raster group: keep the slab of A the running CTAs share at <= 32 MiB
  // (64 MiB for the super-tile kernel: 72B M=8192 sustained, group of 2 / 4 / 8 / 16 super tiles:
  // 1309 / 1357 / 1367 / 1302 TFLOP/s)
  int64_t gm = ((kMB == 2 ? 64ll : 32ll) << 20) / ((int64_t)rows_per_tile * K * (kWMode == kOperandsFp8 ? 1 : 2));
  const int forced_gm = env().group_m;
  if (forced_gm > 0) gm = forced_gm;
  if (gm < 1) gm = 1;
  if (gm > p.m_tiles) gm = p.m_tiles;
  p.group_m = (int)gm;
  const int64_t tiles = (int64_t)p.m_tiles * p.n_tiles;
  int G = d.sm_count / (kCtaGroup * kPairs);
  if constexpr (kPairs == 2) {
    // clusters of four do not tile every GPC: ask how many can be resident at once
    static int max_clusters = -1;  // per (instantiation, process); devices of one process are alike
    if (max_clusters < 0) {
      cudaLaunchConfig_t q;
      memset(&q, 0, sizeof q);
      q.gridDim = dim3((unsigned)d.sm_count / 4 * 4);
      q.blockDim = dim3(kGemmThreads);
      q.dynamicSmemBytes = Cfg::kSmemBytes;
      cudaLaunchAttribute qa[1];
      qa[0].id = cudaLaunchAttributeClusterDimension;
      qa[0].val.clusterDim.x = 4;
      qa[0].val.clusterDim.y = 1;
      qa[0].val.clusterDim.z = 1;
      q.attrs = qa;
      q.numAttrs = 1;
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, gemm_swiglu_kernel<kCtaGroup, kFused, kBN, kAct, kWMode, kPairs>, &q) !=
              cudaSuccess || n < 1) {
        cudaGetLastError();
        n = d.sm_count / 4;
      }
      max_clusters = n;
    }
    if (G > max_clusters) G = max_clusters;
  }
  const TailPlan tail = plan_tail(tiles, G, (K + kBKe - 1) / kBKe, kFused && kBN == 128 && kPairs == 1 && kMB == 1,
                                  split_ws != nullptr && d.sm_count <= 160);
  p.wide_tiles = (int)tail.wide;
  p.total_tiles = (int)tail.total;
  p.tail_ksplit = tail.ksplit;
  p.skew = env().skew;
  p.tail_div = 1;
  if constexpr (kMB == 2) {
    // last partial wave of super tiles: cut every tile into its two row blocks, or into row
    // blocks x 64-column halves, when that many units still fit one wave
    const int64_t rem = tiles % G;
    p.tail_div = super_tail_div(tiles, G, kFused ? 4 : 2);  // (a plain GEMM tile has no column halves)
    if (p.tail_div > 1) {
      p.wide_tiles = (int)(tiles - rem);
      p.total_tiles = (int)(tiles - rem + rem * p.tail_div);
    }
  }
  p.split_ctr = (int*)split_ws;
  p.split_ws = split_ws ? (float*)((char*)split_ws + kSplitCtrBytes) : nullptr;
  const int groups = (int)(p.total_tiles < G ? p.total_tiles : G);
  // one tile per CTA (a short, HBM-bound call): fill the TMA ring before the setup barrier
  p.early_issue = (kCtaGroup == 1 && kFused && tiles <= groups && tail.ksplit == 0 && !env().no_early);
  {
    const int64_t kb = (K + kBKe - 1) / kBKe;
    // (same cap as the decode kernel; M = 128, 0 / 2 / 4 / 8 k-blocks: 1.5B 11.29 / 11.08 / 11.13 /
    // 11.61 us, 7B 41.96 / 41.37 / 40.90 / 40.15 us)
    p.early_prefetch = env().no_prefetch ? 0 : (int)(kb / 3 < 4 ? kb / 3 : 4);
  }
  {
    const uint64_t pol[3] = {sm100::kEvictNormal, sm100::kEvictFirst, sm100::kEvictLast};
    p.w_policy = (p.m_tiles == 1 && !env().no_w_evict_first) ? sm100::kEvictFirst : sm100::kEvictNormal;
    p.a_policy = sm100::kEvictNormal;
    if (env().w_policy >= 0 && env().w_policy < 3) p.w_policy = pol[env().w_policy];
    if (env().a_policy >= 0 && env().a_policy < 3) p.a_policy = pol[env().a_policy];
    // Y larger than half of L2 cannot stay for a consumer anyway: let its lines leave first
    // (72B M=8192 / 7B M=4096 sustained: 1408 -> 1415, 1404 -> 1415 TFLOP/s; noise-level, kept)
    p.y_policy = (M * N * 2 > (64ll << 20)) ? sm100::kEvictFirst : sm100::kEvictNormal;
    if (env().y_policy >= 0 && env().y_policy < 3) p.y_policy = pol[env().y_policy];
  }
  p.clk = g_clk.load(std::memory_order_relaxed);
  p.scale_gate = scale_gate;
  p.scale_up = scale_up;
#ifdef SWIGLU_TRACE
  p.trace = g_trace;
#endif

  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof cfg);
  cfg.gridDim = dim3((unsigned)(groups * kCtaGroup * kPairs));
  cfg.blockDim = dim3(kGemmThreads);
  cfg.dynamicSmemBytes = Cfg::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attrs[2];
  int na = 0;
  if (kCtaGroup == 2) {
    attrs[na].id = cudaLaunchAttributeClusterDimension;
    attrs[na].val.clusterDim.x = 2 * kPairs;
    attrs[na].val.clusterDim.y = 1;
    attrs[na].val.clusterDim.z = 1;
    ++na;
  }
  if (pdl_enabled()) {
    attrs[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attrs[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = attrs;
  cfg.numAttrs = na;
  CUDA_TRY(cudaLaunchKernelEx(&cfg, gemm_swiglu_kernel<kCtaGroup, kFused, kBN, kAct, kWMode, kPairs, kMB>,
                              ta, tb1, tb2, ty, p));
  return SWIGLU_OK;
}

// Split-K factor of the small-M kernel (cluster size S), fitted to the measured sweep in
// profiles/r01_smallm_ksplit_sweep.md:
//  * at least as many 128-column tiles as SMs: no split (S = 1) -- except MP = 64, whose ring
//    is only two stages deep, where two co-resident half-K CTAs per SM keep more bytes in flight;
//  * fewer tiles than SMs: fill the co-resident CTA slots, but never more than 4 CTAs per
//    cluster (clusters of 5-8 do not all fit at once and run in a second wave) and never fewer
//    than 4 k-blocks per CTA (the cluster barrier + DSMEM reduction cost grows with S).
int smallm_ksplit(int sm_count, int ctas_per_sm, int mp, int64_t n_tiles, int64_t k_blocks) {
  const int forced = env().ksplit;
  const int64_t slots = (int64_t)ctas_per_sm * sm_count;
  int64_t s;
  if (n_tiles >= sm_count) {
    s = (mp == 64 && 2 * n_tiles <= slots) ? 2 : 1;
  } else {
    s = slots / n_tiles;
    if (s > 4) s = 4;
    while (s > 1 && k_blocks / s < 4) --s;
  }
  if (forced > 0) s = forced;
  if (s > 8) s = 8;
  if (s > k_blocks) s = k_blocks;
  if (s < 1) s = 1;
  return (int)s;
}

template <int MP, int kAct, int kWMode, bool kStoreGU = false, bool kDeep = false, bool kStack = false>
int launch_smallm_mp(const DeviceState& d, const void* A, const void* W1, const void* W2,
                     void* Y, void* U, int64_t M, int64_t N, int64_t K, cudaStream_t stream,
                     int probe = 0, float scale_gate = 1.0f, float scale_up = 1.0f) {
  using namespace swiglu;
  // Stacked 64-column tile (one CTA per SM, no cluster): when the 128-column tiles cannot fill
  // the GPU but the 64-column ones fit one wave -- 0.5B and 1.5B-class N -- the GPU fills without
  // a cluster split of K.
  if constexpr (!kStack && !kDeep && MP <= 32) {
    const int64_t nt128 = (N + 127) / 128, nt64 = (N + 63) / 64;
    // (not for prepacked weights: there the 128-column forms already send every weight load ahead
    // of the grid dependency and measure faster -- 1.5B M=16: 10.9 vs 12.2 us, 0.5B: 6.1 vs 6.6)
    const bool automatic = env().smallm_stack < 0 && nt128 < d.sm_count && nt64 <= 2 * d.sm_count &&
                           env().smallm_deep < 0 && kWMode != kWeightsPacked;
    if (env().smallm_stack == 1 || automatic)
      return launch_smallm_mp<MP, kAct, kWMode, kStoreGU, false, true>(d, A, W1, W2, Y, U, M, N, K, stream,
                                                                       probe, scale_gate, scale_up);
  }
  // Deep-ring form (one CTA per SM, six stages): taken when it is instantiated for this
  // (MP, weights) and some S <= 4 puts n-tiles x S on at most one CTA per SM.
  if constexpr (!kStack && !kDeep && !kStoreGU && MP <= 32 && (kWMode == kWeightsKN || kWMode == kWeightsPacked)) {
    const int64_t nt = (N + 127) / 128;
    const bool fits = nt < d.sm_count && (env().ksplit <= 0 || nt * env().ksplit <= d.sm_count);
    // automatic: only with prepacked (constant) weights and when the CTA's whole K-range fits the
    // ring, so that every weight byte is in flight before griddepcontrol.wait (0.5B: 6.8 -> 6.1 us;
    // with 12 k-blocks per CTA at 1.5B the two-CTA form stays ahead: profiles/r02_decode_study.md)
    const int64_t s_deep = smallm_ksplit(d.sm_count, 1, MP, nt, (K + 63) / 64);
    const bool resident = ((K + 63) / 64 + s_deep - 1) / s_deep <= SmallCfg<MP, true>::kStages;
    const bool automatic = env().smallm_deep < 0 && kWMode == kWeightsPacked && resident;
    if (fits && (env().smallm_deep == 1 || automatic))
      return launch_smallm_mp<MP, kAct, kWMode, kStoreGU, true>(d, A, W1, W2, Y, U, M, N, K, stream,
                                                                probe, scale_gate, scale_up);
  }
  constexpr bool kWK = (kWMode == kWeightsNK);
  constexpr int kBKe = (kWMode == kOperandsFp8) ? 128 : BK;
  CUtensorMap ta, tw1, tw2;
  int rc;
  if constexpr (kWMode == kOperandsFp8) {
    if ((rc = make_tmap_u8(&ta, A, K, M, MP))) return rc;
    if ((rc = make_tmap_u8(&tw1, W1, K, N, 64))) return rc;
    if ((rc = make_tmap_u8(&tw2, W2, K, N, 64))) return rc;
  } else if ((rc = make_tmap(&ta, A, K, M, 64, MP))) {
    return rc;
  }
  if constexpr (kWMode == kOperandsFp8) {
  } else if constexpr (kWMode == kWeightsPacked) {
    if ((rc = make_tmap_packed(&tw1, W1, K, packed_slabs(N), kStack ? 2 : 4))) return rc;  // W1 = Wp
    tw2 = tw1;
  } else {
    if ((rc = make_tmap(&tw1, W1, kWK ? K : N, kWK ? N : K, 64, 64))) return rc;
    if ((rc = make_tmap(&tw2, W2, kWK ? K : N, kWK ? N : K, 64, 64))) return rc;
  }
  using Cfg = SmallCfg<MP, kDeep, kStack>;
  const int64_t n_tiles = (N + Cfg::kTileN - 1) / Cfg::kTileN, k_blocks = (K + kBKe - 1) / kBKe;
  SmallParams p;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  p.ksplit = smallm_ksplit(d.sm_count, Cfg::kCtasPerSm, MP, n_tiles, k_blocks);
  if constexpr (kStack) {
    // stacked tile: a cluster only when the 64-column tiles alone leave half the SMs idle
    // (0.5B: 76 tiles -> S = 2; 1.5B: 140 tiles -> S = 1, measured 11.5 vs 12.4 us at M = 16)
    int64_t s = (d.sm_count + n_tiles / 2) / n_tiles;
    if (s > 4) s = 4;
    while (s > 1 && k_blocks / s < 4) --s;
    if (s < 1) s = 1;
    if (env().ksplit > 0) s = env().ksplit > 8 ? 8 : env().ksplit;
    if (s > k_blocks) s = k_blocks;
    p.ksplit = (int)s;
  }
  p.ldy = N;
  p.U = (uint16_t*)U;
  p.probe = probe;
  p.scale_gate = scale_gate;
  p.scale_up = scale_up;
  p.clk = g_clk.load(std::memory_order_relaxed);
  // L2 prefetch ahead of the grid dependency: at most ~32 MiB over the whole grid
  const int64_t grid = n_tiles * p.ksplit;
  int64_t pf = (32ll << 20) / (grid * 2 * Cfg::kWBytes);
  if (pf > kSmallPrefetchMax) pf = kSmallPrefetchMax;
  // ... and no more than 4 k-blocks or a third of the CTA's K-range: the prefetch only has to
  // cover the start-up latency behind griddepcontrol.wait; anything more competes with the
  // PREVIOUS call's weight stream for HBM (1.5B M=16, cap 0 / 2 / 4 / 8 / 14 k-blocks: 10.66 /
  // 10.44 / 10.42 / 10.46 / 11.51 us; 0.5B: 6.10 / 5.61 / 5.79 / 6.11 / 6.10; 7B: 40.8 / 40.0 / 39.5 /
  // 39.7 / 39.7 -- profiles/r02b_decode_stack_sweep.md)
  {
    const int64_t kb_per_cta = (k_blocks + p.ksplit - 1) / p.ksplit;
    int64_t cap = kb_per_cta / 3 < 4 ? kb_per_cta / 3 : 4;
    if (cap < 1) cap = 1;
    if (pf > cap) pf = cap;
  }
  if (env().no_prefetch) pf = 0;
  p.prefetch_blocks = (int)pf;
  // prepacked weights: two ring stages of real weight loads go out ahead of the grid dependency
  // (all of the ring / 4 / 2 / 1 / 0 stages, M = 16: 0.5B 6.25 / - / 5.97 / 6.06 / 6.39 us, 1.5B
  // 10.18 / - / 9.95 / 10.40 / 11.12 us: like the L2 prefetch, more only fights the previous call)
  p.packed_pre = 2;
#ifdef SWIGLU_TRACE
  p.trace = g_trace;
#endif
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof cfg);
  cfg.gridDim = dim3((unsigned)(n_tiles * p.ksplit));
  cfg.blockDim = dim3(kSmallThreads);
  cfg.dynamicSmemBytes = Cfg::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attrs[2];
  int na = 0;
  if (p.ksplit > 1) {
    attrs[na].id = cudaLaunchAttributeClusterDimension;
    attrs[na].val.clusterDim.x = (unsigned)p.ksplit;
    attrs[na].val.clusterDim.y = 1;
    attrs[na].val.clusterDim.z = 1;
    ++na;
  }
  if (pdl_enabled()) {
    attrs[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attrs[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = attrs;
  cfg.numAttrs = na;
  CUDA_TRY(cudaLaunchKernelEx(&cfg, smallm_swiglu_kernel<MP, kAct, kWMode, kStoreGU, kDeep, kStack>, ta, tw1,
                              tw2, (uint16_t*)Y, p));
  return SWIGLU_OK;
}

template <int kAct, int kWMode, bool kStoreGU = false>
int launch_smallm(const DeviceState& d, const void* A, const void* W1, const void* W2, void* Y,
                  void* U, int64_t M, int64_t N, int64_t K, cudaStream_t stream, int probe = 0,
                  float sg = 1.0f, float su = 1.0f) {
  if (M <= 16) return launch_smallm_mp<16, kAct, kWMode, kStoreGU>(d, A, W1, W2, Y, U, M, N, K, stream, probe, sg, su);
  if (M <= 32) return launch_smallm_mp<32, kAct, kWMode, kStoreGU>(d, A, W1, W2, Y, U, M, N, K, stream, probe, sg, su);
  if (M <= 64) return launch_smallm_mp<64, kAct, kWMode, kStoreGU>(d, A, W1, W2, Y, U, M, N, K, stream, probe, sg, su);
  return launch_smallm_mp<128, kAct, kWMode, kStoreGU>(d, A, W1, W2, Y, U, M, N, K, stream, probe, sg, su);
}

template <int kAct>
int launch_act_mul(const DeviceState& d, const void* G, const void* U, void* Y, int64_t elems,
                   cudaStream_t stream) {
  const int64_t n_vec = elems / 8;  // N % 8 == 0 so M*N % 8 == 0
  int64_t blocks = (n_vec + 255) / 256;
  const int64_t cap = (int64_t)d.sm_count * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof cfg);
  cfg.gridDim = dim3((unsigned)blocks);
  cfg.blockDim = dim3(256);
  cfg.stream = stream;
  cudaLaunchAttribute attrs[1];
  int na = 0;
  if (pdl_enabled()) {
    attrs[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attrs[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = attrs;
  cfg.numAttrs = na;
  CUDA_TRY(cudaLaunchKernelEx(&cfg, swiglu::silu_mul_kernel<kAct>, (const uint4*)G,
                              (const uint4*)U, (uint4*)Y, n_vec));
  return SWIGLU_OK;
}
int launch_silu_mul(const DeviceState& d, const void* G, const void* U, void* Y, int64_t elems,
                    int act, cudaStream_t stream) {
  using namespace swiglu;
  switch (act) {
    case kActSilu: return launch_act_mul<kActSilu>(d, G, U, Y, elems, stream);
    case kActGelu: return launch_act_mul<kActGelu>(d, G, U, Y, elems, stream);
    case kActGeluTanh: return launch_act_mul<kActGeluTanh>(d, G, U, Y, elems, stream);
    case kActRelu: return launch_act_mul<kActRelu>(d, G, U, Y, elems, stream);
  }
  return fail(SWIGLU_ERR_UNSUPPORTED, "unknown activation %d", act);
}

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

size_t workspace_for(int64_t M, int64_t N, int64_t K, int unfused, int variant) {
  if (M <= 0 || N <= 0 || K <= 0) return 0;
  if (unfused) return 2 * round_up((size_t)M * N * 2, 256);  // Gate and Up, bf16
  if (variant < 0) variant = select_fused(M, N, K);
  // The 128-column large-M kernels can cut their last partial wave in K through a workspace
  // (optional: without it they fall back to 64-column half tiles).  Sized for 148 SMs here --
  // this query makes no CUDA call.  The decode kernel reduces on chip (DSMEM): no workspace.
  if (variant == kFused1Cta || variant == kFused2Cta) {
    const int cg = variant == kFused2Cta ? 2 : 1;
    const int64_t tiles = ((M + 128 * cg - 1) / (128 * cg)) * ((N + 127) / 128);
    if (plan_tail(tiles, 148 / cg, (K + 63) / 64, true, true).ksplit >= 2) return kSplitWsBytes;
  }
  return 0;
}

// Library-owned buffer of `stream` in `pool`, at least `need` bytes.  Allocation and growth are
// STREAM-ORDERED (cudaMallocAsync / cudaFreeAsync on `stream`): the old block is released only
// after the work already enqueued on `stream` that may still use it, and nothing here
// synchronises.  Never under stream capture: a captured graph would keep a pointer the next
// growth frees, so capture needs the _ex form with a caller workspace (include/swiglu_mlp.h).
int ensure_stream_buffer(std::map<cudaStream_t, DeviceState::Buf>& pool, size_t need,
                         cudaStream_t stream, void** out) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(stream, &cap);
  if (cap != cudaStreamCaptureStatusNone)
    return fail(SWIGLU_ERR_WORKSPACE,
                "the library-owned workspace (%zu bytes) cannot be used while the stream is "
                "capturing; use the _ex form with a caller workspace", need);
  std::lock_guard<std::mutex> lk(g_mu);
  DeviceState::Buf& b = pool[stream];
  if (need > b.bytes) {
    if (b.ptr) {
      CUDA_TRY(cudaFreeAsync(b.ptr, stream));
      b.ptr = nullptr;
      b.bytes = 0;
    }
    CUDA_TRY(cudaMallocAsync(&b.ptr, need, stream));
    b.bytes = need;
  }
  *out = b.ptr;
  return SWIGLU_OK;
}

// Return every library-owned buffer of `pool` that belongs to `stream` (or to any stream).
int release_pool(std::map<cudaStream_t, DeviceState::Buf>& pool, bool all, cudaStream_t stream) {
  for (auto it = pool.begin(); it != pool.end();) {
    if (all || it->first == stream) {
      if (it->second.ptr) {
        if (all) CUDA_TRY(cudaFree(it->second.ptr));  // the caller has synchronised the device
        else CUDA_TRY(cudaFreeAsync(it->second.ptr, stream));
      }
      it = pool.erase(it);
    } else {
      ++it;
    }
  }
  return SWIGLU_OK;
}

template <int kAct, int kWK>
int launch_fused_l(const DeviceState& d, int variant, const void* A, const void* W1,
                   const void* W2, void* Y, int64_t M, int64_t N, int64_t K, cudaStream_t stream,
                   void* split_ws) {
  switch (variant) {
    case kFused1Cta: return launch_gemm<1, true, 128, kAct, kWK>(d, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kFused2Cta: return launch_gemm<2, true, 128, kAct, kWK>(d, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kFusedSmallM: return launch_smallm<kAct, kWK>(d, A, W1, W2, Y, nullptr, M, N, K, stream);
    case kFused1CtaN64: return launch_gemm<1, true, 64, kAct, kWK>(d, A, W1, W2, Y, M, N, K, stream);
    case kFused2Cta4: return launch_gemm<2, true, 128, kAct, kWK, 2>(d, A, W1, W2, Y, M, N, K, stream);
    case kFused2CtaMB2: return launch_gemm<2, true, 128, kAct, kWK, 1, 2>(d, A, W1, W2, Y, M, N, K, stream);
  }
  return fail(SWIGLU_ERR_UNSUPPORTED, "unknown fused variant %d", variant);
}
template <int kAct>
int launch_fused(const DeviceState& d, int variant, int layout, const void* A, const void* W1,
                 const void* W2, void* Y, int64_t M, int64_t N, int64_t K, cudaStream_t stream,
                 void* split_ws) {
  switch (layout) {
    case kWeightsNK: return launch_fused_l<kAct, kWeightsNK>(d, variant, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kWeightsPacked: return launch_fused_l<kAct, kWeightsPacked>(d, variant, A, W1, W2, Y, M, N, K, stream, split_ws);
  }
  return launch_fused_l<kAct, kWeightsKN>(d, variant, A, W1, W2, Y, M, N, K, stream, split_ws);
}

// Library-owned K-split workspace of `stream`: FIXED size (never regrown, so a captured graph's
// pointer stays valid until swiglu_release), counters zeroed once in stream order.  Not created
// while the stream is capturing: the caller then gets no K split (half tiles instead) unless it
// passes its own workspace through the _ex form.
void* split_workspace(DeviceState& d, cudaStream_t stream) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = d.split_ws.find(stream);
  if (it != d.split_ws.end()) return it->second.ptr;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(stream, &cap);
  if (cap != cudaStreamCaptureStatusNone) return nullptr;
  void* ptr = nullptr;
  if (cudaMallocAsync(&ptr, kSplitWsBytes, stream) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  if (cudaMemsetAsync(ptr, 0, kSplitCtrBytes, stream) != cudaSuccess) {
    cudaGetLastError();
    cudaFreeAsync(ptr, stream);
    return nullptr;
  }
  d.split_ws[stream] = DeviceState::Buf{ptr, kSplitWsBytes};
  return ptr;
}

// layout: SWIGLU_WEIGHTS_KN / _NK, or kWeightsPacked (internal: W1 = W2 = the packed buffer).
// ws / own_ws: the optional K-split workspace (see plan_tail): the caller's (own_ws == false; used
// if it is large enough, ignored otherwise) or the library's per-stream one.
int run_fused(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
              int64_t K, int variant, int act, int layout, cudaStream_t stream,
              void* ws = nullptr, size_t ws_bytes = 0, bool own_ws = true) {
  if (layout != SWIGLU_WEIGHTS_KN && layout != SWIGLU_WEIGHTS_NK && layout != kWeightsPacked)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown weight layout %d", layout);
  int rc = validate(A, W1, W2, Y, M, N, K);
  if (rc) return rc;
  if (layout == kWeightsPacked && M > 0) {
    // the packed buffer is 2 * K * pad128(N) elements: re-check aliasing against its real size
    const int64_t pb = packed_slabs(N) * packed_rows(K) * 128;
    if (overlaps(Y, M * N * 2, W1, pb)) return fail(SWIGLU_ERR_ALIASING, "Y overlaps Wp");
  }
  if (act < 0 || act >= swiglu::kNumActs)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown activation %d", act);
  if (variant < -1 || variant >= kNumFused)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown fused variant %d", variant);
  if (variant == kFusedSmallM && M > swiglu::kSmallMMax)
    return fail(SWIGLU_ERR_UNSUPPORTED, "variant %s handles M <= %d only",
                kFusedNames[kFusedSmallM], swiglu::kSmallMMax);
  if (M == 0) return SWIGLU_OK;
  DeviceState* d;
  if ((rc = get_device_state(&d))) return rc;
  if (variant < 0) variant = select_fused(M, N, K);
  void* split_ws = nullptr;
  if (workspace_for(M, N, K, 0, variant) > 0) {
    if (own_ws) split_ws = split_workspace(*d, stream);
    else if (ws && ws_bytes >= kSplitWsBytes && !((uintptr_t)ws & 255u)) split_ws = ws;
  }
  using namespace swiglu;
  switch (act) {
    case kActSilu: return launch_fused<kActSilu>(*d, variant, layout, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kActGelu: return launch_fused<kActGelu>(*d, variant, layout, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kActGeluTanh: return launch_fused<kActGeluTanh>(*d, variant, layout, A, W1, W2, Y, M, N, K, stream, split_ws);
    case kActRelu: return launch_fused<kActRelu>(*d, variant, layout, A, W1, W2, Y, M, N, K, stream, split_ws);
  }
  return fail(SWIGLU_ERR_UNSUPPORTED, "unknown activation %d", act);
}

int run_unfused(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
                int64_t K, void* ws, size_t ws_bytes, bool own_ws, int variant, int act,
                int layout, cudaStream_t stream) {
  if (layout != SWIGLU_WEIGHTS_KN && layout != SWIGLU_WEIGHTS_NK)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown weight layout %d", layout);
  int rc = validate(A, W1, W2, Y, M, N, K);
  if (rc) return rc;
  if (act < 0 || act >= swiglu::kNumActs)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown activation %d", act);
  if (variant < -1 || variant >= kNumUnfused)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown unfused variant %d", variant);
  if (variant == kUnfusedSmallM && M > swiglu::kSmallMMax)
    return fail(SWIGLU_ERR_UNSUPPORTED, "variant %s handles M <= %d only",
                kUnfusedNames[kUnfusedSmallM], swiglu::kSmallMMax);
  if (M == 0) return SWIGLU_OK;
  const size_t need = workspace_for(M, N, K, 1, variant);
  if (!own_ws) {
    if (!ws || ws_bytes < need || ((uintptr_t)ws & 255u))
      return fail(SWIGLU_ERR_WORKSPACE, "workspace needs %zu bytes, 256-byte aligned", need);
  }
  DeviceState* d;
  if ((rc = get_device_state(&d))) return rc;
  if (own_ws && (rc = ensure_stream_buffer(d->workspace, need, stream, &ws))) return rc;
  if (variant < 0) variant = select_unfused(M, N, K);
  void* G = ws;
  void* U = (char*)ws + need / 2;
  using namespace swiglu;
  if (variant == kUnfusedSmallM) {
    rc = layout ? launch_smallm<kActSilu, kWeightsNK, true>(*d, A, W1, W2, G, U, M, N, K, stream)
                : launch_smallm<kActSilu, kWeightsKN, true>(*d, A, W1, W2, G, U, M, N, K, stream);
    if (rc) return rc;
  } else if (variant == kUnfused1Cta && !layout) {
    if ((rc = launch_gemm<1, false>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<1, false>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  } else if (variant == kUnfused1Cta) {
    if ((rc = launch_gemm<1, false, 128, kActSilu, kWeightsNK>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<1, false, 128, kActSilu, kWeightsNK>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  } else if (variant == kUnfused2CtaMB2 && !layout) {
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsKN, 1, 2>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsKN, 1, 2>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  } else if (variant == kUnfused2CtaMB2) {
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsNK, 1, 2>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsNK, 1, 2>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  } else if (!layout) {
    if ((rc = launch_gemm<2, false>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<2, false>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  } else {
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsNK>(*d, A, W1, W1, G, M, N, K, stream))) return rc;
    if ((rc = launch_gemm<2, false, 128, kActSilu, kWeightsNK>(*d, A, W2, W2, U, M, N, K, stream))) return rc;
  }
  return launch_silu_mul(*d, G, U, Y, M * N, act, stream);
}

// Device address of g_static_scratch on the CURRENT device, resolved once per device.
std::mutex g_static_mu;
void* g_static_addr[64] = {nullptr};
int static_scratch_address(void** out) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(SWIGLU_ERR_CUDA, "device index %d out of range", dev);
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_addr[dev]) {
    void* ptr = nullptr;
    CUDA_TRY(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));  // `dev` is current
    if (!ptr || ((uintptr_t)ptr & 255u))
      return fail(SWIGLU_ERR_CUDA, "static scratch resolved to a bad address %p", ptr);
    g_static_addr[dev] = ptr;
  }
  *out = g_static_addr[dev];
  return SWIGLU_OK;
}

}  // namespace

// ====================================================================== C ABI
extern "C" {

int swiglu_validate(const void* A, const void* W1, const void* W2, const void* Y, int64_t M,
                    int64_t N, int64_t K) {
  return validate(A, W1, W2, Y, M, N, K);
}

int swiglu_mlp(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
               int64_t K, void* stream) {
  return run_fused(A, W1, W2, Y, M, N, K, -1, swiglu::kActSilu, 0, (cudaStream_t)stream);
}

int swiglu_mlp_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
                  int64_t K, void* workspace, size_t workspace_bytes, int variant,
                  void* stream) {
  // optional: only the K split of the last wave uses it (swiglu_workspace_bytes says when)
  return run_fused(A, W1, W2, Y, M, N, K, variant, swiglu::kActSilu, 0, (cudaStream_t)stream,
                   workspace, workspace_bytes, false);
}

int swiglu_mlp_unfused(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                       int64_t N, int64_t K, void* stream) {
  return run_unfused(A, W1, W2, Y, M, N, K, nullptr, 0, true, -1, swiglu::kActSilu, 0,
                     (cudaStream_t)stream);
}

int swiglu_mlp_unfused_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                          int64_t N, int64_t K, void* workspace, size_t workspace_bytes,
                          int variant, void* stream) {
  return run_unfused(A, W1, W2, Y, M, N, K, workspace, workspace_bytes, false, variant,
                     swiglu::kActSilu, 0, (cudaStream_t)stream);
}

int swiglu_mlp_unfused_static(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                              int64_t N, int64_t K, void* stream) {
  int rc = validate(A, W1, W2, Y, M, N, K);  // no CUDA call yet
  if (rc) return rc;
  if (M == 0) return SWIGLU_OK;
  const size_t need = workspace_for(M, N, K, 1, -1);
  if (need > (size_t)SWIGLU_STATIC_SCRATCH_BYTES)
    return fail(SWIGLU_ERR_WORKSPACE,
                "M=%lld x N=%lld needs %zu bytes of Gate/Up scratch; the static scratch of "
                "swiglu_mlp_unfused_static holds %u (use swiglu_mlp_unfused_ex with a caller workspace)",
                (long long)M, (long long)N, need, (unsigned)SWIGLU_STATIC_SCRATCH_BYTES);
  void* scratch = nullptr;
  if ((rc = static_scratch_address(&scratch))) return rc;
  return run_unfused(A, W1, W2, Y, M, N, K, scratch, SWIGLU_STATIC_SCRATCH_BYTES, false, -1,
                     swiglu::kActSilu, 0, (cudaStream_t)stream);
}

int swiglu_glu_mlp(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
                   int64_t K, int activation, void* stream) {
  return run_fused(A, W1, W2, Y, M, N, K, -1, activation, 0, (cudaStream_t)stream);
}

int swiglu_glu_mlp_unfused(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                           int64_t N, int64_t K, int activation, void* stream) {
  return run_unfused(A, W1, W2, Y, M, N, K, nullptr, 0, true, -1, activation, 0,
                     (cudaStream_t)stream);
}

int swiglu_glu_mlp_layout(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                          int64_t N, int64_t K, int activation, int weight_layout, int unfused,
                          int variant, void* stream) {
  if (weight_layout != SWIGLU_WEIGHTS_KN && weight_layout != SWIGLU_WEIGHTS_NK)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown weight layout %d", weight_layout);
  if (unfused)
    return run_unfused(A, W1, W2, Y, M, N, K, nullptr, 0, true, variant, activation,
                       weight_layout, (cudaStream_t)stream);
  return run_fused(A, W1, W2, Y, M, N, K, variant, activation, weight_layout,
                   (cudaStream_t)stream);
}

int swiglu_glu_mlp_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                      int64_t N, int64_t K, int activation, int variant, void* stream) {
  return run_fused(A, W1, W2, Y, M, N, K, variant, activation, 0, (cudaStream_t)stream);
}

size_t swiglu_packed_weight_bytes(int64_t N, int64_t K) {
  if (N <= 0 || K <= 0 || (N % 8) || (K % 8)) return 0;
  return (size_t)packed_slabs(N) * (size_t)packed_rows(K) * 128;
}

int swiglu_pack_weights(const void* W1, const void* W2, void* Wp, int64_t N, int64_t K,
                        int weight_layout, void* stream) {
  if (weight_layout != SWIGLU_WEIGHTS_KN && weight_layout != SWIGLU_WEIGHTS_NK)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown weight layout %d", weight_layout);
  // same shape / pointer rules as a compute call with one row (Wp plays the part of Y)
  int rc = validate(W1, W1, W2, Wp, 1, N, K);
  if (rc == SWIGLU_ERR_ALIASING) rc = SWIGLU_OK;  // checked against the real sizes below
  if (rc) return rc;
  const int64_t wb = K * N * 2, pb = (int64_t)swiglu_packed_weight_bytes(N, K);
  if (overlaps(Wp, pb, W1, wb) || overlaps(Wp, pb, W2, wb))
    return fail(SWIGLU_ERR_ALIASING, "Wp overlaps W1 or W2");
  DeviceState* d;
  if ((rc = get_device_state(&d))) return rc;
  const long long total_vec = pb / 16;
  long long blocks = (total_vec + 255) / 256;
  const long long cap = (long long)d->sm_count * 16;
  if (blocks > cap) blocks = cap;
  if (weight_layout == SWIGLU_WEIGHTS_NK)
    swiglu::pack_weights_kernel<true><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(
        (const uint16_t*)W1, (const uint16_t*)W2, (uint16_t*)Wp, (int)N, (int)K, (int)packed_rows(K), total_vec);
  else
    swiglu::pack_weights_kernel<false><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(
        (const uint16_t*)W1, (const uint16_t*)W2, (uint16_t*)Wp, (int)N, (int)K, (int)packed_rows(K), total_vec);
  CUDA_TRY(cudaGetLastError());
  return SWIGLU_OK;
}

int swiglu_mlp_packed(const void* A, const void* Wp, void* Y, int64_t M, int64_t N, int64_t K,
                      void* stream) {
  return run_fused(A, Wp, Wp, Y, M, N, K, -1, swiglu::kActSilu, swiglu::kWeightsPacked,
                   (cudaStream_t)stream);
}

int swiglu_glu_mlp_packed(const void* A, const void* Wp, void* Y, int64_t M, int64_t N, int64_t K,
                          int activation, int variant, void* stream) {
  return run_fused(A, Wp, Wp, Y, M, N, K, variant, activation, swiglu::kWeightsPacked,
                   (cudaStream_t)stream);
}

// FP8 (E4M3) operands; see include/swiglu_mlp.h.
static int run_fp8(const void* A8, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
                   int64_t K, float sg, float su, int variant, cudaStream_t stream) {
  if (M < 0 || N <= 0 || K <= 0)
    return fail(SWIGLU_ERR_BAD_SHAPE, "bad shape M=%lld N=%lld K=%lld (need M>=0, N>0, K>0)",
                (long long)M, (long long)N, (long long)K);
  if (M > INT32_MAX - 256 || N > INT32_MAX - 256 || K > INT32_MAX - 256 ||
      mul_overflows(M, K, INT64_MAX / 4) || mul_overflows(K, N, INT64_MAX / 4) ||
      mul_overflows(M, N, INT64_MAX / 4))
    return fail(SWIGLU_ERR_BAD_SHAPE, "shape too large M=%lld N=%lld K=%lld", (long long)M,
                (long long)N, (long long)K);
  if ((K % 16) != 0 || (N % 8) != 0)
    return fail(SWIGLU_ERR_UNSUPPORTED,
                "FP8: K=%lld must be a multiple of 16 and N=%lld of 8 (16-byte row pitch for TMA)",
                (long long)K, (long long)N);
  if (!(sg == sg) || !(su == su)) return fail(SWIGLU_ERR_UNSUPPORTED, "a scale is NaN");
  if (variant < -1 || variant >= kNumFused)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown fused variant %d", variant);
  if (variant == kFusedSmallM && M > swiglu::kSmallMMax)
    return fail(SWIGLU_ERR_UNSUPPORTED, "variant %s handles M <= %d only",
                kFusedNames[kFusedSmallM], swiglu::kSmallMMax);
  if (M == 0) return SWIGLU_OK;
  if (!A8 || !W1 || !W2 || !Y) return fail(SWIGLU_ERR_NULL_POINTER, "A, W1, W2 or Y is NULL");
  if (((uintptr_t)A8 | (uintptr_t)W1 | (uintptr_t)W2 | (uintptr_t)Y) & 15u)
    return fail(SWIGLU_ERR_MISALIGNED, "A, W1, W2 and Y must be 16-byte aligned");
  if (overlaps(Y, M * N * 2, A8, M * K) || overlaps(Y, M * N * 2, W1, K * N) ||
      overlaps(Y, M * N * 2, W2, K * N))
    return fail(SWIGLU_ERR_ALIASING, "Y overlaps an input");
  DeviceState* d;
  int rc;
  if ((rc = get_device_state(&d))) return rc;
  if (variant < 0) variant = select_fused(M, N, K / 2);  // a k-block is 128 one-byte elements
  using namespace swiglu;
  void* split_ws = workspace_for(M, N, K / 2, 0, variant) > 0 ? split_workspace(*d, stream) : nullptr;
  switch (variant) {
    case kFused1Cta:
      return launch_gemm<1, true, 128, kActSilu, kOperandsFp8>(*d, A8, W1, W2, Y, M, N, K, stream, split_ws, sg, su);
    case kFused2Cta:
      return launch_gemm<2, true, 128, kActSilu, kOperandsFp8>(*d, A8, W1, W2, Y, M, N, K, stream, split_ws, sg, su);
    case kFusedSmallM:
      return launch_smallm<kActSilu, kOperandsFp8>(*d, A8, W1, W2, Y, nullptr, M, N, K, stream, 0, sg, su);
    case kFused1CtaN64:
      return launch_gemm<1, true, 64, kActSilu, kOperandsFp8>(*d, A8, W1, W2, Y, M, N, K, stream, nullptr, sg, su);
    case kFused2Cta4:
      return launch_gemm<2, true, 128, kActSilu, kOperandsFp8, 2>(*d, A8, W1, W2, Y, M, N, K, stream, nullptr, sg, su);
    case kFused2CtaMB2:
      return launch_gemm<2, true, 128, kActSilu, kOperandsFp8, 1, 2>(*d, A8, W1, W2, Y, M, N, K, stream, nullptr, sg, su);
  }
  return fail(SWIGLU_ERR_UNSUPPORTED, "unknown fused variant %d", variant);
}

int swiglu_mlp_fp8(const void* A8, const void* W1_8, const void* W2_8, void* Y, int64_t M,
                   int64_t N, int64_t K, float scale_gate, float scale_up, void* stream) {
  return run_fp8(A8, W1_8, W2_8, Y, M, N, K, scale_gate, scale_up, -1, (cudaStream_t)stream);
}

int swiglu_mlp_fp8_ex(const void* A8, const void* W1_8, const void* W2_8, void* Y, int64_t M,
                      int64_t N, int64_t K, float scale_gate, float scale_up, int variant,
                      void* stream) {
  return run_fp8(A8, W1_8, W2_8, Y, M, N, K, scale_gate, scale_up, variant, (cudaStream_t)stream);
}

int swiglu_launch_floor_probe(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                              int64_t N, int64_t K, void* stream) {
  int rc = validate(A, W1, W2, Y, M, N, K);
  if (rc) return rc;
  if (M == 0) return SWIGLU_OK;
  if (M > swiglu::kSmallMMax)
    return fail(SWIGLU_ERR_UNSUPPORTED, "the launch-floor probe mirrors the small-M kernel: M <= %d",
                swiglu::kSmallMMax);
  DeviceState* d;
  if ((rc = get_device_state(&d))) return rc;
  return launch_smallm<swiglu::kActSilu, swiglu::kWeightsKN>(*d, A, W1, W2, Y, nullptr, M, N, K,
                                                             (cudaStream_t)stream, /*probe=*/1);
}

const char* swiglu_activation_name(int activation) {
  switch (activation) {
    case SWIGLU_ACT_SILU: return "silu";
    case SWIGLU_ACT_GELU: return "gelu";
    case SWIGLU_ACT_GELU_TANH: return "gelu_tanh";
    case SWIGLU_ACT_RELU: return "relu";
  }
  return nullptr;
}

int swiglu_silu_mul(const void* G, const void* U, void* Y, int64_t elems, void* stream) {
  return swiglu_act_mul(G, U, Y, elems, SWIGLU_ACT_SILU, stream);
}

int swiglu_act_mul(const void* G, const void* U, void* Y, int64_t elems, int activation,
                   void* stream) {
  if (activation < 0 || activation >= swiglu::kNumActs)
    return fail(SWIGLU_ERR_UNSUPPORTED, "unknown activation %d", activation);
  if (elems < 0) return fail(SWIGLU_ERR_BAD_SHAPE, "elems=%lld < 0", (long long)elems);
  if (elems % 8) return fail(SWIGLU_ERR_UNSUPPORTED, "elems=%lld must be a multiple of 8", (long long)elems);
  if (elems == 0) return SWIGLU_OK;
  if (!G || !U || !Y) return fail(SWIGLU_ERR_NULL_POINTER, "G, U or Y is NULL");
  if (((uintptr_t)G | (uintptr_t)U | (uintptr_t)Y) & 15u)
    return fail(SWIGLU_ERR_MISALIGNED, "G, U and Y must be 16-byte aligned");
  DeviceState* d;
  int rc = get_device_state(&d);
  if (rc) return rc;
  return launch_silu_mul(*d, G, U, Y, elems, activation, (cudaStream_t)stream);
}

size_t swiglu_workspace_bytes(int64_t M, int64_t N, int64_t K, int unfused, int variant) {
  return workspace_for(M, N, K, unfused, variant);
}

int swiglu_num_variants(int unfused) { return unfused ? (int)kNumUnfused : (int)kNumFused; }

const char* swiglu_variant_name(int unfused, int variant) {
  if (variant < 0 || variant >= (unfused ? (int)kNumUnfused : (int)kNumFused)) return nullptr;
  return unfused ? kUnfusedNames[variant] : kFusedNames[variant];
}

int swiglu_selected_variant(int64_t M, int64_t N, int64_t K, int unfused) {
  return unfused ? select_unfused(M, N, K) : select_fused(M, N, K);
}

int swiglu_launches_per_call(int64_t M, int64_t N, int64_t K, int unfused, int variant) {
  if (M <= 0) return 0;
  if (!unfused) return 1;
  if (variant < 0) variant = select_unfused(M, N, K);
  return variant == kUnfusedSmallM ? 2 : 3;  // merged Gate|Up GEMM, or two GEMMs; + elementwise
}

int swiglu_mlp_host(const void* A_host, const void* W1_host, const void* W2_host, void* Y_host,
                    int64_t M, int64_t N, int64_t K, int unfused, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  // validate shapes/pointers with the host pointers (alignment of host buffers is irrelevant)
  if (M < 0 || N <= 0 || K <= 0) return validate(nullptr, nullptr, nullptr, nullptr, M, N, K);
  if ((K % 8) || (N % 8)) return validate(nullptr, nullptr, nullptr, nullptr, M, N, K);
  if (M == 0) return SWIGLU_OK;
  if (!A_host || !W1_host || !W2_host || !Y_host)
    return fail(SWIGLU_ERR_NULL_POINTER, "a host pointer is NULL");
  DeviceState* d;
  int rc = get_device_state(&d);
  if (rc) return rc;
  const size_t ab = round_up((size_t)M * K * 2, 256), wb = round_up((size_t)K * N * 2, 256),
               yb = round_up((size_t)M * N * 2, 256);
  const size_t need = ab + 2 * wb + yb;
  void* scratch;
  if ((rc = ensure_stream_buffer(d->host_scratch, need, stream, &scratch))) return rc;
  char* base = (char*)scratch;
  void *dA = base, *dW1 = base + ab, *dW2 = base + ab + wb, *dY = base + ab + 2 * wb;
  CUDA_TRY(cudaMemcpyAsync(dA, A_host, (size_t)M * K * 2, cudaMemcpyHostToDevice, stream));
  CUDA_TRY(cudaMemcpyAsync(dW1, W1_host, (size_t)K * N * 2, cudaMemcpyHostToDevice, stream));
  CUDA_TRY(cudaMemcpyAsync(dW2, W2_host, (size_t)K * N * 2, cudaMemcpyHostToDevice, stream));
  rc = unfused ? swiglu_mlp_unfused(dA, dW1, dW2, dY, M, N, K, stream_v)
               : swiglu_mlp(dA, dW1, dW2, dY, M, N, K, stream_v);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(Y_host, dY, (size_t)M * N * 2, cudaMemcpyDeviceToHost, stream));
  CUDA_TRY(cudaStreamSynchronize(stream));
  return SWIGLU_OK;
}

int swiglu_mlp_host_batched(const void* const* A_host, void* const* Y_host, const int64_t* M,
                            int count, const void* W1_host, const void* W2_host, int64_t N,
                            int64_t K, int unfused, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (count < 0) return fail(SWIGLU_ERR_BAD_SHAPE, "count=%d < 0", count);
  if (N <= 0 || K <= 0 || (K % 8) || (N % 8))
    return validate(nullptr, nullptr, nullptr, nullptr, 0, N, K);
  if (count == 0) return SWIGLU_OK;
  if (!A_host || !Y_host || !M || !W1_host || !W2_host)
    return fail(SWIGLU_ERR_NULL_POINTER, "a host pointer is NULL");
  int64_t rows = 0;
  for (int i = 0; i < count; ++i) {
    if (M[i] < 0 || M[i] > INT32_MAX - 256)
      return fail(SWIGLU_ERR_BAD_SHAPE, "bad batch size M[%d]=%lld", i, (long long)M[i]);
    if (M[i] > 0 && (!A_host[i] || !Y_host[i]))
      return fail(SWIGLU_ERR_NULL_POINTER, "A_host[%d] or Y_host[%d] is NULL", i, i);
    rows += M[i];
  }
  if (rows == 0) return SWIGLU_OK;
  DeviceState* d;
  int rc = get_device_state(&d);
  if (rc) return rc;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(stream, &cap);
  if (cap != cudaStreamCaptureStatusNone)
    return fail(SWIGLU_ERR_UNSUPPORTED, "the host-buffer forms synchronise; not capturable");
  // One pipeline per DEVICE at a time (it owns that device's copy streams and events).
  std::lock_guard<std::mutex> host_lk(d->host_mu);
  if (!d->s_in) {
    CUDA_TRY(cudaStreamCreateWithFlags(&d->s_in, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&d->s_out, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&d->ev_a, cudaEventDisableTiming));
    for (int b = 0; b < 2; ++b) {
      CUDA_TRY(cudaEventCreateWithFlags(&d->ev_in[b], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&d->ev_cmp[b], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&d->ev_out[b], cudaEventDisableTiming));
    }
  }
  // Column chunks of the weights: H2D of chunk j+1 and D2H of chunk j-1 run under the kernels
  // of chunk j (the path has no dependency between output columns).
  const int want_chunks = env().host_chunks;
  int64_t nc = round_up((size_t)((N + want_chunks - 1) / want_chunks), 128);
  if (nc < 512) nc = 512;
  if (nc > N) nc = N;
  const int chunks = (int)((N + nc - 1) / nc);
  const size_t a_bytes = round_up((size_t)rows * K * 2, 256);
  const size_t w_bytes = round_up((size_t)K * nc * 2, 256);
  // One Y buffer holds every batch's [M[i], nc] block, each block padded to 256 bytes.
  size_t y_bytes = 0;
  for (int i = 0; i < count; ++i)
    if (M[i] > 0) y_bytes += round_up((size_t)M[i] * nc * 2, 256);
  void* scratch;
  if ((rc = ensure_stream_buffer(d->host_scratch, a_bytes + 4 * w_bytes + 2 * y_bytes, stream,
                                 &scratch)))
    return rc;
  char* dA = (char*)scratch;
  char* dW = dA + a_bytes;                // [2 buffers][W1c | W2c]
  char* dY = dW + 4 * w_bytes;            // [2 buffers][sum_i pad256(M[i] x nc)]

  // The enqueue phase.  On ANY failure the copies and kernels already enqueued still reference
  // the library's scratch and the caller's host buffers: drain all three streams before
  // returning the error, so the caller may free its buffers as soon as the call is back.
  auto enqueue = [&]() -> int {
    // everything the caller enqueued on `stream` so far comes first
    CUDA_TRY(cudaEventRecord(d->ev_a, stream));
    CUDA_TRY(cudaStreamWaitEvent(d->s_in, d->ev_a, 0));
    CUDA_TRY(cudaStreamWaitEvent(d->s_out, d->ev_a, 0));
    size_t off = 0;
    for (int i = 0; i < count; ++i) {
      if (M[i] == 0) continue;
      CUDA_TRY(cudaMemcpyAsync(dA + off, A_host[i], (size_t)M[i] * K * 2, cudaMemcpyHostToDevice,
                               d->s_in));
      off += (size_t)M[i] * K * 2;
    }
    for (int j = 0; j < chunks; ++j) {
      const int b = j & 1;
      const int64_t n0 = (int64_t)j * nc, ncj = (n0 + nc <= N) ? nc : N - n0;
      char* w1c = dW + (size_t)b * 2 * w_bytes;
      char* w2c = w1c + w_bytes;
      char* yc = dY + (size_t)b * y_bytes;
      // H2D: the weight columns [n0, n0 + ncj), packed dense [K, ncj]
      if (j >= 2) CUDA_TRY(cudaStreamWaitEvent(d->s_in, d->ev_cmp[b], 0));  // buffer b consumed
      CUDA_TRY(cudaMemcpy2DAsync(w1c, (size_t)ncj * 2, (const char*)W1_host + n0 * 2,
                                 (size_t)N * 2, (size_t)ncj * 2, (size_t)K,
                                 cudaMemcpyHostToDevice, d->s_in));
      CUDA_TRY(cudaMemcpy2DAsync(w2c, (size_t)ncj * 2, (const char*)W2_host + n0 * 2,
                                 (size_t)N * 2, (size_t)ncj * 2, (size_t)K,
                                 cudaMemcpyHostToDevice, d->s_in));
      CUDA_TRY(cudaEventRecord(d->ev_in[b], d->s_in));
      // compute on the caller's stream
      CUDA_TRY(cudaStreamWaitEvent(stream, d->ev_in[b], 0));
      if (j >= 2) CUDA_TRY(cudaStreamWaitEvent(stream, d->ev_out[b], 0));  // Y buffer b drained
      size_t a_off = 0, y_off = 0;
      for (int i = 0; i < count; ++i) {
        if (M[i] == 0) continue;
        const int r = unfused
                          ? swiglu_mlp_unfused(dA + a_off, w1c, w2c, yc + y_off, M[i], ncj, K, stream_v)
                          : swiglu_mlp(dA + a_off, w1c, w2c, yc + y_off, M[i], ncj, K, stream_v);
        if (r) return r;
        a_off += (size_t)M[i] * K * 2;
        y_off += round_up((size_t)M[i] * nc * 2, 256);
      }
      CUDA_TRY(cudaEventRecord(d->ev_cmp[b], stream));
      // D2H: scatter the chunk's columns into each batch's Y
      CUDA_TRY(cudaStreamWaitEvent(d->s_out, d->ev_cmp[b], 0));
      y_off = 0;
      for (int i = 0; i < count; ++i) {
        if (M[i] == 0) continue;
        CUDA_TRY(cudaMemcpy2DAsync((char*)Y_host[i] + n0 * 2, (size_t)N * 2, yc + y_off,
                                   (size_t)ncj * 2, (size_t)ncj * 2, (size_t)M[i],
                                   cudaMemcpyDeviceToHost, d->s_out));
        y_off += round_up((size_t)M[i] * nc * 2, 256);
      }
      CUDA_TRY(cudaEventRecord(d->ev_out[b], d->s_out));
    }
    return SWIGLU_OK;
  };
  rc = enqueue();
  const cudaError_t e_in = cudaStreamSynchronize(d->s_in);
  const cudaError_t e_out = cudaStreamSynchronize(d->s_out);
  const cudaError_t e_cmp = cudaStreamSynchronize(stream);
  if (rc) return rc;  // g_err holds the enqueue failure
  if (e_in != cudaSuccess) return fail_cuda(e_in, "cudaStreamSynchronize(copy-in stream)");
  if (e_out != cudaSuccess) return fail_cuda(e_out, "cudaStreamSynchronize(copy-out stream)");
  if (e_cmp != cudaSuccess) return fail_cuda(e_cmp, "cudaStreamSynchronize(stream)");
  return SWIGLU_OK;
}

int swiglu_release_stream(void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(SWIGLU_ERR_CUDA, "device index %d out of range", dev);
  std::lock_guard<std::mutex> lk(g_mu);
  DeviceState& d = g_dev[dev];
  int rc;
  if ((rc = release_pool(d.workspace, false, stream))) return rc;
  if ((rc = release_pool(d.split_ws, false, stream))) return rc;
  return release_pool(d.host_scratch, false, stream);
}

int swiglu_release(void) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(SWIGLU_ERR_CUDA, "device index %d out of range", dev);
  CUDA_TRY(cudaDeviceSynchronize());  // nothing of ours may still be running on the buffers
  DeviceState& d = g_dev[dev];
  std::lock_guard<std::mutex> host_lk(d.host_mu);  // lock order: host_mu, then g_mu
  std::lock_guard<std::mutex> lk(g_mu);
  int rc;
  if ((rc = release_pool(d.workspace, true, nullptr))) return rc;
  if ((rc = release_pool(d.split_ws, true, nullptr))) return rc;
  if ((rc = release_pool(d.host_scratch, true, nullptr))) return rc;
  if (d.s_in) {
    cudaStreamDestroy(d.s_in);
    cudaStreamDestroy(d.s_out);
    cudaEventDestroy(d.ev_a);
    for (int b = 0; b < 2; ++b) {
      cudaEventDestroy(d.ev_in[b]);
      cudaEventDestroy(d.ev_cmp[b]);
      cudaEventDestroy(d.ev_out[b]);
    }
    d.s_in = d.s_out = nullptr;
  }
  return SWIGLU_OK;
}

void swiglu_reload_env(void) { load_env(); }

void swiglu_set_clock_probe(void* device_u64x2) {
  g_clk.store((unsigned long long*)device_u64x2, std::memory_order_relaxed);
}

int swiglu_tensor_map_cache_stats(uint64_t* hits, uint64_t* misses) {
  if (hits) *hits = t_tmap_hits;
  if (misses) *misses = t_tmap_misses;
  return kTmapSlots;
}

#ifdef SWIGLU_TRACE
void swiglu_debug_set_trace(void* device_buffer) { g_trace = (unsigned long long*)device_buffer; }
#endif

const char* swiglu_last_error(void) { return g_err; }

const char* swiglu_status_string(int status) {
  switch (status) {
    case SWIGLU_OK: return "SWIGLU_OK";
    case SWIGLU_ERR_NULL_POINTER: return "SWIGLU_ERR_NULL_POINTER";
    case SWIGLU_ERR_BAD_SHAPE: return "SWIGLU_ERR_BAD_SHAPE";
    case SWIGLU_ERR_UNSUPPORTED: return "SWIGLU_ERR_UNSUPPORTED";
    case SWIGLU_ERR_MISALIGNED: return "SWIGLU_ERR_MISALIGNED";
    case SWIGLU_ERR_ALIASING: return "SWIGLU_ERR_ALIASING";
    case SWIGLU_ERR_ARCH: return "SWIGLU_ERR_ARCH";
    case SWIGLU_ERR_WORKSPACE: return "SWIGLU_ERR_WORKSPACE";
    case SWIGLU_ERR_CUDA: return "SWIGLU_ERR_CUDA";
  }
  return "SWIGLU_ERR_UNKNOWN";
}

const char* swiglu_version(void) { return "swiglu_b200 0.1.0 (sm_100a)"; }

}  // extern "C"
