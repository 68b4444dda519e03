/*
 * swiglu_mlp.h -- C ABI of libswiglu_b200.so: the fused gated MLP of arxiv/paper_2607_02521
 * ("Tile-Level Activation Overlap for Efficient LLM Inference") for NVIDIA B200 (sm_100a).
 *
 * Operation (section 3.1, Eq. 1-3; problem statement line 74:
 * "accept the same input tensors (A, W1, W2) and produce the same output (Y) as the
 * unfused baseline"):
 *
 *     Gate = A . W1,   Up = A . W2,   Y = SiLU(Gate) (.) Up,   SiLU(x) = x * sigma(x)
 *
 * Numeric contract ("BF16 precision throughout", line 370 "FP32
 * arithmetic on register-resident values ... BF16 conversion only at the final store"):
 * bf16 inputs, fp32 accumulation over all of K on the tensor cores, SiLU and the product in
 * fp32, ONE round-to-nearest-even conversion to bf16 at the store.  In the fused entry
 * point Gate and Up never exist in HBM.
 *
 * Layout: everything dense row-major, no strides.
 *     A  : M x K bf16, K contiguous         (device pointer, 16-byte aligned)
 *     W1 : K x N bf16, N contiguous         (device pointer, 16-byte aligned)
 *     W2 : K x N bf16, N contiguous         (device pointer, 16-byte aligned)
 *     Y  : M x N bf16, N contiguous         (device pointer, 16-byte aligned, written)
 * K and N must be multiples of 8 (16-byte row pitch, a TMA requirement); M is arbitrary.
 *
 * All pointers are DEVICE pointers on the current CUDA device unless a parameter says
 * "host".  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 * Every compute entry point is asynchronous: it returns after enqueueing on `stream`.
 *
 * Ownership: the caller owns A, W1, W2, Y and any workspace and keeps them valid until the
 * enqueued work has completed.  swiglu_mlp_unfused (8-argument form) and the host-buffer forms
 * use a library-owned, lazily grown, PER-STREAM device buffer.  It is allocated and regrown
 * with stream-ordered allocation (cudaMallocAsync / cudaFreeAsync on `stream`), so growth never
 * synchronises and never frees memory that earlier work on that stream still uses.  A stream
 * that is being captured is refused (SWIGLU_ERR_WORKSPACE): use the _ex forms with a caller
 * workspace under CUDA-graph capture, or swiglu_mlp_unfused_static (scratch in a static device
 * array of the library: no allocation at all, bounded size).  swiglu_release_stream /
 * swiglu_release give the buffers back.  The fused entry points need no workspace and are always
 * capturable (the optional K split of their last wave uses a fixed-size per-stream buffer when
 * one may be created, or the caller's through swiglu_mlp_ex; under capture it is skipped).
 *
 * Errors: a swiglu_status return code; the library never throws, aborts or prints, and the
 * device-pointer compute entry points never synchronise (the host-buffer forms and
 * swiglu_release do, and say so).  Argument validation happens before any CUDA call, so the validation
 * codes (1-5) can be exercised on a host without a GPU.  M == 0 is SWIGLU_OK and launches
 * nothing.  There is NO CPU fallback: without an sm_100 device the compute entry points
 * return SWIGLU_ERR_ARCH or SWIGLU_ERR_CUDA.
 *
 * Determinism: same inputs + same variant => bitwise identical Y (split-K partial sums
 * are combined in a fixed order).  Thread safety: entry points may be called concurrently
 * from several host threads.
 */
#ifndef SWIGLU_MLP_H_
#define SWIGLU_MLP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SWIGLU_OK = 0,
  SWIGLU_ERR_NULL_POINTER = 1, /* A, W1, W2 or Y is NULL while M > 0                    */
  SWIGLU_ERR_BAD_SHAPE = 2,    /* M < 0, N <= 0, K <= 0, or a byte count overflows int64 */
  SWIGLU_ERR_UNSUPPORTED = 3,  /* K % 8 != 0 or N % 8 != 0; or an unknown variant id     */
  SWIGLU_ERR_MISALIGNED = 4,   /* a base pointer is not 16-byte aligned                  */
  SWIGLU_ERR_ALIASING = 5,     /* Y overlaps A, W1 or W2                                 */
  SWIGLU_ERR_ARCH = 6,         /* current device is not compute capability 10.x          */
  SWIGLU_ERR_WORKSPACE = 7,    /* _ex: workspace NULL / misaligned / too small           */
  SWIGLU_ERR_CUDA = 8          /* a CUDA runtime/driver call failed: swiglu_last_error() */
} swiglu_status;

/*
 * Fused path (Eq. 1-3; the paper's Kernel-1/Kernel-2 idea, lines 124-169, rebuilt
 * for sm_100a): Y = bf16(SiLU(A.W1) * (A.W2)), Gate/Up held only in tensor memory.
 * The kernel variant is picked per (M, N, K) from a measured table.
 */
int swiglu_mlp(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
               int64_t K, void* stream);

/*
 * Unfused comparison path (two GEMMs that write Gate and Up
 * to HBM as bf16, then an elementwise SiLU-multiply kernel).  Built from this library's own
 * tcgen05 GEMM and elementwise kernels, no cuBLAS.  For M <= 128 the two GEMMs are one merged
 * Gate|Up launch of the same swap-AB split-K streaming kernel the fused path uses (so the
 * comparison isolates fusion, not tile shapes).  Needs 2*M*N*2 bytes of workspace
 * (library-owned in this form).
 */
int swiglu_mlp_unfused(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                       int64_t N, int64_t K, void* stream);

/*
 * Explicit-workspace / forced-variant forms.
 *   workspace       : device pointer, 256-byte aligned, or NULL if workspace_bytes == 0
 *   workspace_bytes : size of that buffer; must be >= swiglu_workspace_bytes(...) for the
 *                     variant that will run
 *   variant         : -1 = automatic (same choice as the 8-argument form), otherwise an id
 *                     in [0, swiglu_num_variants(unfused))
 */
int swiglu_mlp_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                  int64_t N, int64_t K, void* workspace, size_t workspace_bytes, int variant,
                  void* stream);
int swiglu_mlp_unfused_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                          int64_t N, int64_t K, void* workspace, size_t workspace_bytes,
                          int variant, void* stream);

/*
 * No-allocation form of the unfused path, for callers that cannot allocate device memory (code
 * under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same
 * arguments, result and kernels as swiglu_mlp_unfused, but the bf16 Gate / Up scratch
 * (2 * round_up(M*N*2, 256) bytes) lives in ONE file-scope `static __device__` array of
 * SWIGLU_STATIC_SCRATCH_BYTES (32 MiB) inside the library: every GPU that loads the library holds
 * those 32 MiB until the process exits.  The call makes no cudaMalloc / cudaMallocAsync / cudaFree
 * and no allocating library call; its only set-up is one cudaGetSymbolAddress per device.
 *   - Sizes whose scratch exceeds the array (M*N > ~8.39 M elements, e.g. more than 283 rows at
 *     N = 29568) are rejected with SWIGLU_ERR_WORKSPACE before any CUDA call; use
 *     swiglu_mlp_unfused_ex with a caller workspace for those.
 *   - Every call on a device shares the array, which keeps the previous call's contents.  Nothing
 *     in it has to start at zero: the GEMMs write every Gate / Up element of [0,M) x [0,N) before
 *     the elementwise kernel reads it.  Calls that OVERLAP on the GPU (two streams, two host
 *     threads, a graph replayed next to an eager call) race on it: the caller must serialise them.
 */
#define SWIGLU_STATIC_SCRATCH_BYTES (32u << 20)
int swiglu_mlp_unfused_static(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                              int64_t N, int64_t K, void* stream);

/*
 * Other gated activations of the GLU family ("gated linear unit variants
 * (GEGLU, SwiGLU, ReGLU)"; line 392 future-work item 4): Y = bf16(act(A.W1) * (A.W2)) with the
 * same tensors, layout, numeric contract (fp32 activation on the fp32 accumulators, one RNE
 * rounding) and dispatch as swiglu_mlp.  SWIGLU_ACT_SILU makes these identical to swiglu_mlp /
 * swiglu_mlp_unfused.  An unknown activation id returns SWIGLU_ERR_UNSUPPORTED.
 */
typedef enum {
  SWIGLU_ACT_SILU = 0,      /* x * sigma(x)                       SwiGLU (the paper's Eq. 3)   */
  SWIGLU_ACT_GELU = 1,      /* x * Phi(x) = x/2 * erfc(-x/sqrt 2) GeGLU, exact form            */
  SWIGLU_ACT_GELU_TANH = 2, /* x/2 * (1 + tanh(sqrt(2/pi) (x + 0.044715 x^3)))  GeGLU, tanh form */
  SWIGLU_ACT_RELU = 3       /* max(x, 0)                          ReGLU                        */
} swiglu_activation;

int swiglu_glu_mlp(const void* A, const void* W1, const void* W2, void* Y, int64_t M, int64_t N,
                   int64_t K, int activation, void* stream);
int swiglu_glu_mlp_unfused(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                           int64_t N, int64_t K, int activation, void* stream);
/* Forced fused variant (-1 = automatic); no fused variant needs a workspace. */
int swiglu_glu_mlp_ex(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                      int64_t N, int64_t K, int activation, int variant, void* stream);
/*
 * Weight layout.  SWIGLU_WEIGHTS_KN is the paper's and every other entry point's: W1, W2 are
 * K x N row-major.  SWIGLU_WEIGHTS_NK takes them as N x K row-major
 * (K contiguous) -- the layout nn.Linear and the serving stacks the paper targets keep their
 * projections in (lines 72-74) -- so a checkpoint's gate_proj / up_proj can be passed as they
 * are.  Everything else (A, Y, numeric contract, dispatch, errors) is as for swiglu_glu_mlp;
 * `unfused` != 0 runs the comparison path, `variant` = -1 is automatic.
 */
typedef enum { SWIGLU_WEIGHTS_KN = 0, SWIGLU_WEIGHTS_NK = 1 } swiglu_weight_layout;
int swiglu_glu_mlp_layout(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                          int64_t N, int64_t K, int activation, int weight_layout, int unfused,
                          int variant, void* stream);

/*
 * Prepacked, tile-interleaved weights (Kernel-2 "interleaves W1
 * and W2 ... a one-time preprocessing step").  The paper interleaves
 * single columns for its Epilogue Visitor Tree; the unit that matters on sm_100a is the
 * 64-column slab (one 128-byte swizzled TMA box row = one UMMA operand atom), so W_fused is
 *
 *     Wp[t][s][k][c]   t < ceil(N/128) column tiles, s in {g0, u0, g1, u1}, k < Kp, c < 64
 *                    = W1[k][128 t + 64 (s>>1) + c]  for s even (Gate slabs), k < K
 *                    = W2[k][128 t + 64 (s>>1) + c]  for s odd  (Up slabs), k < K
 *                    = 0 for columns >= N and for the padding rows K <= k < Kp   (bf16, slab-major)
 *
 * Kp = K + 8 if K/8 is even, else K + 16: the padding makes the slab pitch Kp * 128 B an odd
 * number of KiB, which spreads the slabs over the memory channels (with K = 5120 the unpadded
 * 640 KiB pitch cost 10 % at decode sizes).  swiglu_packed_weight_bytes(N, K) =
 * 4 * ceil(N/128) * Kp * 128 bytes.  One 3-D TMA box then
 * brings a whole Gate|Up stage (instead of four boxes from two tensors), every 8 KB slab block is
 * contiguous in HBM, and the accumulator columns come out as g0 u0 g1 u1.
 *
 * swiglu_pack_weights: device pointers; W1, W2 in `weight_layout` (SWIGLU_WEIGHTS_KN or _NK);
 *   Wp 16-byte aligned (128-byte recommended), not overlapping W1 / W2.  Asynchronous on
 *   `stream`.  Its time is NOT part of any swiglu_mlp_packed timing (the paper excludes the
 *   interleave from its timings too, lines 159, 167).
 * swiglu_mlp_packed / swiglu_glu_mlp_packed: as swiglu_mlp / swiglu_glu_mlp_ex with (W1, W2)
 *   replaced by Wp.  CONTRACT: a packed buffer is a CONSTANT while calls that read it are in
 *   flight or being enqueued.  It must have been written by ordinary stream work (a copy, or a
 *   kernel that does not signal programmatic launch completion before its last write to Wp;
 *   swiglu_pack_weights is such a kernel), so "pack, then swiglu_mlp_packed on the same stream"
 *   is safe without a synchronisation.  In exchange the decode kernel issues its weight loads
 *   BEFORE griddepcontrol.wait: under programmatic dependent launch the weight stream of call
 *   i+1 overlaps the tail of call i, and only the activation tile waits for the previous kernel.
 */
size_t swiglu_packed_weight_bytes(int64_t N, int64_t K); /* 0 for bad N, K */
int swiglu_pack_weights(const void* W1, const void* W2, void* Wp, int64_t N, int64_t K,
                        int weight_layout, void* stream);
int swiglu_mlp_packed(const void* A, const void* Wp, void* Y, int64_t M, int64_t N, int64_t K,
                      void* stream);
int swiglu_glu_mlp_packed(const void* A, const void* Wp, void* Y, int64_t M, int64_t N,
                          int64_t K, int activation, int variant, void* stream);

/*
 * FP8 operands ("For FP8 ... we expect even larger relative gains since the
 * elementwise overhead grows relative to the faster GEMMs"; line 392 future-work item 2;
 * SURVEY.md 8(f) N5).  The paper gives no method detail; the contract taken (R19):
 *
 *     Y = bf16( SiLU(scale_gate * (A8 . W1_8^T)) * (scale_up * (A8 . W2_8^T)) )
 *
 *     A8   : M x K  OCP FP8 E4M3 ("e4m3fn") bytes, K contiguous        (device, 16-byte aligned)
 *     W1_8 : N x K  E4M3 bytes, K contiguous -- the [N,K] layout FP8 checkpoints store
 *     W2_8 : N x K  E4M3 bytes, K contiguous
 *     Y    : M x N  bf16, N contiguous                                  (written)
 *     scale_gate, scale_up : fp32 host scalars, the folded per-tensor dequantisation scales
 *                            (s_A * s_W1 and s_A * s_W2)
 *
 * K must be a multiple of 16 and N of 8.  tcgen05.mma kind::f8f6f4, fp32 accumulation over all
 * of K, scales / SiLU / product in fp32 on the accumulators, one RNE rounding to bf16; Gate and
 * Up never exist in HBM.  Same dispatch, variants (`variant`, -1 = automatic) and error
 * behaviour as swiglu_mlp_ex; SiLU only.  NaN codes (0x7F, 0xFF) in the inputs are out of
 * contract.
 */
int swiglu_mlp_fp8(const void* A8, const void* W1_8, const void* W2_8, void* Y, int64_t M,
                   int64_t N, int64_t K, float scale_gate, float scale_up, void* stream);
int swiglu_mlp_fp8_ex(const void* A8, const void* W1_8, const void* W2_8, void* Y, int64_t M,
                      int64_t N, int64_t K, float scale_gate, float scale_up, int variant,
                      void* stream);

/*
 * Launch-floor probe (measurement aid): enqueues the decode kernel that swiglu_mlp would pick
 * for this (M <= 128, N, K) -- same grid, cluster dimensions, shared memory, tensor-map
 * parameters, barrier initialisation, TMEM allocation and programmatic-dependent-launch
 * attribute -- with its body reduced to prologue + griddepcontrol.wait + teardown: no loads, no
 * MMAs, no reduction, no stores (Y is not written).  Timing a chain of these gives the
 * launch-to-launch floor of a dependent kernel chain that the real kernel's time sits on.
 */
int swiglu_launch_floor_probe(const void* A, const void* W1, const void* W2, void* Y, int64_t M,
                              int64_t N, int64_t K, void* stream);

/* Elementwise stage with a chosen activation: Y[i] = bf16(act(G[i]) * U[i]); see swiglu_silu_mul. */
int swiglu_act_mul(const void* G, const void* U, void* Y, int64_t elems, int activation,
                   void* stream);
const char* swiglu_activation_name(int activation); /* "silu", "gelu", ...; NULL for a bad id */

/*
 * The elementwise stage of the unfused path on its own (read Gate,
 * read Up, write Y; the "standalone SwiGLU" the paper profiles for its effective bandwidth,
 * line 321): Y[i] = bf16(SiLU(float(G[i])) * float(U[i])) for i < elems.  G, U, Y: device
 * pointers to bf16, 16-byte aligned; Y may alias G or U exactly (in place) but not partially;
 * elems must be a multiple of 8.  Asynchronous on `stream`.
 */
int swiglu_silu_mul(const void* G, const void* U, void* Y, int64_t elems, void* stream);

/* Bytes of workspace the given variant (-1 = automatic) needs; 0 if none or bad arguments.
 * `unfused` != 0 asks about swiglu_mlp_unfused. */
size_t swiglu_workspace_bytes(int64_t M, int64_t N, int64_t K, int unfused, int variant);

/* Variant table (fused: unfused == 0).  Names are static strings; NULL for a bad id.
 * (SURVEY.md 8(b) proposed these three without the `unfused` argument; the unfused path has
 * its own variant table, so the argument selects which table is meant.) */
int swiglu_num_variants(int unfused);
const char* swiglu_variant_name(int unfused, int variant);
/* The variant `-1` resolves to for this shape (host-only table lookup, no CUDA call). */
int swiglu_selected_variant(int64_t M, int64_t N, int64_t K, int unfused);

/* Number of kernel launches one call with this shape/variant enqueues (for accounting). */
int swiglu_launches_per_call(int64_t M, int64_t N, int64_t K, int unfused, int variant);

/* Validation only (codes 0-5), no CUDA call: what the compute entry points check first. */
int swiglu_validate(const void* A, const void* W1, const void* W2, const void* Y, int64_t M,
                    int64_t N, int64_t K);

/*
 * Host-buffer convenience form: A, W1, W2, Y are HOST pointers (pageable or pinned).  Copies
 * the inputs to the device, runs swiglu_mlp (unfused == 0) or swiglu_mlp_unfused, copies Y
 * back and synchronises `stream` before returning.  Device scratch is library-owned.
 */
int swiglu_mlp_host(const void* A_host, const void* W1_host, const void* W2_host,
                    void* Y_host, int64_t M, int64_t N, int64_t K, int unfused, void* stream);

/*
 * Host-buffer batch form: ONE pair of weight matrices and `count` activation batches that share
 * them (the batches of one serving step).  A_host[i] is M[i] x K bf16, Y_host[i] is M[i] x N
 * bf16; all HOST pointers (pinned memory gives copy/compute overlap; pageable works).  The
 * weights cross PCIe once per call, in column chunks: while the kernels of chunk j run on
 * `stream`, chunk j+1 is uploaded and chunk j-1's output columns are downloaded on internal
 * copy streams (output columns are independent, Eq. 1-3).  Synchronises before
 * returning; not capturable.  Device scratch is library-owned (per stream); concurrent calls
 * on one device are serialised.  M[i] == 0 batches are skipped.
 */
int swiglu_mlp_host_batched(const void* const* A_host, void* const* Y_host, const int64_t* M,
                            int count, const void* W1_host, const void* W2_host, int64_t N,
                            int64_t K, int unfused, void* stream);

/*
 * Library-owned memory ("workspace ... mutex-guarded").
 * swiglu_release_stream: stream-ordered free of the buffers the library keeps for `stream` on
 *   the current device (call it before destroying a stream you passed to swiglu_mlp_unfused or
 *   a host-buffer form; a later stream that reuses the handle simply allocates afresh).  Does
 *   not synchronise.
 * swiglu_release: cudaDeviceSynchronize(), then frees every library-owned buffer, copy stream
 *   and event of the current device.  The library stays usable; the next call re-allocates.
 */
int swiglu_release_stream(void* stream);
int swiglu_release(void);

/*
 * Experiment overrides (SWIGLU_VARIANT, SWIGLU_UNFUSED_VARIANT, SWIGLU_KSPLIT, SWIGLU_GROUP_M,
 * SWIGLU_HOST_CHUNKS, SWIGLU_NO_PDL, SWIGLU_NO_PREFETCH, SWIGLU_NO_EARLY, SWIGLU_NO_TAIL_SPLIT,
 * SWIGLU_NO_TAIL_KSPLIT, SWIGLU_TAIL_KSPLIT, SWIGLU_NO_W_EVICT_FIRST, SWIGLU_NO_TMAP_CACHE,
 * SWIGLU_SMALLM_DEEP, SWIGLU_SMALLM_STACK, SWIGLU_SKEW, SWIGLU_W_POLICY, SWIGLU_A_POLICY, SWIGLU_Y_POLICY) are read
 * from the environment once, at the
 * first call into the library.  swiglu_reload_env re-reads them (sweeps and tests; not
 * thread-safe against concurrent compute calls).
 */
void swiglu_reload_env(void);

/*
 * Measurement aid ("log the SM clock during each run"): while a device buffer
 * of two uint64 is registered here, CTA 0 of every GEMM-class kernel this library launches
 * (fused, unfused GEMMs; not the elementwise kernel) overwrites it at exit with
 * {SM cycles elapsed, nanoseconds elapsed (%globaltimer)} between its entry and exit, so
 * cycles / ns is the SM clock in GHz that launch really ran at.  Process-wide; NULL switches it
 * off.  The caller owns the buffer and keeps it valid while launches (or captured graphs) that
 * saw it may run.
 */
void swiglu_set_clock_probe(void* device_u64x2);

/* Calling thread's tensor-map cache counters (a0: CUtensorMaps are encoded once per distinct
 * (pointer, shape, box) and fetched from a thread-local cache afterwards); returns the number
 * of cache slots.  Either pointer may be NULL. */
int swiglu_tensor_map_cache_stats(uint64_t* hits, uint64_t* misses);

/* Message for the calling thread's most recent non-OK return; static/thread-local storage. */
const char* swiglu_last_error(void);
const char* swiglu_status_string(int status);
const char* swiglu_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SWIGLU_MLP_H_ */
