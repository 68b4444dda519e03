/*
 * swiglu_oracle.c -- CPU oracle for the gated-MLP hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code, header, table or helper with the CUDA path under
 * paper_2607_02521_b200/csrc/, and neither side includes the other.
 *
 * What it computes (section 3.1, Eq. 1-3):
 *
 *     Gate = A x W1            (Eq. 1)      A  in R^{M x K}
 *     Up   = A x W2            (Eq. 2)      W1, W2 in R^{K x N}
 *     Y    = SiLU(Gate) (.) Up (Eq. 3)      SiLU(x) = x * sigma(x)      (line 94)
 *
 * The method is exact ("produce the same output (Y) as the unfused
 * baseline"), so the oracle is the plain definition written out, in fp64, from the same
 * bf16 input bits the GPU sees (BASELINE.json north_star: "accumulates in fp64 from the
 * same bf16 inputs").  The result is NOT rounded to bf16: y_ref stays in fp64 and the
 * tolerance |y - y_ref| <= 2e-3 + 1.6e-2*|y_ref| is applied by the caller.
 *
 * Loop structure: outputs are independent, so they are handed out to threads as
 * (row m, panel of <= PANEL consecutive columns n).  Inside one unit every output's two
 * dot products are summed with k ascending, exactly as Eq. 1-2 are written; no split of
 * the k sum, no reassociation, no fused multiply-add is requested (-ffp-contract=off is
 * passed by the build), no -ffast-math.  Each product of two bf16 values has at most a
 * 16-bit significand and is exact in fp64; only the k-sum rounds (<= K * 2^-53 relative
 * to sum |terms|).
 *
 * Pins (tests/test_oracle_pins.py): brute-force Fraction arithmetic on tiny shapes; the
 * hand-worked 2x2x2 example in tests/golden/; SiLU closed forms from 50-digit decimal
 * arithmetic; SiLU(x)-SiLU(-x)=x reducing Y to two library fp64 matmuls; A=0 => Y=0;
 * W2=W1 => Y=G*SiLU(G) >= 0; exact scaling / permutation / prefix properties.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PANEL 256 /* columns per work unit: partition of independent outputs, not of any sum */

/* bf16 -> fp64, exact: a bf16 is the upper 16 bits of an IEEE-754 binary32. */
static inline double bf16_bits_to_f64(uint16_t h) {
  uint32_t w = ((uint32_t)h) << 16;
  float f;
  memcpy(&f, &w, sizeof f);
  return (double)f;
}

/* SiLU(x) = x * sigma(x) = x / (1 + exp(-x))   (line 169 gives the same
 * form x * (1 + exp(-x))^-1).  For x < 0 the algebraically identical x*e^x/(1+e^x) is used
 * so exp never overflows (reading R3): finite x gives a finite result. */
double swiglu_oracle_silu(double x) {
  if (x >= 0.0) {
    return x / (1.0 + exp(-x));
  } else {
    double e = exp(x);
    return x * e / (1.0 + e);
  }
}

/*
 * The other gated activations of the GLU family the paper names ("gated
 * linear unit variants (GEGLU, SwiGLU, ReGLU)", Shazeer 2020; line 392 future-work item 4:
 * "generalization to other gated activations (GeGLU, ReGLU)"): Y = act(Gate) (.) Up with
 *   act 0  SiLU       x * sigma(x)                                   (Eq. 3, the paper's)
 *   act 1  GELU       x * Phi(x) = 0.5 * x * erfc(-x / sqrt(2))      (GeGLU, exact form)
 *   act 2  GELU-tanh  0.5 * x * (1 + tanh(sqrt(2/pi) * (x + 0.044715 x^3)))   (GeGLU, the
 *          tanh approximation most frameworks ship; reading R17), evaluated as
 *          x * sigma(2 * sqrt(2/pi) * (x + 0.044715 x^3)), the same function
 *   act 3  ReLU       max(x, 0)                                      (ReGLU)
 * GELU is written with erfc so that the negative tail keeps its relative accuracy.
 */
double swiglu_oracle_activation(int act, double x) {
  switch (act) {
    case 0: return swiglu_oracle_silu(x);
    case 1: return 0.5 * x * erfc(-x / sqrt(2.0));
    case 2: {
      /* 0.5*(1 + tanh(u)) = sigma(2u) exactly; written through exp so that the negative tail
       * does not cancel (1 + tanh(u) loses all its digits for u << 0).  DESIGN.md R17. */
      const double c = sqrt(2.0 / acos(-1.0));
      const double z = 2.0 * c * (x + 0.044715 * x * x * x);
      if (z >= 0.0) return x / (1.0 + exp(-z));
      const double e = exp(z);
      return x * e / (1.0 + e);
    }
    case 3: return x > 0.0 ? x : 0.0;
  }
  return NAN;
}

/* One work unit: row m, columns [n0, n1).  gate/up are caller-provided scratch of PANEL. */
static void unit(const uint16_t *A, const uint16_t *W1, const uint16_t *W2, double *Y,
                 int64_t N, int64_t K, int64_t m, int64_t n0, int64_t n1, double *gate,
                 double *up, int act) {
  const int64_t w = n1 - n0;
  for (int64_t j = 0; j < w; ++j) {
    gate[j] = 0.0;
    up[j] = 0.0;
  }
  for (int64_t k = 0; k < K; ++k) { /* k ascending: the sums of Eq. 1 and Eq. 2 */
    const double a = bf16_bits_to_f64(A[m * K + k]);
    const uint16_t *w1 = W1 + k * N + n0; /* W[k, n], row-major [K, N] */
    const uint16_t *w2 = W2 + k * N + n0;
    for (int64_t j = 0; j < w; ++j) {
      gate[j] += a * bf16_bits_to_f64(w1[j]); /* Eq. 1 */
      up[j] += a * bf16_bits_to_f64(w2[j]);   /* Eq. 2 */
    }
  }
  for (int64_t j = 0; j < w; ++j) {
    Y[m * N + n0 + j] = swiglu_oracle_activation(act, gate[j]) * up[j]; /* Eq. 3 (act 0) */
  }
}

/*
 * Y[M,N] (fp64, row-major) = SiLU(A.W1) (.) (A.W2), A[M,K], W1/W2[K,N] given as bf16 bit
 * patterns (uint16), row-major, dense.  nthreads <= 0 means "all OpenMP threads".
 * Returns the number of threads used, or -1 on bad arguments.
 */
int swiglu_oracle_act(const uint16_t *A, const uint16_t *W1, const uint16_t *W2, double *Y,
                      int64_t M, int64_t N, int64_t K, int act, int nthreads) {
  if (M < 0 || N < 0 || K < 0 || act < 0 || act > 3) return -1;
  if (M == 0 || N == 0) return 0;
  if (!A && K > 0) return -1;
  if ((!W1 || !W2) && K > 0) return -1;
  if (!Y) return -1;
  const int64_t panels = (N + PANEL - 1) / PANEL;
  const int64_t units = M * panels;
  int used = 1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  if ((int64_t)nthreads > units) nthreads = (int)units;
  used = nthreads;
#pragma omp parallel num_threads(nthreads)
#endif
  {
    double gate[PANEL], up[PANEL];
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
    for (int64_t u = 0; u < units; ++u) {
      /* panel-major so that threads working at the same time share a W panel in cache */
      const int64_t p = u / M, m = u % M;
      const int64_t n0 = p * PANEL;
      const int64_t n1 = (n0 + PANEL < N) ? n0 + PANEL : N;
      unit(A, W1, W2, Y, N, K, m, n0, n1, gate, up, act);
    }
  }
  return used;
}

int swiglu_oracle(const uint16_t *A, const uint16_t *W1, const uint16_t *W2, double *Y,
                  int64_t M, int64_t N, int64_t K, int nthreads) {
  return swiglu_oracle_act(A, W1, W2, Y, M, N, K, 0, nthreads);
}

/*
 * Sampled form for full-size shapes: the same computation for a list of `count` rows
 * (row indices into A) only.  Ysub is [count, N] fp64.  Rows are independent (Eq. 1-3
 * act row-wise on A), so Ysub[i,:] == Y[rows[i],:] of the full result.
 */
int swiglu_oracle_rows_act(const uint16_t *A, const uint16_t *W1, const uint16_t *W2,
                           double *Ysub, const int64_t *rows, int64_t count, int64_t M,
                           int64_t N, int64_t K, int act, int nthreads) {
  if (M < 0 || N < 0 || K < 0 || count < 0 || act < 0 || act > 3) return -1;
  if (count == 0 || N == 0) return 0;
  if (!rows || !Ysub) return -1;
  if ((!A || !W1 || !W2) && K > 0) return -1;
  for (int64_t i = 0; i < count; ++i)
    if (rows[i] < 0 || rows[i] >= M) return -1;
  const int64_t panels = (N + PANEL - 1) / PANEL;
  const int64_t units = count * panels;
  int used = 1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  if ((int64_t)nthreads > units) nthreads = (int)units;
  used = nthreads;
#pragma omp parallel num_threads(nthreads)
#endif
  {
    double gate[PANEL], up[PANEL];
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
    for (int64_t u = 0; u < units; ++u) {
      const int64_t p = u / count, i = u % count;
      const int64_t n0 = p * PANEL;
      const int64_t n1 = (n0 + PANEL < N) ? n0 + PANEL : N;
      /* write row i of Ysub from row rows[i] of A: shift the base pointers accordingly */
      unit(A + rows[i] * K, W1, W2, Ysub + i * N, N, K, 0, n0, n1, gate, up, act);
    }
  }
  return used;
}

int swiglu_oracle_rows(const uint16_t *A, const uint16_t *W1, const uint16_t *W2,
                       double *Ysub, const int64_t *rows, int64_t count, int64_t M,
                       int64_t N, int64_t K, int nthreads) {
  return swiglu_oracle_rows_act(A, W1, W2, Ysub, rows, count, M, N, K, 0, nthreads);
}

/*
 * FP8 operands ("FP8 ... we expect even larger relative gains"; line 392
 * future-work item 2).  The paper gives no method detail, so the reading
 * taken (R19) is the one FP8 serving stacks use: A and both weight matrices are
 * OCP FP8 E4M3 ("e4m3fn": 1 sign, 4 exponent bits with bias 7, 3 mantissa bits, no infinities,
 * S.1111.111 = NaN), weights in the [N, K] layout checkpoints store (K contiguous), one
 * dequantisation scale per projection folded into two fp32 scalars:
 *
 *     Gate = scale_gate * (A8 . W1_8^T),  Up = scale_up * (A8 . W2_8^T),  Y = SiLU(Gate) (.) Up
 *
 * Same plain definition as above, fp64, k ascending; each product of two e4m3 values has an
 * 8-bit significand and is exact.  The result is NOT rounded.
 */
double swiglu_oracle_e4m3_to_f64(uint8_t b) {
  const int sign = b >> 7, e = (b >> 3) & 15, m = b & 7;
  double v;
  if (e == 15 && m == 7) return NAN;                 /* the only non-finite code (no inf) */
  if (e == 0) v = ldexp((double)m / 8.0, -6);         /* subnormal: m/8 * 2^(1-7)           */
  else v = ldexp(1.0 + (double)m / 8.0, e - 7);       /* normal: (1 + m/8) * 2^(e-7)        */
  return sign ? -v : v;
}

/* rows[i] of Y for i < count (rows == NULL: row i itself); Ysub is [count, N] fp64. */
int swiglu_oracle_fp8_rows(const uint8_t* A, const uint8_t* W1, const uint8_t* W2, double* Ysub,
                           const int64_t* rows, int64_t count, int64_t M, int64_t N, int64_t K,
                           double scale_gate, double scale_up, int nthreads) {
  if (M < 0 || N < 0 || K < 0 || count < 0) return -1;
  if (count == 0 || N == 0) return 0;
  if ((!A || !W1 || !W2) && K > 0) return -1;
  if (!Ysub) return -1;
  for (int64_t i = 0; i < count; ++i) {
    const int64_t m = rows ? rows[i] : i;
    if (m < 0 || m >= M) return -1;
  }
  int used = 1;
  const int64_t units = count * N;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  if ((int64_t)nthreads > units) nthreads = (int)units;
  used = nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(static)
#endif
  for (int64_t idx = 0; idx < units; ++idx) {        /* one output (row i, column n) at a time */
    const int64_t i = idx / N, n = idx % N;
    const int64_t m = rows ? rows[i] : i;
    double gate = 0.0, up = 0.0;
    for (int64_t k = 0; k < K; ++k) {                /* k ascending: the sums of Eq. 1, Eq. 2 */
      const double a = swiglu_oracle_e4m3_to_f64(A[m * K + k]);
      gate += a * swiglu_oracle_e4m3_to_f64(W1[n * K + k]);   /* W[n, k], row-major [N, K] */
      up += a * swiglu_oracle_e4m3_to_f64(W2[n * K + k]);
    }
    Ysub[i * N + n] = swiglu_oracle_silu(scale_gate * gate) * (scale_up * up);   /* Eq. 3 */
  }
  return used;
}

/*
 * The one-time weight interleave ("W_fused"): Kernel-2
 * "interleaves W1 and W2" ahead of time so that a Gate column and its Up column reach the same
 * tile.  The paper does not print the layout; the reading taken (R18) interleaves
 * 64-column slabs inside 128-column tiles:
 *
 *     Wp[t][s][k][c],  t < ceil(N/128), s in {0,1,2,3} = {gate 0, up 0, gate 1, up 1},
 *                      k < Kp, c < 64
 *       = W1[k][128 t + 64 (s/2) + c]   if s is even and k < K
 *       = W2[k][128 t + 64 (s/2) + c]   if s is odd and k < K
 *       = 0                             where that column is >= N, or k >= K (padding rows)
 *
 * Kp = K + 8 if ceil(K/8) is even, else K + 16: every slab carries 8 or 16 rows of zero padding
 * so that the distance between slabs, Kp x 128 bytes, is an odd number of KiB (address spread
 * over the memory channels; not part of the method, only of the buffer's geometry).
 *
 * Pure index work on 16-bit patterns, written as the definition: one loop per index.
 * Pins (tests/test_oracle_pack_pins.py): every (k, n) of W1 and of W2 appears exactly once, at
 * the stated position (checked by an independent inverse walk), padding is zero, a tiny case
 * written out by hand in tests/golden/.
 */
int64_t swiglu_oracle_pack_rows(int64_t K) { return K + ((((K + 7) / 8) % 2 == 0) ? 8 : 16); }

int swiglu_oracle_pack(const uint16_t* W1, const uint16_t* W2, uint16_t* Wp, int64_t N, int64_t K) {
  if (!W1 || !W2 || !Wp || N <= 0 || K <= 0) return -1;
  const int64_t tiles = (N + 127) / 128, Kp = swiglu_oracle_pack_rows(K);
  for (int64_t t = 0; t < tiles; ++t)
    for (int64_t s = 0; s < 4; ++s)
      for (int64_t k = 0; k < Kp; ++k)
        for (int64_t c = 0; c < 64; ++c) {
          const int64_t n = 128 * t + 64 * (s / 2) + c;
          const uint16_t* W = (s % 2 == 0) ? W1 : W2;
          Wp[((t * 4 + s) * Kp + k) * 64 + c] = (n < N && k < K) ? W[k * N + n] : (uint16_t)0;
        }
  return 0;
}

int swiglu_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
