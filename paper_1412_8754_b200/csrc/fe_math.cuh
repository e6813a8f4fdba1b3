// fe_math.cuh -- fp64 device math for the thermal term of Eq. 5.
//
// Per (k, band, q, h, Delta) term the k-sum kernel needs
//     u = exp(-x1/T), v = exp(-x2/T)  with 0 <= x1 <= x2,     l = ln(1 + w),  w = u + v + u v  in [0, 3].
// Both functions are range-restricted and branch-free (arguments are finite by construction), so they
// compile to straight-line FP64-pipe code plus a few integer / shared-memory instructions that issue in
// the FP64 pipe's shadow (a warp-wide DFMA occupies the 16-lane FP64 unit of an SM sub-partition for two
// issue cycles, so every other issue slot is free for the ALU, LSU and XU pipes).
//
// Accuracy:  what enters Omega is  m + T*l  with m = max(R,|d|) >= x1, so the
// ABSOLUTE error of l matters (times T).  exp: <= 2 ulp + |x| * 1.2e-16 relative (single-constant range
// reduction; |x| e^{-|x|} <= 0.37, so <= 4e-17 absolute in l).  log: <= 1.2e-16 absolute (rounding of 1 + w)
// + 2e-18 (truncation).  tests/test_fe_gpu.py::test_device_math checks both against numpy on 10^6 points.
//
// Build with -DFE_MATH_LIBDEVICE to use CUDA's exp()/log1p() instead (cross-check build).
#pragma once
#include <cuda_runtime.h>

namespace fe {

constexpr int kExpTabN = 64;    // 2^(j/64), j = 0..63
constexpr int kLogTabN = 260;   // index = exponent and top 7 mantissa bits of y in [1, 4]: 0..256 reachable, padded

struct MathTabs {               // global copy; kernels stage the parts they use in shared memory
  double  exp2_j64[kExpTabN];
  double  exp2_j256[256];       // 2^(j/256), j = 0..255 (factored kernel)
  double2 log_tab[kLogTabN];    // .x = 2^-e / c,  .y = -ln(.x) rounded   (c = centre of the 1/128-wide mantissa bin)
};

#ifdef FE_MATH_LIBDEVICE

__device__ __forceinline__ double exp_nonpos(double x, const MathTabs&) { return exp(x); }
__device__ __forceinline__ double log_1p_w(double w, const MathTabs&) { return log1p(w); }
__device__ __forceinline__ void exp_em1_nonpos(double x, const MathTabs&, double& u, double& em) { u = exp(x); em = expm1(x); }

#else

// exp(x) for finite x <= 0.   x = n (ln2/64) + r, n = rint(x 64/ln2), |r| <= ln2/128 = 5.42e-3;
// exp(x) = 2^(n>>6) * 2^((n&63)/64) * exp(r); exp(r) - 1 by degree-5 Taylor (truncation r^6/720 < 3.6e-17).
__device__ __forceinline__ double exp_nonpos(double x, const MathTabs& tb) {
  const double L2E64 = 92.33248261689366;        // 64/ln2
  const double LN2_64 = 0.010830424696249145;    // ln2/64
  const double MAGIC = 6755399441055744.0;       // 1.5 * 2^52
  x = fmax(x, -720.0);                           // keeps n in int range and 2^k normal; exp(-720) ~ 2e-313 ~ 0
  double t = fma(x, L2E64, MAGIC);
  int n = __double2loint(t);
  double nf = t - MAGIC;
  double r = fma(nf, -LN2_64, x);
  double p = fma(r, 8.3333333333333332e-03, 4.1666666666666664e-02);
  p = fma(p, r, 1.6666666666666666e-01);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = p * r;                                     // exp(r) - 1
  double s = tb.exp2_j64[n & 63];
  double y = fma(s, p, s);                       // in [1, 2)
  int k = n >> 6;                                // floor(n / 64) in [-1039, 0]
  k = max(k, -1000);
  return __hiloint2double(__double2hiint(y) + (k << 20), __double2loint(y));
}

// u = exp(x) and em = exp(x) - 1 for finite x <= 0, both without branches and em without cancellation.  Same reduction as
// exp_nonpos: exp(x) = c (1 + p), c = 2^(n>>6) 2^((n&63)/64), p = exp(r) - 1, so  exp(x) - 1 = (c - 1) + c p.  c - 1 is an
// exact subtraction (c in (0, 1]); for |x| < ln2/128 it is 0 and em = p keeps full relative accuracy (x -> 0: em -> x); else
// |em| >= 5.4e-3 and the table value's rounding (2^-53) is 2e-14 of it.  Used by the pair-susceptibility kernel for
// tanh(|x|/2T) = -em / (1 + u) of states near the Fermi level and for (1 - exp(-2z)) / z through its removable singularity.
__device__ __forceinline__ void exp_em1_nonpos(double x, const MathTabs& tb, double& u, double& em) {
  const double L2E64 = 92.33248261689366;        // 64/ln2
  const double LN2_64 = 0.010830424696249145;    // ln2/64
  const double MAGIC = 6755399441055744.0;       // 1.5 * 2^52
  x = fmax(x, -720.0);
  const double t = fma(x, L2E64, MAGIC);
  const int n = __double2loint(t);
  const double r = fma(t - MAGIC, -LN2_64, x);
  double p = fma(r, 8.3333333333333332e-03, 4.1666666666666664e-02);
  p = fma(p, r, 1.6666666666666666e-01);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = p * r;                                     // exp(r) - 1
  const double s = tb.exp2_j64[n & 63];
  const int k = max(n >> 6, -1000);
  const double c = __hiloint2double(__double2hiint(s) + (k << 20), __double2loint(s));
  u = fma(c, p, c);
  em = fma(c, p, c - 1.0);
}

// ln(1 + w), 0 <= w <= 3.   y = 1 + w in [1, 4]; idx = top 8 bits below the leading one of y (with exponent),
// table gives inv = 2^-e/c and lnc = -ln(inv);  r = y*inv - 1 (one FMA, |r| <= 2^-8 + 2^-52);
// ln y = lnc + r + r^2 q(r),  q = -1/2 + r/3 - r^2/4 + r^3/5 - r^4/6   (degree-6 Taylor of ln(1+r): next term
// r^7/7 < 2.1e-18 absolute).
__device__ __forceinline__ double log_1p_w(double w, const MathTabs& tb) {
  double y = 1.0 + w;
  int idx = (__double2hiint(y) - 0x3ff00000) >> 13;     // 0 .. 256 for y in [1, 4]
  double2 ct = tb.log_tab[idx];
  double r = fma(y, ct.x, -1.0);
  double q = fma(r, -1.6666666666666666e-01, 0.2);
  q = fma(q, r, -0.25);
  q = fma(q, r, 3.3333333333333331e-01);
  q = fma(q, r, -0.5);
  double r2 = r * r;
  return fma(r2, q, r) + ct.y;
}

#endif

}  // namespace fe
