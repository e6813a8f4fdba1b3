// fe_ksum_sp.cuh -- K1s: the paper's single-precision builds:
//   SP   : Eq. 4 and Eq. 5 per (k, band, q, h, Delta) term literally, every operation in binary32
//          (1 sqrt, 2 exp, 2 log per term, as in Algorithm 2), accurate expf / log1pf / sqrtf;
//   SPFM : the same with the fast intrinsics (__expf, __logf, rsqrt.approx).
// Only the sum over k is kept in double (reading G20), with the fixed tree of K1, so results do not depend
// on the float summation order and can be compared with a CPU evaluation of the same float expressions.  Geometry = K1 (fe_ksum_kernel):
// block = (iq, h-tile, Delta-tile, k-chunk), thread = one kx column x strided ky rows x a 4 x 4 (h, Delta) tile.
// Writes partial[chunk][q,h,Delta] = - sum_k sum_bands [ f(E+) + f(E-) + C ]  (fe_finish_kernel with S = 0).
#pragma once
#include "fe_kernels.cuh"

namespace fe {

constexpr int kSpTH = 4, kSpTD = 4;

template <int NB>
__device__ __forceinline__ void band_energies_sp(const float (&t)[4], float cx, float sx, float cy, float sy, float (&E)[NB]) {
  if (NB == 1) {
    E[0] = -2.0f * t[0] * (cx + cy);
  } else {
    const float T11 = -2.0f * (t[0] * cx + t[1] * cy) - 4.0f * t[2] * cx * cy;     // A.1
    const float T22 = -2.0f * (t[1] * cx + t[0] * cy) - 4.0f * t[2] * cx * cy;     // A.2
    const float T12 = -4.0f * t[3] * sx * sy;                                      // A.3
    const float avg = 0.5f * (T11 + T22), dif = 0.5f * (T11 - T22);
    const float rad = sqrtf(dif * dif + T12 * T12);
    E[0] = avg + rad;                                                              // A.4
    E[NB - 1] = avg - rad;
  }
}

template <bool FAST>
__device__ __forceinline__ float thermal_sp(float x, float T, float neg_beta) {   // f(x) = -T ln(1 + e^{-x/T}), stable
  const float ax = fabsf(x);
  const float u = FAST ? __expf(ax * neg_beta) : expf(ax * neg_beta);
  const float l = FAST ? __logf(1.0f + u) : log1pf(u);
  return fminf(x, 0.0f) - T * l;
}

struct SpConsts { float t[4]; float mu, eta_scale, T; };

template <int NB, int FORM, bool FAST>
__global__ void __launch_bounds__(kThreads) fe_ksum_sp_kernel(const KsumParams P, const SpConsts sc) {
  constexpr int TH = kSpTH, TD = kSpTD;
  __shared__ double red[kWarps][TH * TD];
  int b = blockIdx.x;
  const int chunk = b % P.ksplit;  b /= P.ksplit;
  const int td = b % P.ntile_d;    b /= P.ntile_d;
  const int th = b % P.ntile_h;
  const int iq = b / P.ntile_h;
  const int cg = chunk % P.ncg, rs = chunk / P.ncg;
  const int bx = 1 << P.bx_log2;
  const int col = cg * bx + (threadIdx.x & (bx - 1));
  const int rsub = threadIdx.x >> P.bx_log2;
  const int by = kThreads >> P.bx_log2;
  const bool valid = col < P.N;

  float hv[TH], dv[TD];                       // P.d2 holds Delta itself for this kernel (the SP build squares in float)
#pragma unroll
  for (int i = 0; i < TH; ++i) hv[i] = (float)P.h[min(th * TH + i, P.nh - 1)];
#pragma unroll
  for (int j = 0; j < TD; ++j) dv[j] = (float)P.d2[min(td * TD + j, P.nd - 1)];
  double acc[TH][TD];
#pragma unroll
  for (int i = 0; i < TH; ++i)
#pragma unroll
    for (int j = 0; j < TD; ++j) acc[i][j] = 0.0;

  if (valid) {
    const double4 ctd = P.coltab[(size_t)iq * P.N + col];
    const float cx = (float)ctd.x, sx = (float)ctd.y, cxq = (float)ctd.z, sxq = (float)ctd.w;
    const double4* rt = P.rowtab + (size_t)iq * P.N;
    const int r0 = rs * P.rows_per_chunk;
    const int r1 = min(P.N, r0 + P.rows_per_chunk);
    const float T = sc.T, nbeta = -1.0f / sc.T;
    for (int r = r0 + rsub; r < r1; r += by) {
      const double4 rrd = rt[r];
      const float cy = (float)rrd.x, sy = (float)rrd.y, cyq = (float)rrd.z, syq = (float)rrd.w;
      float Ek[NB], Eq[NB];
      band_energies_sp<NB>(sc.t, cx, sx, cy, sy, Ek);          // E(k)
      band_energies_sp<NB>(sc.t, cxq, sxq, cyq, syq, Eq);      // E(k - q) = E(-k + q)
      float eta = sc.eta_scale;                                // eta(k)
      if (FORM == 1) eta *= cx * cy;
#pragma unroll
      for (int e = 0; e < NB; ++e) {
        if (!((P.mc.band_mask >> e) & 1)) continue;
        const float xk = Ek[e] - sc.mu, xq = Eq[e] - sc.mu;
#pragma unroll
        for (int i = 0; i < TH; ++i) {
          const float a = xk - hv[i], bdn = xq + hv[i];        // xi_up(k), xi_down(-k+q)
          const float hd = 0.5f * (a - bdn), hs = 0.5f * (a + bdn);
          const float cst = P.mc.const_mode == 0 ? bdn : xk + hv[i];
#pragma unroll
          for (int j = 0; j < TD; ++j) {
            const float gap = dv[j] * eta;
            const float rad2 = hs * hs + gap * gap;
            float root;
            if (FAST) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(rad2 + 1e-37f)); root = rad2 * y; }
            else root = sqrtf(rad2);                                                             // Eq. 4
            const float term = thermal_sp<FAST>(hd + root, T, nbeta) + thermal_sp<FAST>(hd - root, T, nbeta) + cst;   // Eq. 5
            acc[i][j] -= (double)term;
          }
        }
      }
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int i = 0; i < TH; ++i)
#pragma unroll
    for (int j = 0; j < TD; ++j) {
      const double v = warp_sum(acc[i][j]);
      if (lane == 0) red[warp][i * TD + j] = v;
    }
  __syncthreads();
  if (threadIdx.x < TH * TD) {
    const int i = threadIdx.x / TD, j = threadIdx.x % TD;
    const int ih = th * TH + i, id = td * TD + j;
    if (ih < P.nh && id < P.nd) {
      double tot = 0.0;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) tot += red[w][threadIdx.x];
      const size_t nout = (size_t)P.nq * P.nh * P.nd;
      P.partial[(size_t)chunk * nout + ((size_t)iq * P.nh + ih) * P.nd + id] = tot;
    }
  }
}

}  // namespace fe
