// fe_chi.cuh -- static Cooper-pair susceptibility chi_{eps eps'}(q) of Appendix C, Eqs. C.2-C.3
// at omega -> 0, "calculated numerically similarly to the procedure used for free energy":
//
//   chi_{eps eps'}(q) = (1/N^2) sum_k eta(-k-q)^2 g(a, b),   a = E_eps(k) - mu - h,   b = E_eps'(-k-q) - mu + h,
//   g(a, b) = [f(-a) - f(b)] / (a + b) = [tanh(a/2T) + tanh(b/2T)] / (2 (a + b)),   f = Fermi function.
//
// E and eta are even, so -k-q is k+q: the trig tables are built by fe_trig_kernel with the list -q, and for the
// three-band model fe_bands3_kernel fills the band tables from them.  Same k-sum skeleton as the free energy:
// k-points generated from the tables (never stored), per-thread serial sums over a fixed k -> thread map, fixed
// shuffle tree, fixed warp order, fixed chunk order in the finish kernel: deterministic, no atomics.
//
// g has a removable singularity at a + b = 0 and its numerator cancels when a ~ -b.  It is evaluated without
// cancellation from u = exp(-|a|/T), v = exp(-|b|/T):
//   a b > 0 :  g = [ (1-u)/(1+u) + (1-v)/(1+v) ] / (2 (|a| + |b|))
//   else    :  tanh x + tanh y = 2 (v - u) / ((1+u)(1+v)) for x > 0 >= y, and v - u = -w expm1(-2|s|) sgn(s) with
//              s = (a + b)/2T, w = max(u, v):   g = w E(|s|) / (2T (1+u)(1+v)),  E(z) = -expm1(-2z)/z,  E(0) = 2.
#pragma once
#include "fe_kernels.cuh"

namespace fe {

struct ChiSide { double x, ax, u, opu, th; };   // energy, |energy|, exp(-|x|/T), 1 + u, tanh(|x|/2T)

__device__ __forceinline__ ChiSide chi_side(double x, double neg_beta, const MathTabs& tabs) {
  ChiSide s;
  s.x = x; s.ax = fabs(x);
  const double t = s.ax * neg_beta;            // -|x|/T <= 0
  double em;                                   // u - 1 without cancellation for |x| << T (states on the Fermi surface):
  exp_em1_nonpos(t, tabs, s.u, em);            // tanh(|x|/2T) = (1-u)/(1+u); branch-free (fe_math.cuh)
  s.opu = 1.0 + s.u;
  s.th = -em * rcp_nr(s.opu);
  return s;
}

__device__ __forceinline__ double chi_pair_factor(const ChiSide& a, const ChiSide& b, double inv2T, const MathTabs& tabs) {
  if (a.x * b.x > 0.0) return (a.th + b.th) * rcp_nr(2.0 * (a.ax + b.ax));
  const double z = fabs(a.x + b.x) * inv2T;
  const double w = fmax(a.u, b.u);
  const double rz = rcp_nr(fmax(z, 1e-300));
  double E = rz;                                           // z > 20: 1 - exp(-2z) = 1 to fp64 (most opposite-sign pairs at low T)
  if (z <= 20.0) {
    double e2, em;
    exp_em1_nonpos(-2.0 * z, tabs, e2, em);                // em = exp(-2z) - 1: -> -2z for z -> 0; branch-free inside
    E = z == 0.0 ? 2.0 : -em * rz;                         // (a select)
  }
  return w * E * inv2T * rcp_nr(a.opu * b.opu);
}

// grid = (nchunk, nq), 256 threads.  partial[(chunk*nq + iq)*NB*NB + e*NB + f]
template <int NB, int FORM>
__global__ void __launch_bounds__(kThreads) fe_chi_kernel(ModelConsts mc, double T, double hz, int N, int nq,
                                                          unsigned long long kc,
                                                          const double4* __restrict__ coltab,
                                                          const double4* __restrict__ rowtab,
                                                          const double* __restrict__ etab,
                                                          const double* __restrict__ shift,
                                                          const MathTabs* __restrict__ gtabs,
                                                          double* __restrict__ partial) {
  __shared__ MathTabs tabs;                                  // only the 2^(j/64) table is used here
  for (int i = threadIdx.x; i < kExpTabN; i += kThreads) tabs.exp2_j64[i] = gtabs->exp2_j64[i];
  __syncthreads();
  const int iq = blockIdx.y, chunk = blockIdx.x;
  const unsigned long long nk = (unsigned long long)N * N;
  const unsigned long long k0 = (unsigned long long)chunk * kc, k1 = min(nk, k0 + kc);
  const double neg_beta = -1.0 / T, inv2T = 0.5 / T;
  double acc[NB * NB];
#pragma unroll
  for (int i = 0; i < NB * NB; ++i) acc[i] = 0.0;
  for (unsigned long long kk = k0 + threadIdx.x; kk < k1; kk += kThreads) {
    const int row = (int)(kk / (unsigned)N), col = (int)(kk - (unsigned long long)row * (unsigned)N);
    const double4 ct = coltab[(size_t)iq * N + col], rr = rowtab[(size_t)iq * N + row];
    double Ek[NB], Eq[NB];
    if constexpr (NB == 3) {
      // q on the k-grid (the paper's FBZ map): E(k + q) is table 0 read at the shifted index, as in the paper's
      // "generate matrices E for k in FBZ"; otherwise the per-q table built by fe_bands3_kernel
      const double sc = shift[iq];
      size_t base = (size_t)(-sc) * 3 * nk, kq = kk;           // off-grid: sc = -(table index)
      if (sc >= 0.0) {
        const long long code = (long long)sc;
        const int sx = (int)(code % N), sy = (int)(code / N);
        int c2 = col + sx, r2 = row + sy;
        if (c2 >= N) c2 -= N;
        if (r2 >= N) r2 -= N;
        base = 0; kq = (size_t)r2 * N + c2;
      }
#pragma unroll
      for (int e = 0; e < 3; ++e) {
        Ek[e] = etab[(size_t)e * nk + kk];
        Eq[e] = etab[base + (size_t)e * nk + kq];
      }
    } else {
      band_energies<NB>(mc, ct.x, ct.y, rr.x, rr.y, Ek);     // E(k)
      band_energies<NB>(mc, ct.z, ct.w, rr.z, rr.w, Eq);     // E(k + q) = E(-k - q)
    }
    double g2 = mc.eta_scale;                                // eta(-k-q) = eta(k+q)             (C.2)
    if (FORM == 1) g2 *= ct.z * rr.z;
    g2 *= g2;
    ChiSide A[NB], B[NB];
#pragma unroll
    for (int e = 0; e < NB; ++e) {
      A[e] = chi_side(Ek[e] - mc.mu - hz, neg_beta, tabs);         // E_{eps k up}
      B[e] = chi_side(Eq[e] - mc.mu + hz, neg_beta, tabs);         // E_{eps',-k-q,down}
    }
#pragma unroll
    for (int e = 0; e < NB; ++e)
#pragma unroll
      for (int f = 0; f < NB; ++f) acc[e * NB + f] = fma(g2, chi_pair_factor(A[e], B[f], inv2T, tabs), acc[e * NB + f]);
  }
  __shared__ double red[NB * NB][kWarps];
#pragma unroll
  for (int i = 0; i < NB * NB; ++i) {
    const double w = warp_sum(acc[i]);
    if ((threadIdx.x & 31) == 0) red[i][threadIdx.x >> 5] = w;
  }
  __syncthreads();
  if (threadIdx.x < NB * NB) {
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) tot += red[threadIdx.x][w];
    partial[((size_t)chunk * nq + iq) * (NB * NB) + threadIdx.x] = tot;
  }
}

// chi[o] = (sum over chunks in index order) / N^2,  o in [0, nq*NB*NB)
__global__ void fe_chi_finish_kernel(int nout, int nchunk, double inv_nk, const double* __restrict__ partial,
                                     double* __restrict__ chi) {
  const int o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= nout) return;
  double s = 0.0;
  for (int c = 0; c < nchunk; ++c) s += partial[(size_t)c * nout + o];
  chi[o] = s * inv_nk;
}

}  // namespace fe
