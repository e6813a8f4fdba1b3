// fe_bands3.cuh -- three-band model (Appendix B): numerical band diagonalisation on the device
// and the per-q eigenvalue tables in HBM that the paper proposes for models with more than two bands
// ("precalculate the eigenvalues for every momentum vector k in FBZ and store them in memory").
//
//   KB  fe_bands3_kernel : etab[y][e][k],  y = 0: E_e(k);  y = 1 + iq: E_e(k - q_iq) = E_e(-k + q_iq)
//   KS3 fe_ssum3_kernel  : spart[iq][chunk] = sum_k sum_e s  from the tables (the table-fed twin of fe_ssum_kernel)
//
// T_k is complex Hermitian with T^{13}, T^{23} purely imaginary (B.5, B.6) and T^{12} real (B.4); the unitary
// diag(1, 1, -i) maps it to the REAL symmetric matrix [[T11, T12, a], [T12, T22, b], [a, b, T33]] with
// T^{13} = i a, T^{23} = i b, which has the same eigenvalues.  They are found by cyclic Jacobi rotations with the
// classical update formulas (Rutishauser), at most kSweeps sweeps, and sorted ascending (band e = e-th eigenvalue).
#pragma once
#include "fe_kernels.cuh"

namespace fe {

struct Band3Consts { double t[12]; double e0; };   // t[i-1] = t_i of PAPER.md:273

__device__ __forceinline__ void jacobi_rotate(double& app, double& aqq, double& apq, double& arp, double& arq) {
  // zero a_pq; r is the third index.  t = tan(theta) of the smaller rotation angle.
  if (fabs(apq) < 1e-280) { apq = 0.0; return; }    // (also keeps the reciprocal below finite)
  double tau = (aqq - app) * rcp_nr(2.0 * apq);
  tau = fmin(fmax(tau, -1e150), 1e150);             // tau^2 stays finite; t ~ 1/(2 tau) there
  const double t = copysign(1.0, tau) * rcp_nr(fabs(tau) + sqrt_pos(fma(tau, tau, 1.0)));
  const double c = rsqrt_nr(fma(t, t, 1.0)), s = t * c;
  app = fma(-t, apq, app);
  aqq = fma(t, apq, aqq);
  apq = 0.0;
  const double xp = arp, xq = arq;
  arp = fma(c, xp, -s * xq);
  arq = fma(s, xp, c * xq);
}

// Eigenvalues (ascending) of B.1-B.6 at the k whose trig values are (cx, sx, cy, sy).
__device__ __forceinline__ void band3_energies(const Band3Consts& bc, double cx, double sx, double cy, double sy,
                                               double (&E)[3]) {
  const double* t = bc.t;
  const double c2x = fma(2.0 * cx, cx, -1.0), c2y = fma(2.0 * cy, cy, -1.0);      // cos 2k
  const double cc = cx * cy;
  const double common = fma(4.0 * t[2], cc, 4.0 * t[11] * (c2x * c2y));
  const double aniso = 2.0 * t[10] * (c2x - c2y);
  double a11 = fma(2.0 * t[1], cx, 2.0 * t[0] * cy) + common + aniso;               // B.1
  double a22 = fma(2.0 * t[0], cx, 2.0 * t[1] * cy) + common - aniso;               // B.2
  double a33 = bc.e0 + 2.0 * t[4] * (cx + cy) + 4.0 * t[5] * cc + 2.0 * t[8] * (c2x + c2y) +
               4.0 * t[9] * fma(c2x, cy, cx * c2y);                                 // B.3
  double a12 = 4.0 * t[3] * (sx * sy);                                              // B.4
  double a13 = sx * fma(4.0 * t[7], cy, 2.0 * t[6]);                                // B.5 / i
  double a23 = sy * fma(4.0 * t[7], cx, 2.0 * t[6]);                                // B.6 / i
  constexpr int kSweeps = 8;                       // quadratic convergence: 4-5 sweeps reach fp64 for any 3x3
  const double scale = fabs(a11) + fabs(a22) + fabs(a33) + fabs(a12) + fabs(a13) + fabs(a23);
#pragma unroll 1
  for (int sweep = 0; sweep < kSweeps; ++sweep) {
    if (fabs(a12) + fabs(a13) + fabs(a23) <= 1e-22 * scale) break;
    jacobi_rotate(a11, a22, a12, a13, a23);        // (p, q, r) = (1, 2, 3)
    jacobi_rotate(a11, a33, a13, a12, a23);        // (1, 3, 2): a_r p = a12, a_r q = a23 (= a32)
    jacobi_rotate(a22, a33, a23, a12, a13);        // (2, 3, 1)
  }
  double e0 = a11, e1 = a22, e2 = a33, x;
  if (e0 > e1) { x = e0; e0 = e1; e1 = x; }
  if (e1 > e2) { x = e1; e1 = e2; e2 = x; }
  if (e0 > e1) { x = e0; e0 = e1; e1 = x; }
  E[0] = e0; E[1] = e1; E[2] = e2;
}

// KB: grid = (ceil(N*N / 256), ny).  y0 = index of the first table this launch writes (0: the unshifted grid).
// slot (nullable): slot[iq] >= 0 marks a q on the k-grid whose table is not needed (the caller reads table 0 shifted);
// slot[iq] = -t < 0 sends the table of q_iq to table index t >= 1 (tables are then allocated for off-grid q only).
__global__ void __launch_bounds__(256) fe_bands3_kernel(Band3Consts bc, int N, int y0,
                                                        const double4* __restrict__ coltab,
                                                        const double4* __restrict__ rowtab,
                                                        const double* __restrict__ slot,
                                                        double* __restrict__ etab) {
  const size_t nk = (size_t)N * N;
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nk) return;
  const int y = y0 + blockIdx.y;
  int ytab = y;
  if (y > 0 && slot) {
    const double c = slot[y - 1];
    if (c >= 0.0) return;
    ytab = (int)(-c);
  }
  const int row = (int)(k / (unsigned)N), col = (int)(k - (size_t)row * N);
  const int iq = y == 0 ? 0 : y - 1;
  const double4 ct = coltab[(size_t)iq * N + col], rt = rowtab[(size_t)iq * N + row];
  double E[3];
  if (y == 0) band3_energies(bc, ct.x, ct.y, rt.x, rt.y, E);
  else        band3_energies(bc, ct.z, ct.w, rt.z, rt.w, E);
  double* out = etab + (size_t)ytab * 3 * nk + k;
  out[0] = E[0]; out[nk] = E[1]; out[2 * nk] = E[2];
}

// KS3: as fe_ssum_kernel, bands read from the tables.  grid = (nchunk, nq).
__global__ void __launch_bounds__(kThreads) fe_ssum3_kernel(ModelConsts mc, int N, int rows_per_chunk,
                                                            const double* __restrict__ etab,
                                                            double* __restrict__ spart) {
  const int iq = blockIdx.y, chunk = blockIdx.x;
  const size_t nk = (size_t)N * N;
  const size_t k0 = (size_t)chunk * rows_per_chunk * N;
  const size_t k1 = min(nk, k0 + (size_t)rows_per_chunk * N);
  const double* ek = etab;
  const double* eq = etab + (size_t)(1 + iq) * 3 * nk;
  double sum = 0.0, comp = 0.0;
  for (size_t k = k0 + threadIdx.x; k < k1; k += kThreads) {
#pragma unroll
    for (int e = 0; e < 3; ++e) {
      if (!((mc.band_mask >> e) & 1)) continue;
      const double Ek = ek[e * nk + k], Eq = eq[e * nk + k];
      double term = fma(0.5, Ek + Eq, -mc.mu);               // s
      if (mc.const_mode == 1) term += Ek - Eq;              // + 2 d0  (Eq. 5 literal constant)
      const double y = term - comp;
      const double t = sum + y;
      comp = (t - sum) - y;
      sum = t;
    }
  }
  __shared__ double red[kWarps];
  double w = warp_sum(sum);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = w;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
#pragma unroll
    for (int i = 0; i < kWarps; ++i) tot += red[i];
    spart[(size_t)iq * gridDim.x + chunk] = tot;
  }
}

}  // namespace fe
