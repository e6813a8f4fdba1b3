// fe_ksum_coop.cuh -- K1c: the k-sum in factored form, BLOCK-COOPERATIVE (default, FE_EVAL_COOP).
//
// Same quantity as K1 / K1f (fe_kernels.cuh):  P[chunk][q,h,Delta] = sum_{k in chunk, band} T ln Z,
//     Z_ij = A_j + B_i,   A_j = 2cosh(R_j/T),  B_i = 2cosh((d0 - h_i)/T),   R_j = sqrt(s^2 + Delta_j^2 eta_k^2)
// (Eq. 4 / Eq. 5 of the paper, in the cosh form derived in DESIGN.md section 1).
//
// K1f lets every thread own one k column and recompute the TD + TH exponentials of its own (h, Delta) tile, which
// is half of its FP64 work.  Here a block owns ONE (h, Delta) block tile of WH x WD values and a contiguous chunk of
// k-points, and its threads share the exponentials through shared memory:
//
//   P0  (once per NT k-points, one k per thread)  dispersion A.1-A.4 at k and k-q, s, d0, eta^2 per band, and the
//       block tile's exponent bounds -> a 32-byte header per (k, band) "slot": {s^2, eta^2, d0, Eref, flags}.
//   P1  (per sub-batch of KB k-points)  the SLOTS x (WD + WH) exponentials A_j, B_i, one item per thread at a time,
//       scaled by 2^-Eref and stored as plain doubles:  WD + WH exponentials per slot for the whole block
//       instead of (TD + TH) per thread.
//   P2  every thread owns a fixed TH x TD register tile of the block tile for ALL k of the chunk and does, per slot,
//       TD + TH shared-memory loads (LDS.128, mostly broadcast) and TH*TD x { DADD, DMUL }:
//           accP_ij *= (A'_j + B'_i)                       running product, exponent taken out via Eref
//       so there is no cross-thread reduction at all: P_ij = T (ln2 * exponent sum + ln accP_ij) is written
//       straight to partial[chunk][...].  Deterministic by construction (fixed k order per accumulator).
//
// Exponent handling.  Values are m 2^e, m in [0.997, 2.51), e = int32 (R/T reaches 10^4..10^9).  Per slot the
// header carries hi/lo bounds of e over the block tile computed from R(Delta_min), R(Delta_max), min/max |d0 - h|:
// every pair sum lies in [2^lo, 2^(hi+2)).  Fast slots (hi - lo <= kSpread): values are scaled by 2^-Eref with Eref
// centred between lo and hi, so each factor changes log2(accP) by at most spread/2 + 3; all threads track the
// same drift bound and renormalise accP (exponent moved to an integer sum) before 1000 binades are reached.
// Robust slots (wider spread, e.g. an h list spanning thousands of T): mantissa and exponent are stored
// separately and each pair uses its own E = max(eA_j, eB_i), summed per pair in shared memory.
#pragma once
#include "fe_kernels.cuh"

namespace fe {

struct CoopParams {
  ModelConsts mc;
  FactoredConsts fc;
  double T;
  int32_t N, nq, nh, nd;
  int32_t ntile_h, ntile_d, ksplit;
  int32_t debug_flags;                 // bit 0: every slot takes the robust path (tests)
  unsigned long long kc;               // k-points per chunk (multiple of the block size)
  unsigned long long nk;               // N*N
  const double4* coltab;               // [nq][N] {cos kx, sin kx, cos(kx-qx), sin(kx-qx)}
  const double4* rowtab;               // [nq][N] {cos ky, sin ky, cos(ky-qy), sin(ky-qy)}
  const double* h;                     // [nh]
  const double* d2;                    // [nd]  Delta^2
  const MathTabs* tabs;
  double* partial;                     // [ksplit][nq*nh*nd]
};

struct __align__(16) CoopHdr {         // one per (k, band) slot
  double s2, g2, d0;
  int eref;                            // fast: centred reference exponent
  int flags;                           // bit 0 skip, bit 1 robust, bits 8.. = drift step
};
constexpr int kCoopSkip = 1, kCoopRobust = 2;

template <int TH, int TD, int LH, int NW, int KB, int NB>
struct CoopGeom {
  static constexpr int NT = NW * 32;           // threads per block
  static constexpr int LD = 32 / LH;           // lanes of a warp along Delta
  static constexpr int NTD = NW * LD;          // threads along Delta
  static constexpr int WH = TH * LH;           // block tile, h
  static constexpr int WD = TD * NTD;          // block tile, Delta
  static constexpr int W = WD + WH;            // exponentials per slot
  static constexpr int SLOTS = KB * NB;        // slots per sub-batch
  static constexpr int BUF_DOUBLES = SLOTS * W + SLOTS;      // values + one int2 {eref, flags} per slot
  static constexpr size_t smem_bytes =
      sizeof(CoopHdr) * NT * NB + 2 * sizeof(double) * (size_t)BUF_DOUBLES + 2 * sizeof(int) * (size_t)SLOTS * W +
      sizeof(int) * (size_t)TH * TD * NT + sizeof(double) * (256 + WD + WH + 8);
};

// P1 for one kind of item (A_j: KIND 0, B_i: KIND 1) of one sub-batch: U independent chains per thread so that the
// sqrt / exp dependency chains of different items interleave in the FP64 pipe.
template <int KIND, int SLOTS, int WD, int WH, int NT, int U>
__device__ __forceinline__ void coop_p1(const CoopHdr* __restrict__ hdr_b, const double* __restrict__ list_s,
                                        const double* __restrict__ tab256, const FactoredConsts& fc,
                                        double* __restrict__ val, int* __restrict__ ev, int tid) {
  constexpr int W = WD + WH, CNT = KIND == 0 ? WD : WH, OFF = KIND == 0 ? 0 : WD;
  const double MAGIC = 6755399441055744.0;
  for (int it0 = tid; it0 < SLOTS * CNT; it0 += U * NT) {
    double x[U], m[U];
    int e[U], eref[U], flags[U], pos[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int it = it0 + u * NT;
      const bool act = it < SLOTS * CNT;
      const int itc = act ? it : it0;
      const int sl = itc / CNT, idx = itc - sl * CNT;
      const CoopHdr hd = hdr_b[sl];
      pos[u] = sl * W + OFF + idx;
      eref[u] = hd.eref;
      flags[u] = act ? hd.flags : kCoopSkip;
      if (KIND == 0) x[u] = fma(list_s[idx], hd.g2, hd.s2);       // Eq. 4 radicand                (S5)
      else           x[u] = fabs(hd.d0 - list_s[idx]);            // |d_i| = |d0 - h_i|
    }
    if (KIND == 0) {
#pragma unroll
      for (int u = 0; u < U; ++u) x[u] = sqrt_pos(x[u]);           // R_j
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const double t = fma(x[u], fc.c1, MAGIC);
      e[u] = exp_k(t);
      m[u] = exp_mant(x[u], t, fc, tab256);                        // e^{x/T} = m 2^e
    }
    if (KIND == 1) {
#pragma unroll
      for (int u = 0; u < U; ++u) m[u] = cosh_fix(m[u], e[u]);     // + e^{-x/T}: |d|/T is small on whole FFLO lines
    } else {
      bool any = false;
#pragma unroll
      for (int u = 0; u < U; ++u) any |= e[u] < 28;
      if (any) {
#pragma unroll
        for (int u = 0; u < U; ++u) m[u] = cosh_fix(m[u], e[u]);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (flags[u] & kCoopSkip) continue;
      if (flags[u] & kCoopRobust) { val[pos[u]] = m[u]; ev[pos[u]] = e[u]; }
      else                        val[pos[u]] = scale2(m[u], e[u] - eref[u]);
    }
  }
}

template <int NB, int FORM, int TH, int TD, int LH, int NW, int KB, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB) fe_ksum_coop_kernel(const CoopParams P) {
  using G = CoopGeom<TH, TD, LH, NW, KB, NB>;
  constexpr int NT = G::NT, WH = G::WH, WD = G::WD, W = G::W, SLOTS = G::SLOTS, BPS = NT / KB;
  static_assert(NT % KB == 0 && TD % 2 == 0 && TH % 2 == 0 && W % 2 == 0 && G::BUF_DOUBLES % 2 == 0, "geometry");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  CoopHdr* const hdr_s = reinterpret_cast<CoopHdr*>(smem_raw);                       // [NT*NB]
  double* const buf_s = reinterpret_cast<double*>(hdr_s + NT * NB);                  // 2 x {[SLOTS][W] values, [SLOTS] int2}
  double* const tab256 = buf_s + 2 * G::BUF_DOUBLES;                                 // [256]
  double* const d2_s = tab256 + 256;                                                 // [WD]
  double* const h_s = d2_s + WD;                                                     // [WH]
  double* const rng_s = h_s + WH;                                                    // hmin hmax d2min d2max (+pad)
  int* const ev_s = reinterpret_cast<int*>(rng_s + 8);                               // 2 x [SLOTS][W] (robust slots)
  int* const accE_s = ev_s + 2 * SLOTS * W;                                          // [TH*TD][NT]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int b = blockIdx.x;
  const int chunk = b % P.ksplit;  b /= P.ksplit;
  const int td = b % P.ntile_d;    b /= P.ntile_d;
  const int th = b % P.ntile_h;
  const int iq = b / P.ntile_h;

  // thread's register tile inside the block tile
  const int tdx = warp * G::LD + (lane % G::LD);
  const int thx = lane / G::LD;

  for (int i = tid; i < 256; i += NT) tab256[i] = P.tabs->exp2_j256[i];
  for (int i = tid; i < WD; i += NT) d2_s[i] = P.d2[min(td * WD + i, P.nd - 1)];
  for (int i = tid; i < WH; i += NT) h_s[i] = P.h[min(th * WH + i, P.nh - 1)];
  int* const myE = accE_s + tid;
#pragma unroll
  for (int pq = 0; pq < TH * TD; ++pq) myE[pq * NT] = 0;
  __syncthreads();
  if (warp == 0) {   // ranges of the block tile's lists (any order)
    double hmn = h_s[0], hmx = h_s[0], dmn = d2_s[0], dmx = d2_s[0];
    for (int i = lane; i < WH; i += 32) { hmn = fmin(hmn, h_s[i]); hmx = fmax(hmx, h_s[i]); }
    for (int i = lane; i < WD; i += 32) { dmn = fmin(dmn, d2_s[i]); dmx = fmax(dmx, d2_s[i]); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      hmn = fmin(hmn, __shfl_xor_sync(0xffffffffu, hmn, o));
      hmx = fmax(hmx, __shfl_xor_sync(0xffffffffu, hmx, o));
      dmn = fmin(dmn, __shfl_xor_sync(0xffffffffu, dmn, o));
      dmx = fmax(dmx, __shfl_xor_sync(0xffffffffu, dmx, o));
    }
    if (lane == 0) { rng_s[0] = hmn; rng_s[1] = hmx; rng_s[2] = dmn; rng_s[3] = dmx; }
  }
  __syncthreads();
  const double hmin = rng_s[0], hmax = rng_s[1], d2min = rng_s[2], d2max = rng_s[3];

  double accP[TH][TD];
#pragma unroll
  for (int i = 0; i < TH; ++i)
#pragma unroll
    for (int j = 0; j < TD; ++j) accP[i][j] = 1.0;
  int accEc = 0;     // exponent sum common to all pairs (fast slots)
  int drift = 0;     // bound on |log2 accP| since the last renormalisation (same value in every thread)

  const double MAGIC = 6755399441055744.0;
  const FactoredConsts& fc = P.fc;
  const unsigned long long kbeg = (unsigned long long)chunk * P.kc;
  const unsigned long long kend = min(P.nk, kbeg + P.kc);
  const int nbatch = (int)((kend - kbeg + KB - 1) / KB);       // sub-batches of KB k-points (kc < 2^31 KB)
  const bool force_robust = (P.debug_flags & 1) != 0;

  // ---------------- P0: one k-point per thread -> NB slot headers (for NT consecutive k-points) ----------------
  auto p0 = [&](int superbatch) {
    const unsigned long long kidx = kbeg + (unsigned long long)superbatch * NT + tid;
    const bool valid = kidx < kend;
    const unsigned long long kk = valid ? kidx : kbeg;
    const int row = (int)(kk / (unsigned)P.N), col = (int)(kk - (unsigned long long)row * (unsigned)P.N);
    const double4 ct = P.coltab[(size_t)iq * P.N + col];
    const double4 rr = P.rowtab[(size_t)iq * P.N + row];
    double Ek[NB], Eq[NB];
    band_energies<NB>(P.mc, ct.x, ct.y, rr.x, rr.y, Ek);     // E(k)                       (S2)
    band_energies<NB>(P.mc, ct.z, ct.w, rr.z, rr.w, Eq);     // E(k - q) = E(-k + q)
    double g2 = P.mc.eta_scale;                              // eta(k)                     (S4)
    if (FORM == 1) g2 *= ct.x * rr.x;
    g2 *= g2;
#pragma unroll
    for (int e = 0; e < NB; ++e) {
      CoopHdr hd;
      const double s = fma(0.5, Ek[e] + Eq[e], -P.mc.mu);    // (a + b)/2                  (S3)
      const double d0 = 0.5 * (Ek[e] - Eq[e]);               // (a - b)/2 + h
      const double s2 = fma(s, s, 1e-300);
      hd.s2 = s2; hd.g2 = g2; hd.d0 = d0;
      // exponent bounds over the block tile: R in [R(d2min), R(d2max)], |d0 - h| in [ymin, ymax]
      const double Rmax = sqrt_pos(fma(d2max, g2, s2));
      const double Rmin = sqrt_pos(fma(d2min, g2, s2));
      const double dlo = d0 - hmax, dhi = d0 - hmin;
      const double ymax = fmax(fabs(dlo), fabs(dhi));
      const double ymin = fmax(0.0, fmax(dlo, -dhi));
      const int eAhi = exp_k(fma(Rmax, fc.c1, MAGIC)), eAlo = exp_k(fma(Rmin, fc.c1, MAGIC));
      const int eBhi = exp_k(fma(ymax, fc.c1, MAGIC)), eBlo = exp_k(fma(ymin, fc.c1, MAGIC));
      // a value m 2^e has m in [0.997, 2.51); one unit of slack for rounding at the range ends
      const int hi = max(eAhi, eBhi) + 1, lo = max(eAlo, eBlo) - 1;
      const int spread = hi - lo;                            // every pair sum is in [2^lo, 2^(hi+2))
      const bool robust = force_robust || spread > kSpread;
      hd.eref = hi - (spread >> 1);
      int flags = robust ? (kCoopRobust | (3 << 8)) : (((spread >> 1) + 4) << 8);
      if (!valid || !((P.mc.band_mask >> e) & 1)) flags = kCoopSkip;
      hd.flags = flags;
      hdr_s[tid * NB + e] = hd;
    }
  };

  // ---------------- P1: the SLOTS x (WD + WH) exponentials of sub-batch `bt` into buffer bt & 1 ----------------
  auto p1 = [&](int bt) {
    const CoopHdr* const hdr_b = hdr_s + (bt % BPS) * SLOTS;
    double* const val = buf_s + (bt & 1) * G::BUF_DOUBLES;
    int* const ev = ev_s + (bt & 1) * SLOTS * W;
    if (tid < SLOTS) reinterpret_cast<int2*>(val + SLOTS * W)[tid] = make_int2(hdr_b[tid].eref, hdr_b[tid].flags);
    coop_p1<0, SLOTS, WD, WH, NT, 4>(hdr_b, d2_s, tab256, fc, val, ev, tid);
    coop_p1<1, SLOTS, WD, WH, NT, 4>(hdr_b, h_s, tab256, fc, val, ev, tid);
  };

  p0(0);
  __syncthreads();
  p1(0);
  __syncthreads();

#pragma unroll 1
  for (int bt = 0; bt < nbatch; ++bt) {
    if (bt + 1 < nbatch) {
      if ((bt + 1) % BPS == 0) {        // next sub-batch starts a new group of NT k-points: its headers first
        p0((bt + 1) / BPS);
        __syncthreads();
      }
      p1(bt + 1);
    }
    // ---------------- P2: TH x TD pairs per thread and slot, from buffer bt & 1 ----------------
    const double* const val = buf_s + (bt & 1) * G::BUF_DOUBLES;
    const int* const ev = ev_s + (bt & 1) * SLOTS * W;
    const int2* const efs = reinterpret_cast<const int2*>(val + SLOTS * W);
#pragma unroll 1
    for (int sl = 0; sl < SLOTS; ++sl) {
      const int2 ef = efs[sl];
      const int flags = ef.y;
      if (flags & kCoopSkip) continue;
      const int step = flags >> 8;
      if (drift + step > kDriftLimit) {
#pragma unroll
        for (int i = 0; i < TH; ++i)
#pragma unroll
          for (int j = 0; j < TD; ++j) {
            const int hi = __double2hiint(accP[i][j]);
            const int ex = (hi >> 20) - 1023;
            myE[(i * TD + j) * NT] += ex;
            accP[i][j] = __hiloint2double(hi - (ex << 20), __double2loint(accP[i][j]));
          }
        drift = 0;
      }
      drift += step;
      const double* const va = val + sl * W + tdx * TD;
      const double* const vb = val + sl * W + WD + thx * TH;
      if (!(flags & kCoopRobust)) {
        accEc += ef.x;
        double a[TD];
#pragma unroll
        for (int j = 0; j < TD; j += 2) {
          const double2 v = *reinterpret_cast<const double2*>(va + j);
          a[j] = v.x; a[j + 1] = v.y;
        }
        constexpr int HC = TH < 8 ? TH : 8;
#pragma unroll
        for (int i0 = 0; i0 < TH; i0 += HC) {
          double bb[HC];
#pragma unroll
          for (int i = 0; i < HC; i += 2) {
            const double2 v = *reinterpret_cast<const double2*>(vb + i0 + i);
            bb[i] = v.x; bb[i + 1] = v.y;
          }
#pragma unroll
          for (int i = 0; i < HC; ++i)
#pragma unroll
            for (int j = 0; j < TD; ++j) accP[i0 + i][j] *= (a[j] + bb[i]);
        }
      } else {
        const int* const ea = ev + sl * W + tdx * TD;
        const int* const eb = ev + sl * W + WD + thx * TH;
#pragma unroll
        for (int i = 0; i < TH; ++i) {
          const double mB = vb[i];
          const int eB = eb[i];
#pragma unroll
          for (int j = 0; j < TD; ++j) {
            const int eA = ea[j];
            const int E = max(eA, eB);
            accP[i][j] *= (scale2(va[j], eA - E) + scale2(mB, eB - E));
            myE[(i * TD + j) * NT] += E;
          }
        }
      }
    }
    __syncthreads();     // buffer bt & 1 may be rewritten (by P1 of sub-batch bt + 2), buffer (bt + 1) & 1 is complete
  }

  // P_ij = T (ln2 * exponent sum + ln accP_ij); every thread owns its (h, Delta) pairs for the whole chunk
  const double LN2_HI = 6.93147180369123816490e-01, LN2_LO = 1.90821492927058770002e-10;
  const size_t nout = (size_t)P.nq * P.nh * P.nd;
#pragma unroll
  for (int i = 0; i < TH; ++i) {
    const int ih = th * WH + thx * TH + i;
#pragma unroll
    for (int j = 0; j < TD; ++j) {
      const int id = td * WD + tdx * TD + j;
      const int hi = __double2hiint(accP[i][j]);
      const int ex = (hi >> 20) - 1023;
      const double mant = __hiloint2double(hi - (ex << 20), __double2loint(accP[i][j]));
      const double ed = (double)accEc + (double)(myE[(i * TD + j) * NT] + ex);
      const double lnz = fma(ed, LN2_HI, fma(ed, LN2_LO, log(mant)));
      if (ih < P.nh && id < P.nd)
        P.partial[(size_t)chunk * nout + ((size_t)iq * P.nh + ih) * P.nd + id] = P.T * lnz;
    }
  }
}

}  // namespace fe
