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
//   P0  (once per NT k-points, one k per thread)  dispersion A.1-A.4 at k and k-q (three-band model: the
//       eigenvalues of B.1-B.6 read from the per-q tables of fe_bands3.cuh), s, d0, eta^2 per band, and the
//       block tile's exponent bounds -> a 32-byte header per (k, band) "slot": {s^2, eta^2, d0, Eref, flags}.
//   P1  (per sub-batch of KB k-points)  the SLOTS x (WD + WH) exponentials A_j, B_i: a thread keeps a fixed Delta_j
//       (and a fixed h_i) and walks the slots, four independent sqrt / exp chains at a time; results are scaled by
//       2^-Eref and stored as plain doubles: WD + WH exponentials per slot for the whole block instead of
//       (TD + TH) per thread.  Written into one of two buffers while P2 reads the other (one barrier per sub-batch).
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
#include <type_traits>

#include "fe_kernels.cuh"

namespace fe {

struct CoopParams {
  ModelConsts mc;
  FactoredConsts fc;
  double T;
  int32_t N, nq, nh, nd;
  int32_t ntile_h, ntile_d, ksplit;
  int32_t debug_flags;                 // bit 0: every slot takes the robust path (tests)
  int32_t early_out;                   // 1: A-dominated slots bypass the pair products (FE_EVAL_COOP_EO)
  unsigned long long kc;               // k-points per chunk (multiple of the block size)
  unsigned long long nk;               // N*N
  // Mirror-symmetry reduction (fe_set_symmetry; PAPER.md:157 uses E(-k) = E(k) in the same spirit): when every q of the
  // launch is invariant under a mirror M of the lattice (E, eta invariant under M as well), the terms at k and M k are equal
  // and only the k-points with M k "above" k are summed, with weight 2; the fixed points of M keep weight 1.
  //   sym 0: none.  1: k_y -> -k_y (all q_y = 0).  2: k_x -> -k_x (all q_x = 0).  3: k_x <-> k_y (all q_x = q_y).
  // The reduced index set is [0, n2) (weight 2) followed by [n2, n2 + n1) (weight 1); chunks 0 .. ksplit2 - 1 cover the
  // first part, the others the second, so a chunk has one weight.
  int32_t sym, ksplit2;
  unsigned long long n2, n1;
  const double4* coltab;               // [nq][N] {cos kx, sin kx, cos(kx-qx), sin(kx-qx)}
  const double4* rowtab;               // [nq][N] {cos ky, sin ky, cos(ky-qy), sin(ky-qy)}
  const double* h;                     // [nh]
  const double* d2;                    // [nd]  Delta^2
  const MathTabs* tabs;
  const double* etab;                  // NB == 3 only: [1 + nq][3][N*N] band tables, y = 0: E(k), 1 + iq: E(k - q)
  double* partial;                     // [ksplit][nq*nh*nd]
  unsigned long long* kind_counts;     // NULL, or 5 device counters {dense, A-dominated (list), B-dominated, padding, A-dominated
                                       // (moment series)} slots, summed over all blocks of the launch (fe_enable_slot_counts)
};

struct __align__(16) CoopHdr {         // one per (k, band) slot
  double s2, g2, d0;
  int eref;                            // fast: centred reference exponent
  int flags;                           // bit 0 skip, bit 1 robust, bits 8.. = drift step
};
constexpr int kCoopSkip = 1, kCoopRobust = 2;
// A slot is "A-dominated" when over the whole block tile the binary exponent of 2cosh(R_j/T) exceeds that of 2cosh(|d_i|/T)
// by kDomGap or more (mantissas are in [0.997, 2.51), so A_j / B_i > 2^(kDomGap - 1.4)): then T ln Z_ij is replaced by R_j
// for every pair.  What is neglected per term is T ln(1 + B_i/A_j) + T ln(1 + e^{-2R_j/T}) < T 2^-(kDomGap - 1.4) (1 + tiny),
// and a slot can only be dominated if e^{R_j/T} > 2^(kDomGap - 1.4), i.e. T < R_j / ((kDomGap - 1.4) ln 2): the neglected part
// is below R_j 2^-42.6 / (42.6 ln 2) = 5.1e-15 R_j -- 200 times inside the 1e-12 parity bound even if EVERY dominated pair sat
// exactly at the threshold, and it is one-signed (P is underestimated).  Pairs are in fact spread over thousands of T beyond
// the threshold (a fraction ~ T ln 2 / bandwidth of them lies within one binade of it), so the sum of what is neglected is
// ~1e-17 of the sum: below the rounding noise of the dense path (2e-15 .. 6e-14 observed in the parity tests).  Same bound
// for the B-dominated slots (T ln Z_ij = |d_i|).  Measured on config 4: gap 50 -> 44 turns 8 % (T = 0.01) of the dense
// slots into dominated ones.
constexpr int kDomGap = 44;
// A-dominated slots whose radicand is dominated by s^2 over the whole tile, eps_j = Delta_j^2 g / s^2 <= 1/16, are not even
// square-rooted per Delta_j:  R_j = |s| sqrt(1 + eps_j) = |s| sum_m c_m eps_j^m  (binomial series, c_m = binom(1/2, m)), so
//     sum_k R_j(k) = sum_m c_m Delta_j^(2m) M_m,      M_m = sum_k |s_k| x_k^m,   x_k = g_k / s_k^2,
// and the thread that owns k in P0 adds its kMomN moments once for ALL Delta_j of the tile (2 FP64 instructions per order
// instead of 7 per Delta_j); the polynomial in Delta_j^2 is evaluated once per block.  Truncation after m = kMomN - 1 = 12:
// |c_13| (1/16)^13 / (1 - 1/16) < 2^-59 relative to R_j.  On config 4, 95 - 98 % of the A-dominated slots qualify.
constexpr int kMomN = 13;
constexpr double kMomEps = 0.0625;
__device__ __constant__ const double kMomC[kMomN] = {1.0, 0.5, -0.125, 0.0625, -5.0 / 128, 7.0 / 256, -21.0 / 1024, 33.0 / 2048,
                                                      -429.0 / 32768, 715.0 / 65536, -2431.0 / 262144, 4199.0 / 524288,
                                                      -29393.0 / 4194304};

template <int TH, int TD, int LH, int NW, int KB, int NB>
struct CoopGeom {
  static constexpr int NT = NW * 32;           // threads per block
  static constexpr int LD = 32 / LH;           // lanes of a warp along Delta
  static constexpr int NTD = NW * LD;          // threads along Delta
  static constexpr int WH = TH * LH;           // block tile, h
  static constexpr int WD = TD * NTD;          // block tile, Delta
  static constexpr int PADB = LH > 1 ? 2 : 0;  // B rows of the LH thread rows are 2 doubles apart in banks
  // A' part of a slot row: TD/2 blocks of 2 NTD doubles (the two values a thread fetches with one LDS.128 are adjacent).
  // The blocks are SA = 2 NTD + 8 doubles apart: thread t STORES A'_t at ((t % TD) / 2) SA + (t / TD) 2 + (t & 1), so the 16
  // lanes of a half-warp hit {0..7} and {SA..SA+7}, 16 distinct 8-byte banks (with SA = 2 NTD they collided two by two)
  static constexpr int SA = 2 * NTD + (TD > 2 ? 8 : 0);
  static constexpr int AW = (TD / 2 - 1) * SA + 2 * NTD;     // doubles of the A' part
  static constexpr int W = AW + LH * (TH + PADB);            // doubles per slot row
  static constexpr int SLOTS = KB * NB;        // slots per sub-batch
  static constexpr int BUF_DOUBLES = SLOTS * W + SLOTS;      // values + one int2 {eref, flags} per slot
  static constexpr int DPAD = 16;              // room behind the A-dominated list: its neutral padding (< 8) + one prefetch round (8)
  static constexpr int HTOT = NT * NB + 2 * SLOTS + DPAD;   // header array: dense slots compacted at the front (behind the < SLOTS
                                               // slots carried over from the previous group), B- then A-dominated slots at the back
  // Shapes with all 32 lanes of a warp along Delta (LH = 1: WD = 512) have wide slot rows; with the moment arrays they would
  // take 118 KB of shared memory, one block per SM (measured on config 5: the FP64 pipe below 40 %).  For them the Delta^2
  // list of the tile and the 2^(j/256) table are read from global memory (4 + 2 KB, L1-resident) instead of a shared copy.
  // (Likewise the 8 x 4 register-tile shape, whose launch bound is three blocks per SM: 77 -> 74 KB.)
  static constexpr bool SLIM = LH == 1 || TH * TD < 64;
  static constexpr size_t smem_bytes =
      sizeof(CoopHdr) * HTOT + 2 * sizeof(double) * (size_t)BUF_DOUBLES + 2 * sizeof(int) * (size_t)SLOTS * W +
      sizeof(int) * (size_t)TH * TD * NT + sizeof(double) * ((SLIM ? 0 : 256 + WD) + WH + 8 + WD + NT + kMomN * NT + kMomN * NW) +
      sizeof(int) * 2 * (NW + 2);
  // position of A_j (j = index in the block tile's Delta list) in a slot row: the two doubles a thread reads with
  // one LDS.128 are adjacent and consecutive threads follow each other, so a warp's load is one 128-byte wavefront
  __host__ __device__ static constexpr int posA(int jg) { return ((jg % TD) / 2) * SA + (jg / TD) * 2 + (jg & 1); }
  __host__ __device__ static constexpr int posB(int ib) { return AW + ib + (ib / TH) * PADB; }
};

// m 2^(e - eref) for m in [0.997, 2.51); shifts below -1000 are clamped there (the value is then < 2^-500 of its
// partner in every pair of a fast slot, so what it is exactly does not matter)
__device__ __forceinline__ double coop_scale(double m, int shift) {
  return __hiloint2double(__double2hiint(m) + (max(shift, -1000) << 20), __double2loint(m));
}

// Index i of the symmetry-reduced k set -> (row, col) = (k_y, k_x) grid indices (CoopParams.sym).
__host__ __device__ __forceinline__ void coop_sym_index(int sym, int N, unsigned long long n2, unsigned long long i, int& row, int& col) {
  const unsigned uN = (unsigned)N;
  if (sym == 1) {                      // rows 1 .. (N-1)/2 twice; rows 0 and (N even) N/2 once
    if (i < n2) { row = 1 + (int)(i / uN); col = (int)(i % uN); }
    else { const unsigned long long j = i - n2; row = j < uN ? 0 : N / 2; col = (int)(j % uN); }
  } else if (sym == 2) {               // columns 1 .. (N-1)/2 twice; columns 0 and (N even) N/2 once
    const unsigned M = (unsigned)((N - 1) / 2);
    if (i < n2) { row = (int)(i / M); col = 1 + (int)(i % M); }
    else { const unsigned long long j = i - n2; col = j < uN ? 0 : N / 2; row = (int)(j % uN); }
  } else {                             // strict upper triangle col > row twice (row-major, row r holds N-1-r points); diagonal once
    if (i < n2) {
      const double b = 2.0 * N - 1.0;
      long long r = (long long)((b - sqrt(b * b - 8.0 * (double)i)) * 0.5);
      if (r < 0) r = 0;
      if (r > N - 2) r = N - 2;
      // first index of row r: f(r) = r (2N - 1 - r) / 2; correct the rounding of the square root
      while (r > 0 && (unsigned long long)(r * (2LL * N - 1 - r) / 2) > i) --r;
      while ((unsigned long long)((r + 1) * (2LL * N - 2 - r) / 2) <= i) ++r;
      row = (int)r;
      col = (int)(r + 1 + (long long)(i - (unsigned long long)(r * (2LL * N - 1 - r) / 2)));
    } else { row = col = (int)(i - n2); }
  }
}

// SYM = 1: instance for the symmetry-reduced k set (P.sym = 1, 2, 3); SYM = 0 never looks at P.sym (the kernel sits at
// 255 registers: the index mapping is kept out of the full-zone instance so that its register allocation is untouched)
template <int NB, int FORM, int TH, int TD, int LH, int NW, int KB, int MINB, int SYM = 0>
__global__ void __launch_bounds__(NW * 32, MINB) fe_ksum_coop_kernel(const CoopParams P) {
  using G = CoopGeom<TH, TD, LH, NW, KB, NB>;
  constexpr int NT = G::NT, WH = G::WH, WD = G::WD, W = G::W, SLOTS = G::SLOTS, BPS = NT / KB;
  constexpr int U = 4;                         // independent chains per thread in P1
  static_assert(NT % KB == 0 && TD % 2 == 0 && TH % 4 == 0 && W % 2 == 0 && G::BUF_DOUBLES % 2 == 0, "geometry");
  static_assert(WD % NT == 0 && NT % WH == 0, "P1 mapping");

  extern __shared__ __align__(16) unsigned char smem_raw[];
  CoopHdr* const hdr_s = reinterpret_cast<CoopHdr*>(smem_raw);                       // [HTOT]
  double* const buf_s = reinterpret_cast<double*>(hdr_s + G::HTOT);                  // 2 x {[SLOTS][W] values, [SLOTS] int2}
  double* const tab256_s = buf_s + 2 * G::BUF_DOUBLES;                               // [256]   (not for SLIM shapes)
  double* const d2_s = tab256_s + 256;                                               // [WD]    (not for SLIM shapes)
  double* const h_s = G::SLIM ? tab256_s : d2_s + WD;                                // [WH]
  const double* const tab256 = G::SLIM ? P.tabs->exp2_j256 : tab256_s;
  double* const rng_s = h_s + WH;                                                    // hmin hmax d2min d2max (+pad)
  double* const accR_s = rng_s + 8;                                                  // [WD] sums of R_j over A-dominated slots
  double* const accB_s = accR_s + WD;                                                // [NT / WH][WH] sums of |d_i| over B-dominated slots
  double* const mom_s = accB_s + NT;                                                 // [kMomN][NT] moments M_m, one column per thread
  double* const momred_s = mom_s + kMomN * NT;                                       // [kMomN][NW] their per-warp sums
  int* const ev_s = reinterpret_cast<int*>(momred_s + kMomN * NW);                   // 2 x [SLOTS][W] (robust slots)
  int* const accE_s = ev_s + 2 * SLOTS * W;                                          // [TH*TD][NT]
  int* const scan_s = accE_s + TH * TD * NT;                                         // [2][NW + 2] compaction scan

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int b = blockIdx.x;
  const int chunk = b % P.ksplit;  b /= P.ksplit;
  const int td = b % P.ntile_d;    b /= P.ntile_d;
  const int th = b % P.ntile_h;
  const int iq = b / P.ntile_h;

  // thread's register tile inside the block tile
  const int tdx = warp * G::LD + (lane % G::LD);
  const int thx = lane / G::LD;

  // Delta_j^2 of the block tile, j = index in the tile (entries past the end of the list repeat the last one)
  auto d2at = [&](int i) -> double {
    if constexpr (G::SLIM) return P.d2[min(td * WD + i, P.nd - 1)];
    else return d2_s[i];
  };
  if constexpr (!G::SLIM) {
    for (int i = tid; i < 256; i += NT) tab256_s[i] = P.tabs->exp2_j256[i];
    for (int i = tid; i < WD; i += NT) d2_s[i] = P.d2[min(td * WD + i, P.nd - 1)];
  }
  for (int i = tid; i < WH; i += NT) h_s[i] = P.h[min(th * WH + i, P.nh - 1)];
  for (int i = tid; i < WD; i += NT) accR_s[i] = 0.0;
  accB_s[tid] = 0.0;
#pragma unroll
  for (int m = 0; m < kMomN; ++m) mom_s[m * NT + tid] = 0.0;
  int* const myE = accE_s + tid;
#pragma unroll
  for (int pq = 0; pq < TH * TD; ++pq) myE[pq * NT] = 0;
  __syncthreads();
  if (warp == 0) {   // ranges of the block tile's lists (any order)
    double hmn = h_s[0], hmx = h_s[0], dmn = d2at(0), dmx = dmn;
    for (int i = lane; i < WH; i += 32) { hmn = fmin(hmn, h_s[i]); hmx = fmax(hmx, h_s[i]); }
    for (int i = lane; i < WD; i += 32) { const double v = d2at(i); dmn = fmin(dmn, v); dmx = fmax(dmx, v); }
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
  unsigned long long kbeg = (unsigned long long)chunk * P.kc;
  unsigned long long kend = min(P.nk, kbeg + P.kc);
  if constexpr (SYM != 0) {                      // one weight per chunk: chunks < ksplit2 hold the points counted twice
    if (chunk < P.ksplit2) kend = min(P.n2, kbeg + P.kc);
    else { kbeg = P.n2 + (unsigned long long)(chunk - P.ksplit2) * P.kc; kend = min(P.n2 + P.n1, kbeg + P.kc); }
  }
  const bool force_robust = (P.debug_flags & 1) != 0;

  // ---------------- P0: one k-point per thread -> NB slot headers (for NT consecutive k-points) ----------------
  // The NT*NB slots of a group are sorted into three kinds.  DENSE slots are compacted, in k order, to the front of
  // hdr_s, behind the `nleft` (< SLOTS) dense slots the previous groups left over; only whole sub-batches of SLOTS are
  // handed to P1 / P2, the remainder is carried into the next group (the last group of the chunk pads it with neutral
  // skip slots: one padded sub-batch per chunk instead of one per group); A-DOMINATED slots (early-out mode only)
  // go to the back of hdr_s and are summed right here, sum_k R_j per Delta_j of the block tile, by the thread that
  // owns Delta_j (no exponential, no pair work), B-DOMINATED slots likewise as sum_k |d0 - h_i| per h_i; skip slots (k past the chunk end, masked band) are dropped.
  // Returns (to every thread, through the barriers) the number of dense sub-batches of the group and whether any
  // of its dense slots needs the robust path.
  const bool early_out = P.early_out != 0;
  // dense slots carried over: count (< SLOTS) | may be robust << 8 | position in hdr_s << 9 (one register across the main loop)
  int carry_state = 0;
  auto p0 = [&](int superbatch, bool last_group, int& nsub_out) -> bool {
    const int nleft = carry_state & 0xff;
    const bool left_robust = (carry_state >> 8) & 1;
    CoopHdr carried;                                         // thread tid < nleft moves carried slot tid to the front
    if (tid < nleft) carried = hdr_s[(carry_state >> 9) + tid];
    const unsigned long long kidx = kbeg + (unsigned long long)superbatch * NT + tid;
    const bool valid = kidx < kend;
    unsigned long long kk = valid ? kidx : kbeg;
    int row, col;
    if constexpr (SYM == 0) {
      row = (int)(kk / (unsigned)P.N); col = (int)(kk - (unsigned long long)row * (unsigned)P.N);
    } else {
      coop_sym_index(P.sym, P.N, P.n2, kk, row, col);
      kk = (unsigned long long)row * (unsigned)P.N + col;
    }
    const double4 ct = P.coltab[(size_t)iq * P.N + col];
    const double4 rr = P.rowtab[(size_t)iq * P.N + row];
    double Ek[NB], Eq[NB];
    if constexpr (NB == 3) {                                 // three-band model: numerically diagonalised bands
#pragma unroll                                               // from the per-q tables in HBM
      for (int e = 0; e < 3; ++e) {
        Ek[e] = P.etab[(size_t)e * P.nk + kk];
        Eq[e] = P.etab[((size_t)(1 + iq) * 3 + e) * P.nk + kk];
      }
    } else {
      band_energies<NB>(P.mc, ct.x, ct.y, rr.x, rr.y, Ek);   // E(k)                       (S2)
      band_energies<NB>(P.mc, ct.z, ct.w, rr.z, rr.w, Eq);   // E(k - q) = E(-k + q)
    }
    double g2 = P.mc.eta_scale;                              // eta(k)                     (S4)
    if (FORM == 1) g2 *= ct.x * rr.x;
    g2 *= g2;
    bool any_robust = false;
    CoopHdr hd[NB];
    int kind[NB];                                            // 0 dropped, 1 dense, 2 A-dominated, 3 B-dominated
    int cnt = 0;                                             // dense | A-dominated << 10 | B-dominated << 20 (each <= NT NB < 1024)
    int nser = 0;                                            // A-dominated slots of this thread taken by the moment series
#pragma unroll
    for (int e = 0; e < NB; ++e) {
      const double s = fma(0.5, Ek[e] + Eq[e], -P.mc.mu);    // (a + b)/2                  (S3)
      const double d0 = 0.5 * (Ek[e] - Eq[e]);               // (a - b)/2 + h
      const double s2 = fma(s, s, 1e-300);
      hd[e].s2 = s2; hd[e].g2 = g2; hd[e].d0 = d0;
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
      hd[e].eref = hi - (spread >> 1);
      hd[e].flags = robust ? (kCoopRobust | (3 << 8)) : (((spread >> 1) + 4) << 8);
      kind[e] = 1;
      if (early_out && !force_robust && eAlo - eBhi >= kDomGap) kind[e] = 2;
      if (early_out && !force_robust && eBlo - eAhi >= kDomGap) kind[e] = 3;
      if (!valid || !((P.mc.band_mask >> e) & 1)) kind[e] = 0;
      if (kind[e] == 2 && d2max * g2 <= kMomEps * s2) {       // A-dominated and eps_j <= 1/16 for every Delta_j of the tile:
        kind[e] = 4;                                         // its R_j enter through the moments, not the list (kMomN)
        const double x = g2 * rcp_nr(s2);
        double t = fabs(s);
#pragma unroll
        for (int m = 0; m < kMomN; ++m) {
          mom_s[m * NT + tid] += t;                          // (this thread's own column)
          t *= x;
        }
        ++nser;
      }
      any_robust |= kind[e] == 1 && robust;
      cnt += kind[e] == 1 ? 1 : (kind[e] == 2 ? (1 << 10) : (kind[e] == 3 ? (1 << 20) : 0));
    }
    // block-wide exclusive scan of (dense, dominated) counts in slot order (tid, e)
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += v;
    }
    if (lane == 31) scan_s[warp] = incl;
    __syncthreads();
    int base = 0, total = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const int v = scan_s[w];
      if (w < warp) base += v;
      total += v;
    }
    const int ndense = total & 0x3ff, ndom = (total >> 10) & 0x3ff, ndomB = total >> 20;
    const int nfront = nleft + ndense;                       // dense slots waiting at the front of hdr_s
    const int nsub = last_group ? (nfront + SLOTS - 1) / SLOTS : nfront / SLOTS;
    const int off = base + incl - cnt;                       // exclusive prefix of the three counts
    int pd = nleft + (off & 0x3ff);                          // first dense position of this thread
    if (tid < nleft) hdr_s[tid] = carried;                   // (every thread has read its carried slot before the scan's barrier)
    constexpr int DEND = G::HTOT - G::DPAD;                  // end of the A-dominated list
    int pm = DEND - ndom + ((off >> 10) & 0x3ff);            // first A-dominated position (back of the array)
    int pb = DEND - ndom - ndomB + (off >> 20);              // first B-dominated position (just before them)
#pragma unroll
    for (int e = 0; e < NB; ++e) {
      if (kind[e] == 1) hdr_s[pd++] = hd[e];
      else if (kind[e] == 2) hdr_s[pm++] = hd[e];
      else if (kind[e] == 3) hdr_s[pb++] = hd[e];
    }
    const int npad = last_group ? nsub * SLOTS - nfront : 0;
    if (tid < npad) {                                        // neutral padding of the chunk's last sub-batch
      CoopHdr z;
      z.s2 = 1.0; z.g2 = 0.0; z.d0 = 0.0; z.eref = 0; z.flags = kCoopSkip;
      hdr_s[nfront + tid] = z;
    }
    if (tid < ((8 - (ndom & 7)) & 7)) {                      // the A-dominated list is summed 8 entries at a time: pad it with
      CoopHdr z;                                             // entries that add sqrt(1e-300) = 1e-150 to a sum of O(1) terms
      z.s2 = 1e-300; z.g2 = 0.0; z.d0 = 0.0; z.eref = 0; z.flags = kCoopSkip;
      hdr_s[DEND + tid] = z;
    }
    const bool rob = (__syncthreads_or(any_robust) != 0) || left_robust;
    {
      const int nl = last_group ? 0 : nfront - nsub * SLOTS;
      carry_state = nl | ((rob && nl > 0) ? 0x100 : 0) | ((nsub * SLOTS) << 9);
    }
    if (P.kind_counts != nullptr && tid == 0) {              // diagnostics only (fe_enable_slot_counts): what the launch was made of
      if (ndense) atomicAdd(P.kind_counts + 0, (unsigned long long)ndense);
      if (ndom) atomicAdd(P.kind_counts + 1, (unsigned long long)ndom);
      if (ndomB) atomicAdd(P.kind_counts + 2, (unsigned long long)ndomB);
      if (npad) atomicAdd(P.kind_counts + 3, (unsigned long long)npad);
    }
    if (P.kind_counts != nullptr) {                          // (uniform branch) series slots: one atomic per warp
      const unsigned ws = __reduce_add_sync(0xffffffffu, (unsigned)nser);
      if (lane == 0 && ws) atomicAdd(P.kind_counts + 4, (unsigned long long)ws);
    }
    // A-dominated slots: T ln Z_ij = R_j for the whole tile (kDomGap); this thread owns Delta_j, j = tid + r NT
    if (ndom > 0) {
      // entries 0 .. ndom - 1, then the neutral padding up to a multiple of 8; the fetch runs one round ahead (the last
      // round reads 8 entries past the padding: still inside hdr_s, never used)
      const double2* const dm = reinterpret_cast<const double2*>(&hdr_s[DEND - ndom].s2);   // entry i at dm[2 i]: {s2, g2}
#pragma unroll 1
      for (int r = 0; r < WD / NT; ++r) {
        const double d2 = d2at(tid + r * NT);
        constexpr int UD = 8;                                // independent sqrt chains, fixed order
        double acc[UD];
        double2 g[UD];
        const double2* p = dm;
#pragma unroll
        for (int u = 0; u < UD; ++u) { acc[u] = 0.0; g[u] = p[2 * u]; }
#pragma unroll 1
        for (int i = 0; i < ndom; i += UD) {
          double2 n[UD];
          p += 2 * UD;
#pragma unroll
          for (int u = 0; u < UD; ++u) n[u] = p[2 * u];
#pragma unroll
          for (int u = 0; u < UD; ++u) acc[u] += sqrt_pos(fma(d2, g[u].y, g[u].x));       // R_j, Eq. 4 radicand   (S5)
#pragma unroll
          for (int u = 0; u < UD; ++u) g[u] = n[u];
        }
        const double a0 = acc[0] + acc[4], a1 = acc[1] + acc[5], a2 = acc[2] + acc[6], a3 = acc[3] + acc[7];
        accR_s[tid + r * NT] += (a0 + a1) + (a2 + a3);
      }
    }
    // B-dominated slots (2cosh(|d_i|/T) exceeds 2cosh(R_j/T) by 2^kDomGap over the whole tile): T ln Z_ij = |d0 - h_i|
    // for every Delta_j.  Thread (half, ib) = (tid / WH, tid % WH) sums every (NT / WH)-th entry for its h_i.
    if (ndomB > 0) {
      const CoopHdr* const db = hdr_s + (DEND - ndom - ndomB);
      const double hv = h_s[tid % WH];
      double a0 = 0.0, a1 = 0.0;
      int i = tid / WH;
#pragma unroll 1
      for (; i + NT / WH < ndomB; i += 2 * (NT / WH)) {
        a0 += fabs(db[i].d0 - hv);
        a1 += fabs(db[i + NT / WH].d0 - hv);
      }
      if (i < ndomB) a0 += fabs(db[i].d0 - hv);
      accB_s[tid] += a0 + a1;
    }
    nsub_out = nsub;
    return rob;
  };

  // ---------------- P1: the SLOTS x (WD + WH) exponentials of sub-batch `j` of the group into buffer `par` ----------------
  // A thread keeps its Delta_j^2 (WD/NT of them) and its h_i and walks the slots, U independent chains at a time.
  // ROB: some slot of this group of NT k-points is robust -> per-slot flag test, robust slots store (m, e).
  auto p1 = [&](int j, int par, auto rob_tag) {
    constexpr bool ROB = decltype(rob_tag)::value;
    const CoopHdr* const hdr_b = hdr_s + j * SLOTS;
    double* const val = buf_s + par * G::BUF_DOUBLES;
    int* const ev = ev_s + par * SLOTS * W;
    if (tid < SLOTS) reinterpret_cast<int2*>(val + SLOTS * W)[tid] = make_int2(hdr_b[tid].eref, hdr_b[tid].flags);
    // skip slots (k past the end of the chunk, masked band) get the neutral pair A' = 1, B' = 0: factor exactly 1
    auto put = [&](int pos, double m, int e, int eref, int flags, double neutral) {
      if (ROB && (flags & kCoopRobust)) { val[pos] = m; ev[pos] = e; }
      else val[pos] = (flags & kCoopSkip) ? neutral : coop_scale(m, e - eref);
    };
    // ---- A_j = 2cosh(R_j/T) ----
#pragma unroll 1
    for (int r = 0; r < WD / NT; ++r) {
      const int jg = tid + r * NT;
      const double d2 = d2at(jg);
      const int pos = G::posA(jg);
#pragma unroll 1
      for (int sl0 = 0; sl0 < SLOTS; sl0 += U) {
        double x[U], m[U];
        int e[U], eref[U], flags[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int sl = min(sl0 + u, SLOTS - 1);
          const double2 sg = *reinterpret_cast<const double2*>(&hdr_b[sl].s2);
          const int2 ef = *reinterpret_cast<const int2*>(&hdr_b[sl].eref);
          eref[u] = ef.x; flags[u] = ef.y;
          x[u] = sqrt_pos(fma(d2, sg.y, sg.x));                      // R_j, Eq. 4 radicand           (S5)
        }
        bool fix = false;
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const double t = fma(x[u], fc.c1, MAGIC);
          e[u] = exp_k(t);
          m[u] = exp_mant(x[u], t, fc, tab256);                      // e^{R/T} = m 2^e
          fix |= e[u] < 28;
        }
        if (fix) {
#pragma unroll
          for (int u = 0; u < U; ++u) m[u] = cosh_fix(m[u], e[u]);   // + e^{-R/T}
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (sl0 + u < SLOTS) put((sl0 + u) * W + pos, m[u], e[u], eref[u], flags[u], 1.0);
      }
    }
    // ---- B_i = 2cosh((d0 - h_i)/T): NT / WH slots per pass ----
    {
      constexpr int SPP = NT / WH, PASSES = (SLOTS + SPP - 1) / SPP;
      const int ib = tid % WH, slb = tid / WH;
      const double hv = h_s[ib];
      const int pos = G::posB(ib);
#pragma unroll 1
      for (int p0i = 0; p0i < PASSES; p0i += U) {
        double x[U], m[U];
        int e[U], eref[U], flags[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int sl = min(slb + (p0i + u) * SPP, SLOTS - 1);
          const double d0 = hdr_b[sl].d0;
          const int2 ef = *reinterpret_cast<const int2*>(&hdr_b[sl].eref);
          eref[u] = ef.x; flags[u] = ef.y;
          x[u] = fabs(d0 - hv);                                      // |d_i| = |d0 - h_i|
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const double t = fma(x[u], fc.c1, MAGIC);
          e[u] = exp_k(t);
          m[u] = cosh_fix(exp_mant(x[u], t, fc, tab256), e[u]);      // |d|/T is small on whole lines of the zone
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int sl = slb + (p0i + u) * SPP;
          if (sl < SLOTS) put(sl * W + pos, m[u], e[u], eref[u], flags[u], 0.0);
        }
      }
    }
  };

  // Sub-batches are consumed group by group; a group (NT k-points) has `nsub` dense sub-batches after compaction,
  // possibly none.  `next_group` runs P0 on the following groups until one has dense work (or the chunk ends).
  const int ngroups = (int)((kend - kbeg + NT - 1) / NT);
  int group_next = 0;                            // next group P0 has not seen yet
  auto next_group = [&](int& nsub_out, bool& robust_out) -> bool {
    while (group_next < ngroups) {
      int ns = 0;
      const bool last = group_next + 1 == ngroups;
      const bool rob = p0(group_next++, last, ns);
      if (ns > 0) { nsub_out = ns; robust_out = rob; return true; }
    }
    return false;
  };
  int nsub = 0;                                  // dense sub-batches of the current group
  bool sb_robust = false;
  bool cur_exists = next_group(nsub, sb_robust);
  if (cur_exists) {
    if (sb_robust) p1(0, 0, std::true_type{}); else p1(0, 0, std::false_type{});
  }
  __syncthreads();

  constexpr int HC = TH / 2;                     // the h half-tile handled between two shared-memory fetches
  static_assert(HC % 2 == 0, "half tile");
  // renormalisation: the exponent field of every accP moves into its integer sum (biased: 1023 per call, removed at
  // the end through nrenorm); one shift, one shared-memory reduction and one logic op per accumulator
  int nrenorm = 0;
  auto renorm = [&]() {
#pragma unroll
    for (int i = 0; i < TH; ++i)
#pragma unroll
      for (int j = 0; j < TD; ++j) {
        const int hi = __double2hiint(accP[i][j]);
        atomicAdd(&myE[(i * TD + j) * NT], hi >> 20);
        accP[i][j] = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(accP[i][j]));
      }
    ++nrenorm;
    drift = 0;
  };

  // P1 work that a thread does while it walks the slots of the CURRENT sub-batch in P2 (fused path): per slot its
  // WD / NT values A_j of the same slot number of the NEXT sub-batch, and every SPPE-th slot one value B_i.
  constexpr int RA = WD / NT;
  constexpr int SPP = NT / WH, SPPE = SPP < SLOTS ? SPP : SLOTS;       // slots between two B items of a thread
  static_assert(SLOTS % SPPE == 0 && SPPE <= 4, "fused P1 mapping");
  double d2r[RA];
  int posAr[RA];
#pragma unroll
  for (int r = 0; r < RA; ++r) { d2r[r] = d2at(tid + r * NT); posAr[r] = G::posA(tid + r * NT); }
  const int ibB = tid % WH, slbB = tid / WH, posBr = G::posB(ibB);
  const double hvB = h_s[ibB];

  double xa[RA], ta[RA];                         // stage-1 state of the fused P1 (carried across sub-batches)
  int2 efn = make_int2(0, 0);
  bool have_s1 = false;
  bool cur_robust = sb_robust;                   // robust slots among the group of the sub-batch being consumed
  int j = 0, par = 0;                            // current sub-batch: index in its group, buffer it sits in
#pragma unroll 1
  while (cur_exists) {
    // the sub-batch after this one: the next of the same group, else the first of the next group with dense work
    // (P0 may overwrite the headers now: P1 of every sub-batch of the current group is complete)
    bool nxt_robust = cur_robust, nxt_exists = true;
    int jn = j + 1, nsub_n = nsub;
    if (jn == nsub) { jn = 0; nxt_exists = next_group(nsub_n, nxt_robust); }
    // exponent bookkeeping of the whole sub-batch at once (fused path): sum of the slots' reference exponents and of
    // their drift steps; if the steps of one sub-batch alone could exceed the drift limit (very wide tiles at very
    // low T) the sub-batch takes the plain path below, which checks the drift slot by slot
    int sumE = 0, sumStep = 0;
    {
      const int2* const efc = reinterpret_cast<const int2*>(buf_s + par * G::BUF_DOUBLES + SLOTS * W);
#pragma unroll
      for (int sl = 0; sl < SLOTS; ++sl) { const int2 ef = efc[sl]; sumE += ef.x; sumStep += ef.y >> 8; }
    }
    const bool fused = !cur_robust && !(nxt_exists && nxt_robust) && sumStep <= kDriftLimit;
    if (!fused && nxt_exists) {
      if (nxt_robust) p1(jn, par ^ 1, std::true_type{}); else p1(jn, par ^ 1, std::false_type{});
    }
    // ---------------- P2: TH x TD pairs per thread and slot, from buffer `par` ----------------
    const double* const val = buf_s + par * G::BUF_DOUBLES;
    const int* const ev = ev_s + par * SLOTS * W;
    const int2* const efs = reinterpret_cast<const int2*>(val + SLOTS * W);
    const double* const va0 = val + tdx * 2;                          // + sl W + p 2 NTD
    const double* const vb0 = val + G::AW + thx * (TH + G::PADB);     // + sl W + i
    auto load_a = [&](double (&a)[TD], int sl) {
#pragma unroll
      for (int pp = 0; pp < TD / 2; ++pp) {
        const double2 v = *reinterpret_cast<const double2*>(va0 + sl * W + pp * G::SA);
        a[2 * pp] = v.x; a[2 * pp + 1] = v.y;
      }
    };
    auto load_b = [&](double (&bb)[HC], int sl, int i0) {
#pragma unroll
      for (int i = 0; i < HC; i += 2) {
        const double2 v = *reinterpret_cast<const double2*>(vb0 + sl * W + i0 + i);
        bb[i] = v.x; bb[i + 1] = v.y;
      }
    };
    double a[TD], b0[HC];
    load_a(a, 0);
    load_b(b0, 0, 0);

    if (fused) {
      // next sub-batch's headers and buffer (it may not exist: then this writes the idle buffer from stale,
      // finite headers, which nobody reads)
      const CoopHdr* const hdr_n = hdr_s + jn * SLOTS;
      double* const valn = buf_s + (par ^ 1) * G::BUF_DOUBLES;
      if (tid < SLOTS) reinterpret_cast<int2*>(valn + SLOTS * W)[tid] = make_int2(hdr_n[tid].eref, hdr_n[tid].flags);
      // The P1 chains are split in two stages that run one slot apart, so that each is short and independent of
      // the other: stage 1 (sqrt, range reduction) of slot sl + 1 and stage 2 (polynomial, scaling, store) of slot sl.
      // (stage 1 of a sub-batch's slot 0 is done at the end of the previous iteration when its headers already
      // exist, i.e. inside a group of NT k-points: `have_s1`)
      if (!have_s1) {
        const double2 sg = *reinterpret_cast<const double2*>(&hdr_n[0].s2);
        efn = *reinterpret_cast<const int2*>(&hdr_n[0].eref);
#pragma unroll
        for (int r = 0; r < RA; ++r) {
          xa[r] = sqrt_pos(fma(d2r[r], sg.y, sg.x));                  // R_j, Eq. 4 radicand          (S5)
          ta[r] = fma(xa[r], fc.c1, MAGIC);
        }
      }
      const bool carry = nxt_exists && jn + 1 < nsub_n;               // the sub-batch after next shares its header group
      const CoopHdr* const hdr_nn = hdr_s + (jn + 1) * SLOTS;
      double mb = 0.0, xb = 0.0, tb = 0.0, vbB = 0.0;
      int ebB = 0;
      int2 efb = make_int2(0, 0);
      const double* pa = va0;                                         // this thread's A' / B' of the current slot
      const double* pb = vb0;
      double* pvn = valn;                                             // row of the slot being produced
      const CoopHdr* hn = hdr_n;
      // B' is fetched in chunks of QC values, one chunk ahead of its use (two rotating register buffers)
      constexpr int QC = 4, NQ = TH / QC;
      static_assert(TH % QC == 0 && NQ % 2 == 0, "chunking");
      double bq[2][QC];
      auto load_q = [&](double (&dst)[QC], const double* src) {
#pragma unroll
        for (int i = 0; i < QC; i += 2) {
          const double2 v = *reinterpret_cast<const double2*>(src + i);
          dst[i] = v.x; dst[i + 1] = v.y;
        }
      };
#pragma unroll
      for (int i = 0; i < QC; ++i) bq[0][i] = b0[i];
      if (drift + sumStep > kDriftLimit) renorm();                    // skip slots: step 0, Eref 0, factors 1
      drift += sumStep;
      accEc += sumE;
#pragma unroll 1
      for (int sl0 = 0; sl0 < SLOTS; sl0 += SPPE) {
        const int slB = slbB + (sl0 / SPPE) * SPP;                    // slot of this pass's B item
#pragma unroll
        for (int us = 0; us < SPPE; ++us) {
          const int sl = sl0 + us;
          // ---- one straight-line block: P2 of slot sl interleaved with the P1 chains for the next sub-batch ----
          double an[TD], ma[RA];
          int ea[RA];
          const int2 efa = efn;
          const CoopHdr* const hnn = (sl + 1 < SLOTS) ? hn + 1 : (carry ? hdr_nn : hn);
#pragma unroll
          for (int c = 0; c < NQ; ++c) {
            // fetch the next chunk: of this slot, or (last chunk) the first one of the next slot, and its A'
            if (c + 1 < NQ) load_q(bq[(c + 1) & 1], pb + (c + 1) * QC);
            else            load_q(bq[(c + 1) & 1], pb + W);
            if (c == NQ - 2) {
#pragma unroll
              for (int pp = 0; pp < TD / 2; ++pp) {
                const double2 v = *reinterpret_cast<const double2*>(pa + W + pp * G::SA);
                an[2 * pp] = v.x; an[2 * pp + 1] = v.y;
              }
            }
            // P1 pieces, spread over the chunks
            if (c == 0) {                                             // stage 2 of slot sl's A_j
#pragma unroll
              for (int r = 0; r < RA; ++r) {
                ea[r] = exp_k(ta[r]);
                ma[r] = exp_mant(xa[r], ta[r], fc, tab256);           // e^{R/T} = m 2^e
              }
              if (us == 0) {                                          // B_i of slot slB, stage 1
                const CoopHdr* const hb = hdr_n + min(slB, SLOTS - 1);
                xb = fabs(hb->d0 - hvB);                              // |d_i| = |d0 - h_i|
                efb = *reinterpret_cast<const int2*>(&hb->eref);
                tb = fma(xb, fc.c1, MAGIC);
              }
            }
            if (c == 1) {                                             // stage 1 of slot sl + 1's A_j
              const double2 sg = *reinterpret_cast<const double2*>(&hnn->s2);
              efn = *reinterpret_cast<const int2*>(&hnn->eref);
#pragma unroll
              for (int r = 0; r < RA; ++r) {
                xa[r] = sqrt_pos(fma(d2r[r], sg.y, sg.x));            // R_j, Eq. 4 radicand          (S5)
                ta[r] = fma(xa[r], fc.c1, MAGIC);
              }
              if (us == 0) mb = exp_mant(xb, tb, fc, tab256);
            }
            if (c == NQ - 1 && us == 0) {                             // B_i: + e^{-|d|/T}, among the pair work of this chunk
              ebB = exp_k(tb);
              vbB = cosh_fix(mb, ebB);
            }
#pragma unroll
            for (int i = 0; i < QC; ++i)
#pragma unroll
              for (int j = 0; j < TD; ++j) accP[c * QC + i][j] *= (a[j] + bq[c & 1][i]);
          }
#pragma unroll
          for (int r = 0; r < RA; ++r) {
            if (ea[r] < 28) ma[r] = cosh_fix(ma[r], ea[r]);           // + e^{-R/T} (rare)
            pvn[posAr[r]] = (efa.y & kCoopSkip) ? 1.0 : coop_scale(ma[r], ea[r] - efa.x);
          }
          if (us == SPPE - 1) {                                       // B_i, store
            if (slB < SLOTS) valn[slB * W + posBr] = (efb.y & kCoopSkip) ? 0.0 : coop_scale(vbB, ebB - efb.x);
          }
#pragma unroll
          for (int j = 0; j < TD; ++j) a[j] = an[j];
          pa += W; pb += W; pvn += W; hn = hnn;
        }
      }
      have_s1 = carry;
    } else {
      have_s1 = false;
#pragma unroll 1
      for (int sl = 0; sl < SLOTS; ++sl) {
        const int2 ef = efs[sl];
        const int flags = ef.y;
        double b1[HC], an[TD];
        load_b(b1, sl, HC);                                             // second half of this slot
        const bool fast = !(flags & (kCoopSkip | kCoopRobust));
        if (!(flags & kCoopSkip)) {
          const int step = flags >> 8;
          if (drift + step > kDriftLimit) renorm();
          drift += step;
        }
        if (fast) {
          accEc += ef.x;
#pragma unroll
          for (int i = 0; i < HC; ++i)
#pragma unroll
            for (int j = 0; j < TD; ++j) accP[i][j] *= (a[j] + b0[i]);
        }
        const int nsl = min(sl + 1, SLOTS - 1);                         // fetch the next slot's A and first B half
        load_a(an, nsl);
        load_b(b0, nsl, 0);
        if (fast) {
#pragma unroll
          for (int i = 0; i < HC; ++i)
#pragma unroll
            for (int j = 0; j < TD; ++j) accP[HC + i][j] *= (a[j] + b1[i]);
        } else if (flags & kCoopRobust) {
          const double* const vb = vb0 + sl * W;
          const int* const eb = ev + G::AW + thx * (TH + G::PADB) + sl * W;
#pragma unroll
          for (int j = 0; j < TD; ++j) {
            const int pa = sl * W + (j / 2) * G::SA + tdx * 2 + (j & 1);
            const double mA = val[pa];
            const int eA = ev[pa];
#pragma unroll
            for (int i = 0; i < TH; ++i) {
              const int eB = eb[i];
              const int E = max(eA, eB);
              accP[i][j] *= (scale2(mA, eA - E) + scale2(vb[i], eB - E));
              myE[(i * TD + j) * NT] += E;
            }
          }
        }
#pragma unroll
        for (int j = 0; j < TD; ++j) a[j] = an[j];
      }
    }
    cur_robust = nxt_robust; cur_exists = nxt_exists; j = jn; nsub = nsub_n; par ^= 1;
    __syncthreads();     // buffer `par ^ 1` may be rewritten (by P1 of the sub-batch after next), buffer `par` is complete
  }

  // Moment series of the A-dominated slots (kMomN): column sums in a fixed order (shuffle tree per warp, then the warps in
  // index order), then sum_m c_m Delta_j^(2m) M_m per Delta_j of the tile (Horner in Delta_j^2), added to the list sums.
  if (early_out) {
#pragma unroll
    for (int m = 0; m < kMomN; ++m) {
      const double v = warp_sum(mom_s[m * NT + tid]);
      if (lane == 0) momred_s[m * NW + warp] = v;
    }
    __syncthreads();
    for (int jg = tid; jg < WD; jg += NT) {
      const double d2 = d2at(jg);
      double poly = 0.0;
#pragma unroll
      for (int m = kMomN - 1; m >= 0; --m) {
        double M = momred_s[m * NW];
#pragma unroll
        for (int w = 1; w < NW; ++w) M += momred_s[m * NW + w];
        poly = fma(poly, d2, kMomC[m] * M);
      }
      accR_s[jg] += poly;
    }
    __syncthreads();
  }

  // P_ij = T (ln2 * exponent sum + ln accP_ij); every thread owns its (h, Delta) pairs for the whole chunk
  const double LN2_HI = 6.93147180369123816490e-01, LN2_LO = 1.90821492927058770002e-10;
  const size_t nout = (size_t)P.nq * P.nh * P.nd;
  const double weight = (SYM != 0 && chunk < P.ksplit2) ? 2.0 : 1.0;
#pragma unroll
  for (int i = 0; i < TH; ++i) {
    const int ih = th * WH + thx * TH + i;
    double sumB = 0.0;                                         // B-dominated slots, fixed order over the partial sums
#pragma unroll
    for (int hf = 0; hf < NT / WH; ++hf) sumB += accB_s[hf * WH + thx * TH + i];
    double v[TD];
#pragma unroll
    for (int j = 0; j < TD; ++j) {
      const int hi = __double2hiint(accP[i][j]);
      const int ex = (hi >> 20) - 1023;
      const double mant = __hiloint2double(hi - (ex << 20), __double2loint(accP[i][j]));
      const double ed = (double)accEc + (double)(myE[(i * TD + j) * NT] - 1023 * nrenorm + ex);
      const double lnz = fma(ed, LN2_HI, fma(ed, LN2_LO, log(mant)));
      v[j] = weight * fma(P.T, lnz, accR_s[tdx * TD + j] + sumB);
    }
    // a thread's TD Delta values are consecutive in memory: one 32-byte store per (thread, h) when the row length keeps
    // them 32-byte aligned (nd % 4 == 0; the group is then wholly inside or outside the list), else one double at a time
    const int id0 = td * WD + tdx * TD;
    double* dst = P.partial + (size_t)chunk * nout + ((size_t)iq * P.nh + ih) * P.nd + id0;
    if (ih < P.nh) {
      if (TD == 4 && (P.nd & 3) == 0) {
        if (id0 < P.nd)
          asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" :: "l"(dst), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[TD - 1]) : "memory");
      } else {
#pragma unroll
        for (int j = 0; j < TD; ++j)
          if (id0 + j < P.nd) dst[j] = v[j];
      }
    }
  }
}

}  // namespace fe
