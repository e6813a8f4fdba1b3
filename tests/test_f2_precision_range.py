"""SURVEY 8(f-2), the measured statement behind DESIGN.md section 11 f-2: why the pair products of the factored k-sum
cannot simply be moved to binary32.

The factored kernels keep, per (k, band) slot and block tile, A_j = 2cosh(R_j/T) and B_i = 2cosh(|d_i|/T) scaled by ONE
reference exponent, and multiply the sums A'_j + B'_i into running products.  The pair sums of a slot span
2^spread, spread = hi - lo with hi = max exponent of any A_j or B_i of the tile, lo = exponent of the smallest pair sum
(fe_ksum_coop.cuh, P0).  binary64 absorbs up to 900 binades per slot (kSpread); binary32 has 2^-126 .. 2^127 in total,
for the factor AND the running product.  This test evaluates that spread for the slots of config 4 that survive the
early-out (the ones that need pair products at all), from the oracle's band energies on a k
sub-grid, and pins the numbers DESIGN.md quotes.  CPU only."""
import math

import numpy as np

from paper_1412_8754_b200 import workloads as W

LN2 = math.log(2.0)


def dense_slot_spreads(oracle, w, T, nk=128, WH=64, WD=128, gap=44):
    k = 2.0 * np.pi * np.arange(nk) / nk
    out = []
    ntot = ndense = 0
    for iq in (0, w.nq // 3, (2 * w.nq) // 3, w.nq - 1):
        qx, qy = w.q[iq]
        Ek = np.array([[oracle.band_energies(w.params, kx, ky) for kx in k] for ky in k])
        Eq = np.array([[oracle.band_energies(w.params, kx - qx, ky - qy) for kx in k] for ky in k])
        eta2 = np.array([[oracle.eta(w.params, kx, ky) ** 2 for kx in k] for ky in k])
        for e in range(w.nbands):
            s = 0.5 * (Ek[..., e] + Eq[..., e]) - w.params["mu"]
            d0 = 0.5 * (Ek[..., e] - Eq[..., e])
            for th in range(max(1, w.nh // WH)):
                hh = w.h[th * WH:(th + 1) * WH]
                ymax = np.maximum(np.abs(d0 - hh.min()), np.abs(d0 - hh.max()))
                ymin = np.maximum(0.0, np.maximum(d0 - hh.max(), hh.min() - d0))
                for td in range(max(1, w.nd // WD)):
                    dd = w.delta[td * WD:(td + 1) * WD]
                    Rmin = np.sqrt(s * s + dd.min() ** 2 * eta2)
                    Rmax = np.sqrt(s * s + dd.max() ** 2 * eta2)
                    a_dom = (Rmin - ymax) / (T * LN2) >= gap
                    b_dom = (ymin - Rmax) / (T * LN2) >= gap
                    dense = ~a_dom & ~b_dom
                    hi, lo = np.maximum(Rmax, ymax), np.maximum(Rmin, ymin)       # exponents / (T ln2) of the extreme pair sums
                    out.append(((hi - lo) / (T * LN2))[dense])
                    ntot += s.size
                    ndense += int(dense.sum())
    return np.concatenate(out), ndense / ntot


def test_pair_sums_of_dense_slots_exceed_the_binary32_range(oracle):
    w = W.config(4)
    sp_cold, frac_cold = dense_slot_spreads(oracle, w, 0.001)
    sp_warm, frac_warm = dense_slot_spreads(oracle, w, 0.01)
    # early-out leaves ~12 % (T = 0.001) / ~21 % (T = 0.01) of the slots for the pair products
    assert 0.09 < frac_cold < 0.15 and 0.17 < frac_warm < 0.26
    # T = 0.001: the median dense slot spans more binades than binary32 has on one side of 1 (126), one in ten spans > 350;
    # less than half of them would fit a +-100-binade window that still leaves room for the running product to drift
    assert np.median(sp_cold) > 126 and np.percentile(sp_cold, 90) > 350
    assert np.mean(sp_cold <= 100) < 0.45
    # T = 0.01: the spreads are small (< 60 binades), but there the pair products are ~75 % of the step and every slot
    # still has to carry its running product through thousands of factors: 64 renormalisations per thread every few slots
    assert sp_warm.max() < 60
    # binary64 as used by the kernels: every one of these slots is a "fast" slot (spread <= kSpread = 900)
    assert sp_cold.max() < 900


def test_dense_share_by_block_tile_and_per_pair(oracle):
    """The figures DESIGN.md section 5 quotes for the early-out classification of config 4 (dominance gap 2^50, as measured
    when the 32 x 256 tile was introduced): share of (k, band) slots that stay dense per 64 x 128 tile, per 32 x 256 tile and
    per single (h, Delta) pair.  A narrower tile along h leaves fewer slots dense at low T; at T = 0.01 the window is as
    wide as the h range and the tile hardly matters.  (The per-pair case is evaluated on every 8th h and 32nd Delta.)"""
    w = W.config(4)
    got = {}
    for T in (0.001, 0.01):
        for WH, WD in ((64, 128), (32, 256)):
            got[T, WH, WD] = dense_slot_spreads(oracle, w, T, nk=96, WH=WH, WD=WD, gap=50)[1]
        sub = W.Workload("cfg4_sub", w.params, w.N, w.T, w.q, w.h[::8].copy(), w.delta[::32].copy())
        got[T, 1, 1] = dense_slot_spreads(oracle, sub, T, nk=96, WH=1, WD=1, gap=50)[1]
    assert 0.105 < got[0.001, 64, 128] < 0.13 and 0.075 < got[0.001, 32, 256] < 0.10 and 0.015 < got[0.001, 1, 1] < 0.03
    assert 0.20 < got[0.01, 64, 128] < 0.23 and 0.18 < got[0.01, 32, 256] < 0.21 and 0.15 < got[0.01, 1, 1] < 0.19
    assert got[0.001, 32, 256] < 0.8 * got[0.001, 64, 128] and got[0.01, 32, 256] > 0.88 * got[0.01, 64, 128]
