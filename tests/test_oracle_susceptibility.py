"""Pins for the oracle's static Cooper-pair susceptibility (Appendix C).

What fixes it: the Lehmann (spectral) sum of the pair correlator on the 4-state Fock space of one (k up, -k-q down)
pair; the closed form in the atomic limit; the thermodynamic identity chi = [cond N^2/U - Omega''(Delta=0)/2] / N^2
with the already pinned Omega (which fixes the spin, momentum and form-factor conventions of C.2 against Eq. 3/5);
the Thouless criterion U chi(Tc) = 1 against the oracle's own minimum search.  CPU only.
"""
import math

import numpy as np
import pytest

from paper_1412_8754_b200 import workloads as W

PI = math.pi
ONE = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(1.0,), mu=-0.4, U=2.0)
TWO = W.model_params(U=4.0)
THREE = W.model_params(model=W.MODEL_THREE_BAND, mu=W.THREE_BAND_MU, U=1.5)


def lehmann_pair_response(a, b, T):
    """Static response of P = c_2 c_1 for H = a n_1 + b n_2 from the spectral sum
    sum_{m,n} |<m|P^+|n>|^2 (w_n - w_m) / (E_m - E_n),  w = Boltzmann weights: only |0> -> |12> contributes."""
    E = np.array([0.0, a, b, a + b])                       # |0>, |1>, |2>, |12>
    w = np.exp(-(E - E.min()) / T)
    w /= w.sum()
    return (w[0] - w[3]) / (E[3] - E[0])


def test_pair_term_is_the_lehmann_sum(oracle):
    rng = np.random.default_rng(1)
    for a, b, T in zip(rng.uniform(-2, 2, 300), rng.uniform(-2, 2, 300), rng.choice([0.01, 0.1, 1.0], 300)):
        ref = lehmann_pair_response(a, b, T)
        assert abs(oracle.pair_term(a, b, T) - ref) <= 1e-12 * max(1.0, abs(ref)) + 1e-13 / abs(a + b)
    # removable singularity at a + b = 0: limit -f'(a), continuous through it
    for a, T in ((0.3, 0.1), (0.0, 0.05), (-1.2, 0.4)):
        lim = 1.0 / (4 * T * math.cosh(a / (2 * T)) ** 2)
        assert abs(oracle.pair_term(a, -a, T) - lim) < 1e-14 * max(lim, 1)
        assert abs(oracle.pair_term(a, -a + 1e-7, T) - lim) < 1e-5 * max(lim, 1)
        # rounding-noise-sized sums (perfect nesting E(k+Q) = -E(k) in floating point) stay on the limit
        for e in (1e-16, -3e-17, 1e-12, 0.9e-6 * T, 1.1e-6 * T, 1e-5 * T):
            mid = 1.0 / (4 * T * math.cosh((2 * a - e) / (4 * T)) ** 2)          # -f' at the midpoint (a - b)/2
            assert abs(oracle.pair_term(a, -a + e, T) - mid) < 1e-9 * mid, e
    # deep in the Fermi sea / far above it and huge |x|/T: no overflow, 1/(|a|+|b|) for same-sign pairs
    assert abs(oracle.pair_term(3.0, 2.0, 1e-4) - 1 / 5.0) < 1e-15
    assert abs(oracle.pair_term(-3.0, -2.0, 1e-4) - 1 / 5.0) < 1e-15
    assert oracle.pair_term(3.0, -2.0, 1e-4) == 0.0       # blocked: one state empty, the other full


def test_atomic_limit_closed_form(oracle):
    """t = 0: every k has a = -mu - h, b = -mu + h; eta = 1: chi = [tanh(a/2T) + tanh(b/2T)] / (2 (a + b))."""
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(0.0,), mu=0.3, U=1.0)
    T, h = 0.07, 0.11
    a, b = -0.3 - h, -0.3 + h
    ref = (math.tanh(a / (2 * T)) + math.tanh(b / (2 * T))) / (2 * (a + b))
    got = oracle.pair_susceptibility(p, 6, T, [(0.0, 0.0), (0.4, -1.0)], h)
    assert np.allclose(got.reshape(-1), ref, rtol=1e-14, atol=0)
    # s+- form factor at t = 0: chi = <eta(-k-q)^2> * same = eta_scale^2 / 4 for on-grid q
    p2 = dict(p, form_factor=W.FORM_SPM, eta_scale=4.0)
    got = oracle.pair_susceptibility(p2, 8, T, [(2 * PI * 3 / 8, 2 * PI / 8)], h)
    assert abs(got[0, 0, 0] - 4.0 * ref) < 1e-13 * abs(4.0 * ref)


def _chi_from_curvature(oracle, pe, N, T, q, h, dD=2e-3):
    om = oracle.omega_column(pe, N, T, q, h, [0.0, dD, 2 * dD])
    curv = (-om[2] + 16 * om[1] - 15 * om[0]) / (6 * dD * dD)            # even function: 4th-order stencil for Omega''
    return 1.0 / pe["U"] - curv / (2 * N * N)


@pytest.mark.parametrize("p,N", [(ONE, 12), (TWO, 10), (THREE, 8)], ids=["one", "two", "three"])
def test_chi_is_curvature_of_omega_at_delta_zero(oracle, p, N):
    """d^2 Omega_eps / d Delta^2 at Delta = 0 = 2 cond_mult N^2 / U - 2 sum_k eta(k)^2 g(xi_{k up}, xi_{-k+q' down})
    (differentiate Eq. 5 twice; g = thermal factor of C.3).  C.2 is sum_k eta(-k-q)^2 g(xi_{k up}, xi_{-k-q down}):
    (i) eta = 1: the same sum with q' = -q, any real q;
    (ii) eta = cos kx cos ky and q on the grid: relabel k -> -k-q (a permutation of the grid; E, eta even): the pair
         becomes (k down, -k-q up), i.e. Omega'' at q' = -q with the spins exchanged, h -> -h."""
    T, h = 0.12, 0.07
    nb = W.NBANDS[p["model"]]
    # (i)
    q = (0.35, -0.2)
    ps = dict(p, form_factor=W.FORM_S)
    chi = oracle.pair_susceptibility(ps, N, T, [q], h)[0]
    for e in range(nb):
        ref = _chi_from_curvature(oracle, dict(ps, band_mask=1 << e, cond_mult=1.0), N, T, (-q[0], -q[1]), h)
        assert abs(chi[e, e] - ref) < 2e-6 * abs(ref), (e, chi[e, e], ref)
    # (ii)
    q = (2 * PI * 2 / N, 2 * PI * (N - 3) / N)
    pf = dict(p, form_factor=W.FORM_SPM, eta_scale=1.7)
    chi = oracle.pair_susceptibility(pf, N, T, [q], h)[0]
    for e in range(nb):
        pe = dict(pf, band_mask=1 << e, cond_mult=1.0)
        ref = _chi_from_curvature(oracle, pe, N, T, (-q[0], -q[1]), -h)
        assert abs(chi[e, e] - ref) < 2e-6 * abs(ref), (e, chi[e, e], ref)
        # the identity really pins the spin assignment: without the exchange the number is different
        wrong = _chi_from_curvature(oracle, pe, N, T, (-q[0], -q[1]), h)
        assert abs(chi[e, e] - wrong) > 1e-4 * abs(chi[e, e])


def test_interband_elements_and_symmetry(oracle):
    """chi_{eps eps'}(q, h) with bands from LAPACK on independently built matrices; and the exchange symmetry
    chi_{eps eps'}(q, h) = chi_{eps' eps}(q, -h) for eta = 1 (relabel k -> -k-q; E and eta are even)."""
    from test_oracle_three_band import hk
    N, T, h, q = 6, 0.05, 0.03, (0.3, 0.7)
    p = dict(THREE, form_factor=W.FORM_S)
    ref = np.zeros((3, 3))
    for j in range(N):
        for i in range(N):
            kx, ky = 2 * PI * i / N, 2 * PI * j / N
            a = np.linalg.eigvalsh(hk(p["tb3"], kx, ky)) - p["mu"] - h
            b = np.linalg.eigvalsh(hk(p["tb3"], -kx - q[0], -ky - q[1])) - p["mu"] + h
            for e in range(3):
                for f in range(3):
                    ref[e, f] += lehmann_pair_response(a[e], b[f], T) / N**2
    got = oracle.pair_susceptibility(p, N, T, [q], h)[0]
    assert np.max(np.abs(got - ref) / np.abs(ref)) < 1e-11
    # exchange symmetry needs the shifted grid to be the grid: on-grid q
    qg = (2 * PI * 2 / N, 2 * PI * 5 / N)
    a_ = oracle.pair_susceptibility(p, N, T, [qg], h)[0]
    b_ = oracle.pair_susceptibility(p, N, T, [qg], -h)[0]
    assert np.max(np.abs(a_ - b_.T) / np.abs(a_)) < 1e-12
    assert np.all(got > 0)


def test_thouless_criterion_matches_minimum_search(oracle):
    """One band, q = h = 0, second-order transition: Delta* > 0 on a fine grid iff U chi > 1 (cond_mult = 1)."""
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(1.0,), mu=0.0, U=2.0)
    N = 32
    d = np.linspace(0.0, 0.2, 81)
    seen = set()
    for T in (0.02, 0.06, 0.10, 0.14, 0.20, 0.30):
        chi = oracle.pair_susceptibility(p, N, T, [(0.0, 0.0)], 0.0)[0, 0, 0]
        om = oracle.omega_column(p, N, T, (0.0, 0.0), 0.0, d)
        ordered = int(np.argmin(om)) > 0
        assert ordered == (p["U"] * chi > 1.0), (T, chi, int(np.argmin(om)))
        seen.add(ordered)
    assert seen == {True, False}
