"""Pins for the CPU oracle (oracle/fe_oracle.c): checks against what the paper and the mathematics fix.

None of these re-types the oracle's own Eq. 4 / Eq. 5 evaluation.  They use: the values the paper
prints (tests/golden/paper_constants.json), closed forms, many-body partition functions, and
brute-force numerical diagonalisation (numpy.linalg.eigvalsh) of the orbital-basis / real-space
Bogoliubov-de Gennes matrices.  Labels O1..O12 follow SURVEY.md 8(c) / DESIGN.md "Oracle pins".
Runs on CPU only (-m "not gpu").
"""
import json
import math
import os

import numpy as np
import pytest

from paper_1412_8754_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.json")
PI = math.pi


# ----------------------------------------------------------------------------------------------
# independent helpers (numpy; orbital-basis matrices, never the oracle's closed forms)
# ----------------------------------------------------------------------------------------------
def kgrid(N):
    k = 2.0 * PI * np.arange(N) / N
    return np.meshgrid(k, k, indexing="xy")  # KX[j, i] = k[i], KY[j, i] = k[j]


def orbital_matrix(t, kx, ky):
    """2x2 orbital-basis hopping matrix T_k of the two-band model, Eqs. A.1-A.3."""
    t1, t2, t3, t4 = t
    T11 = -2 * (t1 * np.cos(kx) + t2 * np.cos(ky)) - 4 * t3 * np.cos(kx) * np.cos(ky)
    T22 = -2 * (t2 * np.cos(kx) + t1 * np.cos(ky)) - 4 * t3 * np.cos(kx) * np.cos(ky)
    T12 = -4 * t4 * np.sin(kx) * np.sin(ky)
    M = np.empty(np.shape(kx) + (2, 2))
    M[..., 0, 0], M[..., 1, 1], M[..., 0, 1], M[..., 1, 0] = T11, T22, T12, T12
    return M


def bands_numeric(p, kx, ky):
    """Band energies by NUMERICAL diagonalisation (ascending), shape (..., nb)."""
    if p["model"] == 1:
        return (-2 * p["t"][0] * (np.cos(kx) + np.cos(ky)))[..., None]
    return np.linalg.eigvalsh(orbital_matrix(p["t"], kx, ky))


def softplus_f(x, T):
    """f(x) = -T ln(1 + e^{-x/T}) via numpy's logaddexp (a library routine, not the oracle's form)."""
    return -T * np.logaddexp(0.0, -np.asarray(x) / T)


def neumaier(x):
    return math.fsum(np.asarray(x, dtype=np.float64).ravel().tolist())


def rel(a, b):
    return abs(a - b) / max(abs(a), abs(b), 1e-300)


TWO = W.model_params()                       # paper's two-band constants, s+-, U=2, cond_mult=2
ONE = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(1.0,), mu=0.0, U=2.0)


# ----------------------------------------------------------------------------------------------
# values the paper prints
# ----------------------------------------------------------------------------------------------
def test_paper_constants_are_the_workload_constants():
    g = json.load(open(GOLD))
    t = g["two_band_hoppings"]
    assert W.TWO_BAND_T == (t["t1"], t["t2"], t["t3"], t["t4"])
    assert W.TWO_BAND_MU == g["two_band_half_filling"]["mu"]


def test_O9_filling_is_two_at_mu_1p54(oracle):
    """two electrons per site at mu = 1.54 -- pins sign/order of t1..t4 in A.1-A.3/A.4."""
    g = json.load(open(GOLD))["two_band_half_filling"]
    N = 128
    count = 0
    for j in range(N):
        for i in range(N):
            E = oracle.band_energies(TWO, 2 * PI * i / N, 2 * PI * j / N)
            count += 2 * int(np.sum(E < g["mu"]))        # two spins
    n = count / N**2
    assert abs(n - g["electrons_per_site"]) < 1e-2, n
    # same through the full pipeline: n = -dOmega/dmu at Delta = 0, low T (thermodynamic identity)
    N, T, dmu = 256, 0.002, 1e-3
    om = []
    for mu in (g["mu"] + dmu, g["mu"] - dmu):
        p = W.model_params(mu=mu)
        om.append(oracle.omega_column(p, N, T, (0.0, 0.0), 0.0, [0.0])[0])
    n_fd = -(om[0] - om[1]) / (2 * dmu) / N**2
    assert abs(n_fd - g["electrons_per_site"]) < 1e-2, n_fd
    # a wrong sign of t3 or swapped t1/t2 ordering moves n far from 2:
    bad = W.model_params(t=(-1.0, 1.3, +0.85, -0.85))
    cnt = sum(2 * int(np.sum(oracle.band_energies(bad, 2 * PI * i / 64, 2 * PI * j / 64) < 1.54))
              for i in range(64) for j in range(64)) / 64**2
    assert abs(cnt - 2.0) > 0.2


def test_O10_pocket_signs_and_form_factor(oracle):
    """PAPER.md:230 (E+ electron-like, E- hole-like), :53 (hole pocket at Gamma, sign reversal of cos kx cos ky)."""
    mu = W.TWO_BAND_MU
    Eg = oracle.band_energies(TWO, 0.0, 0.0)
    Ex = oracle.band_energies(TWO, PI, 0.0)
    assert Eg[0] >= Eg[1] and Ex[0] >= Ex[1]              # [0] is the '+' band
    assert Eg[1] - mu > 0                                 # hole-like band is empty at Gamma -> hole pocket
    assert abs((Eg[1] - mu) - 1.26) < 1e-12               # -(t1+t2)*2 - 4 t3 - mu = 2.8 - 1.54 (degenerate at Gamma)
    assert abs((Ex[0] - mu) - (-0.34)) < 1e-12            # electron-like '+' band is occupied at X -> electron pocket
    assert abs(Ex[1] - (-8.0)) < 1e-12
    assert oracle.eta(TWO, 0.0, 0.0) == 1.0
    assert oracle.eta(TWO, PI, 0.0) == -1.0               # s+-: sign reversal between pockets
    assert oracle.eta(ONE, 0.3, 1.1) == 1.0
    assert abs(oracle.eta(W.model_params(eta_scale=4.0), 0.3, 1.1) - 4 * math.cos(0.3) * math.cos(1.1)) < 1e-15


def test_A4_closed_form_vs_numerical_diagonalisation(oracle):
    """Eq. A.4 against eigvalsh of the orbital matrix A.1-A.3 at random k, incl. perturbed hoppings."""
    rng = np.random.default_rng(0)
    for p in (TWO, W.model_params(t=W.perturbed_hoppings(3))):
        for kx, ky in rng.uniform(-7, 7, size=(200, 2)):
            E = oracle.band_energies(p, kx, ky)
            ref = np.linalg.eigvalsh(orbital_matrix(p["t"], kx, ky))
            assert abs(E[0] - ref[1]) < 1e-13 and abs(E[1] - ref[0]) < 1e-13


# ----------------------------------------------------------------------------------------------
# O1  Delta = 0 normal state
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p", [ONE, TWO], ids=["one", "two"])
@pytest.mark.parametrize("q", [(0.0, 0.0), (2 * PI * 3 / 24, 2 * PI * 5 / 24), (0.37, -0.11)],
                         ids=["q0", "qgrid", "qoff"])
def test_O1_normal_state(oracle, p, q):
    """At Delta = 0 {E+, E-} = {a, -b}, so Omega = sum f(xi_up(k)) + f(xi_dn(-k+q)): free fermions."""
    N, T, h = 24, 0.05, 0.13
    KX, KY = kgrid(N)
    Eup = bands_numeric(p, KX, KY) - p["mu"] - h
    Edn = bands_numeric(p, -KX + q[0], -KY + q[1]) - p["mu"] + h
    ref = neumaier(softplus_f(Eup, T)) + neumaier(softplus_f(Edn, T))
    got = oracle.omega_column(p, N, T, q, h, [0.0])[0]
    assert rel(got, ref) < 1e-13
    if q != (0.37, -0.11):
        # on-grid q: the shifted grid is the grid, so the down sum is over the unshifted k
        Edn0 = bands_numeric(p, KX, KY) - p["mu"] + h
        ref0 = neumaier(softplus_f(Eup, T)) + neumaier(softplus_f(Edn0, T))
        assert rel(got, ref0) < 1e-13
        # and the literal Eq. 5 constant (const_mode 1) is then the same number
        p1 = dict(p, const_mode=1)
        assert rel(oracle.omega_column(p1, N, T, q, h, [0.0])[0], got) < 1e-13


def test_const_mode_1_is_eq5_literal(oracle):
    """const_mode 1 replaces sum_k xi_dn(-k+q) by sum_k xi_dn(k) (Eq. 5 as printed): a Delta-independent shift."""
    N, T, h, q = 20, 0.02, 0.07, (0.41, 0.23)
    KX, KY = kgrid(N)
    d = [0.0, 0.1, 0.3]
    # one band at a time (band_mask): E_+ and E_- are not trigonometric polynomials, the readings differ
    for mask, col in ((1, 1), (2, 0)):              # eigvalsh is ascending: column 1 is E_+, column 0 is E_-
        pm = dict(TWO, band_mask=mask, cond_mult=1.0)
        shift = neumaier(bands_numeric(TWO, KX, KY)[..., col]) \
            - neumaier(bands_numeric(TWO, -KX + q[0], -KY + q[1])[..., col])
        o0 = oracle.omega_column(pm, N, T, q, h, d)
        o1 = oracle.omega_column(dict(pm, const_mode=1), N, T, q, h, d)
        assert np.allclose(o1 - o0, shift, rtol=0, atol=1e-10)
        assert abs(shift) > 1e-6
    # both bands together: E_+ + E_- = T11 + T22 IS a trigonometric polynomial of degree < N, so its
    # grid sum is shift-invariant and the two readings coincide (to rounding) for any q
    o0 = oracle.omega_column(TWO, N, T, q, h, d)
    o1 = oracle.omega_column(dict(TWO, const_mode=1), N, T, q, h, d)
    assert np.allclose(o1, o0, rtol=1e-13, atol=0)


# ----------------------------------------------------------------------------------------------
# O2 / O12  many-body partition function of one (k up, -k+q down) pair; atomic limit closed form
# ----------------------------------------------------------------------------------------------
def pair_grand_potential(a, b, gap, T):
    """-T ln Z of H = a n_up + b n_dn + gap (c_up c_dn + h.c.) on the 4 Fock states {0, up, dn, updn}."""
    M = np.array([[0.0, gap], [gap, a + b]])
    lv = np.concatenate([np.linalg.eigvalsh(M), [a, b]])
    m = lv.min()
    return m - T * math.log(np.sum(np.exp(-(lv - m) / T)))


def test_O12_eq4_eq5_equal_pair_partition_function(oracle):
    """f(E+) + f(E-) + b == -T ln Tr exp(-H_pair/T): pins Eq. 4, the thermal term and the constant of Eq. 5."""
    rng = np.random.default_rng(1)
    for _ in range(300):
        a, b = rng.uniform(-3, 3, 2)
        gap = rng.uniform(-1, 1)
        T = 10 ** rng.uniform(-2.5, 0)
        Ep, Em = oracle.quasiparticle(a, b, gap)
        got = oracle.thermal(Ep, T) + oracle.thermal(Em, T) + b
        ref = pair_grand_potential(a, b, gap, T)
        assert abs(got - ref) < 1e-12 * max(1.0, abs(ref))


def test_thermal_stable_form(oracle):
    """f(x) = -T ln(1+exp(-x/T)): library logaddexp, limits f -> x (x << 0), f -> 0 (x >> 0), f(0) = -T ln 2."""
    T = 0.001
    for x in (-5.0, -0.8, -1e-3, -1e-9, 0.0, 1e-9, 1e-3, 0.8, 5.0):
        assert abs(oracle.thermal(x, T) - float(softplus_f(x, T))) <= 1e-15 * max(1.0, abs(x))
    assert oracle.thermal(-5.0, T) == -5.0          # exp(-5000) underflows: no overflow, no NaN
    assert oracle.thermal(5.0, T) == 0.0 or abs(oracle.thermal(5.0, T)) < 1e-300
    assert abs(oracle.thermal(0.0, 0.25) + 0.25 * math.log(2)) < 1e-16


@pytest.mark.parametrize("nb,model", [(1, W.MODEL_ONE_BAND), (2, W.MODEL_TWO_BAND)])
def test_O2_atomic_limit(oracle, nb, model):
    """t = 0, eta = 1: Omega = nb N^2 [-mu - T ln(2cosh(h/T) + 2cosh(sqrt(mu^2+Delta^2)/T))] + cond."""
    N, T, mu, h, U = 7, 0.2, 0.6, 0.35, 1.7
    p = W.model_params(model=model, form_factor=W.FORM_S, t=(0, 0, 0, 0), mu=mu, U=U)
    for D in (0.0, 0.3, -0.9):
        R = math.sqrt(mu * mu + D * D)
        ref = nb * N * N * (-mu - T * math.log(2 * math.cosh(h / T) + 2 * math.cosh(R / T))) \
            + p["cond_mult"] * N * N * D * D / U
        got = oracle.omega_column(p, N, T, (0.3, 0.9), h, [D])[0]
        assert rel(got, ref) < 1e-14
    assert p["cond_mult"] == nb


# ----------------------------------------------------------------------------------------------
# O3  textbook: half-filled free square lattice, E0/site = -16 t / pi^2
# ----------------------------------------------------------------------------------------------
def test_O3_free_square_lattice_ground_state(oracle):
    N, T = 512, 1e-4
    om = oracle.omega_column(ONE, N, T, (0.0, 0.0), 0.0, [0.0])[0]
    assert abs(om / N**2 - (-16.0 / PI**2)) < 1e-4


# ----------------------------------------------------------------------------------------------
# O4  symmetries
# ----------------------------------------------------------------------------------------------
def test_O4_symmetries(oracle):
    N, T = 16, 0.03
    q, h = (0.5, 0.2), 0.11
    d = np.array([0.05, 0.21, 0.4])
    o = oracle.omega_column(TWO, N, T, q, h, d)
    assert np.array_equal(o, oracle.omega_column(TWO, N, T, q, h, -d))                  # Delta -> -Delta, bitwise
    assert np.allclose(o, oracle.omega_column(TWO, N, T, (-q[0], -q[1]), h, d), rtol=1e-14, atol=0)   # q -> -q
    assert np.allclose(o, oracle.omega_column(TWO, N, T, (q[1], q[0]), h, d), rtol=1e-14, atol=0)     # x <-> y
    o0 = oracle.omega_column(TWO, N, T, (0, 0), h, d)
    assert np.allclose(o0, oracle.omega_column(TWO, N, T, (0, 0), -h, d), rtol=1e-14, atol=0)         # h -> -h at q=0
    om = oracle.omega_column(TWO, N, T, q, -h, d)
    assert np.max(np.abs(om - o) / np.abs(o)) > 1e-7        # ... but NOT at q != 0 (spin convention G1 matters)
    # s-wave, on-grid q: h -> -h is again a symmetry
    qg = (2 * PI * 2 / N, 2 * PI * 5 / N)
    a = oracle.omega_column(ONE, N, T, qg, h, d)
    b = oracle.omega_column(ONE, N, T, qg, -h, d)
    assert np.allclose(a, b, rtol=1e-13, atol=0)


def test_spin_convention_G1(oracle):
    """up = +1: xi_up = E - mu - h.  At Delta=0, T->0, one band, a field h>0 lowers Omega by populating up spins;
    with pairing momentum q the up branch is evaluated at k and the down branch at -k+q (checked through O1);
    here: dOmega/dh = -(N_up - N_dn) < 0 for h > 0."""
    N, T = 64, 0.01
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(1.0,), mu=-0.5, U=2.0)
    o = [oracle.omega_column(p, N, T, (0, 0), h, [0.0])[0] for h in (0.19, 0.21)]
    KX, KY = kgrid(N)
    xi = -2 * (np.cos(KX) + np.cos(KY)) + 0.5
    nup = np.sum(1 / (1 + np.exp((xi - 0.2) / T)))
    ndn = np.sum(1 / (1 + np.exp((xi + 0.2) / T)))
    assert nup > ndn
    assert abs((o[1] - o[0]) / 0.02 + (nup - ndn)) < 2e-2 * (nup - ndn)


# ----------------------------------------------------------------------------------------------
# O5  q = 0, h = 0: textbook BCS grand potential
# ----------------------------------------------------------------------------------------------
def test_O5_bcs_reduction(oracle):
    w = W.config(1)
    N, T, U = w.N, w.T[0], w.params["U"]
    KX, KY = kgrid(N)
    xi = -2.0 * (np.cos(KX) + np.cos(KY)) - w.params["mu"]
    for D in (0.0, 0.1, 0.373, 0.5):
        E = np.sqrt(xi**2 + D**2)
        ref = neumaier(xi - E) + neumaier(-2 * T * np.logaddexp(0.0, -E / T)) + N * N * D * D / U
        got = oracle.omega_column(w.params, N, T, (0, 0), 0.0, [D])[0]
        assert rel(got, ref) < 1e-13


# ----------------------------------------------------------------------------------------------
# O6  stationarity == gap equation
# ----------------------------------------------------------------------------------------------
def gap_equation_rhs(p, N, T, q, h, D):
    """dOmega/dDelta from the analytic derivative, bands by numerical diagonalisation."""
    KX, KY = kgrid(N)
    Ek = bands_numeric(p, KX, KY)
    Ekq = bands_numeric(p, -KX + q[0], -KY + q[1])
    eta = p["eta_scale"] * (np.cos(KX) * np.cos(KY) if p["form_factor"] == 1 else np.ones_like(KX))
    s = (Ek + Ekq) / 2 - p["mu"]
    d = (Ek - Ekq) / 2 - h
    R = np.sqrt(s**2 + (D * eta[..., None]) ** 2)
    g = (D * eta[..., None] ** 2 / R) * 0.5 * (np.tanh((R + d) / (2 * T)) + np.tanh((R - d) / (2 * T)))
    return 2 * p["cond_mult"] * N * N * D / p["U"] - neumaier(g)


def test_O6_stationarity_is_gap_equation(oracle):
    N, T, q, h, D = 64, 0.01, (0.2, 0.0), 0.03, 0.11
    p = W.model_params(U=4.0)
    e = 1e-5
    o = oracle.omega_column(p, N, T, q, h, [D - e, D + e])
    fd = (o[1] - o[0]) / (2 * e)
    an = gap_equation_rhs(p, N, T, q, h, D)
    assert rel(fd, an) < 1e-7
    # wrong coupling normalisation (cond_mult 1 instead of 2) would be far off:
    assert rel(fd, gap_equation_rhs(dict(p, cond_mult=1.0), N, T, q, h, D)) > 1e-2


def test_O6_gap_equation_root_is_grid_argmin(oracle):
    """BCS config 1: the root of 1 = (U/N^2) sum tanh(E/2T)/(2E) lies within one grid step of the argmin."""
    w = W.config(1)
    om = oracle.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta)
    idx, ds, _ = oracle.argmin(om, w.delta)
    lo, hi = 0.05, 0.5
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if gap_equation_rhs(w.params, w.N, w.T[0], (0, 0), 0.0, mid) < 0:
            lo = mid
        else:
            hi = mid
    step = w.delta[1] - w.delta[0]
    assert 0 < idx[0, 0] < w.nd - 1
    assert abs(ds[0, 0] - lo) <= step
    # and an interior-minimum two-band grid with a field: same statement
    x = W.interior_minimum(N=32, U=5.0, T=0.01, nq=1, nh=1, nd=128)
    om = oracle.omega_grid(x.params, x.N, x.T[0], x.q, x.h, x.delta)
    idx, ds, _ = oracle.argmin(om, x.delta)
    assert 0 < idx[0, 0] < x.nd - 1
    g_lo = gap_equation_rhs(x.params, x.N, x.T[0], x.q[0], x.h[0], x.delta[idx[0, 0] - 1])
    g_hi = gap_equation_rhs(x.params, x.N, x.T[0], x.q[0], x.h[0], x.delta[idx[0, 0] + 1])
    assert g_lo < 0 < g_hi


# ----------------------------------------------------------------------------------------------
# O7  brute force, real space: 4x4 periodic lattice, FF order parameter, 32x32 BdG matrix
# ----------------------------------------------------------------------------------------------
def real_space_bdg(L, t, mu, h, D, m):
    """H = Psi^+ [[H_up, Dm], [Dm^+, -H_dn^T]] Psi + Tr H_dn,  Psi = (c_up ; c_dn^+),
    hopping -t on nearest neighbours (periodic), pairing sum_j D e^{i q.R_j} c^+_{j up} c^+_{j dn} + h.c.,
    q = 2 pi m / L, which pairs (k up, -k+q dn) as in Eq. 3."""
    n = L * L
    hop = np.zeros((n, n))
    for x in range(L):
        for y in range(L):
            j = x + L * y
            for dx, dy in ((1, 0), (0, 1)):
                jj = (x + dx) % L + L * ((y + dy) % L)
                hop[j, jj] += -t
                hop[jj, j] += -t
    Hup = hop - (mu + h) * np.eye(n)
    Hdn = hop - (mu - h) * np.eye(n)
    ph = np.array([np.exp(1j * 2 * PI * (m[0] * (j % L) + m[1] * (j // L)) / L) for j in range(n)])
    Dm = np.diag(D * ph)
    M = np.block([[Hup.astype(complex), Dm], [Dm.conj().T, -Hdn.T.astype(complex)]])
    return np.linalg.eigvalsh(M), float(np.trace(Hdn))


@pytest.mark.parametrize("m", [(0, 0), (1, 0), (1, 3), (2, 2)])
def test_O7_real_space_bdg_bruteforce(oracle, m):
    L, t, mu, h, D, T, U = 4, 1.0, 0.4, 0.2, 0.7, 0.3, 3.0
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(t,), mu=mu, U=U)
    q = (2 * PI * m[0] / L, 2 * PI * m[1] / L)
    ev, trdn = real_space_bdg(L, t, mu, h, D, m)
    # spectrum: sorted {E+-(k)} from the oracle's Eq. 4 == sorted eigenvalues of the 32x32 matrix
    spec = []
    for j in range(L):
        for i in range(L):
            kx, ky = 2 * PI * i / L, 2 * PI * j / L
            a = oracle.band_energies(p, kx, ky)[0] - mu - h
            b = oracle.band_energies(p, -kx + q[0], -ky + q[1])[0] - mu + h
            spec.extend(oracle.quasiparticle(a, b, D * oracle.eta(p, kx, ky)))
    assert np.max(np.abs(np.sort(spec) - ev)) < 1e-13
    ref = neumaier(softplus_f(ev, T)) + trdn + L * L * D * D / U
    got = oracle.omega_column(p, L, T, q, h, [D])[0]
    assert rel(got, ref) < 1e-13


# ----------------------------------------------------------------------------------------------
# O8  brute force, two-band: per-k 4x4 BdG in the ORBITAL basis (q = 0) and in the band basis (q != 0)
# ----------------------------------------------------------------------------------------------
def test_O8_two_band_orbital_bdg(oracle):
    L, T, h, D, U = 4, 0.15, 0.12, 0.45, 2.5
    p = W.model_params(U=U)
    mu = p["mu"]
    total = 0.0
    for j in range(L):
        for i in range(L):
            kx, ky = 2 * PI * i / L + 0.01, 2 * PI * j / L - 0.02   # generic (non-degenerate) points too
            Tk = orbital_matrix(p["t"], kx, ky)
            g = D * math.cos(kx) * math.cos(ky)
            M = np.block([[Tk - (mu + h) * np.eye(2), g * np.eye(2)],
                          [g * np.eye(2), -(Tk - (mu - h) * np.eye(2)).T]])
            ev = np.linalg.eigvalsh(M)
            E = oracle.band_energies(p, kx, ky)
            spec = []
            for e in range(2):
                spec.extend(oracle.quasiparticle(E[e] - mu - h, E[e] - mu + h, D * oracle.eta(p, kx, ky)))
            assert np.max(np.abs(np.sort(spec) - ev)) < 1e-13
    # full Omega on the true 4x4 grid, q = 0, from orbital-basis diagonalisation only
    for j in range(L):
        for i in range(L):
            kx, ky = 2 * PI * i / L, 2 * PI * j / L
            Tk = orbital_matrix(p["t"], kx, ky)
            g = D * math.cos(kx) * math.cos(ky)
            M = np.block([[Tk - (mu + h) * np.eye(2), g * np.eye(2)],
                          [g * np.eye(2), -(Tk - (mu - h) * np.eye(2)).T]])
            total += float(np.sum(softplus_f(np.linalg.eigvalsh(M), T))) + np.trace(Tk - (mu - h) * np.eye(2))
    total += 2 * L * L * D * D / U
    got = oracle.omega_column(p, L, T, (0, 0), h, [D])[0]
    assert rel(got, total) < 1e-13


def test_O8_band_basis_bdg_offgrid_q(oracle):
    rng = np.random.default_rng(5)
    p = TWO
    mu, h, D = p["mu"], 0.09, 0.33
    for kx, ky, qx, qy in rng.uniform(-3, 3, size=(50, 4)):
        Ek = oracle.band_energies(p, kx, ky)
        Ekq = oracle.band_energies(p, -kx + qx, -ky + qy)
        g = D * oracle.eta(p, kx, ky)
        M = np.block([[np.diag(Ek - mu - h), g * np.eye(2)], [g * np.eye(2), -np.diag(Ekq - mu + h)]])
        spec = []
        for e in range(2):
            spec.extend(oracle.quasiparticle(Ek[e] - mu - h, Ekq[e] - mu + h, g))
        assert np.max(np.abs(np.sort(spec) - np.linalg.eigvalsh(M))) < 1e-13


def test_band_mask_splits_omega(oracle):
    """Omega = sum_eps Omega_eps: the two single-band potentials add up to the total."""
    N, T, q, h = 12, 0.02, (0.3, 0.1), 0.05
    d = [0.0, 0.2]
    tot = oracle.omega_column(TWO, N, T, q, h, d)
    a = oracle.omega_column(dict(TWO, band_mask=1, cond_mult=1.0), N, T, q, h, d)
    b = oracle.omega_column(dict(TWO, band_mask=2, cond_mult=1.0), N, T, q, h, d)
    assert np.allclose(a + b, tot, rtol=1e-13, atol=0)
    assert np.max(np.abs(a - b)) > 1e-3


# ----------------------------------------------------------------------------------------------
# O11  T -> 0 closed form and Pauli-limit blindness
# ----------------------------------------------------------------------------------------------
def test_O11_zero_temperature_limit(oracle):
    N, q, h, D = 32, (0.21, 0.0), 0.08, 0.15
    p = W.model_params(U=4.0)
    KX, KY = kgrid(N)
    Ek = bands_numeric(p, KX, KY)
    Ekq = bands_numeric(p, -KX + q[0], -KY + q[1])
    eta = np.cos(KX) * np.cos(KY)
    s = (Ek + Ekq) / 2 - p["mu"]
    d = (Ek - Ekq) / 2 - h
    R = np.sqrt(s**2 + (D * eta[..., None]) ** 2)
    ref = neumaier(s - np.maximum(R, np.abs(d))) + p["cond_mult"] * N * N * D * D / p["U"]
    got = oracle.omega_column(p, N, 1e-6, q, h, [D])[0]
    assert rel(got, ref) < 1e-9


def test_O11_gapped_state_is_field_blind(oracle):
    """eta = 1, q = 0: for |h| < min_k R - 40 T the fully gapped state does not see the field."""
    w = W.config(1)
    D, T = 0.4, 0.002
    o0 = oracle.omega_column(w.params, w.N, T, (0, 0), 0.0, [D])[0]
    o1 = oracle.omega_column(w.params, w.N, T, (0, 0), 0.3, [D])[0]
    assert rel(o0, o1) < 1e-14
    o2 = oracle.omega_column(w.params, w.N, T, (0, 0), 0.45, [D])[0]      # h > Delta: Pauli limit crossed
    assert rel(o0, o2) > 1e-6


# ----------------------------------------------------------------------------------------------
# argmin, grid layout, error paths
# ----------------------------------------------------------------------------------------------
def test_argmin_linear_search_lowest_index_on_ties(oracle):
    rng = np.random.default_rng(2)
    om = rng.integers(0, 5, size=(6, 7, 40)).astype(np.float64)     # many exact ties
    d = np.linspace(0, 1, 40)
    idx, ds, os_ = oracle.argmin(om, d)
    assert np.array_equal(idx, np.argmin(om, axis=-1).astype(np.int32))   # numpy: first occurrence
    assert np.array_equal(ds, d[idx])
    assert np.array_equal(os_, np.min(om, axis=-1))


def test_argmin_q_outer_loop_of_algorithm_1(oracle):
    """Algorithm 1 lines 1, 6-9 against numpy.argmin on the flattened (q, Delta) axis, with exact
    ties (first occurrence in (iq, id) order wins) and with the condensation-energy reference (reading G17)."""
    rng = np.random.default_rng(4)
    om = rng.integers(-5, 5, size=(6, 7, 9)).astype(np.float64)        # many exact ties
    iq, idd, val = oracle.argmin_q(om)
    flat = om.transpose(1, 0, 2).reshape(7, -1)
    assert np.array_equal(iq * 9 + idd, np.argmin(flat, axis=1))
    assert np.array_equal(val, flat.min(axis=1))
    om = rng.normal(size=(5, 4, 8))
    iq, idd, val = oracle.argmin_q(om, ref_id=2)
    ce = (om - om[:, :, 2:3]).transpose(1, 0, 2).reshape(4, -1)
    assert np.array_equal(iq * 8 + idd, np.argmin(ce, axis=1)) and np.array_equal(val, ce.min(axis=1))
    assert np.all(val <= 0.0)                                          # the reference point itself gives 0
    with pytest.raises(ValueError):
        oracle.argmin_q(om, ref_id=8)
    # physics: on the interior-minimum grid the uniform state (q = 0) wins at h = 0 and is beaten or lost at high h
    w = W.interior_minimum(N=32, U=5.0, T=0.005, nq=4, nh=4, nd=24)
    g = oracle.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta)
    iq, idd, val = oracle.argmin_q(g, ref_id=0)
    assert iq[0] == 0 and idd[0] > 0 and val[0] < 0
    cols_iq, cols_id, _ = oracle.argmin(g, w.delta)
    for ih in range(w.nh):                                             # consistent with the per-(q, h) search
        assert idd[ih] == cols_iq[iq[ih], ih]


def test_grid_is_columns_in_q_h_delta_order(oracle):
    w = W.ragged(N=9, nq=2, nh=3, nd=5)
    om = oracle.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta)
    assert om.shape == (2, 3, 5)
    for iq in range(2):
        for ih in range(3):
            col = oracle.omega_column(w.params, w.N, w.T[0], w.q[iq], w.h[ih], w.delta)
            assert np.array_equal(om[iq, ih], col)


def test_oracle_rejects_bad_input(oracle):
    with pytest.raises(ValueError):
        oracle.omega_column(TWO, 8, 0.0, (0, 0), 0.0, [0.1])          # T = 0 (reading G7)
    with pytest.raises(ValueError):
        oracle.omega_column(dict(TWO, U=0.0), 8, 0.1, (0, 0), 0.0, [0.1])
    with pytest.raises(ValueError):
        oracle.omega_column(dict(TWO, model=4), 8, 0.1, (0, 0), 0.0, [0.1])          # models are 1, 2, 3


def test_survey_anchor_config1(oracle):
    """Config 1 anchors recorded in SURVEY.md 8(c) (independent numpy probe of the survey session)."""
    w = W.config(1)
    om = oracle.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta)
    idx, ds, os_ = oracle.argmin(om, w.delta)
    assert idx[0, 0] == 47
    assert abs(os_[0, 0] / w.N**2 - (-1.63885196927)) < 1e-10
    assert abs(om[0, 0, 0] / w.N**2 - (-1.61938750152)) < 1e-10


def test_magnitude_diagnostic(oracle):
    """feo_omega_column_magnitude (the scale the parity tests measure ill-conditioned sums against): triangle
    inequality against Omega itself; for a completely filled band every term of Eq. 5 is negative, so the magnitude is
    -Omega + 2 x condensation term exactly; in the atomic limit (t = 0) every k contributes the same closed-form term."""
    d = np.array([0.0, 0.13, 0.4])
    q, h = np.array([[0.3, -0.2]]), np.array([0.07])
    for p in (W.model_params(), W.model_params(band_mask=1, cond_mult=1.0), W.model_params(model=W.MODEL_THREE_BAND, mu=W.THREE_BAND_MU, band_mask=4, cond_mult=1.0)):
        om = oracle.omega_grid(p, 12, 0.01, q, h, d)
        mag = oracle.omega_grid_magnitude(p, 12, 0.01, q, h, d)
        assert np.all(mag >= np.abs(om) * (1 - 1e-14))
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(1.0,), mu=9.0, U=2.0)      # filled band
    om = oracle.omega_grid(p, 10, 0.02, q, h, d)[0, 0]
    mag = oracle.omega_grid_magnitude(p, 10, 0.02, q, h, d)[0, 0]
    cond = 1.0 * 100 * d * d / 2.0
    assert np.allclose(mag, -om + 2 * cond, rtol=1e-13, atol=0)
    p = W.model_params(model=W.MODEL_ONE_BAND, form_factor=W.FORM_S, t=(0.0,), mu=-0.3, U=2.0)     # atomic limit
    T, hh = 0.05, 0.07
    mag = oracle.omega_grid_magnitude(p, 6, T, q, np.array([hh]), d)[0, 0]
    R = np.sqrt(0.3 ** 2 + d ** 2)
    f = lambda x: -T * np.logaddexp(0.0, -x / T)        # noqa: E731
    want = 36 * (np.abs(f(-hh + R)) + np.abs(f(-hh - R)) + abs(0.3 + hh)) + 36 * d * d / 2.0
    assert np.allclose(mag, want, rtol=1e-13, atol=0)
