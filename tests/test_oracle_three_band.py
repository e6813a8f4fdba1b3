"""Pins for the oracle's three-band model (Appendix B).

What fixes it: the filling the paper prints (n = 4 at mu = 0.4748), LAPACK (numpy eigvalsh) for the numerical
3x3 diagonalisation, brute-force 6x6 orbital-basis BdG matrices for Eq. 4, and the free-fermion normal state.
CPU only.
"""
import json
import math
import os

import numpy as np
import pytest

from paper_1412_8754_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.json")
PI = math.pi
THREE = W.model_params(model=W.MODEL_THREE_BAND, mu=W.THREE_BAND_MU, U=0.5)


def rel(a, b):
    return abs(a - b) / max(abs(a), abs(b), 1e-300)


def softplus_f(x, T):
    return -T * np.logaddexp(0.0, -np.asarray(x) / T)


def hk(tb3, kx, ky):
    """Independent numpy construction of the Hermitian T_k of Eqs. B.1-B.6 (used with eigvalsh only)."""
    t = (None,) + tuple(tb3[:12])
    e0 = tb3[12]
    cx, cy, sx, sy = math.cos(kx), math.cos(ky), math.sin(kx), math.sin(ky)
    c2x, c2y = math.cos(2 * kx), math.cos(2 * ky)
    H = np.zeros((3, 3), dtype=complex)
    H[0, 0] = 2 * t[2] * cx + 2 * t[1] * cy + 4 * t[3] * cx * cy + 2 * t[11] * (c2x - c2y) + 4 * t[12] * c2x * c2y
    H[1, 1] = 2 * t[1] * cx + 2 * t[2] * cy + 4 * t[3] * cx * cy - 2 * t[11] * (c2x - c2y) + 4 * t[12] * c2x * c2y
    H[2, 2] = e0 + 2 * t[5] * (cx + cy) + 4 * t[6] * cx * cy + 2 * t[9] * (c2x + c2y) + 4 * t[10] * (c2x * cy + cx * c2y)
    H[0, 1] = H[1, 0] = 4 * t[4] * sx * sy
    H[0, 2] = 2j * t[7] * sx + 4j * t[8] * sx * cy
    H[1, 2] = 2j * t[7] * sy + 4j * t[8] * sy * cx
    H[2, 0], H[2, 1] = np.conj(H[0, 2]), np.conj(H[1, 2])
    return H


def test_paper_constants_three_band():
    g = json.load(open(GOLD))
    t = g["three_band_hoppings"]
    assert W.THREE_BAND_T == tuple(t[f"t{i}"] for i in range(1, 13)) + (t["eps0"],)
    assert W.THREE_BAND_MU == g["three_band_filling"]["mu"]


def test_jacobi_eigenvalues_vs_lapack(oracle):
    """feo_herm3_eigvals against numpy.linalg.eigvalsh (zheevd) on random, degenerate and diagonal matrices."""
    rng = np.random.default_rng(11)
    mats = []
    for _ in range(300):
        a = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))
        mats.append((a + a.conj().T) * rng.choice([1e-3, 1.0, 50.0]))
    u = np.linalg.qr(rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3)))[0]
    mats.append(u @ np.diag([1.0, 1.0, 2.0]) @ u.conj().T)            # exact double degeneracy
    mats.append(u @ np.diag([0.3, 0.3, 0.3]) @ u.conj().T)            # multiple of the identity
    mats.append(np.diag([3.0, -1.0, 2.0]).astype(complex))            # already diagonal, unsorted
    mats.append(np.zeros((3, 3), dtype=complex))
    for a in mats:
        a = (a + a.conj().T) / 2
        got = oracle.herm3_eigvals(a)
        ref = np.linalg.eigvalsh(a)
        assert np.max(np.abs(got - ref)) <= 8e-15 * max(1e-3, np.abs(ref).max()), (got, ref)
        assert got[0] <= got[1] <= got[2]


def test_three_band_matrix_is_hermitian_and_even_spectrum(oracle):
    """T_k Hermitian; T_{-k} = conj(T_k) so E(-k) = E(k) -- the property that lets -k+q be k-q."""
    rng = np.random.default_rng(2)
    for kx, ky in rng.uniform(-4, 4, size=(100, 2)):
        H = oracle.three_band_matrix(THREE, kx, ky)
        assert np.array_equal(H, H.conj().T)
        assert np.allclose(oracle.three_band_matrix(THREE, -kx, -ky), H.conj(), atol=1e-16)
        assert np.max(np.abs(oracle.band_energies(THREE, kx, ky) - oracle.band_energies(THREE, -kx, -ky))) < 1e-14
        assert np.max(np.abs(oracle.band_energies(THREE, kx, ky) - np.linalg.eigvalsh(hk(THREE["tb3"], kx, ky)))) < 1e-14
    # x <-> y exchanges the d_xz and d_yz orbitals: same spectrum
    for kx, ky in rng.uniform(-4, 4, size=(50, 2)):
        assert np.max(np.abs(oracle.band_energies(THREE, kx, ky) - oracle.band_energies(THREE, ky, kx))) < 1e-14


def test_filling_is_four_at_mu_0p4748(oracle):
    """n = 4 at mu = 0.4748 -- pins B.1-B.6 and the hopping order; common slips move n visibly."""
    g = json.load(open(GOLD))["three_band_filling"]
    N = 96
    ks = 2 * PI * np.arange(N) / N

    def filling(p):
        c = 0
        for kx in ks:
            for ky in ks:
                c += 2 * int(np.sum(oracle.band_energies(p, kx, ky) < g["mu"]))
        return c / N**2

    n = filling(THREE)
    assert abs(n - g["electrons_per_site"]) < 5e-3, n
    # thermodynamic identity through the whole pipeline: n = -dOmega/dmu at Delta = 0
    T, dmu, N2 = 0.002, 2e-3, 128
    om = [oracle.omega_column(dict(THREE, mu=g["mu"] + s * dmu), N2, T, (0.0, 0.0), 0.0, [0.0])[0] for s in (+1, -1)]
    n_fd = -(om[0] - om[1]) / (2 * dmu) / N2**2
    assert abs(n_fd - g["electrons_per_site"]) < 2e-2, n_fd
    # slips: t1 <-> t2 swapped, eps0 dropped, t7 coupling dropped
    tb = list(W.THREE_BAND_T)
    swapped = tb[:]; swapped[0], swapped[1] = tb[1], tb[0]
    no_e0 = tb[:]; no_e0[12] = 0.0
    for bad in (swapped, no_e0):
        assert abs(filling(W.model_params(model=3, mu=g["mu"], tb3=tuple(bad))) - 4.0) > 0.05


def test_normal_state_three_band(oracle):
    """Delta = 0: Omega = sum f(xi_up(k)) + f(xi_dn(-k+q)) with LAPACK bands of the independently built T_k."""
    N, T, h = 16, 0.02, 0.03
    for q in [(0.0, 0.0), (2 * PI * 3 / 16, 2 * PI / 16), (0.21, -0.4)]:
        acc = []
        for j in range(N):
            for i in range(N):
                kx, ky = 2 * PI * i / N, 2 * PI * j / N
                up = np.linalg.eigvalsh(hk(THREE["tb3"], kx, ky)) - THREE["mu"] - h
                dn = np.linalg.eigvalsh(hk(THREE["tb3"], -kx + q[0], -ky + q[1])) - THREE["mu"] + h
                acc += list(softplus_f(up, T)) + list(softplus_f(dn, T))
        ref = math.fsum(acc)
        got = oracle.omega_column(THREE, N, T, q, h, [0.0])[0]
        assert rel(got, ref) < 1e-13


def test_three_band_orbital_bdg_6x6(oracle):
    """q = 0: intra-band pairing with a common Delta eta(k) is intra-orbital (U U^+ = 1, T_{-k} = conj T_k), so the
    per-k BdG matrix in the ORBITAL basis is [[T_k-(mu+h), g],[g, -(T_k-(mu-h))]]; its spectrum must be the
    oracle's {E+-} of Eq. 4 over the three numerically diagonalised bands, and Omega follows from it."""
    L, T, h, D, U = 4, 0.05, 0.04, 0.11, 0.7
    p = W.model_params(model=3, mu=W.THREE_BAND_MU, U=U)
    mu = p["mu"]
    total = []
    for j in range(L):
        for i in range(L):
            for off in ((0.013, -0.007), (0.0, 0.0)):
                kx, ky = 2 * PI * i / L + off[0], 2 * PI * j / L + off[1]
                Tk = hk(p["tb3"], kx, ky)
                g = D * math.cos(kx) * math.cos(ky)
                M = np.block([[Tk - (mu + h) * np.eye(3), g * np.eye(3)], [g * np.eye(3), -(Tk - (mu - h) * np.eye(3))]])
                ev = np.linalg.eigvalsh(M)
                E = oracle.band_energies(p, kx, ky)
                spec = []
                for e in range(3):
                    spec.extend(oracle.quasiparticle(E[e] - mu - h, E[e] - mu + h, D * oracle.eta(p, kx, ky)))
                assert np.max(np.abs(np.sort(spec) - ev)) < 1e-13
                if off == (0.0, 0.0):
                    total += list(softplus_f(ev, T)) + [float(np.trace(Tk).real) - 3 * (mu - h)]
    ref = math.fsum(total) + 3 * L * L * D * D / U
    got = oracle.omega_column(p, L, T, (0, 0), h, [D])[0]
    assert rel(got, ref) < 1e-13


def test_three_band_band_basis_bdg_offgrid_q(oracle):
    rng = np.random.default_rng(8)
    mu, h, D = THREE["mu"], 0.02, 0.07
    for kx, ky, qx, qy in rng.uniform(-3, 3, size=(40, 4)):
        Ek = oracle.band_energies(THREE, kx, ky)
        Ekq = oracle.band_energies(THREE, -kx + qx, -ky + qy)
        g = D * oracle.eta(THREE, kx, ky)
        M = np.block([[np.diag(Ek - mu - h), g * np.eye(3)], [g * np.eye(3), -np.diag(Ekq - mu + h)]])
        spec = []
        for e in range(3):
            spec.extend(oracle.quasiparticle(Ek[e] - mu - h, Ekq[e] - mu + h, g))
        assert np.max(np.abs(np.sort(spec) - np.linalg.eigvalsh(M))) < 1e-13


def test_three_band_symmetries_and_band_mask(oracle):
    N, T = 12, 0.01
    d = np.array([0.0, 0.03, -0.03])
    a = oracle.omega_column(THREE, N, T, (0.3, 0.1), 0.02, d)
    assert a[1] == a[2]                                                # Omega(Delta) = Omega(-Delta)
    b = oracle.omega_column(THREE, N, T, (0.1, 0.3), 0.02, d)
    assert rel(a[1], b[1]) < 1e-13                                     # x <-> y
    c = oracle.omega_column(THREE, N, T, (-0.3, -0.1), 0.02, d)
    assert rel(a[1], c[1]) < 1e-13                                     # q -> -q
    parts = [oracle.omega_column(dict(THREE, band_mask=1 << e, cond_mult=1.0), N, T, (0.3, 0.1), 0.02, d) for e in range(3)]
    assert np.max(np.abs(sum(parts) - a) / np.abs(a)) < 1e-13          # Omega = sum_eps Omega_eps


def test_three_band_matrix_lattice_symmetries(oracle):
    """A pin of feo_three_band_matrix that does not retype B.1-B.6: what the square lattice and the orbitals fix.
    The xz / yz orbitals swap under k_x <-> k_y and xy maps to itself, so T(k_y, k_x) = P T(k_x, k_y) P^T with P the swap
    of orbitals 1 and 2; under k_x -> -k_x the xz orbital changes sign, T(-k_x, k_y) = D T(k_x, k_y)* D ... in every case
    the SPECTRUM is unchanged.  A slip in one matrix element (t1 and t2 exchanged in one diagonal entry, a sign in the
    t11 term, sin for cos in an off-diagonal entry, a wrong k component) breaks at least one of: Hermiticity,
    2 pi periodicity, the three mirror invariances of the eigenvalues, the orbital-swap identity of the matrix itself,
    inversion T(-k) = T(k)* (time reversal for spinless hoppings)."""
    rng = np.random.default_rng(5)
    P = np.array([[0, 1, 0], [1, 0, 0], [0, 0, 1]], dtype=float)
    for _ in range(200):
        kx, ky = rng.uniform(-PI, PI, size=2)
        M = oracle.three_band_matrix(THREE, kx, ky)
        assert np.abs(M - M.conj().T).max() < 1e-15
        assert np.abs(M - oracle.three_band_matrix(THREE, kx + 2 * PI, ky - 2 * PI)).max() < 1e-13
        ev = np.linalg.eigvalsh(M)
        for k2 in ((ky, kx), (-kx, ky), (kx, -ky), (-kx, -ky)):
            assert np.abs(np.linalg.eigvalsh(oracle.three_band_matrix(THREE, *k2)) - ev).max() < 1e-13
        # the matrix identities behind two of them
        assert np.abs(oracle.three_band_matrix(THREE, ky, kx) - P @ M @ P.T).max() < 1e-14
        assert np.abs(oracle.three_band_matrix(THREE, -kx, -ky) - M.conj()).max() < 1e-14
    # and the band energies the oracle's Omega uses are those eigenvalues, ascending
    kx, ky = 0.3, -1.1
    assert np.abs(oracle.band_energies(THREE, kx, ky) - np.linalg.eigvalsh(oracle.three_band_matrix(THREE, kx, ky))).max() < 1e-13
