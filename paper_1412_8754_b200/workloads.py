"""Seeded, synthetic input generators shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no dispersion, no Eq. 4/5): it only
produces parameter structs-as-dicts and the q / h / Delta lists of the workloads named in
BASELINE.json (`configs`), plus seeded sub-samples of those grids.  Both the oracle
(`oracle/`) and the CUDA path (`paper_1412_8754_b200.fe`) are fed from here so that they
see bit-identical inputs.

The paper's workloads are themselves synthetic parameter scans ("a single
value of q_i and 200 values of Delta_i ... square lattice N x N"), so nothing stands in
for a dataset.  Model constants are the paper's (Appendix A).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# PAPER.md:225 (Appendix A): t1 = -1.0, t2 = 1.3, t3 = t4 = -0.85, mu = 1.54 |t1|.
TWO_BAND_T = (-1.0, 1.3, -0.85, -0.85)
TWO_BAND_MU = 1.54

# PAPER.md:273 (Appendix B): three-band model of Daghofer et al., hoppings in eV, t1..t12 then eps0; n = 4 at mu = 0.4748.
THREE_BAND_T = (-0.08, 0.1825, 0.08375, -0.03, 0.15, 0.15, -0.12, 0.06, 0.0, -0.024, -0.01, 0.0275, 0.75)
THREE_BAND_MU = 0.4748

MODEL_ONE_BAND = 1
MODEL_TWO_BAND = 2
MODEL_THREE_BAND = 3
NBANDS = {MODEL_ONE_BAND: 1, MODEL_TWO_BAND: 2, MODEL_THREE_BAND: 3}
FORM_S = 0        # eta = 1                  (homogeneous BCS)
FORM_SPM = 1      # eta = cos kx cos ky      (s+-)


def model_params(model=MODEL_TWO_BAND, form_factor=FORM_SPM, t=TWO_BAND_T, mu=TWO_BAND_MU,
                 U=2.0, eta_scale=1.0, cond_mult=None, band_mask=None, const_mode=0, tb3=None):
    """Plain dict mirrored field-by-field by both C structs (fe_model_params / feo_params)."""
    nb = NBANDS[model]
    if model == MODEL_THREE_BAND:
        t, tb3 = (), (THREE_BAND_T if tb3 is None else tb3)
    tb3 = tuple(float(x) for x in (tb3 or ())) + (0.0,) * (13 - len(tb3 or ()))
    t4 = tuple(float(x) for x in t) + (0.0,) * (4 - len(t))
    return dict(model=int(model), form_factor=int(form_factor), t=t4, mu=float(mu), U=float(U),
                eta_scale=float(eta_scale),
                cond_mult=float(nb if cond_mult is None else cond_mult),
                band_mask=int((1 << nb) - 1 if band_mask is None else band_mask),
                const_mode=int(const_mode), tb3=tb3)


@dataclass
class Workload:
    """One parameter scan: Omega over (q, h, Delta) on an N x N k-grid at temperature(s) T."""
    name: str
    params: dict
    N: int
    T: tuple                      # one or more temperatures (config 4 has two)
    q: np.ndarray                 # (nq, 2) float64, (qx, qy)
    h: np.ndarray                 # (nh,)   float64
    delta: np.ndarray             # (nd,)   float64
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def nq(self):
        return int(self.q.shape[0])

    @property
    def nh(self):
        return int(self.h.shape[0])

    @property
    def nd(self):
        return int(self.delta.shape[0])

    @property
    def nbands(self):
        return NBANDS[self.params["model"]]

    def k_param_evals(self):
        """k-point x parameter evaluations per temperature (the unit of BASELINE.json's metric)."""
        return self.N * self.N * self.nq * self.nh * self.nd

    def band_evals(self):
        return self.k_param_evals() * self.nbands


def _q_axis(v):          # q = (v, 0)
    v = np.asarray(v, dtype=np.float64)
    return np.stack([v, np.zeros_like(v)], axis=1)


def _q_diag(v):          # q = (v, v)
    v = np.asarray(v, dtype=np.float64)
    return np.stack([v, v], axis=1)


def splitmix64(state):
    """One step of splitmix64; returns (new_state, output).  Used only to draw inputs."""
    mask = (1 << 64) - 1
    state = (state + 0x9E3779B97F4A7C15) & mask
    z = state
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
    z = z ^ (z >> 31)
    return state, z


def perturbed_hoppings(seed, t=TWO_BAND_T, amplitude=0.01):
    """Config 5: t_i <- t_i (1 + amplitude u_i), u_i in [-1, 1) from splitmix64(seed), i = 1..4 in order."""
    state = int(seed) & ((1 << 64) - 1)
    out = []
    for ti in t:
        state, z = splitmix64(state)
        u = ((z >> 11) * 2.0 ** -53) * 2.0 - 1.0
        out.append(ti * (1.0 + amplitude * u))
    return tuple(out)


def config(i, seed=1):
    """BASELINE.json `configs[i-1]`, i = 1..5 (all linspace grids inclusive of both ends)."""
    pi = math.pi
    if i == 1:
        p = model_params(model=MODEL_ONE_BAND, form_factor=FORM_S, t=(1.0,), mu=0.0, U=2.0)
        return Workload("cfg1_bcs_N32", p, 32, (0.01,), _q_axis([0.0]), np.array([0.0]),
                        np.linspace(0.0, 0.5, 64), "BCS one band, q=0, h=0")
    if i == 2:
        return Workload("cfg2_twoband_N128", model_params(), 128, (0.001,), _q_axis([0.0]),
                        np.linspace(0.0, 0.3, 16), np.linspace(0.0, 0.4, 256), "two-band s+-, q=0, h scan")
    if i == 3:
        return Workload("cfg3_fflo_N512", model_params(), 512, (0.001,),
                        _q_axis(np.linspace(0.0, 0.2 * pi, 64)),
                        np.linspace(0.0, 0.3, 32), np.linspace(0.0, 0.4, 256), "FFLO scan q=(qx,0)")
    if i == 4:
        return Workload("cfg4_fflo_N1024", model_params(), 1024, (0.001, 0.01),
                        _q_diag(np.linspace(0.0, 0.2 * pi, 32)),
                        np.linspace(0.0, 0.3, 64), np.linspace(0.0, 0.4, 512),
                        "paper's largest size, q along (1,1); headline roofline config")
    if i == 5:
        p = model_params(t=perturbed_hoppings(seed))
        return Workload(f"cfg5_finite_size_N4096_seed{seed}", p, 4096, (0.0005,),
                        _q_axis(np.linspace(0.0, 0.05 * pi, 16)),
                        np.linspace(0.1, 0.25, 16), np.linspace(0.0, 0.4, 1024),
                        "finite-size elimination, hoppings +-1%", extra=dict(seed=seed))
    if i == 6:     # not in BASELINE.json: SURVEY.md 8(f-1), the shape of config 4 on the three-band model
        b = three_band(N=1024, U=1.5, T=0.001, nq=32, nh=64, nd=512, qdir="diag")
        b.name = "B3_fflo_N1024"
        return b
    if i == 7:     # not in BASELINE.json: config 4's shape on an interior-minimum grid (U = 5: Delta* > 0 on most columns),
        w = interior_minimum(N=1024, U=5.0, T=0.001, nq=32, nh=64, nd=512)      # to show how data-dependent the early-out is
        w.T, w.name, w.q = (0.001, 0.01), "X_U5_fflo_N1024", _q_diag(np.linspace(0.0, 0.2 * pi, 32))
        return w
    if i == 8:     # not in BASELINE.json: config 4 at a high temperature (wide dominance window: more slots stay dense)
        w = config(4)
        w.T, w.name = (0.02,), "cfg4_fflo_N1024_T0.02"
        return w
    raise ValueError(f"no such config: {i}")


def paper_shaped(N=2000):
    """Context run shaped like the paper's benchmark: 1 q, 200 Delta, N x N."""
    return Workload(f"paperP_N{N}", model_params(), N, (0.001,), _q_axis([0.1 * math.pi]),
                    np.array([0.1]), np.linspace(0.0, 0.4, 200), "paper-shaped (Fig. 4) context run")


def interior_minimum(N=128, U=5.0, T=0.001, nq=8, nh=16, nd=256):
    """Extra grids 'X': larger U gives interior minima and first-order jumps in h."""
    return Workload(f"X_U{U:g}_N{N}_T{T:g}", model_params(U=U), N, (T,),
                    _q_axis(np.linspace(0.0, 0.2 * math.pi, nq)),
                    np.linspace(0.0, 0.3, nh), np.linspace(0.0, 0.4, nd), "interior-minimum grid")


def three_band(N=256, U=1.5, T=0.001, nq=8, nh=16, nd=128, qdir="axis"):
    """the three-band model of Appendix B (hoppings in eV, mu = 0.4748) with s+-
    pairing.  U = 1.5 eV gives Delta* ~ 0.044 eV at h = 0 and first-order jumps to Delta* = 0 for h in [0.02, 0.04]."""
    v = np.linspace(0.0, 0.2 * math.pi, nq)
    return Workload(f"B3_U{U:g}_N{N}_T{T:g}", model_params(model=MODEL_THREE_BAND, mu=THREE_BAND_MU, U=U), N, (T,),
                    _q_axis(v) if qdir == "axis" else _q_diag(v),
                    np.linspace(0.0, 0.06, nh), np.linspace(0.0, 0.15, nd), "three-band FFLO scan")


def ragged3(seed=11, N=37, nq=3, nh=5, nd=19):
    """Awkward sizes for the three-band model: odd N, off-grid q of both signs, negative h / Delta."""
    rng = np.random.default_rng(seed)
    return Workload(f"ragged3_s{seed}_N{N}", model_params(model=MODEL_THREE_BAND, mu=THREE_BAND_MU, U=1.3), N, (0.002,),
                    rng.uniform(-0.6, 0.6, size=(nq, 2)), np.sort(rng.uniform(-0.02, 0.06, size=nh)),
                    np.sort(rng.uniform(-0.02, 0.16, size=nd)), "ragged sizes, three bands")


def chi_map(model=MODEL_TWO_BAND, N=256, nside=16, T=0.001, h=0.025, on_grid=True):
    """q map of the static Cooper-pair susceptibility (Appendix C; Fig. C.6 is at h = 0.025 eV,
    k_B T ~ 0, eta = 4 cos kx cos ky): nside x nside q-points over the quadrant [0, pi]^2, snapped to the k-grid
    when on_grid.  Returned as a Workload whose h list holds the single field and whose Delta list is unused."""
    v = np.linspace(0.0, math.pi, nside)
    if on_grid:
        v = 2.0 * math.pi * np.round(v * N / (2.0 * math.pi)) / N
    q = np.stack(np.meshgrid(v, v, indexing="ij"), axis=-1).reshape(-1, 2)
    if model == MODEL_THREE_BAND:
        p = model_params(model=MODEL_THREE_BAND, mu=THREE_BAND_MU, U=1.5, eta_scale=4.0)
    elif model == MODEL_TWO_BAND:
        p = model_params(eta_scale=4.0)
    else:
        p = model_params(model=MODEL_ONE_BAND, form_factor=FORM_S, t=(1.0,), mu=-0.3, U=2.0)
    return Workload(f"chi_m{model}_N{N}_q{nside}x{nside}", p, N, (T,), q, np.array([h]), np.array([0.0]),
                    "pair-susceptibility q map")


def ragged(seed=7, N=45, nq=3, nh=5, nd=37, model=MODEL_TWO_BAND):
    """Deliberately awkward sizes: odd N, list lengths that divide no tile, off-grid q, negative h/Delta."""
    rng = np.random.default_rng(seed)
    q = rng.uniform(-0.7, 0.7, size=(nq, 2))
    h = np.sort(rng.uniform(-0.1, 0.3, size=nh))
    d = np.sort(rng.uniform(-0.05, 0.45, size=nd))
    if model == MODEL_ONE_BAND:
        p = model_params(model=MODEL_ONE_BAND, form_factor=FORM_S, t=(1.0,), mu=-0.3, U=3.0)
    else:
        p = model_params(U=4.5)
    return Workload(f"ragged_s{seed}_N{N}", p, N, (0.004,), q, h, d, "ragged sizes")


def sample_columns(w: Workload, n, cfg_id=0):
    """Seeded distinct (iq, ih) pairs, always containing (0,0) and (nq-1, nh-1)."""
    total = w.nq * w.nh
    n = min(n, total)
    chosen = [(0, 0)]
    if (w.nq - 1, w.nh - 1) not in chosen and n > 1:
        chosen.append((w.nq - 1, w.nh - 1))
    state = 20141231 + cfg_id
    while len(chosen) < n:
        state, z = splitmix64(state)
        c = int(z % total)
        pair = (c // w.nh, c % w.nh)
        if pair not in chosen:
            chosen.append(pair)
    return chosen[:n]


def sample_points(w: Workload, n, cfg_id=0):
    """Seeded distinct (iq, ih, id) triples incl. the grid corners."""
    total = w.nq * w.nh * w.nd
    n = min(n, total)
    chosen = [(0, 0, 0)]
    last = (w.nq - 1, w.nh - 1, w.nd - 1)
    if last not in chosen and n > 1:
        chosen.append(last)
    state = 977 * 20141231 + cfg_id
    while len(chosen) < n:
        state, z = splitmix64(state)
        c = int(z % total)
        tr = (c // (w.nh * w.nd), (c // w.nd) % w.nh, c % w.nd)
        if tr not in chosen:
            chosen.append(tr)
    return chosen[:n]
