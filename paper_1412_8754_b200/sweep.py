"""Outer loops of the paper's Algorithm 1 around the library calls: orchestration only, no arithmetic of the method.

PAPER.md:125: "for each ... (h, T) ... minimizing the free energy over the set of Delta and q", per band
("(q_eps, Delta_eps)") -- the physics loop the paper's driver runs on top of the Omega evaluator.  Here every Omega and
every minimum comes from the CUDA kernels through fe.FreeEnergy (fe_set_temperature, fe_omega_grid, fe_argmin_q); these
helpers only loop over temperatures / bands and stack the small per-h results on the host.
"""
from __future__ import annotations

import numpy as np

from . import fe


def phase_diagram(params: dict, N: int, q, h, delta, T_list, ref_id: int = 0, mode=None):
    """h-T sweep: for every T of T_list and every field h the ground state over (q, Delta).

    One handle; per T: fe_set_temperature -> fe_omega_grid -> fe_argmin_q(ref_id) (ref_id = index of Delta = 0: compares
    condensation energies across q, reading G17; -1 = Omega itself, Algorithm 1 as printed).
    Returns dict(iq, id: int32 (nT, nh); value: float64 (nT, nh); q_star: (nT, nh, 2); delta_star: (nT, nh))."""
    import torch
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    h = np.ascontiguousarray(h, dtype=np.float64).reshape(-1)
    delta = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    T_list = [float(t) for t in T_list]
    iq = np.empty((len(T_list), len(h)), dtype=np.int32)
    idd = np.empty_like(iq)
    val = np.empty((len(T_list), len(h)), dtype=np.float64)
    with fe.FreeEnergy(params, N, T_list[0]) as F:
        if mode is not None:
            F.set_eval_mode(mode)
        omega = torch.empty((q.shape[0], h.shape[0], delta.shape[0]), dtype=torch.float64, device="cuda")
        for it, T in enumerate(T_list):
            F.set_temperature(T)
            F.omega_grid(q, h, delta, out=omega)
            a, b, c = F.argmin_q(omega, ref_id=ref_id)
            torch.cuda.synchronize()
            iq[it], idd[it], val[it] = a.cpu().numpy(), b.cpu().numpy(), c.cpu().numpy()
    return dict(iq=iq, id=idd, value=val, q_star=q[iq], delta_star=delta[idd])


def per_band_minima(params: dict, N: int, T: float, q, h, delta, ref_id: int = 0, mode=None):
    """The paper's per-band minimisation (Omega = sum_eps Omega_eps): one handle per band eps
    (band_mask = 1 << eps, condensation term counted once: cond_mult = 1), each minimised over (q, Delta) per field h.
    Returns a list over bands of dict(iq, id, value) arrays of length nh."""
    nb = {1: 1, 2: 2, 3: 3}[int(params["model"])]
    out = []
    for e in range(nb):
        pe = dict(params, band_mask=1 << e, cond_mult=1.0)
        r = phase_diagram(pe, N, q, h, delta, [T], ref_id=ref_id, mode=mode)
        out.append(dict(iq=r["iq"][0], id=r["id"][0], value=r["value"][0]))
    return out
