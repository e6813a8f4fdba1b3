"""Pins for the oracle's single-precision variant ("DP / SP / SPFM").

The SP function is pinned by the separately pinned double-precision oracle: same inputs, every per-term operation
in binary32, so the two must agree to a few float ulps per term -- and, as the paper reports ("we obtained the same
results with all three approaches"), give the same minima wherever they are resolved.  CPU only.
"""
import numpy as np
import pytest

from paper_1412_8754_b200 import workloads as W

EPS32 = float(np.finfo(np.float32).eps)


@pytest.mark.parametrize("w,T", [(W.config(1), 0.01), (W.config(2), 0.001),
                                 (W.interior_minimum(N=48, U=5.0, T=0.001, nq=3, nh=6, nd=48), 0.001),
                                 (W.ragged(seed=7, N=21, nq=2, nh=4, nd=15), 0.004),
                                 (W.ragged(seed=9, N=24, nq=2, nh=3, nd=9, model=W.MODEL_ONE_BAND), 0.02)],
                         ids=["cfg1", "cfg2", "X", "ragged2", "ragged1"])
def test_sp_oracle_tracks_dp_oracle(oracle, w, T):
    dp = oracle.omega_grid(w.params, w.N, T, w.q, w.h, w.delta)
    sp = oracle.omega_grid_sp(w.params, w.N, T, w.q, w.h, w.delta)
    # per term: a handful of float operations on values up to the band width (~8): <= ~8 ulp_32 each, mostly cancelling
    # in the sum; systematic part bounded by 4 eps32 relative
    err = np.max(np.abs(sp - dp) / np.abs(dp))
    assert err < 4 * EPS32, err
    assert err > 1e-12                                   # it really is a different precision
    srt = np.sort(dp, axis=-1)
    resolved = (srt[..., 1] - srt[..., 0]) > 16 * EPS32 * np.abs(srt[..., 0])
    assert np.array_equal(np.argmin(dp, -1)[resolved], np.argmin(sp, -1)[resolved])
    # where the minimum is flatter than float resolution the SP index is still a DP near-minimum
    pick = np.take_along_axis(dp, np.argmin(sp, -1)[..., None], -1)[..., 0]
    assert np.all(pick - srt[..., 0] <= 8 * EPS32 * np.abs(srt[..., 0]))


def test_sp_oracle_rejects_three_band_and_bad_input(oracle):
    with pytest.raises(ValueError):
        oracle.omega_grid_sp(W.model_params(model=W.MODEL_THREE_BAND, mu=0.4748), 8, 0.01, [(0, 0)], [0.0], [0.1])
    with pytest.raises(ValueError):
        oracle.omega_grid_sp(W.model_params(), 8, 0.0, [(0, 0)], [0.0], [0.1])
