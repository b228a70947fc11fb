"""GPU parity of the flow statistics (mc_tvd_flow_stats / mc_tvd_stats_flow / mc_tvd_stats_read_flow; Eqs. 40-43,
PAPER.md:457-467, the distribution of r = K_e / I_e, and the correlation C of Eq. 49)
against the oracle on the same states."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs

pytestmark = pytest.mark.gpu

FORCE_KEYS = ("Fn_mean", "Fp_mean", "Fb_mean", "Fv_mean", "Fn_rms", "Fp_rms", "Fb_rms", "Fv_rms", "FbFp_mean")


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


def _compare(d, do, h, ho, rms_tol=1e-10):
    # a mean is a sum of signed terms: its error is measured against the rms of the same term
    for t in ("Fn", "Fp", "Fb", "Fv"):
        scale = max(do[t + "_rms"], 1e-300)
        assert abs(d[t + "_mean"] - do[t + "_mean"]) <= rms_tol * scale, t
        assert abs(d[t + "_rms"] - do[t + "_rms"]) <= rms_tol * scale, t
    assert abs(d["FbFp_mean"] - do["FbFp_mean"]) <= rms_tol * do["Fb_rms"]
    assert d["max_r"] == pytest.approx(do["max_r"], rel=1e-12)
    assert d["max_mach"] == pytest.approx(do["max_mach"], rel=1e-12)
    assert d["volume"] == pytest.approx(do["volume"], rel=1e-13)
    # Eq. 49: two sums of squares and one of signed products, measured against their Cauchy-Schwarz bound
    bound = np.sqrt(do["rhouz_sq_mean"] * do["Tsa_sq_mean"])
    assert d["rhouz_sq_mean"] == pytest.approx(do["rhouz_sq_mean"], rel=1e-12)
    assert d["Tsa_sq_mean"] == pytest.approx(do["Tsa_sq_mean"], rel=1e-12)
    assert abs(d["flux_mean"] - do["flux_mean"]) <= 1e-12 * bound
    assert abs(d["corr_C"] - do["corr_C"]) <= 1e-11 and abs(d["corr_C"]) <= 1.0
    # the bin is read off the bit pattern of r; the two sides may round r differently in the last place, which moves
    # a node across a bin edge only if r sits within an ulp of it
    assert h.sum() == ho.sum()
    assert np.abs(h - ho).sum() <= 2


@pytest.mark.parametrize("ndim,nx,ny,nz,stretch,bc_z", [
    (2, 300, 1, 70, None, 0), (2, 301, 1, 40, 1.5, 0), (2, 64, 1, 32, None, 1),
    (3, 60, 21, 19, None, 0), (3, 45, 17, 14, 2.0, 0), (3, 24, 10, 12, None, 1)])
def test_flow_stats_parity(gpu, orc, ndim, nx, ny, nz, stretch, bc_z):
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=stretch)
    params = inputs.make_params(Ra=1e4, bc_z=bc_z)
    X0 = inputs.rough_random_state(grid, params, seed=17 + nx)
    do, ho = orc.flow_stats(orc.Problem(grid, params), X0)
    s = gpu.MCTVD(grid, params, X0)
    d, h = s.flow_stats()
    d2, h2 = s.flow_stats()                                   # a second call starts from a cleared histogram
    nu_conv = s.diagnostics()[0]["nu_conv"]
    s.close()
    if bc_z == 0:     # the average inside Nu_conv of Eq. 22 (another kernel) is the numerator of Eq. 49
        assert np.sqrt(params["Ra"] * params["Pr"]) / params["eps"] * d["flux_mean"] == pytest.approx(nu_conv, rel=1e-10)
    assert do["Fn_rms"] > 0 and do["Fv_rms"] > 0 and (ho[1:] > 0).sum() >= 5
    _compare(d, do, h, ho)
    assert d2 == d and np.array_equal(h2, h)


def test_flow_stats_time_averages(gpu, orc):
    """mc_tvd_stats_flow + mc_tvd_step_stats: the device accumulators against the written-out weighted means of the
    oracle's samples (weights: time since the previous sample), histogram summed over the samples."""
    grid = inputs.make_grid(2, 96, 33, z_stretch=1.5)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.moving_state(grid, params, u_amp=0.1)
    prob = orc.Problem(grid, params)
    n_steps, every = 12, 3
    s = gpu.MCTVD(grid, params, X0)
    s.stats_reset()
    s.stats_flow(True)
    s.step_stats(n_steps, every)
    avg, hist = s.stats_read_flow()
    st = s.stats_read()[0]
    s.close()
    X, t, t_last, wsum = X0, 0.0, 0.0, 0.0
    acc = {k: 0.0 for k in FORCE_KEYS + ("max_mach", "max_r", "flux_mean", "rhouz_sq_mean", "Tsa_sq_mean")}
    hsum = np.zeros(orc.HIST_BINS, dtype=np.int64)
    for n in range(n_steps):
        X, dts, _ = orc.step(prob, X, 1)
        t += dts[0]
        if (n + 1) % every:
            continue
        f, h = orc.flow_stats(prob, X)
        w = t - t_last
        for k in acc:
            acc[k] += w * (f[k] ** 2 if k.endswith("_rms") else f[k])
        hsum += h
        wsum += w
        t_last = t
    want = {k: (np.sqrt(v / wsum) if k.endswith("_rms") else v / wsum) for k, v in acc.items()}
    assert avg["volume"] == pytest.approx(wsum, rel=1e-12) and st["weight"] == pytest.approx(wsum, rel=1e-12)
    for k in FORCE_KEYS:
        scale = want[k[:2] + "_rms"] if k != "FbFp_mean" else want["Fb_rms"]
        assert abs(avg[k] - want[k]) <= 1e-9 * scale, k
    assert avg["max_mach"] == pytest.approx(want["max_mach"], rel=1e-9)
    # Eq. 49 over volume AND time: C from the time-averaged three
    bound = np.sqrt(want["rhouz_sq_mean"] * want["Tsa_sq_mean"])
    assert avg["rhouz_sq_mean"] == pytest.approx(want["rhouz_sq_mean"], rel=1e-9)
    assert avg["Tsa_sq_mean"] == pytest.approx(want["Tsa_sq_mean"], rel=1e-9)
    assert abs(avg["flux_mean"] - want["flux_mean"]) <= 1e-9 * bound
    assert abs(avg["corr_C"] - want["flux_mean"] / bound) <= 1e-9 and avg["corr_C"] != 0.0
    assert hist.sum() == hsum.sum() and np.abs(hist - hsum).sum() <= 4


def test_flow_read_without_samples_is_an_error(gpu):
    grid, params, _ = inputs.config("C1")
    s = gpu.MCTVD(grid, params, inputs.conduction_state(grid, params))
    with pytest.raises(gpu.MCTVDError):
        s.stats_read_flow()
    s.step_stats(2, 1)                                         # flow accumulation is off by default
    with pytest.raises(gpu.MCTVDError):
        s.stats_read_flow()
    s.close()
