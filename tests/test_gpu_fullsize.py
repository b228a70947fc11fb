"""Parity at BASELINE.json's full sizes (configs C2-C5), in the launch configuration bench.py times.

The oracle cannot march 67M-268M nodes in test time, but every operation of the step is local
(stencil radius 2 per operator in the sweep direction and across it):
after s steps the state inside a column window equals the oracle run on that window plus a margin of
2 * (operators per step) * s columns on each periodic side (full z), given the same dt sequence.  So
the GPU runs the whole grid, and the oracle recomputes sampled windows of it -- including windows across
the periodic seam and across tile boundaries -- element by element.  dt itself (a global max) is checked
against the oracle's max over the whole downloaded state.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import parity_err

pytestmark = pytest.mark.gpu

TOL_1STEP = 1e-12


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


def _device_window(s, grid, ix, iy):
    """Columns ix (and rows iy) of every field of the solver's device state, as numpy (nf, nz*wy*wx)."""
    import torch
    nf, nz, ny, nx = s.nf, grid["nz"], grid["ny"], grid["nx"]
    s.stream.synchronize()
    v = s.fields.view(nf, nz, ny, nx)
    ixt = torch.as_tensor(ix, device=v.device)
    iyt = torch.as_tensor(iy, device=v.device)
    w = v.index_select(3, ixt).index_select(2, iyt)
    return w.cpu().numpy().reshape(nf, -1)


def _check_windows(gpu, orc, name, n_steps, windows):
    import psutil
    grid, params, _ = inputs.config(name)
    nf, N = inputs.num_fields(grid), inputs.num_nodes(grid)
    need = 3 * nf * N * 8
    if psutil.virtual_memory().available < need + (8 << 30):
        pytest.skip(f"host memory too small for {name}")
    X0 = inputs.conduction_state(grid, params)
    s = gpu.MCTVD(grid, params, X0)
    ops = 4 if grid["ndim"] == 2 else 6
    margin = 2 * ops * n_steps
    dts = []
    for _ in range(n_steps):
        dts.append(s.dt())
        s.step(1)
    # dt of the initial state: the oracle's global max-reduction on the same array
    prob = orc.Problem(grid, params)
    dt_ref = orc.dt(prob, X0)
    assert abs(dts[0] - dt_ref) <= 4e-16 * dt_ref
    worst = 0.0
    for (i0, wx, j0, wy) in windows:
        i0 %= grid["nx"]
        if grid["ndim"] == 2:
            Xw, gw = inputs.window_x(X0.reshape(nf, -1), grid, i0 - margin, wx + 2 * margin)
            iy = np.array([0])
        else:
            j0 %= grid["ny"]
            Xw, gw = inputs.window_xy(X0.reshape(nf, -1), grid, i0 - margin, wx + 2 * margin, j0 - margin,
                                      wy + 2 * margin)
            iy = (np.arange(wy) + j0) % grid["ny"]
        ref, _, _ = orc.step(orc.Problem(gw, params), Xw, n_steps, dt_in=dts)
        ix = (np.arange(wx) + i0) % grid["nx"]
        gw_out = dict(gw, nx=wx, ny=len(iy))
        got = _device_window(s, grid, ix, iy)
        r = ref.reshape(nf, gw["nz"], gw["ny"], gw["nx"])
        if grid["ndim"] == 2:
            r = r[:, :, :, margin:margin + wx]
        else:
            r = r[:, :, margin:margin + wy, margin:margin + wx]
        err = parity_err(gw_out, params, got, r.reshape(nf, -1)).max()
        worst = max(worst, err)
        assert err <= TOL_1STEP * n_steps, (name, (i0, wx, j0, wy), err)
    # dt after the last step: global max over the whole downloaded state
    dt_gpu = s.dt()
    if psutil.virtual_memory().available > 2 * nf * N * 8 + (8 << 30):
        Xn = s.state()
        dt_ref = orc.dt(prob, Xn)
        assert abs(dt_gpu - dt_ref) <= 4e-16 * dt_ref
        d, Tp, rp, pp = s.diagnostics()
        if N <= 80_000_000:                                   # oracle diagnostics: one serial pass
            do, To, ro, po = orc.diagnostics(prob, Xn)
            assert abs(d["nu_bar"] - do["nu_bar"]) <= 1e-10 * abs(do["nu_bar"])
            assert abs(d["mass"] - do["mass"]) <= 1e-12 * abs(do["mass"])
            np.testing.assert_allclose(Tp, To, rtol=1e-13)
        del Xn
    s.close()
    return worst


def test_c2_windows(gpu, orc):
    # tile boundaries of the 2-D kernels: 124-column march tiles, 28-column lane warps
    _check_windows(gpu, orc, "C2", 2, [(-6, 12, 0, 1), (124 * 7 - 6, 12, 0, 1), (28 * 50 - 6, 12, 0, 1), (3001, 16, 0, 1)])


def test_c3_windows(gpu, orc):
    _check_windows(gpu, orc, "C3", 1, [(-8, 16, 0, 1), (124 * 66 - 8, 16, 0, 1), (9999, 16, 0, 1)])


def test_c4_windows(gpu, orc):
    # 3-D tiles: 28 columns x 8 rows
    _check_windows(gpu, orc, "C4", 1, [(-4, 8, -4, 8), (28 * 9 - 4, 8, 8 * 31 - 4, 8), (301, 8, 77, 8)])


def test_c5_windows(gpu, orc):
    _check_windows(gpu, orc, "C5", 1, [(-4, 8, -4, 8), (28 * 18 - 4, 8, 8 * 63 - 4, 8)])
