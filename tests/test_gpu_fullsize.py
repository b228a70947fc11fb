"""Parity at BASELINE.json's full sizes (configs C2-C5), in the launch configuration bench.py times.

The oracle cannot march 67M-268M nodes in test time, but every operation of the step is local
(stencil radius 2 per operator in the sweep direction and across it):
after s steps the state inside a column window equals the oracle run on that window plus a margin of
2 * (operators per step) * s columns on each periodic side (full z), given the same dt sequence.  So
the GPU runs the whole grid for several steps, and the oracle recomputes sampled windows of it element by
element.  The windows are placed from the kernels' own tiling (mc_tvd_debug_geometry): across the periodic
seam, across interior tile boundaries in x and in y, and -- through the full height of every window -- across
every chunk boundary of the marching direction.  dt (a global max) and the diagnostics are checked against
the oracle on the whole downloaded state.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import parity_err, plate_nusselt_exact

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


def _windows_from_tiling(s, grid, wx, wy):
    """Sample windows (i0, wx, j0, wy) placed on the kernels' own tile boundaries: the periodic seam, an interior
    boundary of each x-tiling in use (L_x's and, where it differs, L_z's), an interior boundary of each y-tiling
    (3-D: L_z's and L_x's rows), and one window away from all of them."""
    nx, ny = grid["nx"], grid["ny"]
    tx = sorted({s.debug_geometry(a)[0] for a in ((0, 2) if grid["ndim"] == 2 else (0, 1, 2))})
    tb = sorted({s.debug_geometry(a)[1] for a in (0, 2)}) if grid["ndim"] == 3 else [1]
    assert all(t > 0 for t in tx + tb), (tx, tb)
    wins = [(-wx // 2, wx, -wy // 2 if ny > 1 else 0, wy)]                      # the seam (both directions in 3-D)
    for n, t in enumerate(tx):
        m = max(1, (nx // t) * (2 + n) // 5)                                     # an interior boundary, not the first
        j0 = (max(1, (ny // tb[0]) // 2) * tb[0] - wy // 2) if ny > 1 else 0
        wins.append((m * t - wx // 2, wx, j0, wy))
    if ny > 1:
        for n, t in enumerate(tb):
            m = max(1, (ny // t) * (3 + n) // 7)
            wins.append((nx // 3 + 1, wx, m * t - wy // 2, wy))
        ch_y = s.debug_geometry(1)[2]                                            # L_y marches along y in chunks
        if 0 < ch_y < ny:
            wins.append((2 * nx // 3 + 3, wx, ch_y * max(1, (ny // ch_y) // 2) - wy // 2, wy))
    return wins, tx, tb


def _check_windows(gpu, orc, name, n_steps, wx, wy=1, state="conduction", max_windows=None):
    import psutil
    grid, params, _ = inputs.config(name)
    nf, N = inputs.num_fields(grid), inputs.num_nodes(grid)
    need = 3 * nf * N * 8
    if psutil.virtual_memory().available < need + (8 << 30):
        pytest.skip(f"host memory too small for {name}")
    X0 = inputs.conduction_state(grid, params) if state == "conduction" else inputs.moving_state(grid, params)
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
    windows, tx, tb = _windows_from_tiling(s, grid, wx, wy)
    chunks = {a: s.debug_geometry(a)[2] for a in ((0, 2) if grid["ndim"] == 2 else (0, 1, 2))}
    if max_windows:
        windows = windows[:max_windows]
    worst = 0.0
    for (i0, wx_, j0, wy_) in windows:
        i0 %= grid["nx"]
        if grid["ndim"] == 2:
            Xw, gw = inputs.window_x(X0.reshape(nf, -1), grid, i0 - margin, wx_ + 2 * margin)
            iy = np.array([0])
        else:
            j0 %= grid["ny"]
            Xw, gw = inputs.window_xy(X0.reshape(nf, -1), grid, i0 - margin, wx_ + 2 * margin, j0 - margin,
                                      wy_ + 2 * margin)
            iy = (np.arange(wy_) + j0) % grid["ny"]
        ref, _, _ = orc.step(orc.Problem(gw, params), Xw, n_steps, dt_in=dts)
        ix = (np.arange(wx_) + i0) % grid["nx"]
        gw_out = dict(gw, nx=wx_, ny=len(iy))
        got = _device_window(s, grid, ix, iy)
        r = ref.reshape(nf, gw["nz"], gw["ny"], gw["nx"])
        if grid["ndim"] == 2:
            r = r[:, :, :, margin:margin + wx_]
        else:
            r = r[:, :, margin:margin + wy_, margin:margin + wx_]
        err = parity_err(gw_out, params, got, r.reshape(nf, -1)).max()
        worst = max(worst, err)
        assert err <= TOL_1STEP * n_steps, (name, (i0, wx_, j0, wy_), err)
    print(f"{name} ({state}), {n_steps} steps: x-tiles {tx}, y-tiles {tb}, chunks {chunks}, {len(windows)} windows, "
          f"worst parity error {worst:.2e} (bound {TOL_1STEP * n_steps:.0e})")
    # dt after the last step and the diagnostics: the oracle on the whole downloaded state
    dt_gpu = s.dt()
    if psutil.virtual_memory().available > 2 * nf * N * 8 + (8 << 30):
        Xn = s.state()
        dt_ref = orc.dt(prob, Xn)
        assert abs(dt_gpu - dt_ref) <= 4e-16 * dt_ref
        d, Tp, rp, pp = s.diagnostics()
        do, To, ro, po = orc.diagnostics(prob, Xn)                # one serial pass, ~20 ns per node
        # Nu within 1e-10 (north_star) of the size of the plate Nusselt numbers (nu_bar is their mean; on the noisy
        # early states the two have opposite signs and nearly cancel).  The reference is the plate gradient of plane
        # means summed in extended precision: on these grids the oracle's plain serial fp64 sums carry ~1e-9 of noise
        # after the 1/(eps dz) amplification of Eq. 23, so the oracle itself is only held to 1e-8.
        nb, nt, nbar = plate_nusselt_exact(grid, params, Xn)
        nu_scale = max(abs(nb), abs(nt), 1.0)
        for k, want in (("nu_bottom", nb), ("nu_top", nt), ("nu_bar", nbar)):
            assert abs(d[k] - want) <= 1e-10 * nu_scale, (k, d[k], want, do[k])
            assert abs(do[k] - want) <= 1e-8 * nu_scale, (k, do[k], want)
        assert abs(d["nu_bulk"] - do["nu_bulk"]) <= 1e-10 * max(abs(do["nu_bulk"]), 1.0)
        for k in ("mass", "energy", "re", "min_rho", "min_T"):
            assert abs(d[k] - do[k]) <= 1e-12 * max(abs(do[k]), 1e-30), (k, d[k], do[k])
        np.testing.assert_allclose(Tp, To, rtol=1e-13)
        np.testing.assert_allclose(rp, ro, rtol=1e-13)
        np.testing.assert_allclose(pp, po, rtol=1e-13)
        del Xn
    s.close()
    return worst


def test_c2_windows(gpu, orc):
    _check_windows(gpu, orc, "C2", 20, wx=12)


def test_c3_windows(gpu, orc):
    _check_windows(gpu, orc, "C3", 5, wx=16)


def test_c3_moving_state(gpu, orc):
    _check_windows(gpu, orc, "C3", 3, wx=16, state="moving", max_windows=2)


def test_c4_windows(gpu, orc):
    _check_windows(gpu, orc, "C4", 3, wx=8, wy=8)


def test_c5_windows(gpu, orc):
    _check_windows(gpu, orc, "C5", 3, wx=8, wy=8)


def test_c5_moving_state(gpu, orc):
    _check_windows(gpu, orc, "C5", 2, wx=8, wy=8, state="moving", max_windows=2)
