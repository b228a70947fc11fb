"""GPU parity on the paper's non-uniform (tangent-hyperbolic) z grid, readings R19 / R20: the CUDA path
through mc_tvd_grid.z_nodes against the CPU oracle, element by element on the same seeded inputs -- every operator,
both directions, both forms of Eq. 34, chunked marches, whole steps with the CFL reduction, and the diagnostics.
Tolerances as on the uniform grid (tests/test_gpu_parity.py)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import parity_err, rel_err

pytestmark = pytest.mark.gpu

TOL_SWEEP = 2e-13
TOL_1STEP = 1e-12
TOL_NU = 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


GRIDS = [
    (2, 300, 1, 70),      # 2-D, even nx: k_march / k_lane2, ragged tiles
    (2, 301, 1, 40),      # 2-D, odd nx: k_lane
    (2, 29, 1, 5),        # smallest plate problem
    (3, 60, 21, 19),      # 3-D: TMA-staged k_march3 (L_z, L_y with z as the tile's second direction), k_lane3
    (3, 45, 17, 14),      # 3-D, odd nx: the register-prefetch k_march3
    (3, 6, 4, 6),
]


@pytest.mark.parametrize("ndim,nx,ny,nz", GRIDS)
@pytest.mark.parametrize("tvd_form", [0, 1])
@pytest.mark.parametrize("stretch", [1.5, 2.5])
def test_sweep_parity_stretched(gpu, orc, ndim, nx, ny, nz, tvd_form, stretch):
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=stretch)
    params = inputs.make_params(Ra=1e4, tvd_form=tvd_form)
    X0 = inputs.rough_random_state(grid, params, seed=21 + nx)
    prob = orc.Problem(grid, params)
    tau = 0.25 * orc.dt(prob, X0)
    for alpha in ((0, 2) if ndim == 2 else (0, 1, 2)):
        for direction in (1, -1):
            ref = orc.sweep(prob, X0, alpha, tau, direction)
            s = gpu.MCTVD(grid, params, X0)
            s.sweep(alpha, direction, tau)
            err = rel_err(s.state(), ref).max()
            s.close()
            assert err <= TOL_SWEEP, (alpha, direction, err)


@pytest.mark.parametrize("ndim,nx,ny,nz", [(2, 300, 1, 70), (3, 60, 21, 19)])
@pytest.mark.parametrize("chunk", [7, 16])
def test_sweep_parity_stretched_chunked(gpu, orc, ndim, nx, ny, nz, chunk):
    """Blocks that start in the middle of the march: the metric of the warm-up levels comes from the tables too."""
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=1.5)
    params = inputs.make_params(Ra=1e4)
    X0 = inputs.rough_random_state(grid, params, seed=5)
    prob = orc.Problem(grid, params)
    tau = 0.25 * orc.dt(prob, X0)
    for alpha in ((0, 2) if ndim == 2 else (0, 1, 2)):
        for direction in (1, -1):
            ref = orc.sweep(prob, X0, alpha, tau, direction)
            s = gpu.MCTVD(grid, params, X0)
            s.debug_set_chunk(chunk)
            s.sweep(alpha, direction, tau)
            err = rel_err(s.state(), ref).max()
            s.close()
            assert err <= TOL_SWEEP, (alpha, direction, err)


@pytest.mark.parametrize("ndim,nx,ny,nz", [(2, 256, 1, 65), (3, 64, 20, 25)])
def test_steps_dt_and_diagnostics_stretched(gpu, orc, ndim, nx, ny, nz):
    """Whole steps of Eq. 30 on the stretched grid from the seeded conduction-plus-noise state: the state after 1 and
    after 10 steps, dt after every step (the fused CFL reduction with the per-level spacing), Nu / Re / totals /
    profiles on an identical state."""
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=1.5)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.conduction_state(grid, params, amplitude=1e-2)
    prob = orc.Problem(grid, params)
    s = gpu.MCTVD(grid, params, X0)
    X = X0
    for n in range(10):
        dt_gpu = s.dt()
        assert dt_gpu == pytest.approx(orc.dt(prob, X), rel=4e-16)
        X, dts, _ = orc.step(prob, X, 1)
        s.step(1)
        if n == 0:
            assert parity_err(grid, params, s.state(), X).max() <= TOL_1STEP
    Y = s.state()
    assert parity_err(grid, params, Y, X).max() <= 10 * TOL_1STEP
    d, Tp, rp, pp = s.diagnostics()
    do, To, ro, po = orc.diagnostics(prob, Y)
    s.close()
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk"):
        assert d[k] == pytest.approx(do[k], rel=TOL_NU), k
    for k in ("re", "mass", "energy", "max_mach", "min_rho", "min_T"):
        assert d[k] == pytest.approx(do[k], rel=1e-11), k
    assert np.allclose(Tp, To, rtol=1e-13) and np.allclose(rp, ro, rtol=1e-13) and np.allclose(pp, po, rtol=1e-13)


def test_mass_is_conserved_on_the_stretched_grid(gpu):
    """The device path keeps the cell-height-weighted mass between the plates to round-off (R19 / R20), as the oracle does."""
    grid = inputs.make_grid(3, 48, 33, 24, z_stretch=1.5)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.rough_random_state(grid, params, seed=9, rough=0.02)
    s = gpu.MCTVD(grid, params, X0)
    m0 = s.diagnostics()[0]["mass"]
    s.step(20)
    m1 = s.diagnostics()[0]["mass"]
    s.close()
    assert abs(m1 - m0) <= 1e-13 * m0


def test_bad_node_heights_are_rejected(gpu):
    grid = inputs.make_grid(2, 16, 9, z_stretch=1.5)
    params = inputs.make_params()
    X0 = inputs.conduction_state(grid, params)
    bad = dict(grid, z_nodes=grid["z_nodes"][::-1].copy())
    with pytest.raises(gpu.MCTVDError) as e:
        gpu.MCTVD(bad, params, X0)
    assert e.value.code == -1
    with pytest.raises(gpu.MCTVDError):
        gpu.MCTVD(grid, inputs.make_params(bc_z=1), X0)
