"""GPU parity: the CUDA path (through the C ABI, include/mc_tvd.h) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star):
field-max-normalised error <= 1e-12 after 1 step, <= 1e-9 after 100 steps, Nu within 1e-10 relative.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import parity_err, rel_err, ulp_perturbed

pytestmark = pytest.mark.gpu

TOL_SWEEP = 2e-13      # one operator L_alpha: a handful of roundings on O(1) fields
TOL_1STEP = 1e-12      # parity_err norm
TOL_100STEP = 1e-9
TOL_NU = 1e-10
COND_FACTOR = 2.0      # field-max norm: at most twice the oracle's own response to 1-ulp input noise (measured on
                       # B200: 0.6-1.0 times it after 1 step, 0.8 after 100; the values are printed by the C1 tests)


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


def _solver(gpu, grid, params, X0):
    return gpu.MCTVD(grid, params, X0)


# ---- one operator L_alpha(tau) (Eqs. 31-39), every axis, both directions, both z boundaries ------
SWEEP_GRIDS = [
    (2, 300, 1, 70),      # 2-D, even nx: 3 march tiles (124 outputs) / 5 two-node lane warps (60 outputs), ragged tails
    (2, 301, 1, 40),      # 2-D, odd nx: the one-node-per-lane x-sweep (11 lane warps of 28 outputs)
    (2, 29, 1, 5),        # smallest plate problem, one ragged tile
    (3, 60, 21, 19),      # 3-D: 3 x-tiles, 3 b-tiles (8 outputs) with ragged tails, walls in b for Ly
    (3, 30, 9, 33),       # ragged the other way
    (3, 45, 17, 14),      # 3-D, odd nx: no TMA (16-byte row strides), the register-prefetch k_march3
    (2, 4, 1, 5),         # the smallest boxes the ABI accepts: a tile wraps the periodic seam several times
    (3, 6, 4, 6),
]


def _state(kind, grid, params, seed):
    """smooth: a few Fourier modes (the limiter stays at phi = 1 almost everywhere, the TVD term is ~0);
    rough: the same plus node-to-node noise, which switches the TVD term on along every axis."""
    if kind == "rough":
        return inputs.rough_random_state(grid, params, seed=seed)
    return inputs.smooth_random_state(grid, params, seed=seed)


def _tvd_active_fraction(orc, grid, params, X0, alpha, tau, direction, ref):
    """Fraction of nodes on which the TVD term of Eqs. 34-39 changes the operator's result (oracle, tvd on vs off)."""
    off = orc.sweep(orc.Problem(grid, dict(params, tvd_off=1)), X0, alpha, tau, direction)
    return float((np.abs(ref - off).max(axis=0) > 1e-9).mean())


@pytest.mark.parametrize("ndim,nx,ny,nz", SWEEP_GRIDS)
@pytest.mark.parametrize("bc_z", [0, 1])
@pytest.mark.parametrize("tvd_form", [0, 1])
@pytest.mark.parametrize("kind", ["smooth", "rough"])
def test_sweep_parity(gpu, orc, ndim, nx, ny, nz, bc_z, tvd_form, kind):
    grid = inputs.make_grid(ndim, nx, nz, ny)
    params = inputs.make_params(Ra=1e4, bc_z=bc_z, tvd_form=tvd_form)
    X0 = _state(kind, grid, params, 11 + nx + bc_z)
    prob = orc.Problem(grid, params)
    tau = 0.25 * orc.dt(prob, X0)
    for alpha in ((0, 2) if ndim == 2 else (0, 1, 2)):
        for direction in (1, -1):
            ref = orc.sweep(prob, X0, alpha, tau, direction)
            if kind == "rough":
                # the limiter must really be exercised: along every axis, both directions, both forms of Eq. 34
                # (between plates only the interior interfaces carry a dissipation flux, R11)
                frac = _tvd_active_fraction(orc, grid, params, X0, alpha, tau, direction, ref)
                assert frac >= (0.2 if bc_z == 0 and nz <= 6 else 0.5), (alpha, direction, frac)
            s = _solver(gpu, grid, params, X0)
            s.sweep(alpha, direction, tau)
            err = rel_err(s.state(), ref).max()
            s.close()
            assert err <= TOL_SWEEP, (kind, alpha, direction, err)


@pytest.mark.parametrize("ndim,nx,ny,nz,stretch", [(2, 300, 1, 70, None), (2, 301, 1, 40, 1.5), (3, 60, 21, 19, None),
                                                   (3, 45, 17, 14, None), (3, 30, 9, 33, 2.0)])
@pytest.mark.parametrize("tvd_form", [0, 1])
def test_sweep_parity_advective_courant_number(gpu, orc, ndim, nx, ny, nz, stretch, tvd_form):
    """co_mode = 1 (R5, second reading of Eq. 39's local Courant number: |u_alpha| tau / dx): every operator on
    a rough state, where the TVD term is active and differs from the co_mode = 0 result; then one whole step."""
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=stretch)
    params = inputs.make_params(Ra=1e4, tvd_form=tvd_form, co_mode=1)
    X0 = inputs.rough_random_state(grid, params, seed=23 + nx)
    prob = orc.Problem(grid, params)
    tau = 0.25 * orc.dt(prob, X0)
    for alpha in ((0, 2) if ndim == 2 else (0, 1, 2)):
        for direction in (1, -1):
            ref = orc.sweep(prob, X0, alpha, tau, direction)
            other = orc.sweep(orc.Problem(grid, dict(params, co_mode=0)), X0, alpha, tau, direction)
            assert rel_err(other, ref).max() > 1e-6                      # the switch matters on this state
            s = _solver(gpu, grid, params, X0)
            s.sweep(alpha, direction, tau)
            err = rel_err(s.state(), ref).max()
            s.close()
            assert err <= TOL_SWEEP, (alpha, direction, err)
    ref, dts, _ = orc.step(prob, X0, 1)
    s = _solver(gpu, grid, params, X0)
    s.step(1)
    err = parity_err(grid, params, s.state(), ref).max()
    s.close()
    assert err <= TOL_1STEP, err


def test_bad_co_mode_is_rejected(gpu):
    grid = inputs.make_grid(2, 16, 9)
    params = inputs.make_params(co_mode=2)
    with pytest.raises(gpu.MCTVDError) as e:
        gpu.MCTVD(grid, params, inputs.conduction_state(grid, inputs.make_params()))
    assert e.value.code == -1


@pytest.mark.parametrize("ndim,nx,ny,nz", [(2, 300, 1, 70), (3, 60, 21, 19)])
@pytest.mark.parametrize("chunk", [7, 16])
@pytest.mark.parametrize("tvd_form", [0, 1])
def test_sweep_parity_chunked(gpu, orc, ndim, nx, ny, nz, chunk, tvd_form):
    """Blocks that start in the middle of the marching direction (4-level warm-up), on a rough state so that the
    TVD stencil of the warm-up levels (dX of the levels below the chunk) matters."""
    grid = inputs.make_grid(ndim, nx, nz, ny)
    params = inputs.make_params(Ra=1e4, tvd_form=tvd_form)
    X0 = inputs.rough_random_state(grid, params, seed=5)
    prob = orc.Problem(grid, params)
    tau = 0.25 * orc.dt(prob, X0)
    for alpha in ((0, 2) if ndim == 2 else (0, 1, 2)):
        for direction in (1, -1):
            ref = orc.sweep(prob, X0, alpha, tau, direction)
            assert _tvd_active_fraction(orc, grid, params, X0, alpha, tau, direction, ref) >= 0.5
            s = _solver(gpu, grid, params, X0)
            s.debug_set_chunk(chunk)
            s.sweep(alpha, direction, tau)
            err = rel_err(s.state(), ref).max()
            s.close()
            assert err <= TOL_SWEEP, (alpha, direction, err)


def test_tvd_off_and_paper_direction(gpu, orc):
    grid = inputs.make_grid(3, 40, 13, 12)
    for over in (dict(tvd_off=1), dict(dir_mode=0), dict(lambda_coef=2.0 / 3.0)):
        params = inputs.make_params(Ra=1e3, **over)
        X0 = inputs.smooth_random_state(grid, params, seed=3)
        prob = orc.Problem(grid, params)
        ref, dts, _ = orc.step(prob, X0, 1)
        s = _solver(gpu, grid, params, X0)
        s.step(1)
        assert rel_err(s.state(), ref).max() <= TOL_1STEP, over
        s.close()


# ---- config C1 (BASELINE.json configs[0]): 1 step, 100 steps, dt, Nu ------------------------------
@pytest.fixture(scope="module")
def c1(orc):
    grid, params, steps = inputs.config("C1")
    X0 = inputs.conduction_state(grid, params)
    prob = orc.Problem(grid, params)
    ref1, dts1, _ = orc.step(prob, X0, 1)
    ref100, dts100, t100 = orc.step(prob, X0, steps)
    # conditioning of the map itself: the oracle against the oracle on an input moved by <= 1 ulp
    Xu = ulp_perturbed(X0)
    cond1 = rel_err(orc.step(prob, Xu, 1)[0], ref1)
    cond100 = rel_err(orc.step(prob, Xu, steps)[0], ref100)
    return dict(grid=grid, params=params, steps=steps, X0=X0, prob=prob, ref1=ref1, ref100=ref100,
                dts=dts100, t100=t100, cond1=cond1, cond100=cond100)


def test_c1_one_step(gpu, orc, c1):
    s = _solver(gpu, c1["grid"], c1["params"], c1["X0"])
    dt0 = s.dt()
    assert abs(dt0 - c1["dts"][0]) <= 4e-16 * dt0
    s.step(1)
    X = s.state()
    s.close()
    assert parity_err(c1["grid"], c1["params"], X, c1["ref1"]).max() <= TOL_1STEP
    # field-max norm: rho and E meet the tolerance outright; the momenta (max ~8e-4 here) are bounded by
    # the conditioning of the step, measured on the oracle itself
    fm = rel_err(X, c1["ref1"])
    print("C1, 1 step: parity_err", parity_err(c1["grid"], c1["params"], X, c1["ref1"]), "field-max", fm,
          "oracle 1-ulp conditioning", c1["cond1"])
    assert fm[0] <= TOL_1STEP and fm[-1] <= TOL_1STEP
    assert np.all(fm <= np.maximum(TOL_1STEP, COND_FACTOR * c1["cond1"])), (fm, c1["cond1"])


def test_c1_100_steps_and_diagnostics(gpu, orc, c1):
    s = _solver(gpu, c1["grid"], c1["params"], c1["X0"])
    s.step(c1["steps"])
    X = s.state()
    assert parity_err(c1["grid"], c1["params"], X, c1["ref100"]).max() <= TOL_100STEP
    fm = rel_err(X, c1["ref100"])
    print("C1, 100 steps: parity_err", parity_err(c1["grid"], c1["params"], X, c1["ref100"]), "field-max", fm,
          "oracle 1-ulp conditioning", c1["cond100"])
    assert np.all(fm <= np.maximum(TOL_100STEP, COND_FACTOR * c1["cond100"])), (fm, c1["cond100"])
    d, Tp, rp, pp = s.diagnostics()
    assert d["step"] == c1["steps"]
    assert abs(d["time"] - c1["t100"]) <= 1e-9 * c1["t100"]
    # Nu on an IDENTICAL state (the downloaded GPU state): tolerance 1e-10 relative
    do, To, ro, po = orc.diagnostics(c1["prob"], X)
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk"):
        assert abs(d[k] - do[k]) <= TOL_NU * abs(do[k]), (k, d[k], do[k])
    for k in ("re", "u_rms", "mass", "energy", "max_mach", "min_rho", "min_T"):
        assert abs(d[k] - do[k]) <= 1e-12 * max(abs(do[k]), 1e-30), (k, d[k], do[k])
    for k in ("nu_conv", "nu_K", "mom_x", "mom_z"):          # sums that cancel: absolute on their scale
        scale = {"nu_conv": 1.0, "nu_K": 1.0, "mom_x": do["mass"], "mom_z": do["mass"]}[k]
        assert abs(d[k] - do[k]) <= 1e-10 * scale, (k, d[k], do[k])
    np.testing.assert_allclose(Tp, To, rtol=1e-13)
    np.testing.assert_allclose(rp, ro, rtol=1e-13)
    np.testing.assert_allclose(pp, po, rtol=1e-13)
    assert abs(d["dt"] - orc.dt(c1["prob"], X)) <= 4e-16 * d["dt"]
    # end to end: Nu of the GPU run against Nu of the oracle run
    dref, *_ = orc.diagnostics(c1["prob"], c1["ref100"])
    assert abs(d["nu_bar"] - dref["nu_bar"]) <= 1e-7 * abs(dref["nu_bar"])
    s.close()


def test_step_host_matches_step(gpu, orc, c1):
    import torch
    s = _solver(gpu, c1["grid"], c1["params"], c1["X0"])
    s.step(3)
    a = s.state().copy()
    hin = torch.from_numpy(c1["X0"].reshape(-1).copy()).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    s.step_host(hin, hout, 3)
    assert np.array_equal(hout.numpy().reshape(a.shape), a)      # same kernels, same order: bit-equal
    s.close()


@pytest.mark.parametrize("name,n,every", [("C1", 24, 3), ("3d", 9, 2)])
def test_time_averages(gpu, orc, name, n, every):
    """mc_tvd_step_stats / mc_tvd_stats_read against the oracle's twin: the same samples, the
    same weights; the two states differ by the parity error of n steps, so do the averages."""
    if name == "C1":
        grid, params, _ = inputs.config("C1")
    else:
        grid, params = inputs.make_grid(3, 64, 20, 24), inputs.make_params(Ra=1e5)
    X0 = inputs.conduction_state(grid, params, amplitude=1e-2)
    prob = orc.Problem(grid, params)
    ref, ro, To, rho_o, po = orc.step_stats(prob, X0, n, every)
    s = _solver(gpu, grid, params, X0)
    s.step_stats(n, every)
    st, Tp, rp, pp = s.stats_read()
    assert st["samples"] == n // every == ro["samples"]
    assert abs(st["t_end"] - ro["t_end"]) <= 1e-12 * ro["t_end"] and abs(st["weight"] - ro["weight"]) <= 1e-12 * ro["weight"]
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk", "re", "u_rms", "nu_bar_sq", "re_sq"):
        assert abs(st[k] - ro[k]) <= 1e-9 * max(abs(ro[k]), 1.0), (k, st[k], ro[k])
    for k in ("nu_conv", "nu_K"):
        assert abs(st[k] - ro[k]) <= 1e-9, (k, st[k], ro[k])
    np.testing.assert_allclose(Tp, To, rtol=1e-12)
    np.testing.assert_allclose(rp, rho_o, rtol=1e-12)
    np.testing.assert_allclose(pp, po, rtol=1e-12)
    assert parity_err(grid, params, s.state(), ref).max() <= n * TOL_1STEP
    # sampling in one call or call by call is the same thing, bit for bit; a reset starts a new span
    s2 = _solver(gpu, grid, params, X0)
    for _ in range(n):
        s2.step_stats(1, every)
    st2, Tp2, _, _ = s2.stats_read()
    assert st2 == st and np.array_equal(Tp2, Tp)
    s2.stats_reset()
    with pytest.raises(gpu.MCTVDError):
        s2.stats_read()                                   # no sample yet
    s2.step_stats(every, every)
    st3, *_ = s2.stats_read()
    assert st3["samples"] == 1 and st3["t_begin"] == st["t_end"] if n % every == 0 else st3["samples"] == 1
    s.close(); s2.close()


def test_3d_steps(gpu, orc):
    """A 3-D box with plates, 3 full steps of Eq. 30 (18 sweeps), CFL dt from the fused reduction."""
    grid = inputs.make_grid(3, 64, 20, 24)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.conduction_state(grid, params, amplitude=1e-2)
    prob = orc.Problem(grid, params)
    ref, dts, t = orc.step(prob, X0, 3)
    s = _solver(gpu, grid, params, X0)
    s.step(1)
    ref1, _, _ = orc.step(prob, X0, 1)
    assert parity_err(grid, params, s.state(), ref1).max() <= TOL_1STEP
    s.step(2)
    assert parity_err(grid, params, s.state(), ref).max() <= 3 * TOL_1STEP
    d, *_ = s.diagnostics()
    assert abs(d["time"] - t) <= 1e-12 * t
    do, *_ = orc.diagnostics(prob, s.state())
    assert abs(d["nu_bar"] - do["nu_bar"]) <= TOL_NU * abs(do["nu_bar"])
    s.close()


@pytest.mark.parametrize("ndim,nx,ny,nz,chunk", [(2, 300, 1, 70, 0), (2, 300, 1, 70, 9), (3, 60, 21, 19, 0), (3, 60, 21, 19, 5)])
def test_cfl_reduction_is_exact_every_step(gpu, orc, ndim, nx, ny, nz, chunk):
    """The CFL max-reduction is folded into the last operator behind a division-free filter that skips
    nodes which cannot raise the maximum already recorded (csrc/mc_common.cuh cfl_can_skip).  It must stay
    EXACT: after every step dt equals the oracle's dt of the same (downloaded) state to an ulp or two, on a
    state whose fastest node is in the interior and moves, with several marching chunks per column."""
    grid = inputs.make_grid(ndim, nx, nz, ny)
    params = inputs.make_params(Ra=1e4)
    X0 = inputs.smooth_random_state(grid, params, seed=23)
    prob = orc.Problem(grid, params)
    s = _solver(gpu, grid, params, X0)
    s.debug_set_chunk(chunk)
    assert abs(s.dt() - orc.dt(prob, X0)) <= 4e-16 * s.dt()
    for _ in range(6):
        s.step(1)
        dt_gpu = s.dt()
        assert abs(dt_gpu - orc.dt(prob, s.state())) <= 4e-16 * dt_gpu
    s.close()


# ---- properties that hold at any size --------------------------------------------------------------
def test_uniform_state_is_a_fixed_point(gpu):
    """Every flux difference and dX is exactly zero: the state must not change in a single bit."""
    from tests.helpers import ideal_gas_params, state_from_primitives
    for ndim, nx, ny, nz in [(2, 130, 1, 40), (3, 60, 12, 10)]:
        grid = inputs.make_grid(ndim, nx, nz, ny)
        params = ideal_gas_params(mu_override=1e-2, K_override=1e-2)
        X0 = state_from_primitives(grid, params, 1.3, 0.4, 0.0 if ndim == 2 else -0.2, 0.1, 0.9)
        s = _solver(gpu, grid, params, X0)
        s.step(5)
        assert np.array_equal(s.state(), X0)
        s.close()


def test_mass_conserved_with_plates(gpu):
    grid, params, _ = inputs.config("C1")
    X0 = inputs.conduction_state(grid, params, amplitude=1e-2)
    s = _solver(gpu, grid, params, X0)
    m0 = s.diagnostics()[0]["mass"]
    s.step(50)
    m1 = s.diagnostics()[0]["mass"]
    assert abs(m1 - m0) <= 1e-12 * abs(m0)
    s.close()


# ---- error behaviour of the C ABI -------------------------------------------------------------------
def test_nonfinite_state_is_reported(gpu):
    grid = inputs.make_grid(2, 64, 16)
    params = inputs.make_params()
    X0 = inputs.conduction_state(grid, params)
    bad = X0.copy()
    bad[0, 37] = -1.0                      # non-positive rho
    s = _solver(gpu, grid, params, bad)
    with pytest.raises(gpu.MCTVDError) as e:
        s.dt()
    assert e.value.code == -4
    s.close()
    bad = X0.copy()
    bad[3, 100] = np.nan
    s = _solver(gpu, grid, params, bad)
    with pytest.raises(gpu.MCTVDError) as e:
        s.dt()
    assert e.value.code == -4
    s.close()


def test_workspace_too_small(gpu):
    import ctypes as C
    import torch
    lib = gpu.load_library()
    grid = inputs.make_grid(2, 64, 16)
    g, p = gpu.make_grid(grid), gpu.make_params(inputs.make_params())
    wb = lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(p))
    f = torch.zeros(4 * 64 * 16, dtype=torch.float64, device="cuda")
    w = torch.zeros(wb // 8, dtype=torch.float64, device="cuda")
    h = C.c_void_p()
    rc = lib.mc_tvd_init(C.byref(g), C.byref(p), f.data_ptr(), w.data_ptr(), wb - 8, None, C.byref(h))
    assert rc == -3 and not h.value
    rc = lib.mc_tvd_init(C.byref(g), C.byref(p), f.data_ptr() + 8, w.data_ptr(), wb, None, C.byref(h))
    assert rc == -1 and not h.value
