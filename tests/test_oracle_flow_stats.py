"""Pins of the oracle's flow statistics (oracle.flow_stats: the z-momentum balance terms of Eqs. 40-43, PAPER.md:457-467,
and the distribution of r = K_e / I_e, Fig. 5) against closed forms.  No GPU needed."""
import numpy as np
import pytest
import sympy as sp

from paper_2411_10372_b200 import inputs
from tests.helpers import state_from_primitives


def cell_heights(z):
    w = np.empty_like(z)
    w[1:-1] = 0.5 * (z[2:] - z[:-2])
    w[0], w[-1] = 0.5 * (z[1] - z[0]), 0.5 * (z[-1] - z[-2])
    return w


def test_conduction_state_balances_buoyancy_and_pressure(orc):
    """Hydrostatic conduction state: F_n = F_v = 0, <F_b> = g <rho> over the interior cells, and <F_p> = <F_b> (Eq. 44,
    PAPER.md:469).  For the configs' parameters rho = 1 - z/2 is linear, the trapezoid recursion of the input recipe is
    exact and the central difference of p balances rho g to round-off; for gamma = 1.4 (rho = T^1.8) the balance is
    approached at second order."""
    for gam, exact in ((5.0 / 3.0, True), (1.4, False)):
        gap = []
        for nz in (17, 33, 65):
            g = inputs.make_grid(2, 8, nz)
            p = inputs.make_params(Ra=1e6, gamma=gam)
            X = inputs.conduction_state(g, p, amplitude=0.0)
            f, _ = orc.flow_stats(orc.Problem(g, p), X)
            w = cell_heights(inputs.z_nodes(g, p))[1:-1]
            rho = X[0].reshape(nz, 8)[1:-1, 0]
            assert f["Fb_mean"] == pytest.approx(10.0 * np.sum(w * rho) / np.sum(w), rel=1e-13)
            assert f["volume"] == pytest.approx(np.sum(w), rel=1e-14)
            assert f["Fn_mean"] == 0.0 and f["Fv_rms"] == 0.0 and f["max_mach"] == 0.0
            assert f["FbFp_mean"] == pytest.approx(f["Fb_mean"] - f["Fp_mean"], abs=1e-15)
            gap.append(abs(f["FbFp_mean"]))
        if exact:
            assert max(gap) < 1e-13, gap
        else:
            assert gap[0] < 1e-2 and gap[0] / gap[1] > 3.5 and gap[1] / gap[2] > 3.5, gap


def _analytic_forces(ndim, lam, mu, g_val, R):
    """F_n, F_p, F_b, F_v of Eqs. 40-43 for a smooth synthetic flow, by symbolic differentiation of the definitions."""
    x, y, z = sp.symbols("x y z")
    ky = 2 * sp.pi if ndim == 3 else 0
    ux = sp.Rational(3, 10) * sp.sin(2 * sp.pi * x) * sp.cos(sp.pi * z) * sp.cos(ky * y)
    uy = sp.Rational(1, 5) * sp.cos(2 * sp.pi * x) * sp.sin(ky * y) * sp.sin(sp.pi * z) if ndim == 3 else sp.Integer(0)
    uz = sp.Rational(1, 4) * sp.cos(2 * sp.pi * x) * sp.sin(sp.pi * z) * sp.cos(ky * y)
    rho = 1 + sp.Rational(1, 5) * sp.cos(2 * sp.pi * x) * sp.cos(sp.pi * z)
    T = 1 + sp.Rational(1, 10) * sp.sin(2 * sp.pi * x) * z * (1 - z)
    u = (ux, uy, uz)
    X = (x, y, z)
    div = sum(sp.diff(u[i], X[i]) for i in range(3))
    Fn = rho * sum(u[i] * sp.diff(uz, X[i]) for i in range(3))
    Fp = -sp.diff(R * rho * T, z)
    Fb = rho * g_val
    tau = [mu * (sp.diff(uz, X[i]) + sp.diff(u[i], z) + (lam * div if i == 2 else 0)) for i in range(3)]
    Fv = sum(sp.diff(tau[i], X[i]) for i in range(3))
    fns = [sp.lambdify((x, y, z), e, "numpy") for e in (rho, ux, uy, uz, T, Fn, Fp, Fb, Fv)]
    return fns


@pytest.mark.parametrize("ndim,stretch", [(2, None), (2, 1.5), (3, 1.5)])
@pytest.mark.parametrize("lam", [-2.0 / 3.0, 2.0 / 3.0])
def test_force_terms_converge_to_their_definitions(orc, ndim, stretch, lam):
    """A smooth synthetic flow with non-zero divergence, variable rho and T between plates: the volume means and
    root-mean-squares of F_n, F_p, F_b, F_v approach those of the analytic fields (same nodes, same weights) at second
    order.  Pins every term of Eqs. 40-43 incl. the (1 + lambda) d_z div u part of the viscous force, on the uniform and
    on the stretched grid."""
    mu, gv = 0.02, 10.0
    p = inputs.make_params(Ra=1e4, lambda_coef=lam, mu_override=mu)
    R = inputs.closure_constants(p)["R"]
    fns = _analytic_forces(ndim, lam, mu, gv, R)
    errs = []
    for n in (16, 32, 64):
        g = inputs.make_grid(ndim, n, n + 1, n // 2 if ndim == 3 else 1, lx=1.0, ly=1.0, z_stretch=stretch)
        zz = inputs.z_nodes(g, p)
        Z, Y, Xc = np.meshgrid(zz, np.arange(g["ny"]) / g["ny"], np.arange(n) / n, indexing="ij")
        rho, ux, uy, uz, T, Fn, Fp, Fb, Fv = [np.broadcast_to(f(Xc, Y, Z), Z.shape) for f in fns]
        X = state_from_primitives(g, p, rho, ux, uy, uz, R * rho * T)
        f, _ = orc.flow_stats(orc.Problem(g, p), X)
        w = cell_heights(zz)[1:-1, None, None]
        mean = lambda F: float(np.sum(w * F[1:-1]) / (np.sum(w) * g["nx"] * g["ny"]))
        e = []
        for name, F in (("Fn", Fn), ("Fp", Fp), ("Fb", Fb), ("Fv", Fv)):
            rms = np.sqrt(mean(F * F))
            e.append(abs(f[name + "_mean"] - mean(F)) / rms)
            e.append(abs(f[name + "_rms"] - rms) / rms)
        errs.append(max(e))
    assert errs[0] < 0.1, errs             # (n = 16 on the stretched 3-D grid: 0.07)
    assert errs[0] / errs[1] > 3.3 and errs[1] / errs[2] > 3.3, errs


def test_histogram_of_r_and_the_largest_mach_number(orc):
    """Uniform rho and T; |u| chosen node by node so that r = u^2 / (2 c_v T) sits in the middle of a quarter-octave,
    r = 2^e (1 + m/4 + 1/8): the node must land in bin 4 (e + 32) + m.  r = 0 and r < 2^-32 go to bin 0, r >= 1 to the last
    bin.  The largest Mach number from its definition."""
    g = inputs.make_grid(2, 16, 9)
    p = inputs.make_params(gamma=1.4, eps=1.0, D=1.0 / 1.4, g_override=0.0, T_bot=1.0, T_top=1.0)   # c_v = 1, R = 0.4
    es = [-40, -32, -31, -20, -10, -3, -1, 0, 3]
    want = np.zeros(128, dtype=np.int64)
    ux = np.zeros((9, 1, 16))
    for row, e in enumerate(es):
        for i in range(16):
            m = i % 4
            if i < 12:
                ux[row, 0, i] = np.sqrt(2.0 * 2.0 ** e * (1 + m / 4 + 1 / 8))      # T = 1, c_v = 1: r = u^2 / 2
                want[min(127, max(0, 4 * (e + 32) + m))] += 1
            else:
                want[0] += 1                                                       # a node at rest
    X = state_from_primitives(g, p, 1.0, ux, 0.0, 0.0, 0.4)
    f, h = orc.flow_stats(orc.Problem(g, p), X)
    assert h.sum() == 144 and np.array_equal(h, want)
    assert f["max_r"] == pytest.approx(0.5 * ux.max() ** 2, rel=1e-13)
    assert f["max_mach"] == pytest.approx(ux.max() / np.sqrt(1.4 * 0.4), rel=1e-13)


@pytest.mark.parametrize("ndim", [2, 3])
@pytest.mark.parametrize("phase,want", [(0.0, 1.0), (np.pi / 3, 0.5), (np.pi / 2, 0.0), (np.pi, -1.0), (2.0, np.cos(2.0))])
def test_correlation_of_mass_flux_and_superadiabatic_temperature(orc, ndim, phase, want):
    """Eq. 49.  rho u_z = A sin(pi z) cos(2 pi x) and T_sa = T - (1 - D z) = B sin(pi z) cos(2 pi x +
    phase): on a uniform grid the trapezoid rule integrates these trigonometric products exactly, so
    <rho u_z T_sa> = A B cos(phase) / 4, <(rho u_z)^2> = A^2 / 4, <T_sa^2> = B^2 / 4 and C = cos(phase) to round-off --
    the sign, the T_A(z) that is subtracted, the half cells at the plates and the normalisation all enter."""
    A, B = 0.03, 0.02
    g = inputs.make_grid(ndim, 16, 13, 8 if ndim == 3 else 1, lx=1.0, ly=1.0)
    p = inputs.make_params(Ra=1e5, D=0.4)
    R = inputs.closure_constants(p)["R"]
    zz = inputs.z_nodes(g, p)
    Z, Y, Xc = np.meshgrid(zz, np.arange(g["ny"]) / g["ny"], np.arange(16) / 16, indexing="ij")
    rho = 1.0 + 0.3 * np.cos(2 * np.pi * Xc) * Z + 0.1 * np.sin(2 * np.pi * Y)
    mz = A * np.sin(np.pi * Z) * np.cos(2 * np.pi * Xc)
    T = (1.0 - p["D"] * Z) + B * np.sin(np.pi * Z) * np.cos(2 * np.pi * Xc + phase)
    X = state_from_primitives(g, p, rho, 0.05 * np.sin(2 * np.pi * Xc), 0.0, mz / rho, R * rho * T)
    f, _ = orc.flow_stats(orc.Problem(g, p), X)
    assert f["flux_mean"] == pytest.approx(A * B * np.cos(phase) / 4, abs=1e-17)
    assert f["rhouz_sq_mean"] == pytest.approx(A * A / 4, rel=1e-13)
    assert f["Tsa_sq_mean"] == pytest.approx(B * B / 4, rel=1e-11)          # (T_sa is a difference of O(1) numbers)
    assert f["corr_C"] == pytest.approx(want, abs=1e-11)


@pytest.mark.parametrize("ndim,stretch", [(2, None), (3, None), (2, 1.5), (3, 2.0)])
def test_correlation_agrees_with_nu_conv_and_is_bounded(orc, ndim, stretch):
    """<rho u_z T_sa>_V of Eq. 49 is the average inside Nu_conv of Eq. 22: the two routines must agree,
    on uniform and stretched grids; |C| <= 1 (Cauchy-Schwarz with non-negative weights), and C is unchanged when u_z is
    scaled (it is a normalised correlation) and changes sign with u_z."""
    g = inputs.make_grid(ndim, 12, 11, 10 if ndim == 3 else 1, z_stretch=stretch)
    p = inputs.make_params(Ra=1e5)
    X = inputs.rough_random_state(g, p, seed=17)
    prob = orc.Problem(g, p)
    f, _ = orc.flow_stats(prob, X)
    d = orc.diagnostics(prob, X)[0]
    assert np.sqrt(p["Ra"] * p["Pr"]) / p["eps"] * f["flux_mean"] == pytest.approx(d["nu_conv"], rel=1e-12)
    assert abs(f["corr_C"]) <= 1.0 and f["rhouz_sq_mean"] > 0 and f["Tsa_sq_mean"] > 0
    assert f["corr_C"] == pytest.approx(f["flux_mean"] / np.sqrt(f["rhouz_sq_mean"] * f["Tsa_sq_mean"]), rel=1e-15)
    # scale u_z by -2 at fixed rho, u_x, u_y, T
    nf = X.shape[0]
    rho, mz = X[0], X[nf - 2]
    Y = X.copy()
    Y[nf - 2] = -2.0 * mz
    Y[nf - 1] = X[nf - 1] + 0.5 * (4.0 - 1.0) * mz * mz / rho          # E keeps T: the kinetic energy of u_z grows 4-fold
    f2, _ = orc.flow_stats(prob, Y)
    assert f2["Tsa_sq_mean"] == pytest.approx(f["Tsa_sq_mean"], rel=1e-10)
    assert f2["corr_C"] == pytest.approx(-f["corr_C"], rel=1e-9)
    assert f2["rhouz_sq_mean"] == pytest.approx(4.0 * f["rhouz_sq_mean"], rel=1e-13)


def test_correlation_on_the_stretched_grid_converges(orc):
    """The same closed form (C = cos(phase), <rho u_z T_sa> = A B cos(phase) / 4) on the tanh grid, where the
    cell-height weights (R19) integrate sin^2(pi z) only to second order."""
    A, B, phase = 0.03, 0.02, 0.7
    errs = []
    for n in (16, 32, 64):
        g = inputs.make_grid(2, 16, n + 1, lx=1.0, z_stretch=1.5)
        p = inputs.make_params(Ra=1e5, D=0.4)
        R = inputs.closure_constants(p)["R"]
        zz = inputs.z_nodes(g, p)
        Z, _, Xc = np.meshgrid(zz, np.zeros(1), np.arange(16) / 16, indexing="ij")
        rho = 1.0 + 0.2 * Z
        mz = A * np.sin(np.pi * Z) * np.cos(2 * np.pi * Xc)
        T = (1.0 - p["D"] * Z) + B * np.sin(np.pi * Z) * np.cos(2 * np.pi * Xc + phase)
        X = state_from_primitives(g, p, rho, 0.0, 0.0, mz / rho, R * rho * T)
        f, _ = orc.flow_stats(orc.Problem(g, p), X)
        assert f["corr_C"] == pytest.approx(np.cos(phase), abs=1e-10)       # the weights cancel in the ratio
        errs.append(abs(f["flux_mean"] / (A * B * np.cos(phase) / 4) - 1.0))
    assert errs[0] < 2e-2 and errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5, errs
