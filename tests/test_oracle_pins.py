"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU needed).

BASELINE.json's five checks (uniform state, conservation, Sod tube vs the exact Riemann solution,
second-order convergence, mirror symmetry) plus closed forms that pin every term of Eq. 28:
viscous shear decay (inner and cross derivative halves of tau_ij), acoustic attenuation (the
dilatation coefficient), thermal diffusion (K), viscous heating pattern (the u_j tau_ij work term),
hydrostatic balance (gravity source and the potential energy inside E), and axis-permutation
identities that carry each pin from one sweep direction to the other two.
"""
import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import (advance_to, ideal_gas_params, primitives_of, rel_err, riemann_exact,
                           state_from_primitives)


def periodic_grid(ndim, nx, nz, ny=1, lx=1.0, ly=1.0, lz=1.0):
    return inputs.make_grid(ndim, nx, nz, ny, lx=lx, ly=ly, lz=lz)


# ----------------------------------------------------------------------------- coefficients
def test_coefficients_from_paper_numbers(orc):
    """tests/golden/coefficients.txt: values that Eqs. 14-18 and PAPER.md:204 give for the configs."""
    import os
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "coefficients.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                gold[k] = float(v)
    g, p, _ = inputs.config("C1")
    c = orc.coefficients(orc.Problem(g, p))
    for k in ("R", "cv", "g", "mu", "K"):
        assert c[k] == pytest.approx(gold[k], rel=1e-14), k
    assert p["T_top"] == pytest.approx(gold["T_top"], rel=1e-15)
    assert c["dx"] == 4.0 / 256 and c["dz"] == 1.0 / 63


# ----------------------------------------------------------------------------- check 1: uniform
@pytest.mark.parametrize("ndim", [2, 3])
def test_uniform_state_stays_uniform_bitwise(orc, ndim):
    """Every flux difference and dX of a uniform state is exactly 0 (BASELINE check 1)."""
    g = periodic_grid(ndim, 12, 10, 6 if ndim == 3 else 1)
    p = ideal_gas_params(mu_override=0.01, K_override=0.02)
    X = state_from_primitives(g, p, 1.3, 0.4, -0.2 if ndim == 3 else 0.0, 0.3, 2.0)
    Y, dts, _ = orc.step(orc.Problem(g, p), X, 20)
    assert np.array_equal(X, Y)
    # plates: u = 0, both plates at the gas temperature, no gravity
    p = ideal_gas_params(bc_z=0, mu_override=0.01, K_override=0.02)
    X = state_from_primitives(g, p, 1.3, 0.0, 0.0, 0.0, 1.3 * (p["gamma"] - 1.0))   # T = 1 = T_w
    Y, _, _ = orc.step(orc.Problem(g, p), X, 20)
    assert np.array_equal(X, Y)


# ----------------------------------------------------------------------------- check 2: conservation
@pytest.mark.parametrize("ndim,tvd_form", [(2, 0), (2, 1), (3, 1)])
def test_conservation_periodic(orc, ndim, tvd_form):
    """All-periodic box, g = 0, viscous and conducting: sums of rho, rho*u, E stay constant to
    round-off because flux differences and the TVD term telescope (BASELINE check 2a)."""
    g = periodic_grid(ndim, 24, 20, 16 if ndim == 3 else 1)
    p = ideal_gas_params(mu_override=5e-3, K_override=7e-3, tvd_form=tvd_form)
    X = inputs.smooth_random_state(g, p, seed=7)
    Y, _, _ = orc.step(orc.Problem(g, p), X, 10)
    s0, s1 = X.sum(axis=1), Y.sum(axis=1)
    scale = np.abs(X).sum(axis=1)
    assert np.all(np.abs(s1 - s0) <= 2e-14 * scale), (s1 - s0) / scale
    assert not np.array_equal(X, Y)


def test_mass_conserved_between_plates(orc):
    """Config C1 (plates): trapezoid mass constant to round-off under the conservative half-cell
    closure; horizontal momentum is reported only (the plates exert drag) (BASELINE check 2b)."""
    g, p, _ = inputs.config("C1")
    X = inputs.conduction_state(g, p)
    prob = orc.Problem(g, p)
    d0 = orc.diagnostics(prob, X)[0]
    Y, _, _ = orc.step(prob, X, 25)
    d1 = orc.diagnostics(prob, Y)[0]
    assert abs(d1["mass"] - d0["mass"]) <= 1e-14 * d0["mass"]
    assert d0["mass"] == pytest.approx(3.0, rel=1e-12)     # 4 * integral of the linear rho = 4*(1+0.5)/2
    assert abs(d1["mom_x"]) < 1e-6


# ----------------------------------------------------------------------------- check 3: Sod
def _sod(orc, n, axis, tvd_form, ndim=2, t_end=0.2, co_mode=0):
    """Classical two-state tube (8:1 density, 10:1 pressure, at rest, gamma 1.4), doubled so the
    periodic box holds two mirrored tubes; returns (x, rho(x), u(x), p(x)) along `axis`."""
    gam = 1.4
    x = np.arange(n) * 2.0 / n
    left = (x >= 0.5) & (x < 1.5)
    rho1, p1 = np.where(left, 1.0, 0.125), np.where(left, 1.0, 0.1)
    m = 4
    if axis == 0:
        g = periodic_grid(ndim, n, m, m if ndim == 3 else 1, lx=2.0, ly=m * 2.0 / n, lz=m * 2.0 / n)
        shape = (1, 1, n)
    elif axis == 2:
        g = periodic_grid(ndim, m, n, m if ndim == 3 else 1, lx=m * 2.0 / n, ly=m * 2.0 / n, lz=2.0)
        shape = (n, 1, 1)
    else:
        g = periodic_grid(3, m, m, n, lx=m * 2.0 / n, ly=2.0, lz=m * 2.0 / n)
        shape = (1, n, 1)
    p = ideal_gas_params(gamma=gam, tvd_form=tvd_form, co_mode=co_mode)
    X = state_from_primitives(g, p, rho1.reshape(shape), 0.0, 0.0, 0.0, p1.reshape(shape))
    X, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    prim = primitives_of(g, p, X)
    line = {0: np.s_[1, 0, :], 1: np.s_[1, :, 1], 2: np.s_[:, 0, 1]}[axis]
    return x, prim[0][line], prim[1 + axis][line], prim[5][line]


def test_sod_star_state_golden():
    """The test's own Riemann solver reproduces the star values quoted in tests/golden/sod.txt."""
    _, _, _, ps, us = riemann_exact(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, np.array([0.0]))
    assert ps == pytest.approx(0.30313, abs(1e-5)) and us == pytest.approx(0.92745, abs=1e-5)


@pytest.mark.parametrize("axis,ndim", [(0, 2), (2, 2), (1, 3)])
def test_sod_tube_vs_exact_riemann(orc, axis, ndim):
    """L1(rho) error falls about first order with N and the solution stays oscillation-free
    (BASELINE check 3) along every sweep direction."""
    errs = []
    for n in (100, 200, 400) if axis == 0 else (100, 200):
        x, rho, u, pr = _sod(orc, n, axis, tvd_form=1, ndim=ndim)
        sel = x >= 1.0
        re, ue, pe, _, _ = riemann_exact(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, (x[sel] - 1.5) / 0.2)
        errs.append(np.abs(rho[sel] - re).mean())
        tv = np.abs(np.diff(np.r_[rho, rho[0]])).sum()
        assert rho.max() <= 1.0 * (1 + 1e-3) and rho.min() >= 0.125 * (1 - 1e-3)
        assert tv <= 1.01 * (2 * 0.875)
        # mirrored tube: the initial data are symmetric under i -> n-1-i, the solution nearly so
        assert np.abs(rho - rho[::-1]).mean() < 2e-3
        assert np.abs(u[sel] - ue).mean() < 4 * errs[-1] + 1e-3 and np.abs(pr[sel] - pe).mean() < 2 * errs[-1]
    for a, b in zip(errs, errs[1:]):
        assert 1.6 < a / b < 2.6, errs
    assert errs[0] < 0.02


def test_tvd_form_decision(orc):
    """DESIGN.md R4: Eq. 34 as printed (G of the sum r+ + r-) lets the total variation of the Sod
    density grow by ~75 %, the Davis/Yee form (sum of two G's) keeps it non-increasing; this is why
    tvd_form = 1 is the default."""
    tv0 = 2 * 0.875
    _, rho0, _, _ = _sod(orc, 200, 0, tvd_form=0)
    _, rho1, _, _ = _sod(orc, 200, 0, tvd_form=1)
    tv = lambda r: np.abs(np.diff(np.r_[r, r[0]])).sum()
    assert tv(rho1) <= 1.001 * tv0
    assert tv(rho0) > 1.3 * tv0
    assert inputs.make_params()["tvd_form"] == 1


def test_courant_number_reading_decision(orc):
    """DESIGN.md R5: with the acoustic Courant number (co_mode 0) the Sod density stays free of oscillations (total
    variation non-increasing); with the advective one (co_mode 1) the TVD coefficient is too small at the shock and the
    total variation grows by a few per cent.  This is why co_mode = 0 is the default although the low-Mach validation
    runs need co_mode = 1."""
    tv0 = 2 * 0.875
    tv = lambda r: np.abs(np.diff(np.r_[r, r[0]])).sum()
    _, rho_a, _, _ = _sod(orc, 200, 0, tvd_form=1, co_mode=0)
    _, rho_u, _, _ = _sod(orc, 200, 0, tvd_form=1, co_mode=1)
    assert tv(rho_a) <= 1.001 * tv0
    assert 1.01 * tv0 < tv(rho_u) < 1.10 * tv0
    assert inputs.make_params()["co_mode"] == 0


# ----------------------------------------------------------------------------- check 4: convergence
def _density_wave_error(orc, n, ndim, oblique, tvd_off, t_end=0.4):
    gam = 1.4
    ny = n if (ndim == 3) else 1
    nz = n if oblique else 4
    g = periodic_grid(ndim, n, nz, ny, lx=1.0, ly=1.0, lz=1.0 if oblique else 4.0 / n)
    p = ideal_gas_params(gamma=gam, tvd_off=tvd_off, cfl=0.4)
    x = (np.arange(n) / n)[None, None, :]
    y = (np.arange(ny) / ny)[None, :, None]
    z = (np.arange(nz) / nz)[:, None, None]
    u = (1.0, 0.5 if ndim == 3 else 0.0, 0.75 if oblique else 0.0)
    kz, ky = (1 if oblique else 0), (1 if ndim == 3 else 0)
    phase = lambda t: 2 * np.pi * ((x - u[0] * t) + ky * (y - u[1] * t) + kz * (z - u[2] * t))
    rho0 = 1.0 + 0.2 * np.sin(phase(0.0))
    X = state_from_primitives(g, p, rho0, u[0], u[1], u[2], 1.0)
    X, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    rho = X[0].reshape(nz, ny, n)
    exact = 1.0 + 0.2 * np.sin(phase(t_end)) + 0 * rho
    return np.abs(rho - exact).mean()


@pytest.mark.parametrize("ndim,oblique", [(2, False), (2, True), (3, True)])
def test_second_order_convergence_density_wave(orc, ndim, oblique):
    """Smooth advected density wave, dt ~ dx: L1 error ratio per doubling ~4 without the TVD term
    and >= 3.6 with it (the limiter clips extrema) (BASELINE check 4).  The oblique
    cases exercise the operator splitting of Eq. 30."""
    sizes = (16, 32) if ndim == 3 else (32, 64)
    e_off = [_density_wave_error(orc, n, ndim, oblique, tvd_off=1) for n in sizes]
    assert 3.7 < e_off[0] / e_off[1] < 4.4, e_off
    if ndim == 2:
        sizes = (64, 128)
        e_on = [_density_wave_error(orc, n, ndim, oblique, tvd_off=0) for n in sizes]
        assert e_on[0] / e_on[1] > 3.0, e_on
        assert e_on[1] < 2e-3


# ----------------------------------------------------------------------------- check 5: mirror
def _mirror(X, grid, axis):
    nf = X.shape[0]
    F = X.reshape(nf, grid["nz"], grid["ny"], grid["nx"]).copy()
    ax = {0: 3, 1: 2, 2: 1}[axis]
    F = np.roll(np.flip(F, axis=ax), 1, axis=ax)          # i -> (n - i) mod n
    mom = {0: 1, 1: 2, 2: nf - 2}[axis]
    F[mom] = -F[mom]
    return F.reshape(nf, -1)


@pytest.mark.parametrize("ndim", [2, 3])
def test_mirror_identity(orc, ndim):
    """mirror(L_alpha^{dir}(X)) == L_alpha^{-dir}(mirror X) and, across the sweep,
    mirror_beta(L_alpha^{dir}(X)) == L_alpha^{dir}(mirror_beta X): the forward/backward pair is the
    exact mirror image of the backward/forward pair (BASELINE check 5a, R9)."""
    g = periodic_grid(ndim, 16, 12, 10 if ndim == 3 else 1)
    p = ideal_gas_params(mu_override=4e-3, K_override=6e-3)
    X = inputs.smooth_random_state(g, p, seed=11)
    prob = orc.Problem(g, p)
    axes = (0, 2) if ndim == 2 else (0, 1, 2)
    for a in axes:
        for m in axes:
            for d in (+1, -1):
                lhs = _mirror(orc.sweep(prob, X, a, 0.01, d), g, m)
                rhs = orc.sweep(prob, _mirror(X, g, m), a, 0.01, -d if m == a else d)
                assert np.max(rel_err(lhs, rhs)) < 5e-16, (a, m, d)


def test_symmetric_state_asymmetry_shrinks(orc):
    """A left-right symmetric state stays symmetric up to truncation error, which falls at second
    order (BASELINE check 5b)."""
    asym = []
    for n in (32, 64):
        g = periodic_grid(2, n, n)
        p = ideal_gas_params(tvd_off=1, cfl=0.4)
        x = (np.arange(n) / n)[None, None, :]
        z = (np.arange(n) / n)[:, None, None]
        rho = 1.0 + 0.2 * np.cos(2 * np.pi * x) * (1 + 0.5 * np.sin(2 * np.pi * z))
        ux = 0.3 * np.sin(2 * np.pi * x)
        uz = 0.2 * np.cos(2 * np.pi * x) * np.sin(2 * np.pi * z)
        X = state_from_primitives(g, p, rho, ux, 0.0, uz, 1.0 + 0 * rho)
        assert np.allclose(_mirror(X, g, 0), X, rtol=0, atol=1e-15)
        X = 0.5 * (X + _mirror(X, g, 0))                       # exactly symmetric
        Y, _ = advance_to(orc, orc.Problem(g, inputs.make_params(**{**p, "dir_mode": 0})), X, 0.1)
        asym.append(np.abs(_mirror(Y, g, 0) - Y)[0].max())
    assert asym[0] / asym[1] > 3.0 and asym[1] < 1e-3, asym


# ----------------------------------------------------------------------------- viscous terms
def _shear_decay(orc, n, plane, tvd_off=1, drop=None, t_end=0.4, nu=0.01):
    """Oblique, divergence-free shear wave u = A t sin(k.x) (t perpendicular to k) in a uniform
    low-Mach gas: the amplitude decays as exp(-nu |k|^2 t) exactly when tau_ij carries both
    d_j u_i and d_i u_j.  `plane` picks the two axes spanning k."""
    a1, a2 = plane
    ndim = 2 if 1 not in plane else 3
    dims = {0: n, 1: n, 2: n}
    for a in (0, 1, 2):
        if a not in plane:
            dims[a] = 4 if ndim == 3 else 1
    if ndim == 2:
        dims[1] = 1
    g = periodic_grid(ndim, dims[0], dims[2], dims[1], lx=1.0 if 0 in plane else 4.0 / n,
                      ly=1.0 if 1 in plane else 4.0 / n, lz=1.0 if 2 in plane else 4.0 / n)
    gam = 1.4
    p = ideal_gas_params(gamma=gam, mu_override=nu, tvd_off=tvd_off, cfl=0.5)
    coords = [(np.arange(dims[0]) / dims[0])[None, None, :], (np.arange(dims[1]) / dims[1])[None, :, None],
              (np.arange(dims[2]) / dims[2])[:, None, None]]
    theta = 2 * np.pi * (coords[a1] + coords[a2])
    A = 0.02
    u = [0.0, 0.0, 0.0]
    u[a1] = A / np.sqrt(2) * np.sin(theta)
    u[a2] = -A / np.sqrt(2) * np.sin(theta)
    X = state_from_primitives(g, p, 1.0, u[0], u[1], u[2], 1.0 / gam)      # c_s = 1
    X, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    prim = primitives_of(g, p, X)
    amp = 2 * np.mean((prim[1 + a1] - prim[1 + a2]) / np.sqrt(2) * np.sin(theta + 0 * prim[0]))
    return amp / A, np.exp(-nu * 8 * np.pi**2 * t_end)


@pytest.mark.parametrize("plane", [(0, 2), (0, 1), (1, 2)])
def test_oblique_shear_wave_decay_rate(orc, plane):
    """Pins mu = sqrt(Pr/Ra)'s role and both halves of tau_ij = mu(d_j u_i + d_i u_j) (Eq. 18):
    without the cross-derivative half the wave would decay 1.5x faster, with the wrong sign 2x."""
    got, want = _shear_decay(orc, 48, plane)
    assert got == pytest.approx(want, rel=6e-3), (got, want)
    assert abs(np.log(got) / np.log(want) - 1.0) < 0.02
    got_tvd, _ = _shear_decay(orc, 48, plane, tvd_off=0)
    assert got_tvd == pytest.approx(want, rel=0.05)


@pytest.mark.parametrize("lam", [-2.0 / 3.0, 2.0 / 3.0])
def test_acoustic_attenuation_pins_dilatation_coefficient(orc, lam):
    """A standing sound wave in a viscous, non-conducting gas loses acoustic energy as
    exp(-(2 + lambda) nu k^2 t) (classical absorption, tau_xx = mu (2 + lambda) d_x u_x)."""
    n, nu, gam, A = 64, 0.005, 1.4, 1e-3
    g = periodic_grid(2, n, 4, lz=4.0 / n)
    p = ideal_gas_params(gamma=gam, mu_override=nu, lambda_coef=lam, tvd_off=1)
    x = (np.arange(n) / n)[None, None, :]
    X = state_from_primitives(g, p, 1.0, A * np.sin(2 * np.pi * x), 0.0, 0.0, 1.0 / gam)

    def energy(Y):
        rho, ux, _, _, _, pr = primitives_of(g, p, Y)
        return np.mean(0.5 * rho * ux**2 + (pr - 1.0 / gam) ** 2 / 2.0)     # rho0 c^2 = 1

    t_end = 2.0
    Y, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    rate = np.log(energy(X) / energy(Y)) / t_end
    assert rate == pytest.approx((2.0 + lam) * nu * (2 * np.pi) ** 2, rel=0.03)


def test_thermal_diffusion_rate_pins_K(orc):
    """Isobaric temperature ripple in a gas at rest decays at K k^2/(rho c_p), c_p = gamma c_v:
    pins the -K dT/dx term of the energy flux (Eq. 15) and c_v of Eq. 17."""
    n, K, gam, a = 64, 0.02, 1.4, 1e-3
    g = periodic_grid(2, n, 4, lz=4.0 / n)
    p = ideal_gas_params(gamma=gam, K_override=K, tvd_off=1)
    x = (np.arange(n) / n)[None, None, :]
    T0 = 1.0 / (gam * (gam - 1.0))                                          # c_s = 1 with R = gam-1
    T = T0 * (1 + a * np.sin(2 * np.pi * x))
    pr = 1.0 / gam
    X = state_from_primitives(g, p, pr / ((gam - 1.0) * T), 0.0, 0.0, 0.0, pr)
    t_end = 1.0
    Y, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    Tn = primitives_of(g, p, Y)[4]
    amp = 2 * np.mean((Tn / T0 - 1) * np.sin(2 * np.pi * x + 0 * Tn)) / a
    kappa = K / (1.0 * gam * 1.0)                                           # rho0 = 1, c_v = 1
    assert amp == pytest.approx(np.exp(-kappa * (2 * np.pi) ** 2 * t_end), rel=0.02)


def test_viscous_heating_pattern_pins_work_term(orc):
    """Shear u_x = A sin(kz) heats the gas where the shear is largest: the early temperature rise
    is mu A^2 k^2 cos^2(kz) t/(rho c_v), i.e. a positive cos(2kz) coefficient.  Without the
    u_j tau_ij term of the energy flux (Eq. 15) that coefficient would be negative."""
    n, nu, gam, A = 64, 0.02, 1.4, 0.05
    g = periodic_grid(2, 4, n, lx=4.0 / n)
    p = ideal_gas_params(gamma=gam, mu_override=nu, tvd_off=1)
    z = (np.arange(n) / n)[:, None, None]
    k = 2 * np.pi
    X = state_from_primitives(g, p, 1.0, A * np.sin(k * z), 0.0, 0.0, 1.0 / gam)
    T0 = primitives_of(g, p, X)[4]
    t_end = 0.03                                                           # << acoustic time 0.5
    Y, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    dT = primitives_of(g, p, Y)[4] - T0
    c2 = 2 * np.mean(dT * np.cos(2 * k * z + 0 * dT))
    want = nu * A**2 * k**2 * t_end / 2.0                                   # rho = c_v = 1
    assert 0.7 * want < c2 < 1.1 * want, (c2, want)


# ----------------------------------------------------------------------------- TVD coefficient (Eqs. 34-39)
@pytest.mark.parametrize("tvd_form", [0, 1])
@pytest.mark.parametrize("axis", [0, 2])
def test_stationary_contact_pins_tvd_coefficient(orc, tvd_form, axis):
    """A contact at rest: u = 0, uniform p, one isolated density jump (mu = K = g = 0).  The flux F_alpha is
    then uniform, so every MacCormack difference of Eqs. 31-32 is exactly zero and one operator returns X + T
    (Eq. 33).  At an isolated jump dX_{k+1/2} = (drho, 0, 0, 0) with zero neighbours, so r+_k = r-_{k+1} = 0
    (Eq. 37), phi = 0 and Eq. 34 moves exactly
        +-[G_k + G_{k+1}] drho = +-(1/2)[C(Co_k) + C(Co_{k+1})] drho        (Davis/Yee sum, tvd_form 1)
        +-(1/2) mean(C_k, C_{k+1}) drho                                     (Eq. 34 as printed, tvd_form 0, R6)
    of density across the jump and nothing anywhere else, with Co = c_s tau/dx (R5: u = 0 here) and
    C = Co (1 - Co) for Co <= 0.5, else 0.25 (Eq. 39).  tau is chosen on both branches of
    Eq. 39 and straddling them.  Pins the 1/2 of Eq. 38, Eq. 39, and R5's tau and c_s."""
    gam, p0, rl, rr = 1.4, 1.0, 1.0, 0.25
    n, h = 16, 0.1
    cl, cr = np.sqrt(gam * p0 / rl), np.sqrt(gam * p0 / rr)          # c_s = sqrt(gamma p / rho) on either side
    C = lambda Co: Co * (1.0 - Co) if Co <= 0.5 else 0.25            # Eq. 39
    for tau in (0.01, 0.03, 0.06):                                   # Co = (0.12, 0.24), (0.35, 0.71), (0.71, 1.42)
        if axis == 0:
            g = periodic_grid(2, n, 6, lx=n * h, lz=0.6)
            shape = (1, 1, n)
        else:
            g = periodic_grid(2, 6, n, lx=0.6, lz=n * h)
            shape = (n, 1, 1)
        p = ideal_gas_params(gamma=gam, tvd_form=tvd_form)
        i = np.arange(n)
        heavy = (i >= 4) & (i < 11)                                  # jumps at 3|4 and 10|11
        X = state_from_primitives(g, p, np.where(heavy, rl, rr).reshape(shape), 0.0, 0.0, 0.0, p0)
        for direction in (+1, -1):
            Y = orc.sweep(orc.Problem(g, p), X, axis, tau, direction)
            d = (Y - X).reshape(4, g["nz"], g["nx"])
            assert np.all(d[1:] == 0.0)                              # momenta and E untouched, bit for bit
            line = d[0][:, 2] if axis == 2 else d[0][2, :]
            Cl, Cr = C(cl * tau / h), C(cr * tau / h)
            amount = (0.5 * (Cl + Cr) if tvd_form == 1 else 0.25 * (Cl + Cr)) * (rl - rr)
            want = np.zeros(n)
            want[3], want[4], want[10], want[11] = +amount, -amount, -amount, +amount
            np.testing.assert_allclose(line, want, rtol=0, atol=2e-16)
    # both nodes beyond Co = 0.5: C = 0.25 exactly, so a quarter (an eighth) of the jump crosses
    assert amount == (0.25 if tvd_form == 1 else 0.125) * (rl - rr)


@pytest.mark.parametrize("tvd_form", [0, 1])
@pytest.mark.parametrize("axis", [0, 2])
def test_advective_courant_number_in_the_tvd_coefficient(orc, tvd_form, axis):
    """co_mode = 1, the second reading of the "local Courant number" of Eq. 39 (R5): Co = |u_alpha| tau/dx.
    (a) A contact at rest has Co = 0, C = 0: one operator returns X bit for bit (with co_mode = 0 it does not).
    (b) A contact carried by a uniform flow u along the axis (uniform p, mu = K = g = 0): the TVD term is additive in
    Eq. 33 and computed from X^n alone, so sweep(TVD on) - sweep(TVD off) = T.  At an isolated jump dX_{k+1/2} =
    drho (1, u, u^2/2) in (rho, rho u, E) with zero neighbours, r+- = 0, phi = 0, and Co is the SAME number |u| tau/dx
    at every node, so T = +-C(Co) dX (Davis/Yee sum) or +-C(Co)/2 dX (Eq. 34 as printed), on both branches of Eq. 39."""
    gam, p0, rl, rr = 1.4, 1.0, 1.0, 0.25
    n, h = 16, 0.1
    C = lambda Co: Co * (1.0 - Co) if Co <= 0.5 else 0.25
    if axis == 0:
        g, shape = periodic_grid(2, n, 6, lx=n * h, lz=0.6), (1, 1, n)
    else:
        g, shape = periodic_grid(2, 6, n, lx=0.6, lz=n * h), (n, 1, 1)
    i = np.arange(n)
    heavy = (i >= 4) & (i < 11)
    rho = np.where(heavy, rl, rr).reshape(shape)
    p1 = ideal_gas_params(gamma=gam, tvd_form=tvd_form, co_mode=1)
    X = state_from_primitives(g, p1, rho, 0.0, 0.0, 0.0, p0)
    for direction in (+1, -1):
        assert np.array_equal(orc.sweep(orc.Problem(g, p1), X, axis, 0.03, direction), X)
        p0m = ideal_gas_params(gamma=gam, tvd_form=tvd_form, co_mode=0)
        assert not np.array_equal(orc.sweep(orc.Problem(g, p0m), X, axis, 0.03, direction), X)
    for u, tau in ((0.8, 0.02), (-0.8, 0.02), (2.0, 0.04)):          # Co = 0.16, 0.16, 0.8
        ux, uz = (u, 0.0) if axis == 0 else (0.0, u)
        X = state_from_primitives(g, p1, rho, ux, 0.0, uz, p0)
        off = ideal_gas_params(gamma=gam, tvd_off=1)
        for direction in (+1, -1):
            T = (orc.sweep(orc.Problem(g, p1), X, axis, tau, direction)
                 - orc.sweep(orc.Problem(g, off), X, axis, tau, direction)).reshape(4, g["nz"], g["nx"])
            coef = C(abs(u) * tau / h) * (1.0 if tvd_form == 1 else 0.5)
            dX = (rl - rr) * np.array([1.0, ux, uz, 0.5 * u * u])    # the jump in (rho, rho u_x, rho u_z, E) at fixed p
            for f in range(4):
                line = T[f][:, 2] if axis == 2 else T[f][2, :]
                want = np.zeros(n)
                want[3], want[4], want[10], want[11] = +coef * dX[f], -coef * dX[f], -coef * dX[f], +coef * dX[f]
                np.testing.assert_allclose(line, want, rtol=0, atol=5e-16 * max(1.0, abs(u)) ** 2)


def test_contact_next_to_a_plate_records_R11(orc):
    """DESIGN.md R11 (the paper is silent): the dissipation flux of Eq. 34 is dropped on the two interfaces
    that touch a plate node, whose r+- would need a node outside the box.  A contact at rest sitting on the
    plate-adjacent interface therefore stays put bit for bit, while the same contact one interface further in
    is smoothed.  This records the reading; nothing in the paper pins it."""
    gam, p0 = 1.4, 1.0
    nz = 12
    for k_jump, moves in ((0, False), (1, True), (nz - 2, False), (nz - 3, True)):
        rho = np.where(np.arange(nz) <= k_jump, 1.0, 0.25)
        g = inputs.make_grid(2, 6, nz, lx=0.6, lz=1.1)
        # plates at the local gas temperature T = p / (R rho), R = gamma - 1 in these units
        p = ideal_gas_params(gamma=gam, bc_z=0, T_bot=p0 / ((gam - 1) * rho[0]), T_top=p0 / ((gam - 1) * rho[-1]))
        X = state_from_primitives(g, p, rho[:, None, None], 0.0, 0.0, 0.0, p0)
        for direction in (+1, -1):
            Y = orc.sweep(orc.Problem(g, p), X, 2, 0.01, direction)
            assert np.allclose(Y[1:], X[1:], rtol=0, atol=1e-15)
            assert np.array_equal(Y[0], X[0]) != moves, (k_jump, direction)


# ----------------------------------------------------------------------------- second order in time (Eq. 32's S^P)
_TAYLOR = {}


def _euler_gravity_taylor(gam, g):
    """X, X_t and X_tt of the 1-D inviscid equations with gravity (Eqs. 13-15 along z, PAPER.md:181-185:
    rho_t = -(rho w)_z;  (rho w)_t = -(rho w^2 + p)_z - g rho;  E_t = -(w (E + p))_z with
    E = rho w^2/2 + p/(gamma-1) + rho g z) for the smooth state below, derived symbolically (sympy) from
    the PDE itself -- nothing of the scheme enters."""
    if (gam, g) in _TAYLOR:
        return _TAYLOR[(gam, g)]
    import sympy as sp
    z, s = sp.symbols("z s")
    k = 2 * sp.pi
    G, gg = sp.Float(gam), sp.Float(g)
    rho = 1 + sp.Rational(1, 5) * sp.sin(k * z)
    w = sp.Rational(3, 10) * sp.sin(k * z + 1)
    pr = 1 + sp.Rational(1, 10) * sp.cos(k * z)
    X = (rho, rho * w, rho * w * w / 2 + pr / (G - 1) + rho * gg * z)

    def rhs(r, m, E):
        u = m / r
        p = (G - 1) * (E - m * u / 2 - r * gg * z)
        return (-sp.diff(m, z), -sp.diff(m * u + p, z) - gg * r, -sp.diff(u * (E + p), z))

    Xt = rhs(*X)
    Xtt = [sp.diff(c, s).subs(s, 0) for c in rhs(*[a + s * b for a, b in zip(X, Xt)])]
    out = tuple([sp.lambdify(z, e, "numpy") for e in grp] for grp in (X, Xt, Xtt))
    _TAYLOR[(gam, g)] = out
    return out


@pytest.mark.parametrize("direction", [+1, -1])
def test_one_operator_is_second_order_in_time_with_gravity(orc, direction):
    """the scheme is second order in space AND time.  One operator L_z(tau) applied to a smooth
    state with gravity must then reproduce X + tau X_t + tau^2 X_tt / 2 of the PDE up to O(h^3) when tau ~ dz = h,
    i.e. the local error falls 8x per halving.  The g tau^2 (rho w)_z / 2 part of X_tt only appears if the
    corrector's source is taken at the predicted state (S^P_k in Eq. 32); with S(X^n) the local
    error of rho w is O(h^2) and falls 4x.  (z is periodic here; gravity makes the periodic seam inconsistent,
    so nodes within 4 of it are left out: one operator reaches 2 nodes.)"""
    gam, g = 1.4, 10.0
    f0, ft, ftt = _euler_gravity_taylor(gam, g)
    errs = []
    for n in (32, 64, 128):
        grid = periodic_grid(2, 4, n, lx=4.0 / n, lz=1.0)
        p = ideal_gas_params(gamma=gam, g_override=g, tvd_off=1)
        zz = np.arange(n) / n
        tau = 0.2 / n
        cols = lambda f: np.repeat(np.asarray(f(zz), dtype=float)[:, None], 4, 1).reshape(-1)
        X0 = np.stack([cols(f0[0]), np.zeros(4 * n), cols(f0[1]), cols(f0[2])])
        Y = orc.sweep(orc.Problem(grid, p), X0, 2, tau, direction).reshape(4, n, 4)[:, :, 0]
        sel = slice(4, n - 4)
        e = []
        for i, f in ((0, 0), (1, 2)):                                # rho and rho w
            exact = f0[i](zz) + tau * ft[i](zz) + 0.5 * tau**2 * ftt[i](zz)
            e.append(np.abs(Y[f][sel] - exact[sel]).max())
        errs.append(e)
    errs = np.array(errs)
    ratios = errs[:-1] / errs[1:]
    assert np.all(ratios > 7.0) and np.all(ratios < 9.0), (errs, ratios)
    assert errs[0, 1] < 3e-4


# ----------------------------------------------------------------------------- R7: compact viscous stencil
@pytest.mark.parametrize("a,b", [(0, 2), (2, 0)])
def test_aligned_shear_wave_decays_at_the_compact_stencil_rate(orc, a, b):
    """R7: inside F_alpha the derivative along alpha is one-sided, OPPOSITE to the stage's outer difference, so
    that predictor and corrector each form the compact second difference (f_{k+1} - 2 f_k + f_{k-1})/h^2.  A
    grid-aligned shear wave u_a = A sin(k x_b) in a gas at rest then decays at exactly nu (2 - 2 cos(k h))/h^2
    (the symbol of that stencil; time-stepping error ~1e-5 here).  The same-side rule would give the wide
    stencil (f_{k+2} - 2 f_k + f_{k-2})/(2h)^2-like average, whose rate is smaller by cos(k h): 7.6 % at
    n = 16."""
    gam, nu, A, n, t_end = 1.4, 0.02, 1e-3, 16, 1.0
    dims = {0: 4, 2: 4}
    dims[b] = n
    g = periodic_grid(2, dims[0], dims[2], lx=1.0 if b == 0 else 4.0 / n, lz=1.0 if b == 2 else 4.0 / n)
    p = ideal_gas_params(gamma=gam, mu_override=nu, tvd_off=1, cfl=0.25)
    x = (np.arange(dims[0]) / dims[0])[None, None, :]
    z = (np.arange(dims[2]) / dims[2])[:, None, None]
    s = x if b == 0 else z
    k, h = 2 * np.pi, 1.0 / n
    u = [0.0, 0.0, 0.0]
    u[a] = A * np.sin(k * s)
    X = state_from_primitives(g, p, 1.0, u[0], 0.0, u[2], 1.0 / gam)
    X, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
    ua = primitives_of(g, p, X)[1 + a]
    rate = -np.log(2 * np.mean(ua * np.sin(k * s + 0 * ua)) / A) / t_end
    compact = nu * (2 - 2 * np.cos(k * h)) / h**2
    assert rate == pytest.approx(compact, rel=1e-4), (rate, compact, compact * np.cos(k * h))
    assert abs(rate / (nu * k * k) - 1) < 0.02                       # and it approximates nu k^2


# ----------------------------------------------------------------------------- Eq. 30: the operator sequence
@pytest.mark.parametrize("ndim", [2, 3])
def test_step_is_the_operator_sequence_of_eq30(orc, ndim):
    """Eq. 30: X^(n+1) = L_x L_y L_z L_x L_y L_z X^n, each with dt/2, operators acting right
    to left (no L_y in 2-D).  With R9's alternation the list, in the order of application, is
        L_z(+1), [L_y(+1),] L_x(+1), L_z(-1), [L_y(-1),] L_x(-1),  each with tau = dt/2.
    One step must equal that list of single operators bit for bit, and must differ from the x-first order
    (R8: the operators do not commute on a generic state)."""
    g = inputs.make_grid(ndim, 12, 9, 8 if ndim == 3 else 1)
    p = inputs.make_params(Ra=1e3)
    X = inputs.smooth_random_state(g, p, seed=17)
    prob = orc.Problem(g, p)
    dt = 0.8 * orc.dt(prob, X)
    tau = 0.5 * dt
    z, y, x = 2, 1, 0
    sequence = [(z, +1), (y, +1), (x, +1), (z, -1), (y, -1), (x, -1)]
    if ndim == 2:
        sequence = [(a, d) for a, d in sequence if a != y]
    Y = X
    for alpha, direction in sequence:
        Y = orc.sweep(prob, Y, alpha, tau, direction)
    got, dts, t = orc.step(prob, X, 1, dt_in=[dt])
    assert np.array_equal(got, Y)
    assert dts[0] == dt and t == dt
    W = X
    for alpha, direction in [(a, d) for d in (+1, -1) for a in ((x, z) if ndim == 2 else (x, y, z))]:
        W = orc.sweep(prob, W, alpha, tau, direction)
    assert np.max(rel_err(W, Y)) > 1e-9
    # dir_mode 0 (the paper's fixed backward predictor): both triples with dir = +1
    p0 = inputs.make_params(Ra=1e3, dir_mode=0)
    prob0 = orc.Problem(g, p0)
    Y0 = X
    for alpha, _ in sequence:
        Y0 = orc.sweep(prob0, Y0, alpha, tau, +1)
    assert np.array_equal(orc.step(prob0, X, 1, dt_in=[dt])[0], Y0)


# ----------------------------------------------------------------------------- gravity, plates
def test_hydrostatic_conduction_state_drift_is_second_order(orc):
    """The noise-free conduction state is a steady solution of Eqs. 13-15 (linear T: constant heat
    flux; hydrostatic p).  The discrete drift is truncation error only: small and ~4x smaller per
    grid doubling.  Pins the -rho/eps source (Eq. 14), the z/eps term of E (Eq. 17) and the plate
    treatment."""
    drift = []
    for nz in (33, 65, 129):
        g = inputs.make_grid(2, 8, nz, lx=8.0 / (nz - 1))
        p = inputs.make_params(Ra=1e4)
        X = inputs.conduction_state(g, p, amplitude=0.0)
        Y, _ = advance_to(orc, orc.Problem(g, p), X, 0.05)
        drift.append(np.abs(primitives_of(g, p, Y)[3]).max())
    assert drift[0] < 2e-4
    assert drift[0] / drift[1] > 3.3 and drift[1] / drift[2] > 3.3, drift


def test_discrete_hydrostatic_density_is_polytrope():
    """Input recipe: the hydrostatic polytrope of a linear T is rho = T^m with
    m = gamma D/((gamma-1)(eps+D)) - 1 (from Eqs. 14, 16).  For the configs (gamma = 5/3, eps = 0.1,
    D = 0.4) m = 1 and the trapezoid recursion is exact; for gamma = 1.4 (m = 1.8) it converges at
    second order."""
    for gam, m in ((5.0 / 3.0, 1.0), (1.4, 1.8)):
        err = []
        for nz in (33, 65):
            g = inputs.make_grid(2, 4, nz)
            p = inputs.make_params(gamma=gam)
            X = inputs.conduction_state(g, p, amplitude=0.0)
            rho = X[0].reshape(nz, 4)[:, 0]
            err.append(np.abs(rho - (1 - 0.5 * inputs.z_nodes(g, p)) ** m).max())
        if m == 1.0:
            assert max(err) < 1e-14
        else:
            assert err[1] < 1e-4 and 3.5 < err[0] / err[1] < 4.5, err


def test_plate_values_hold(orc):
    """No-slip, isothermal plates: after any number of steps the plate nodes
    carry zero momentum and exactly the plate temperatures."""
    g = inputs.make_grid(2, 32, 17)
    p = inputs.make_params(Ra=1e5)
    X = inputs.smooth_random_state(g, p, seed=3)
    Y, _, _ = orc.step(orc.Problem(g, p), X, 8)
    rho, ux, _, uz, T, _ = primitives_of(g, p, Y)
    for k, Tw in ((0, p["T_bot"]), (-1, p["T_top"])):
        assert np.all(ux[k] == 0) and np.all(uz[k] == 0)
        assert np.allclose(T[k], Tw, rtol=1e-13, atol=0)
    assert rho.min() > 0


# ----------------------------------------------------------------------------- diagnostics
def test_diagnostics_closed_forms(orc):
    """Conduction state: T_sa = -eps z so Nu_0 = Nu_1 = Nu_bulk = 1 and Re = 0 (Eqs. 22-26)."""
    g, p, _ = inputs.config("C1")
    prob = orc.Problem(g, p)
    X = inputs.conduction_state(g, p, amplitude=0.0)
    d, Tp, rp, pp = orc.diagnostics(prob, X)
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk"):
        assert d[k] == pytest.approx(1.0, abs=1e-11), k
    assert d["re"] == 0.0 and d["u_rms"] == 0.0 and d["nu_conv"] == 0.0 and d["nu_K"] == 0.0
    z = inputs.z_nodes(g, p)
    assert np.allclose(Tp, 1 - 0.5 * z, rtol=1e-13)
    assert np.allclose(pp, 10.0 * rp * Tp, rtol=1e-13)
    assert d["min_T"] == pytest.approx(0.5, rel=1e-13) and d["max_mach"] == 0.0


def test_diagnostics_synthetic_flow(orc):
    """Uniform rho, constant u_z = a, T = T_A + b + c z^2: every mean of Eqs. 22-26 has a closed
    form, and the 2nd-order one-sided plate gradients are exact for a quadratic."""
    g = inputs.make_grid(3, 6, 21, 5)
    p = inputs.make_params(Ra=1e4, Pr=0.7)
    a, b, c = 0.03, 0.05, -0.2
    z = inputs.z_nodes(g, p)[:, None, None]
    T = (1 - p["D"] * z) + b + c * z**2 + np.zeros((21, 5, 6))
    X = inputs.pack(g, np.full_like(T, 1.25), 0 * T, 0 * T, a + 0 * T, T, p)
    d, Tp, rp, pp = orc.diagnostics(orc.Problem(g, p), X)
    sRaPr = np.sqrt(p["Ra"] * p["Pr"])
    zz = z.ravel()
    w = np.full(21, zz[1]); w[0] = w[-1] = zz[1] / 2
    mean_tsa = np.sum(w * (b + c * zz**2)) / np.sum(w)
    assert d["nu_conv"] == pytest.approx(sRaPr / p["eps"] * 1.25 * a * mean_tsa, rel=1e-12)
    assert d["nu_K"] == pytest.approx(p["D"] * sRaPr / 2 * 1.25 * a**3, rel=1e-12)
    assert d["nu_bulk"] == pytest.approx(1 + d["nu_conv"] + d["nu_K"], rel=1e-15)
    assert d["re"] == pytest.approx(np.sqrt(p["Ra"] / p["Pr"]) * a, rel=1e-12)
    assert d["nu_bottom"] == pytest.approx(0.0, abs=1e-11)
    assert d["nu_top"] == pytest.approx(-2 * c / p["eps"], rel=1e-10)
    assert d["nu_bar"] == pytest.approx(0.5 * (d["nu_bottom"] + d["nu_top"]), rel=1e-15)
    assert d["mass"] == pytest.approx(1.25 * 16.0, rel=1e-13)
    assert d["mom_z"] == pytest.approx(1.25 * a * 16.0, rel=1e-13)
    assert np.allclose(rp, 1.25) and np.allclose(Tp, T[:, 0, 0], rtol=1e-14)


def test_dt_rule(orc):
    """R12: dt = cfl / max((|u_a| + c_s)/dx_a); closed form on a uniform state; NaN on bad data."""
    g = periodic_grid(3, 8, 6, 4, lx=2.0, ly=1.0, lz=3.0)
    p = ideal_gas_params(gamma=1.4, cfl=0.5)
    X = state_from_primitives(g, p, 2.0, 0.3, -0.7, 0.1, 2.0 / 1.4)      # c_s = 1
    prob = orc.Problem(g, p)
    want = 0.5 / max(1.3 / (2.0 / 8), 1.7 / (1.0 / 4), 1.1 / (3.0 / 6))
    assert orc.dt(prob, X) == pytest.approx(want, rel=1e-14)
    p2 = ideal_gas_params(gamma=1.4, fixed_dt=1e-3)
    assert orc.dt(orc.Problem(g, p2), X) == 1e-3
    X[0, 5] = -1.0
    assert np.isnan(orc.max_speed(prob, X))


# ----------------------------------------------------------------------------- axis permutations
def test_2d_is_3d_with_ny1_and_y_invariance(orc):
    """A 3-D run of a y-invariant state equals the 2-D run copied along y, bit for bit: every
    y-difference is an exact zero, so L_y is the identity there."""
    g2 = inputs.make_grid(2, 16, 13)
    p = inputs.make_params(Ra=1e4)
    X2 = inputs.smooth_random_state(g2, p, seed=5)
    g3 = inputs.make_grid(3, 16, 13, 4, ly=4 * 4.0 / 16)
    F2 = X2.reshape(4, 13, 1, 16)
    X3 = np.stack([np.repeat(F2[0], 4, 1), np.repeat(F2[1], 4, 1), np.zeros((13, 4, 16)),
                   np.repeat(F2[2], 4, 1), np.repeat(F2[3], 4, 1)]).reshape(5, -1)
    dts = [2e-3] * 3
    Y2, _, _ = orc.step(orc.Problem(g2, p), X2, 3, dt_in=dts)
    Y3, _, _ = orc.step(orc.Problem(g3, p), X3, 3, dt_in=dts)
    G3 = Y3.reshape(5, 13, 4, 16)
    for j in range(4):
        assert np.array_equal(G3[[0, 1, 3, 4], :, j, :].reshape(4, -1), Y2)
    assert np.all(G3[2] == 0)


def _swap_axes(X, grid, a, b):
    """Relabel axes a <-> b of a 3-D state (fields reshaped (nz, ny, nx)); returns (X', grid')."""
    ax = {0: 3, 1: 2, 2: 1}
    F = X.reshape(5, grid["nz"], grid["ny"], grid["nx"]).swapaxes(ax[a], ax[b]).copy()
    F[[1 + a, 1 + b]] = F[[1 + b, 1 + a]]
    n = ["nx", "ny", "nz"]; l = ["lx", "ly", "lz"]
    g = dict(grid)
    g[n[a]], g[n[b]] = grid[n[b]], grid[n[a]]
    g[l[a]], g[l[b]] = grid[l[b]], grid[l[a]]
    return F.reshape(5, -1), g


@pytest.mark.parametrize("a,b", [(0, 1), (0, 2), (1, 2)])
def test_sweeps_are_one_operator_under_axis_relabelling(orc, a, b):
    """L_a on the relabelled state equals the relabelled L_b (all-periodic box, g = 0): the three
    sweeps implement one 1-D operator, so every pin above holds for each of them.  Sums over
    fields and axes change order under the relabelling, hence a few-ulp tolerance."""
    g = periodic_grid(3, 12, 8, 10, lx=1.0, ly=0.9, lz=0.7)
    p = ideal_gas_params(mu_override=4e-3, K_override=6e-3)
    X = inputs.smooth_random_state(g, p, seed=13)
    Xs, gs = _swap_axes(X, g, a, b)
    for d in (+1, -1):
        for sweep_axis in (0, 1, 2):
            mapped = {a: b, b: a}.get(sweep_axis, sweep_axis)
            lhs, _ = _swap_axes(orc.sweep(orc.Problem(g, p), X, sweep_axis, 0.004, d), g, a, b)
            rhs = orc.sweep(orc.Problem(gs, p), Xs, mapped, 0.004, d)
            assert np.max(rel_err(lhs, rhs)) < 1e-14, (sweep_axis, d)


# ----------------------------------------------------------------------------- time averages
def test_time_averages_are_the_weighted_means_of_the_samples(orc):
    """<f>_t = sum_k w_k f_k / sum_k w_k with w_k = t_k - t_{k-1} (time since the previous sample): the twin of
    mc_tvd_step_stats must equal that composition of single steps and instantaneous diagnostics written out
    here, the weights must add up to the elapsed time, and a diagnostic that does not change in time (the plate
    temperature profile of a steady conduction state, Nu = 1) must average to itself."""
    g, p, _ = inputs.config("C1")
    prob = orc.Problem(g, p)
    X0 = inputs.conduction_state(g, p, amplitude=1e-2)
    n, every = 14, 3
    Y, st, Tp, rp, pp = orc.step_stats(prob, X0, n, every)
    X, t, t_last, wsum = X0, 0.0, 0.0, 0.0
    acc = {k: 0.0 for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk", "nu_conv", "nu_K", "re", "u_rms")}
    sq = {"nu_bar": 0.0, "re": 0.0}
    accT = np.zeros(g["nz"])
    for s in range(n):
        X, dts, _ = orc.step(prob, X, 1)
        t += dts[0]
        if (s + 1) % every:
            continue
        d, T_, _, _ = orc.diagnostics(prob, X)
        w = t - t_last
        for k in acc:
            acc[k] += w * d[k]
        for k in sq:
            sq[k] += w * d[k] ** 2
        accT += w * T_
        wsum += w
        t_last = t
    assert np.array_equal(Y, X)
    assert st["samples"] == n // every and st["t_end"] == t_last
    assert st["weight"] == pytest.approx(wsum, rel=1e-15) and st["weight"] == pytest.approx(st["t_end"], rel=1e-14)
    for k in acc:
        assert st[k] == pytest.approx(acc[k] / wsum, rel=1e-14, abs=1e-18), k
    assert st["nu_bar_sq"] == pytest.approx(sq["nu_bar"] / wsum, rel=1e-14)
    assert st["re_sq"] == pytest.approx(sq["re"] / wsum, rel=1e-14)
    np.testing.assert_allclose(Tp, accT / wsum, rtol=1e-14)
    # Eq. 23 is linear in the plane means: the averaged plate Nusselt number is Eq. 23 of the averaged profile
    z = inputs.z_nodes(g, p)
    tsa = Tp - (1.0 - p["D"] * z)
    dz = z[1]
    assert st["nu_bottom"] == pytest.approx(-(-3 * tsa[0] + 4 * tsa[1] - tsa[2]) / (2 * dz) / p["eps"], rel=1e-9)
    # steady conduction state (no noise): every sample is Nu = 1, Re = 0 up to the O(dz^2) drift
    Xs = inputs.conduction_state(g, p, amplitude=0.0)
    _, ss, Ts, _, _ = orc.step_stats(prob, Xs, 6, 2)
    assert ss["nu_bar"] == pytest.approx(1.0, abs=1e-4) and ss["re"] < 1e-2
    np.testing.assert_allclose(Ts, 1 - 0.5 * z, atol=2e-5)           # O(dz^2) drift of the discrete steady state
