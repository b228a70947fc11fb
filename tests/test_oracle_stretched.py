"""Pins of the CPU oracle on the paper's non-uniform z grid ("a non-uniform tangent-hyperbolic grid
in the z-direction"; readings R19 / R20 of DESIGN.md, because the paper prints no formula for it).  No GPU needed.

What fixes the readings: (i) node heights that happen to be uniform must give the uniform-grid scheme back; (ii) the
mass between the plates stays constant to round-off (north_star's conservation check), which holds only if the outer
differences, the plate closure and the TVD term all use the same cell heights; (iii) closed forms of the PDE on the
physical coordinate z -- hydrostatic balance, viscous decay between no-slip plates, the mixed derivative of the
stress -- are approached at second order although the node spacing varies by a factor of five; (iv) the one-sided
plate gradients of Eq. 23 are exact for a quadratic on any spacing."""
import numpy as np
import pytest

from paper_2411_10372_b200 import inputs
from tests.helpers import advance_to, primitives_of, state_from_primitives


def cell_heights(z):
    """The height of the cell each node owns, written from the definition (not from the oracle): half the
    distance between its neighbours, and half the adjacent spacing at a plate node."""
    w = np.empty_like(z)
    w[1:-1] = 0.5 * (z[2:] - z[:-2])
    w[0], w[-1] = 0.5 * (z[1] - z[0]), 0.5 * (z[-1] - z[-2])
    return w


def test_tanh_nodes_recipe():
    z = inputs.tanh_nodes(65, 1.0, 1.5)
    assert z[0] == 0.0 and z[-1] == 1.0 and np.all(np.diff(z) > 0)
    assert np.allclose(z + z[::-1], 1.0, atol=1e-15)                       # symmetric about mid-height
    h = np.diff(z)
    assert h[0] < 0.35 / 64 and h[32] > 1.6 / 64                           # finest at the plates
    assert cell_heights(z).sum() == pytest.approx(1.0, rel=1e-14)


@pytest.mark.parametrize("ndim", [2, 3])
def test_uniform_node_heights_give_the_uniform_scheme(orc, ndim):
    """R19 / R20 reduce to Eqs. 31-39 as printed when z_k = k dz: same state after three steps, same dt, same
    diagnostics, whether the node heights are passed or not."""
    g = inputs.make_grid(ndim, 12, 17, 6 if ndim == 3 else 1)
    p = inputs.make_params(Ra=1e4)
    gz = dict(g, z_nodes=inputs.z_nodes(g, p))
    X = inputs.rough_random_state(g, p, seed=5)
    a, dta, _ = orc.step(orc.Problem(g, p), X, 3)
    b, dtb, _ = orc.step(orc.Problem(gz, p), X, 3)
    assert np.abs(a - b).max() <= 1e-14 * np.abs(a).max()
    assert np.allclose(dta, dtb, rtol=1e-15)
    da, db = orc.diagnostics(orc.Problem(g, p), a)[0], orc.diagnostics(orc.Problem(gz, p), a)[0]
    for k in ("nu_bar", "nu_bulk", "re", "mass", "energy"):
        assert da[k] == pytest.approx(db[k], rel=1e-13), k


@pytest.mark.parametrize("tvd_form", [0, 1])
def test_mass_between_plates_is_conserved_on_the_stretched_grid(orc, tvd_form):
    """Sum of (cell height x rho) over a column telescopes to the plate fluxes, which are zero: constant to round-off
    with the TVD term active on most nodes (rough state).  A mismatch between the heights used by the predictor, the
    corrector, the plate closure (R10) or the TVD weighting (R20) breaks this at the 1e-4 level."""
    g = inputs.make_grid(2, 24, 33, z_stretch=1.5)
    p = inputs.make_params(Ra=1e4, tvd_form=tvd_form)
    X = inputs.rough_random_state(g, p, seed=11, rough=0.02)
    prob = orc.Problem(g, p)
    w = cell_heights(g["z_nodes"])[:, None]
    mass = lambda Y: float(np.sum(w * Y[0].reshape(33, 24)))
    off = orc.step(orc.Problem(g, dict(p, tvd_off=1)), X, 1)[0]
    on = orc.step(prob, X, 1)[0]
    assert np.abs(on - off)[0].max() > 1e-5                                 # the TVD term is at work
    Y, _, _ = orc.step(prob, X, 20)
    assert abs(mass(Y) - mass(X)) <= 2e-14 * mass(X)
    d = orc.diagnostics(prob, Y)[0]
    assert d["mass"] == pytest.approx(mass(Y) * g["lx"] / g["nx"], rel=1e-13)   # the oracle's total uses the same weights


@pytest.mark.parametrize("tvd_form", [0, 1])
def test_contact_at_rest_on_the_stretched_grid_records_R20(orc, tvd_form):
    """A contact at rest between plates (u = 0, uniform p, one density jump between nodes k and k+1 well inside the
    box, mu = K = g = 0): every MacCormack difference vanishes, r+- = 0, and reading R20 moves
        h_{k+1/2} Dh / dzc_k   out of node k  and  h_{k+1/2} Dh / dzc_{k+1}  into node k+1,
    Dh = (1/2)[C(Co_k) + C(Co_{k+1})] drho (Davis/Yee; the mean of the two C's times 1/2 for Eq. 34 as printed), with
    Co_k = c_s tau / dzc_k (the node's cell height).  So the amounts differ at the two nodes but the heights-weighted
    sum is zero.  The paper prints the TVD term for a uniform grid only: this records the reading's closed form."""
    gam, p0, rl, rr = 1.4, 1.0, 1.0, 0.25
    nz, kj, tau = 17, 6, 0.004
    g = inputs.make_grid(2, 6, nz, lx=0.6, z_stretch=1.5)
    z = g["z_nodes"]
    w = cell_heights(z)
    rho = np.where(np.arange(nz) <= kj, rl, rr)
    p = inputs.make_params(gamma=gam, eps=1.0, D=1.0 / gam, g_override=0.0, mu_override=0.0, K_override=0.0,
                           T_bot=p0 / ((gam - 1) * rl), T_top=p0 / ((gam - 1) * rr), tvd_form=tvd_form)
    X = state_from_primitives(g, p, rho[:, None, None], 0.0, 0.0, 0.0, p0)
    C = lambda Co: Co * (1.0 - Co) if Co <= 0.5 else 0.25
    Cl = C(np.sqrt(gam * p0 / rl) * tau / w[kj])
    Cr = C(np.sqrt(gam * p0 / rr) * tau / w[kj + 1])
    Dh = (0.5 * (Cl + Cr) if tvd_form == 1 else 0.25 * (Cl + Cr)) * (rr - rl)
    h = z[kj + 1] - z[kj]
    for direction in (+1, -1):
        Y = orc.sweep(orc.Problem(g, p), X, 2, tau, direction)
        d = (Y - X).reshape(4, nz, 6)
        assert np.abs(d[1:]).max() <= 1e-15
        want = np.zeros(nz)
        want[kj], want[kj + 1] = h * Dh / w[kj], -h * Dh / w[kj + 1]
        np.testing.assert_allclose(d[0][:, 2], want, rtol=0, atol=3e-16)
        assert abs(np.sum(w * d[0][:, 2])) <= 1e-17


def test_hydrostatic_conduction_state_drift_is_second_order_on_the_stretched_grid(orc):
    """The noise-free conduction state (linear T, hydrostatic p) is steady for the PDE; on the stretched grid the
    discrete drift is truncation error, ~4x smaller per doubling (same test as on the uniform grid)."""
    drift = []
    for nz in (33, 65, 129):
        g = inputs.make_grid(2, 8, nz, lx=8.0 / (nz - 1), z_stretch=1.5)
        p = inputs.make_params(Ra=1e6)        # (at Ra = 1e4 the finest plate spacing sits at the explicit diffusive limit)
        X = inputs.conduction_state(g, p, amplitude=0.0)
        Y, _ = advance_to(orc, orc.Problem(g, p), X, 0.05)
        drift.append(np.abs(primitives_of(g, p, Y)[3]).max())
    assert drift[0] < 1e-3            # (1.3e-4 on the uniform grid of 33 levels: the mid-height cells are 1.66x larger here)
    assert drift[0] / drift[1] > 3.3 and drift[1] / drift[2] > 3.3, drift


def test_shear_flow_between_plates_decays_at_the_viscous_rate_on_the_stretched_grid(orc):
    """u_x = A sin(pi z) between no-slip plates, uniform rho and p, no gravity: d_t u_x = nu d_zz u_x, so the profile
    keeps its shape and decays as exp(-nu pi^2 t).  Pins the spacings of the z-sweep's viscous flux (inner one-sided
    difference over the face spacing, outer difference over the cell height): the error of the decayed amplitude
    falls ~4x per doubling; dividing both by the same local spacing would leave an O(1) error where the grid
    stretches."""
    nu, A, t_end = 0.002, 1e-3, 5.0         # (explicit diffusive limit h^2 / 2 nu stays 2x above the acoustic step)
    err = []
    for nz in (17, 33, 65):
        g = inputs.make_grid(2, 4, nz, lx=4.0 / (nz - 1), z_stretch=1.5)
        p = inputs.make_params(gamma=1.4, eps=1.0, D=1.0 / 1.4, g_override=0.0, mu_override=nu, K_override=0.0,
                               T_bot=1.0, T_top=1.0, cfl=0.4, tvd_off=1)     # (the limiter clips the extremum)
        z = g["z_nodes"][:, None, None]
        X = state_from_primitives(g, p, 1.0, A * np.sin(np.pi * z), 0.0, 0.0, 0.4)      # rho = 1, T = 1: plates at T_w
        Y, _ = advance_to(orc, orc.Problem(g, p), X, t_end)
        ux = primitives_of(g, p, Y)[1][:, 0, 0]
        want = A * np.exp(-nu * np.pi**2 * t_end) * np.sin(np.pi * g["z_nodes"])
        err.append(np.abs(ux - want).max() / A)
    assert err[0] < 2e-3
    assert err[0] / err[1] > 3.3 and err[1] / err[2] > 3.3, err


def test_cross_derivative_along_z_in_the_x_sweep_on_the_stretched_grid(orc):
    """One operator L_x on u_x = A sin(2 pi x / lx) sin(pi z), u_z = 0, uniform rho and p, no gravity: the only source
    of vertical momentum is the shear stress, d_t (rho u_z) = mu d_x d_z u_x + mu' d_z d_x u_x's x-sweep part, i.e.
    the x-sweep adds tau mu d_x (d_z u_x) = tau mu A (2 pi / lx) pi cos(2 pi x / lx) cos(pi z).  Pins the central
    z-difference inside F_x (R7) on the stretched grid: divided by z_{k+1} - z_{k-1}, second order."""
    mu, A, lx = 0.05, 1e-3, 1.0
    err = []
    for n in (16, 32, 64):
        g = inputs.make_grid(2, n, n + 1, lx=lx, z_stretch=1.5)
        p = inputs.make_params(gamma=1.4, eps=1.0, D=1.0 / 1.4, g_override=0.0, mu_override=mu, K_override=0.0,
                               T_bot=1.0, T_top=1.0, tvd_off=1)
        z = g["z_nodes"][:, None, None]
        x = (np.arange(n) * lx / n)[None, None, :]
        X = state_from_primitives(g, p, 1.0, A * np.sin(2 * np.pi * x / lx) * np.sin(np.pi * z), 0.0, 0.0, 0.4)
        tau = 1e-4 / n
        Y = orc.sweep(orc.Problem(g, p), X, 0, tau, +1)
        mz = Y[2].reshape(n + 1, n)[1:-1]
        want = (tau * mu * A * (2 * np.pi / lx) * np.pi * np.cos(2 * np.pi * x / lx) * np.cos(np.pi * z))[1:-1, 0, :]
        err.append(np.abs(mz - want).max() / np.abs(want).max())
    assert err[0] < 0.05
    assert err[0] / err[1] > 3.3 and err[1] / err[2] > 3.3, err


def test_diagnostics_closed_forms_on_the_stretched_grid(orc):
    """Conduction state: Nu_0 = Nu_1 = Nu_bulk = 1, Re = 0 on any node spacing.  T = T_A - eps z + q z (1 - z): the
    second-order one-sided plate gradients of Eq. 23 are exact for a quadratic (Nu_0 = 1 - q/eps, Nu_1 = 1 + q/eps),
    and the volume mean of Eq. 22 is the cell-height-weighted sum."""
    g = inputs.make_grid(3, 6, 21, 5, z_stretch=1.5)
    p = inputs.make_params(Ra=1e4, Pr=0.7)
    prob = orc.Problem(g, p)
    d = orc.diagnostics(prob, inputs.conduction_state(g, p, amplitude=0.0))[0]
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk"):
        assert d[k] == pytest.approx(1.0, abs=1e-11), k
    assert d["re"] == 0.0
    q, a = 0.07, 0.03
    z = g["z_nodes"][:, None, None]
    T = 1 - (p["eps"] + p["D"]) * z + q * z * (1 - z) + np.zeros((21, 5, 6))
    X = inputs.pack(g, np.full_like(T, 1.25), 0 * T, 0 * T, a + 0 * T, T, p)
    d, Tp, rp, pp = orc.diagnostics(prob, X)
    assert d["nu_bottom"] == pytest.approx(1 - q / p["eps"], rel=1e-10)
    assert d["nu_top"] == pytest.approx(1 + q / p["eps"], rel=1e-10)
    w = cell_heights(g["z_nodes"])
    zz = g["z_nodes"]
    mean_tsa = np.sum(w * (-p["eps"] * zz + q * zz * (1 - zz))) / np.sum(w)
    assert d["nu_conv"] == pytest.approx(np.sqrt(p["Ra"] * p["Pr"]) / p["eps"] * 1.25 * a * mean_tsa, rel=1e-12)
    assert d["mass"] == pytest.approx(1.25 * 16.0, rel=1e-13)


def test_dt_rule_on_the_stretched_grid(orc):
    """R12 with the cell heights: a gas at rest, s = c_s / min(dx, smallest interior cell height); the plate nodes take
    the full adjacent spacing (their own cell is a half cell), which equals the first interior cell's height only on
    a uniform grid."""
    g = inputs.make_grid(2, 8, 17, lx=8.0, z_stretch=2.0)
    p = inputs.make_params(gamma=1.4, eps=1.0, D=1.0 / 1.4, g_override=0.0, mu_override=0.0, K_override=0.0,
                           T_bot=1.0, T_top=1.0, cfl=0.5)
    X = state_from_primitives(g, p, 2.0, 0.0, 0.0, 0.0, 2.0 / 1.4)          # c_s = 1
    z = g["z_nodes"]
    h_int = 0.5 * (z[2:] - z[:-2])
    want = 0.5 * min(1.0, h_int.min(), z[1] - z[0])
    assert orc.dt(orc.Problem(g, p), X) == pytest.approx(want, rel=1e-14)


def test_periodic_z_rejects_node_heights(orc):
    g = inputs.make_grid(2, 8, 16)
    g["z_nodes"] = np.arange(16) / 16.0
    with pytest.raises(ValueError):
        orc.sweep(orc.Problem(g, inputs.make_params(bc_z=1)), np.ones((4, 128)), 2, 1e-3, 1)
