"""Test-side helpers: analytic reference solutions and state builders for the oracle pins.

Nothing here is used by the product path.  The exact Riemann solver and the closed forms are
written from the textbook definitions (not from the oracle), so they can pin it.
"""
from __future__ import annotations

import numpy as np

from paper_2411_10372_b200 import inputs


def ideal_gas_params(gamma=1.4, **over):
    """Parameters of a plain ideal gas for the test problems: gamma*eps*D = 1 so that c_v = 1 and
    R = gamma - 1; no gravity, no viscosity, no conduction, periodic z."""
    base = dict(gamma=gamma, eps=1.0, D=1.0 / gamma, g_override=0.0, mu_override=0.0, K_override=0.0,
                bc_z=1, T_bot=1.0, T_top=1.0, cfl=0.5)
    base.update(over)
    return inputs.make_params(**base)


def state_from_primitives(grid, params, rho, ux, uy, uz, p):
    """Conserved block from rho, u, p given as arrays broadcastable to (nz, ny, nx)."""
    shp = (grid["nz"], grid["ny"], grid["nx"])
    c = inputs.closure_constants(params)
    rho = np.broadcast_to(np.asarray(rho, dtype=float), shp).copy()
    p = np.broadcast_to(np.asarray(p, dtype=float), shp)
    T = p / (c["R"] * rho)
    b = lambda a: np.broadcast_to(np.asarray(a, dtype=float), shp).copy()
    return inputs.pack(grid, rho, b(ux), b(uy), b(uz), T, params)


def primitives_of(grid, params, X):
    """(rho, ux, uy, uz, T, p) as (nz, ny, nx) arrays -- independent numpy restatement of
    Eqs. 16-17 used only to read test results."""
    c = inputs.closure_constants(params)
    nf = inputs.num_fields(grid)
    shp = (grid["nz"], grid["ny"], grid["nx"])
    F = X.reshape(nf, *shp)
    rho = F[0]
    ux = F[1] / rho
    uy = F[2] / rho if nf == 5 else np.zeros(shp)
    uz = F[nf - 2] / rho
    z = inputs.z_nodes(grid, params)[:, None, None]
    T = (F[nf - 1] / rho - 0.5 * (ux**2 + uy**2 + uz**2) - c["g"] * z) / c["cv"]
    return rho, ux, uy, uz, T, c["R"] * rho * T


def advance_to(orc, prob, X, t_end):
    """March with the CFL rule, clipping the last step to land on t_end."""
    t = 0.0
    n = 0
    while t < t_end * (1 - 1e-13):
        dt = min(orc.dt(prob, X), t_end - t)
        X, _, _ = orc.step(prob, X, 1, dt_in=[dt])
        t += dt
        n += 1
    return X, n


def riemann_exact(rl, ul, pl, rr, ur, pr, gam, xi):
    """Exact solution of the Riemann problem for the ideal-gas Euler equations sampled at
    xi = x/t: Newton iteration on the star pressure, then the standard wave-by-wave sampling."""
    al, ar = np.sqrt(gam * pl / rl), np.sqrt(gam * pr / rr)
    g1, g2 = (gam - 1) / (2 * gam), (gam + 1) / (2 * gam)

    def f(p, rk, pk, ak):
        if p > pk:   # shock
            A, B = 2 / ((gam + 1) * rk), (gam - 1) / (gam + 1) * pk
            q = np.sqrt(A / (p + B))
            return (p - pk) * q, q * (1 - (p - pk) / (2 * (B + p)))
        return 2 * ak / (gam - 1) * ((p / pk) ** g1 - 1), (p / pk) ** (-g2) / (rk * ak)

    p = 0.5 * (pl + pr)
    for _ in range(200):
        fl, dfl = f(p, rl, pl, al)
        fr, dfr = f(p, rr, pr, ar)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p = max(p - dp, 1e-14)
        if abs(dp) < 1e-15 * p:
            break
    fl, _ = f(p, rl, pl, al)
    fr, _ = f(p, rr, pr, ar)
    us = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    rho, u, pp = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm = (gam - 1) / (gam + 1)
    for n, s in enumerate(xi):
        if s <= us:      # left of the contact
            if p > pl:
                sl = ul - al * np.sqrt(g2 * p / pl + g1)
                r_, u_, p_ = (rl, ul, pl) if s < sl else (rl * (p / pl + gm) / (gm * p / pl + 1), us, p)
            else:
                head, tail = ul - al, us - al * (p / pl) ** g1
                if s < head:
                    r_, u_, p_ = rl, ul, pl
                elif s > tail:
                    r_, u_, p_ = rl * (p / pl) ** (1 / gam), us, p
                else:
                    u_ = 2 / (gam + 1) * (al + (gam - 1) / 2 * ul + s)
                    c = 2 / (gam + 1) * (al + (gam - 1) / 2 * (ul - s))
                    r_, p_ = rl * (c / al) ** (2 / (gam - 1)), pl * (c / al) ** (2 * gam / (gam - 1))
        else:
            if p > pr:
                sr = ur + ar * np.sqrt(g2 * p / pr + g1)
                r_, u_, p_ = (rr, ur, pr) if s > sr else (rr * (p / pr + gm) / (gm * p / pr + 1), us, p)
            else:
                head, tail = ur + ar, us + ar * (p / pr) ** g1
                if s > head:
                    r_, u_, p_ = rr, ur, pr
                elif s < tail:
                    r_, u_, p_ = rr * (p / pr) ** (1 / gam), us, p
                else:
                    u_ = 2 / (gam + 1) * (-ar + (gam - 1) / 2 * ur + s)
                    c = 2 / (gam + 1) * (ar - (gam - 1) / 2 * (ur - s))
                    r_, p_ = rr * (c / ar) ** (2 / (gam - 1)), pr * (c / ar) ** (2 * gam / (gam - 1))
        rho[n], u[n], pp[n] = r_, u_, p_
    return rho, u, pp, p, us


def rel_err(a, b):
    """Field-max-normalised error, per field."""
    a = np.asarray(a)
    b = np.asarray(b)
    out = []
    for fa, fb in zip(a, b):
        den = np.max(np.abs(fb))
        out.append(np.max(np.abs(fa - fb)) / den if den > 0 else np.max(np.abs(fa - fb)))
    return np.array(out)


def parity_err(grid, params, got, ref):
    """Per-field parity error, each field on its own physical scale:
    rho and E by their field maximum; a momentum component by max(max|m|, max rho * c_s), the acoustic
    momentum scale -- a momentum field that is still ~1e-4 of that scale (config C1 after one step)
    carries the ulp-level rounding of the O(10) pressure and energy it is differenced from, so its
    own maximum is not a meaningful denominator."""
    got = np.asarray(got)
    ref = np.asarray(ref)
    nf = ref.shape[0]
    rho, _, _, _, T, _ = primitives_of(grid, params, ref)
    c = inputs.closure_constants(params)
    m_scale = float(np.max(rho * np.sqrt(np.abs(params["gamma"] * c["R"] * T))))
    out = []
    for f in range(nf):
        den = np.max(np.abs(ref[f]))
        if 0 < f < nf - 1:
            den = max(den, m_scale)
        out.append(np.max(np.abs(got[f] - ref[f])) / (den if den > 0 else 1.0))
    return np.array(out)


def ulp_perturbed(X, seed=1):
    """X with every entry moved by -1, 0 or +1 unit in the last place (seeded)."""
    rng = np.random.default_rng(seed)
    k = rng.integers(-1, 2, size=X.shape)
    return np.where(k > 0, np.nextafter(X, np.inf), np.where(k < 0, np.nextafter(X, -np.inf), X))


def plate_nusselt_exact(grid, params, X):
    """(nu_bottom, nu_top, nu_bar) of Eqs. 23-24 with the plane means of T summed in extended
    precision: the reference for the Nu tolerance on large grids, where a plain serial fp64 sum of 1e4-1e6 plane
    values (the oracle's) carries more rounding noise than the tolerance once the one-sided plate difference has
    amplified it by 1/(eps dz).  Independent numpy restatement; second-order one-sided differences."""
    T = primitives_of(grid, params, X)[4]
    z = inputs.z_nodes(grid, params)
    dz = z[1] - z[0]
    k = [0, 1, 2, grid["nz"] - 3, grid["nz"] - 2, grid["nz"] - 1]
    m = {j: float(np.sum(T[j].astype(np.longdouble)) / T[j].size) for j in k}
    tsa = {j: m[j] - (1.0 - params["D"] * z[j]) for j in k}                      # T_sa = T - T_A, T_A = 1 - D z (Eq. 19)
    g0 = (-3.0 * tsa[k[0]] + 4.0 * tsa[k[1]] - tsa[k[2]]) / (2.0 * dz)
    g1 = (3.0 * tsa[k[5]] - 4.0 * tsa[k[4]] + tsa[k[3]]) / (2.0 * dz)
    nb, nt = -g0 / params["eps"], -g1 / params["eps"]
    return nb, nt, 0.5 * (nb + nt)
