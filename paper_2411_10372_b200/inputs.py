"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds no part of the method (no flux, no stencil, no limiter, no reduction): it only
builds grids, parameter sets and initial states, on the host, with numpy.  The same arrays are
handed bit-identically to the CPU oracle and to the CUDA library.

Recipe (BASELINE.json `configs`; not in the paper):
  * parameters: gamma = 5/3, Pr = 1, Ra per config, eps = 0.1, D = 0.4 so that the conduction
    profile T = 1 - (eps + D) z runs from 1 (bottom) to 0.5 (top), i.e. the
    config's "T = 1 + Delta (1 - z), Delta = 1" in units of the bottom temperature;
  * rho from the discrete (trapezoid) hydrostatic balance of p = R rho T with rho(0) = 1;
  * u = 0; a seeded uniform perturbation of T with amplitude 1e-3 on interior nodes;
  * E = rho (c_v T + g z) (Eq. 17 with u = 0).
Random numbers: counter-based 64-bit mixing hash of (seed, global node index), top 53 bits.
"""
from __future__ import annotations

import numpy as np

SEED = 20241110

# BASELINE.json `configs`, in order.  steps = the step count the config names.
CONFIGS = {
    "C1": dict(ndim=2, nx=256, ny=1, nz=64, Ra=1e6, steps=100),
    "C2": dict(ndim=2, nx=4096, ny=1, nz=1024, Ra=1e10, steps=1000),
    "C3": dict(ndim=2, nx=16384, ny=1, nz=4096, Ra=1e14, steps=200),
    "C4": dict(ndim=3, nx=512, ny=512, nz=128, Ra=1e8, steps=200),
    "C5": dict(ndim=3, nx=1024, ny=1024, nz=256, Ra=1e11, steps=50),
}


TANH_STRETCH = 1.5      # default stretching of `tanh_nodes` (the paper names the grid but gives no parameter)


def tanh_nodes(nz: int, lz: float = 1.0, stretch: float = TANH_STRETCH) -> np.ndarray:
    """Node heights of a "non-uniform tangent-hyperbolic grid in the z-direction" with nodes on
    both plates: z_k = lz/2 (1 + tanh(s (2k/(nz-1) - 1)) / tanh(s)), finest at the plates.  The paper does not
    state its stretching parameter; s = 1.5 makes the plate spacing about 0.3 of the uniform one."""
    xi = 2.0 * np.arange(nz, dtype=np.float64) / (nz - 1) - 1.0
    z = 0.5 * lz * (1.0 + np.tanh(stretch * xi) / np.tanh(stretch))
    z[0], z[-1] = 0.0, lz
    return z


def make_grid(ndim: int, nx: int, nz: int, ny: int = 1, lx: float = 4.0, ly: float = 4.0,
              lz: float = 1.0, z_stretch: float | None = None) -> dict:
    """Box of aspect ratio 4 by default.  z_stretch: tanh-stretched z nodes (`tanh_nodes`),
    stored under "z_nodes"; None = uniform z."""
    if ndim == 2:
        ny, ly = 1, 1.0
    g = dict(ndim=int(ndim), nx=int(nx), ny=int(ny), nz=int(nz), lx=float(lx), ly=float(ly),
             lz=float(lz))
    if z_stretch is not None:
        g["z_nodes"] = tanh_nodes(nz, lz, z_stretch)
    return g


def make_params(**over) -> dict:
    """Parameter set of the BASELINE configs; keyword arguments override single entries."""
    p = dict(gamma=5.0 / 3.0, Pr=1.0, Ra=1e6, eps=0.1, D=0.4, cfl=0.5, fixed_dt=0.0,
             T_bot=1.0, T_top=None, lambda_coef=-2.0 / 3.0,
             g_override=-1.0, mu_override=-1.0, K_override=-1.0,
             bc_z=0, tvd_form=1, dir_mode=1, tvd_off=0, co_mode=0)
    p.update(over)
    if p["T_top"] is None:
        p["T_top"] = 1.0 - p["eps"] - p["D"]
    return p


def config(name: str, **over):
    """(grid, params, steps) of a BASELINE config."""
    c = CONFIGS[name]
    grid = make_grid(c["ndim"], c["nx"], c["nz"], c["ny"])
    return grid, make_params(Ra=c["Ra"], **over), c["steps"]


def num_fields(grid: dict) -> int:
    return 4 if grid["ndim"] == 2 else 5


def num_nodes(grid: dict) -> int:
    return grid["nx"] * grid["ny"] * grid["nz"]


def closure_constants(params: dict) -> dict:
    """R, c_v, g of the paper's dimensionless closure (Eqs. 14, 16, 17)."""
    ged = params["gamma"] * params["eps"] * params["D"]
    g = params["g_override"] if params["g_override"] >= 0 else 1.0 / params["eps"]
    return dict(R=(params["gamma"] - 1.0) / ged, cv=1.0 / ged, g=g)


def z_nodes(grid: dict, params: dict) -> np.ndarray:
    if grid.get("z_nodes") is not None:
        return np.asarray(grid["z_nodes"], dtype=np.float64)
    nz = grid["nz"]
    dz = grid["lz"] / (nz - 1) if params["bc_z"] == 0 else grid["lz"] / nz
    return np.arange(nz, dtype=np.float64) * dz


def hash_uniform(seed: int, index: np.ndarray) -> np.ndarray:
    """U in [0,1): splitmix64-style finaliser of (seed, index), top 53 bits."""
    with np.errstate(over="ignore"):
        x = index.astype(np.uint64) + np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        x = x ^ (x >> np.uint64(31))
    return (x >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def pack(grid: dict, rho, ux, uy, uz, T, params: dict) -> np.ndarray:
    """Conserved SoA block (nf, N) from node arrays of shape (nz, ny, nx); Eq. 17."""
    c = closure_constants(params)
    z = z_nodes(grid, params)[:, None, None]
    E = rho * (0.5 * (ux * ux + uy * uy + uz * uz) + c["cv"] * T + c["g"] * z)
    fields = [rho, rho * ux] + ([rho * uy] if grid["ndim"] == 3 else []) + [rho * uz, E]
    return np.ascontiguousarray(np.stack([np.broadcast_to(f, rho.shape).reshape(-1) for f in fields]),
                                dtype=np.float64)


def conduction_state(grid: dict, params: dict, seed: int = SEED, amplitude: float = 1e-3,
                     x_offset: int = 0, nx_global: int | None = None) -> np.ndarray:
    """Hydrostatic conduction profile plus seeded T noise; returns X with shape (nf, N).

    x_offset / nx_global let a test build a window [x_offset, x_offset + nx) of a wider periodic
    box with the very same per-node random numbers (3-D windows: x only).
    """
    assert params["bc_z"] == 0
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    nxg = nx if nx_global is None else nx_global
    c = closure_constants(params)
    z = z_nodes(grid, params)
    uniform = grid.get("z_nodes") is None
    Tbar = params["T_bot"] + (params["T_top"] - params["T_bot"]) * z / grid["lz"]
    rho = np.empty(nz)
    rho[0] = 1.0
    for k in range(nz - 1):   # p_{k+1} - p_k = -(dz/2) g (rho_k + rho_{k+1}),  p = R rho Tbar
        dz = (z[1] - z[0]) if uniform else (z[k + 1] - z[k])
        rho[k + 1] = rho[k] * (c["R"] * Tbar[k] - c["g"] * dz / 2) / (c["R"] * Tbar[k + 1] + c["g"] * dz / 2)
    nf = num_fields(grid)
    X = np.zeros((nf, nz, ny * nx), dtype=np.float64)     # momenta stay zero (u = 0)
    jj, ii = np.meshgrid(np.arange(ny, dtype=np.int64), (np.arange(nx, dtype=np.int64) + x_offset) % nxg,
                         indexing="ij")
    plane_idx = (jj * nxg + ii).reshape(-1)
    for k in range(nz):                                   # plane by plane: bounded host memory
        T = np.full(ny * nx, Tbar[k])
        if 0 < k < nz - 1:
            U = hash_uniform(seed, plane_idx + np.int64(k) * ny * nxg)
            T = T + amplitude * (2.0 * U - 1.0)
        X[0, k] = rho[k]
        X[nf - 1, k] = rho[k] * (c["cv"] * T + c["g"] * z[k])   # Eq. 17 with u = 0
    return X.reshape(nf, -1)


def smooth_random_state(grid: dict, params: dict, seed: int = SEED, u_amp: float = 0.3,
                        s_amp: float = 0.2, modes: int = 3) -> np.ndarray:
    """Smooth periodic (x, y) state with non-zero velocity for parity tests.

    rho and T are positive sums of a few seeded Fourier modes; with plates (bc_z = 0) the velocity
    carries a sin(pi z) envelope and T is pinned to the plate temperatures, so the state satisfies
    the boundary conditions.  With bc_z = 1 everything is periodic in z too.
    """
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    rng = np.random.default_rng(seed)
    z = z_nodes(grid, params) / grid["lz"]
    x = np.arange(nx) / nx
    y = np.arange(ny) / ny
    Z, Y, Xc = np.meshgrid(z, y, x, indexing="ij")
    walls = params["bc_z"] == 0

    def field():
        f = np.zeros_like(Z)
        for _ in range(modes):
            kx, ky, kz = rng.integers(0, 3, size=3)
            if grid["ndim"] == 2:
                ky = 0
            ph = rng.uniform(0, 2 * np.pi, size=3)
            zfac = np.cos(np.pi * kz * Z + ph[2]) if walls else np.cos(2 * np.pi * kz * Z + ph[2])
            f += rng.uniform(-1, 1) * np.cos(2 * np.pi * kx * Xc + ph[0]) * np.cos(2 * np.pi * ky * Y + ph[1]) * zfac
        return f / modes

    env = np.sin(np.pi * Z) if walls else np.ones_like(Z)
    rho = 1.0 + s_amp * field()
    ux = u_amp * field() * env
    uy = u_amp * field() * env if grid["ndim"] == 3 else np.zeros_like(Z)
    uz = u_amp * field() * env
    if walls:
        Tlin = params["T_bot"] + (params["T_top"] - params["T_bot"]) * Z
        T = Tlin * (1.0 + s_amp * field() * env)
    else:
        T = params["T_bot"] * (1.0 + s_amp * field())
    return pack(grid, rho, ux, uy, uz, T, params)


def rough_random_state(grid: dict, params: dict, seed: int = SEED, rough: float = 0.05) -> np.ndarray:
    """`smooth_random_state` with seeded node-to-node noise of relative amplitude `rough` on rho, u and T of
    the interior nodes: adjacent differences change sign from node to node, so the limiter ratios r+- of
    Eq. 37 leave [1/2, infinity) on most nodes and the TVD term of Eqs. 34-39 is non-zero along every axis
    (the smooth states keep phi = 1 almost everywhere).  Plate nodes keep u = 0 and T = T_w."""
    nf = num_fields(grid)
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    X = smooth_random_state(grid, params, seed=seed).reshape(nf, nz, ny, nx)
    c = closure_constants(params)
    z = z_nodes(grid, params)[:, None, None]
    rho = X[0]
    u = [X[1 + k] / rho for k in range(nf - 2)]
    T = (X[nf - 1] / rho - 0.5 * sum(v * v for v in u) - c["g"] * z) / c["cv"]
    idx = np.arange(nx * ny * nz, dtype=np.int64).reshape(nz, ny, nx)
    noise = lambda k: 2.0 * hash_uniform(seed + 1000 * (k + 1), idx) - 1.0
    interior = np.ones((nz, 1, 1))
    if params["bc_z"] == 0:
        interior[0] = interior[-1] = 0.0
    rho = rho * (1.0 + rough * noise(0))
    T = T * (1.0 + rough * noise(1) * interior)
    u = [v + rough * noise(2 + k) * interior for k, v in enumerate(u)]
    ux, uz = u[0], u[-1]
    uy = u[1] if nf == 5 else np.zeros_like(rho)
    return pack(grid, rho, ux, uy, uz, T, params)


def moving_state(grid: dict, params: dict, seed: int = SEED, amplitude: float = 1e-3, u_amp: float = 0.05) -> np.ndarray:
    """The conduction-plus-noise state of `conduction_state` set in motion: a smooth, plate-compatible
    velocity field of amplitude u_amp (a few per cent of the sound speed) is added plane by plane, so the
    full-size parity tests also sample a state that moves.  Host memory stays bounded by one z-plane."""
    assert params["bc_z"] == 0
    nf = num_fields(grid)
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    X = conduction_state(grid, params, seed=seed, amplitude=amplitude).reshape(nf, nz, ny * nx)
    zn = z_nodes(grid, params) / grid["lz"]
    x = (np.arange(nx) / nx)[None, :]
    y = (np.arange(ny) / ny)[:, None]
    sx, cx = np.sin(2 * np.pi * 3 * x), np.cos(2 * np.pi * 3 * x)
    sy, cy = np.sin(2 * np.pi * 2 * y), np.cos(2 * np.pi * 2 * y)
    for k in range(1, nz - 1):
        env = np.sin(np.pi * zn[k])
        rho = X[0, k]
        ux = (u_amp * env * (cy + 0 * x) * (1.0 + 0.3 * sx)).reshape(-1)
        uy = (0.6 * u_amp * env * (sx + 0 * y)).reshape(-1)
        uz = (0.8 * u_amp * env * (sx * cy if ny > 1 else sx + 0 * y)).reshape(-1) * np.cos(np.pi * zn[k])
        if nf == 4:
            uy = 0.0 * ux
        X[1, k] = rho * ux
        if nf == 5:
            X[2, k] = rho * uy
        X[nf - 2, k] = rho * uz
        X[nf - 1, k] += 0.5 * rho * (ux * ux + uy * uy + uz * uz)
    return X.reshape(nf, -1)


def window_x(X: np.ndarray, grid: dict, i0: int, width: int):
    """Columns [i0, i0 + width) (periodic in x) of every field; returns (X_window, grid_window).

    The window is itself treated as a periodic box of `width` columns with the same spacing, so a
    local scheme run on it equals the full-box result away from the window's two edges.
    """
    nf = X.shape[0]
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    idx = (np.arange(width) + i0) % nx
    Xw = X.reshape(nf, nz, ny, nx)[:, :, :, idx].reshape(nf, -1).copy()
    gw = dict(grid)
    gw["nx"] = width
    gw["lx"] = grid["lx"] * width / nx
    return Xw, gw


def window_xy(X: np.ndarray, grid: dict, i0: int, wx: int, j0: int, wy: int):
    """Same as window_x for a 3-D box, cutting both periodic directions."""
    nf = X.shape[0]
    nx, ny, nz = grid["nx"], grid["ny"], grid["nz"]
    ix = (np.arange(wx) + i0) % nx
    iy = (np.arange(wy) + j0) % ny
    Xw = X.reshape(nf, nz, ny, nx)[:, :, iy][:, :, :, ix].reshape(nf, -1).copy()
    gw = dict(grid)
    gw.update(nx=wx, ny=wy, lx=grid["lx"] * wx / nx, ly=grid["ly"] * wy / ny)
    return Xw, gw
