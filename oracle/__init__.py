"""CPU ORACLE binding -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes access to ``oracle/mc_tvd_oracle.c`` (plain C99, fp64, single thread),
the step-by-step restatement of the MacCormack-TVD step of arXiv 2411.10372
(PAPER.md:247-309).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_2411_10372_b200`` (the CUDA path)
and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mc_tvd_oracle.c")
_HDR = os.path.join(_HERE, "mc_tvd_oracle.h")
_LIB = os.path.join(_HERE, "libmc_tvd_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, no fast-math)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math",
                               "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double), ("z_nodes", C.POINTER(C.c_double))]


class _Params(C.Structure):
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("Ra", C.c_double), ("eps", C.c_double),
                ("D", C.c_double), ("cfl", C.c_double), ("fixed_dt", C.c_double),
                ("T_bot", C.c_double), ("T_top", C.c_double), ("lambda_coef", C.c_double),
                ("g_override", C.c_double), ("mu_override", C.c_double), ("K_override", C.c_double),
                ("bc_z", C.c_int), ("tvd_form", C.c_int), ("dir_mode", C.c_int), ("tvd_off", C.c_int),
                ("co_mode", C.c_int)]


class _Diag(C.Structure):
    _fields_ = [("time", C.c_double), ("dt", C.c_double), ("step", C.c_longlong),
                ("nu_bottom", C.c_double), ("nu_top", C.c_double), ("nu_bar", C.c_double),
                ("nu_bulk", C.c_double), ("nu_conv", C.c_double), ("nu_K", C.c_double),
                ("re", C.c_double), ("u_rms", C.c_double),
                ("mass", C.c_double), ("mom_x", C.c_double), ("mom_y", C.c_double),
                ("mom_z", C.c_double), ("energy", C.c_double),
                ("max_mach", C.c_double), ("min_rho", C.c_double), ("min_T", C.c_double)]


class _Stats(C.Structure):
    _fields_ = [("t_begin", C.c_double), ("t_end", C.c_double), ("weight", C.c_double), ("samples", C.c_longlong),
                ("nu_bottom", C.c_double), ("nu_top", C.c_double), ("nu_bar", C.c_double),
                ("nu_bulk", C.c_double), ("nu_conv", C.c_double), ("nu_K", C.c_double),
                ("re", C.c_double), ("u_rms", C.c_double), ("nu_bar_sq", C.c_double), ("re_sq", C.c_double)]


class _Forces(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("Fn_mean", "Fp_mean", "Fb_mean", "Fv_mean", "Fn_rms", "Fp_rms", "Fb_rms",
                                          "Fv_rms", "FbFp_mean", "max_mach", "max_r", "volume", "corr_C", "flux_mean",
                                          "rhouz_sq_mean", "Tsa_sq_mean")]


HIST_BINS = 128

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_sweep.restype = C.c_int
        L.orc_sweep.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp, dp, C.c_int, C.c_double, C.c_int]
        L.orc_max_speed.restype = C.c_double
        L.orc_max_speed.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp]
        L.orc_dt.restype = C.c_double
        L.orc_dt.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp, C.c_int, dp, dp, dp]
        L.orc_diagnostics.restype = C.c_int
        L.orc_diagnostics.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp, C.POINTER(_Diag), dp, dp, dp]
        L.orc_step_stats.restype = C.c_int
        L.orc_step_stats.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp, C.c_int, C.c_int, dp,
                                     C.POINTER(_Stats), dp, dp, dp]
        L.orc_flow_stats.restype = C.c_int
        L.orc_flow_stats.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp, C.POINTER(_Forces), C.POINTER(C.c_longlong)]
        L.orc_coefficients.restype = C.c_int
        L.orc_coefficients.argtypes = [C.POINTER(_Grid), C.POINTER(_Params), dp]
        _lib = L
    return _lib


@dataclass
class Problem:
    """Grid and parameters as plain numbers (dicts from the inputs module map onto this)."""
    grid: dict
    params: dict

    def c_grid(self) -> _Grid:
        g = self.grid
        zp = None
        if g.get("z_nodes") is not None:             # non-uniform z (R19): keep the array alive next to the struct
            self._z = np.ascontiguousarray(g["z_nodes"], dtype=np.float64)
            assert self._z.size == int(g["nz"])
            zp = self._z.ctypes.data_as(C.POINTER(C.c_double))
        return _Grid(int(g["ndim"]), int(g["nx"]), int(g.get("ny", 1)), int(g["nz"]),
                     float(g["lx"]), float(g.get("ly", 1.0)), float(g["lz"]), zp)

    def c_params(self) -> _Params:
        p = self.params
        return _Params(p["gamma"], p["Pr"], p["Ra"], p["eps"], p["D"], p["cfl"], p["fixed_dt"],
                       p["T_bot"], p["T_top"], p["lambda_coef"], p["g_override"], p["mu_override"],
                       p["K_override"], int(p["bc_z"]), int(p["tvd_form"]), int(p["dir_mode"]),
                       int(p["tvd_off"]), int(p.get("co_mode", 0)))

    @property
    def nf(self) -> int:
        return 4 if int(self.grid["ndim"]) == 2 else 5

    @property
    def n_nodes(self) -> int:
        g = self.grid
        return int(g["nx"]) * int(g.get("ny", 1)) * int(g["nz"])


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _check(prob: Problem, X: np.ndarray) -> np.ndarray:
    X = np.ascontiguousarray(X, dtype=np.float64)
    assert X.size == prob.nf * prob.n_nodes, (X.size, prob.nf, prob.n_nodes)
    return X


def sweep(prob: Problem, X: np.ndarray, alpha: int, tau: float, direction: int) -> np.ndarray:
    X = _check(prob, X)
    out = np.empty_like(X)
    g, p = prob.c_grid(), prob.c_params()
    rc = lib().orc_sweep(C.byref(g), C.byref(p), _dp(X), _dp(out), alpha, tau, direction)
    if rc:
        raise ValueError(f"orc_sweep failed: {rc}")
    return out


def max_speed(prob: Problem, X: np.ndarray) -> float:
    X = _check(prob, X)
    g, p = prob.c_grid(), prob.c_params()
    return float(lib().orc_max_speed(C.byref(g), C.byref(p), _dp(X)))


def dt(prob: Problem, X: np.ndarray) -> float:
    X = _check(prob, X)
    g, p = prob.c_grid(), prob.c_params()
    return float(lib().orc_dt(C.byref(g), C.byref(p), _dp(X)))


def step(prob: Problem, X: np.ndarray, n_steps: int, dt_in=None):
    """Advance a copy of X by n_steps; returns (X_new, dt_used[n_steps], elapsed_time)."""
    X = _check(prob, X).copy()
    g, p = prob.c_grid(), prob.c_params()
    dts = np.zeros(max(n_steps, 1))
    t = C.c_double(0.0)
    din = None
    if dt_in is not None:
        din = np.ascontiguousarray(dt_in, dtype=np.float64)
        assert din.size >= n_steps
    rc = lib().orc_step(C.byref(g), C.byref(p), _dp(X), n_steps, _dp(din), _dp(dts), C.byref(t))
    if rc:
        raise ValueError(f"orc_step failed: {rc}")
    return X, dts[:n_steps], t.value


def diagnostics(prob: Problem, X: np.ndarray):
    """Returns (dict of scalars, T_prof, rho_prof, p_prof)."""
    X = _check(prob, X)
    g, p = prob.c_grid(), prob.c_params()
    nz = int(prob.grid["nz"])
    d = _Diag()
    Tp, rp, pp = np.zeros(nz), np.zeros(nz), np.zeros(nz)
    rc = lib().orc_diagnostics(C.byref(g), C.byref(p), _dp(X), C.byref(d), _dp(Tp), _dp(rp), _dp(pp))
    if rc:
        raise ValueError(f"orc_diagnostics failed: {rc}")
    return {n: getattr(d, n) for n, _ in _Diag._fields_}, Tp, rp, pp


def step_stats(prob: Problem, X: np.ndarray, n_steps: int, every: int = 1, dt_in=None):
    """Advance a copy of X by n_steps, sampling the diagnostics after every `every`-th step; returns
    (X_new, dict of time averages, <T>_{A,t}, <rho>_{A,t}, <p>_{A,t})."""
    X = _check(prob, X).copy()
    g, p = prob.c_grid(), prob.c_params()
    nz = int(prob.grid["nz"])
    din = None
    if dt_in is not None:
        din = np.ascontiguousarray(dt_in, dtype=np.float64)
        assert din.size >= n_steps
    st = _Stats()
    Tp, rp, pp = np.zeros(nz), np.zeros(nz), np.zeros(nz)
    rc = lib().orc_step_stats(C.byref(g), C.byref(p), _dp(X), n_steps, every, _dp(din), C.byref(st), _dp(Tp),
                              _dp(rp), _dp(pp))
    if rc:
        raise ValueError(f"orc_step_stats failed: {rc}")
    return X, {n: getattr(st, n) for n, _ in _Stats._fields_}, Tp, rp, pp


def flow_stats(prob: Problem, X: np.ndarray):
    """Returns (dict of the force-balance averages of Eqs. 40-43, the extrema and the correlation C of Eq. 49 with its
    three volume averages, histogram of r as int64[HIST_BINS])."""
    X = _check(prob, X)
    g, p = prob.c_grid(), prob.c_params()
    f = _Forces()
    hist = np.zeros(HIST_BINS, dtype=np.int64)
    rc = lib().orc_flow_stats(C.byref(g), C.byref(p), _dp(X), C.byref(f), hist.ctypes.data_as(C.POINTER(C.c_longlong)))
    if rc:
        raise ValueError(f"orc_flow_stats failed: {rc}")
    return {n: getattr(f, n) for n, _ in _Forces._fields_}, hist


def coefficients(prob: Problem) -> dict:
    g, p = prob.c_grid(), prob.c_params()
    o = np.zeros(9)
    rc = lib().orc_coefficients(C.byref(g), C.byref(p), _dp(o))
    if rc:
        raise ValueError("orc_coefficients failed")
    return dict(zip(["R", "cv", "g", "mu", "K", "lam", "dx", "dy", "dz"], o.tolist()))
