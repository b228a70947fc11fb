"""Thin ctypes binding over the C-ABI library libmc_tvd.so (include/mc_tvd.h).

Argument marshalling only: every step of the path (Eqs. 27-39, the CFL reduction,
the diagnostics of Eqs. 22-26) runs in the CUDA kernels behind the C ABI.  PyTorch supplies device
memory and the stream, nothing else.  There is no CPU fallback: if the library cannot be loaded the
import of this module's users fails with the reason.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB_PATH, build_library

_DP = C.POINTER(C.c_double)


class Grid(C.Structure):            # mc_tvd_grid
    _fields_ = [("ndim", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double), ("z_nodes", _DP)]


class Params(C.Structure):          # mc_tvd_params
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("Ra", C.c_double), ("eps", C.c_double),
                ("D", C.c_double), ("cfl", C.c_double), ("fixed_dt", C.c_double),
                ("T_bot", C.c_double), ("T_top", C.c_double), ("lambda_coef", C.c_double),
                ("g_override", C.c_double), ("mu_override", C.c_double), ("K_override", C.c_double),
                ("bc_z", C.c_int), ("tvd_form", C.c_int), ("dir_mode", C.c_int), ("tvd_off", C.c_int),
                ("co_mode", C.c_int)]


class Diag(C.Structure):            # mc_tvd_diag
    _fields_ = [("time", C.c_double), ("dt", C.c_double), ("step", C.c_longlong),
                ("nu_bottom", C.c_double), ("nu_top", C.c_double), ("nu_bar", C.c_double),
                ("nu_bulk", C.c_double), ("nu_conv", C.c_double), ("nu_K", C.c_double),
                ("re", C.c_double), ("u_rms", C.c_double),
                ("mass", C.c_double), ("mom_x", C.c_double), ("mom_y", C.c_double),
                ("mom_z", C.c_double), ("energy", C.c_double),
                ("max_mach", C.c_double), ("min_rho", C.c_double), ("min_T", C.c_double)]


class Stats(C.Structure):           # mc_tvd_stats
    _fields_ = [("t_begin", C.c_double), ("t_end", C.c_double), ("weight", C.c_double), ("samples", C.c_longlong),
                ("nu_bottom", C.c_double), ("nu_top", C.c_double), ("nu_bar", C.c_double),
                ("nu_bulk", C.c_double), ("nu_conv", C.c_double), ("nu_K", C.c_double),
                ("re", C.c_double), ("u_rms", C.c_double), ("nu_bar_sq", C.c_double), ("re_sq", C.c_double)]


class Forces(C.Structure):          # mc_tvd_forces
    _fields_ = [(n, C.c_double) for n in ("Fn_mean", "Fp_mean", "Fb_mean", "Fv_mean", "Fn_rms", "Fp_rms", "Fb_rms",
                                          "Fv_rms", "FbFp_mean", "max_mach", "max_r", "volume", "corr_C", "flux_mean",
                                          "rhouz_sq_mean", "Tsa_sq_mean")]


HIST_BINS = 128                     # MC_TVD_HIST_BINS

# every symbol include/mc_tvd.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "mc_tvd_workspace_bytes": (C.c_size_t, [C.POINTER(Grid), C.POINTER(Params)]),
    "mc_tvd_init": (C.c_int, [C.POINTER(Grid), C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_size_t,
                              C.c_void_p, C.POINTER(C.c_void_p)]),
    "mc_tvd_step": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_sweep": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_double]),
    "mc_tvd_debug_set_chunk": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_debug_geometry": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "mc_tvd_step_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]),
    "mc_tvd_dt": (C.c_int, [C.c_void_p, _DP]),
    "mc_tvd_diagnostics": (C.c_int, [C.c_void_p, C.POINTER(Diag), _DP, _DP, _DP]),
    "mc_tvd_stats_reset": (C.c_int, [C.c_void_p]),
    "mc_tvd_step_stats": (C.c_int, [C.c_void_p, C.c_int, C.c_int]),
    "mc_tvd_stats_read": (C.c_int, [C.c_void_p, C.POINTER(Stats), _DP, _DP, _DP]),
    "mc_tvd_flow_stats": (C.c_int, [C.c_void_p, C.POINTER(Forces), C.POINTER(C.c_longlong)]),
    "mc_tvd_stats_flow": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_stats_read_flow": (C.c_int, [C.c_void_p, C.POINTER(Forces), C.POINTER(C.c_longlong)]),
    "mc_tvd_slab_op": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_slab_reduce": (C.c_int, [C.c_void_p]),
    "mc_tvd_slab_commit": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_slab_buffers": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "mc_tvd_slab_peers": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "mc_tvd_slab_pointers": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                       C.POINTER(C.c_void_p)]),
    "mc_tvd_slab_diag_partial": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "mc_tvd_slab_diag_finish": (C.c_int, [C.c_void_p, C.c_double, C.POINTER(Diag), _DP, _DP, _DP]),
    "mc_tvd_cfl_noalloc": (C.c_int, [C.POINTER(Grid), C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p]),
    "mc_tvd_launch_count": (C.c_longlong, [C.c_void_p]),
    "mc_tvd_timing_enable": (C.c_int, [C.c_void_p, C.c_int]),
    "mc_tvd_timing_read": (C.c_int, [C.c_void_p, _DP, C.POINTER(C.c_longlong)]),
    "mc_tvd_destroy": (C.c_int, [C.c_void_p]),
    "mc_tvd_last_error": (C.c_char_p, []),
}

STATUS = {0: "MC_TVD_OK", -1: "MC_TVD_EINVAL", -2: "MC_TVD_ECUDA", -3: "MC_TVD_ENOMEM",
          -4: "MC_TVD_ENONFINITE", -5: "MC_TVD_EUNSUPPORTED"}


class MCTVDError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{STATUS.get(code, code)}: {message}")
        self.code = code


_lib = None


def declare(lib: C.CDLL) -> C.CDLL:
    """Attach the prototypes of include/mc_tvd.h to a loaded library."""
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)          # AttributeError if the symbol is missing
        fn.restype = res
        fn.argtypes = args
    return lib


def load_library(path: str | None = None) -> C.CDLL:
    """Load libmc_tvd.so, building it with nvcc first if it is missing or stale.  Raises (never
    falls back) when neither works."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    if path is None:
        build_library()                  # no-op unless a source file changed since the last build
        path = LIB_PATH
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2411_10372_b200.build` (needs nvcc)")
    lib = declare(C.CDLL(path))
    if path == LIB_PATH:
        _lib = lib
    return lib


def make_grid(grid: dict) -> Grid:
    """grid["z_nodes"] (optional): nz node heights of the non-uniform z grid; the library copies what it
    needs during mc_tvd_init, the array only has to live until then (it is kept on the returned struct)."""
    g = Grid(int(grid["ndim"]), int(grid["nx"]), int(grid.get("ny", 1)), int(grid["nz"]),
             float(grid["lx"]), float(grid.get("ly", 1.0)), float(grid["lz"]), None)
    if grid.get("z_nodes") is not None:
        z = np.ascontiguousarray(grid["z_nodes"], dtype=np.float64)
        if z.size != g.nz:
            raise ValueError("z_nodes must hold nz values")
        g._z_keepalive = z
        g.z_nodes = z.ctypes.data_as(_DP)
    return g


def make_params(p: dict) -> Params:
    return Params(p["gamma"], p["Pr"], p["Ra"], p["eps"], p["D"], p["cfl"], p["fixed_dt"],
                  p["T_bot"], p["T_top"], p["lambda_coef"], p["g_override"], p["mu_override"],
                  p["K_override"], int(p["bc_z"]), int(p["tvd_form"]), int(p["dir_mode"]),
                  int(p["tvd_off"]), int(p.get("co_mode", 0)))


NOALLOC_MAX_NZ = 4096                 # MC_TVD_NOALLOC_MAX_NZ of include/mc_tvd.h


def cfl_noalloc(grid: dict, params: dict, fields, out, stream=None) -> None:
    """mc_tvd_cfl_noalloc: enqueue the CFL reduction of the state in `fields` (CUDA float64 tensor, nf * N values, read only)
    and write (s, dt) into `out` (CUDA float64 tensor, >= 2 values) -- no handle, no workspace, no allocation: the
    library's fixed scratch array serves (nz <= NOALLOC_MAX_NZ).  Asynchronous on `stream` (default: torch's current
    stream of the tensors' device); calls whose kernels overlap on the GPU race on the scratch."""
    import torch

    if not (fields.is_cuda and out.is_cuda and fields.dtype == torch.float64 and out.dtype == torch.float64):
        raise TypeError("fields and out must be CUDA float64 tensors")
    if not (fields.is_contiguous() and out.is_contiguous()) or out.numel() < 2 or out.device != fields.device:
        raise ValueError("fields and out must be contiguous tensors on one device, out with at least 2 values")
    nf = 4 if int(grid["ndim"]) == 2 else 5
    if fields.numel() != nf * int(grid["nx"]) * int(grid.get("ny", 1)) * int(grid["nz"]):
        raise ValueError("fields does not hold nf * nx * ny * nz values")
    lib = load_library()
    g, p = make_grid(grid), make_params(params)
    with torch.cuda.device(fields.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.mc_tvd_cfl_noalloc(C.byref(g), C.byref(p), fields.data_ptr(), out.data_ptr(), st.cuda_stream)
        if rc == 0 and g.z_nodes:
            st.synchronize()             # the host node heights (kept alive by g) must outlive the upload
    if rc != 0:
        raise MCTVDError(rc, lib.mc_tvd_last_error().decode())


class MCTVD:
    """One solver handle: owns the torch device buffers and the C handle.

    X0: initial conserved state, numpy (nf, N) / flat, or a CUDA float64 torch tensor (copied).
    """

    def __init__(self, grid: dict, params: dict, X0, device="cuda:0", stream=None):
        import torch

        self._torch = torch
        if not torch.cuda.is_available():
            raise RuntimeError("mc_tvd needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load_library()
        self.grid, self.params = dict(grid), dict(params)
        self.nf = 4 if int(grid["ndim"]) == 2 else 5
        self.N = int(grid["nx"]) * int(grid.get("ny", 1)) * int(grid["nz"])
        self.nz = int(grid["nz"])
        self.device = torch.device(device)
        self._g, self._p = make_grid(grid), make_params(params)
        wb = self.lib.mc_tvd_workspace_bytes(C.byref(self._g), C.byref(self._p))
        if wb == 0:
            raise MCTVDError(-1, self.lib.mc_tvd_last_error().decode())
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
            self.fields = torch.empty(self.nf * self.N, dtype=torch.float64, device=self.device)
            self.workspace = torch.empty((wb + 7) // 8, dtype=torch.float64, device=self.device)
            self.set_state(X0)
            h = C.c_void_p()
            rc = self.lib.mc_tvd_init(C.byref(self._g), C.byref(self._p), self.fields.data_ptr(),
                                      self.workspace.data_ptr(), self.workspace.numel() * 8,
                                      self.stream.cuda_stream, C.byref(h))
        self._h = h
        self._check(rc)

    # -- helpers ------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise MCTVDError(rc, self.lib.mc_tvd_last_error().decode())

    def set_state(self, X0):
        """Copy a state into the device fields (does NOT recompute dt; init does that)."""
        torch = self._torch
        if isinstance(X0, torch.Tensor):
            src = X0.to(dtype=torch.float64).reshape(-1)
        else:
            src = torch.from_numpy(np.ascontiguousarray(X0, dtype=np.float64).reshape(-1))
        assert src.numel() == self.nf * self.N, (src.numel(), self.nf, self.N)
        with torch.cuda.stream(self.stream):
            self.fields.copy_(src, non_blocking=False)

    # -- the C ABI, one method per call ---------------------------------------------------------
    def step(self, n_steps: int = 1):
        self._check(self.lib.mc_tvd_step(self._h, int(n_steps)))

    def sweep(self, alpha: int, direction: int, tau: float):
        self._check(self.lib.mc_tvd_sweep(self._h, int(alpha), int(direction), float(tau)))

    def debug_set_chunk(self, levels: int):
        self._check(self.lib.mc_tvd_debug_set_chunk(self._h, int(levels)))

    def debug_geometry(self, alpha: int):
        """(outputs per tile along x, along the second tile direction, levels per chunk) of L_alpha's last launch."""
        tx, tb, ch = C.c_int(), C.c_int(), C.c_int()
        self._check(self.lib.mc_tvd_debug_geometry(self._h, int(alpha), C.byref(tx), C.byref(tb), C.byref(ch)))
        return tx.value, tb.value, ch.value

    def step_host(self, h_in, h_out, n_steps: int):
        """h_in / h_out: CPU float64 torch tensors (pinned for async copies) or numpy arrays."""
        self._check(self.lib.mc_tvd_step_host(self._h, _host_ptr(h_in), _host_ptr(h_out), int(n_steps)))

    def dt(self) -> float:
        v = C.c_double()
        self._check(self.lib.mc_tvd_dt(self._h, C.byref(v)))
        return v.value

    def diagnostics(self):
        """Returns (dict of scalars, T_prof, rho_prof, p_prof) -- same shape as the oracle's."""
        d = Diag()
        Tp, rp, pp = np.zeros(self.nz), np.zeros(self.nz), np.zeros(self.nz)
        self._check(self.lib.mc_tvd_diagnostics(self._h, C.byref(d), Tp.ctypes.data_as(_DP),
                                                rp.ctypes.data_as(_DP), pp.ctypes.data_as(_DP)))
        return {n: getattr(d, n) for n, _ in Diag._fields_}, Tp, rp, pp

    def stats_reset(self):
        self._check(self.lib.mc_tvd_stats_reset(self._h))

    def step_stats(self, n_steps: int, every: int = 1):
        self._check(self.lib.mc_tvd_step_stats(self._h, int(n_steps), int(every)))

    def stats_read(self):
        """Returns (dict of time averages, <T>_{A,t}, <rho>_{A,t}, <p>_{A,t}) -- same shape as the oracle's."""
        st = Stats()
        Tp, rp, pp = np.zeros(self.nz), np.zeros(self.nz), np.zeros(self.nz)
        self._check(self.lib.mc_tvd_stats_read(self._h, C.byref(st), Tp.ctypes.data_as(_DP), rp.ctypes.data_as(_DP),
                                               pp.ctypes.data_as(_DP)))
        return {n: getattr(st, n) for n, _ in Stats._fields_}, Tp, rp, pp

    def flow_stats(self):
        """Returns (dict of the force-balance averages of Eqs. 40-43 and the extrema, histogram of r as int64[HIST_BINS])."""
        f = Forces()
        hist = np.zeros(HIST_BINS, dtype=np.int64)
        self._check(self.lib.mc_tvd_flow_stats(self._h, C.byref(f), hist.ctypes.data_as(C.POINTER(C.c_longlong))))
        return {n: getattr(f, n) for n, _ in Forces._fields_}, hist

    def stats_flow(self, enable: bool = True):
        self._check(self.lib.mc_tvd_stats_flow(self._h, int(bool(enable))))

    def stats_read_flow(self):
        """Time averages of the flow statistics since the last stats_reset: (dict, summed histogram)."""
        f = Forces()
        hist = np.zeros(HIST_BINS, dtype=np.int64)
        self._check(self.lib.mc_tvd_stats_read_flow(self._h, C.byref(f), hist.ctypes.data_as(C.POINTER(C.c_longlong))))
        return {n: getattr(f, n) for n, _ in Forces._fields_}, hist

    # -- slab decomposition hooks (used by paper_2411_10372_b200.slab) ------------------------------------------
    def slab_op(self, op: int):
        self._check(self.lib.mc_tvd_slab_op(self._h, int(op)))

    def slab_reduce(self):
        self._check(self.lib.mc_tvd_slab_reduce(self._h))

    def slab_commit(self, advance: bool):
        self._check(self.lib.mc_tvd_slab_commit(self._h, int(bool(advance))))

    def slab_buffers(self):
        """Device addresses of the handle's two state buffers (d_fields, its copy in the workspace)."""
        a, b = C.c_void_p(), C.c_void_p()
        self._check(self.lib.mc_tvd_slab_buffers(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def slab_peers(self, lo, hi, own_lo: int, own_hi: int, halo: int):
        """lo / hi: slab_buffers() of the ranks below / above (None, None switches the fused halo push off)."""
        if lo is None and hi is None:
            self._check(self.lib.mc_tvd_slab_peers(self._h, None, None, None, None, 0, 0, 0))
        else:
            self._check(self.lib.mc_tvd_slab_peers(self._h, lo[0], lo[1], hi[0], hi[1], int(own_lo), int(own_hi), int(halo)))

    def _view(self, ptr: int, count: int, dtype):
        """A torch view of `count` 8-byte elements at device address ptr, which lies inside self.fields or self.workspace."""
        for t in (self.fields, self.workspace):
            off = ptr - t.data_ptr()
            if 0 <= off and off + 8 * count <= t.numel() * 8:
                assert off % 8 == 0
                return t[off // 8: off // 8 + count].view(dtype)
        raise RuntimeError("pointer outside the handle's buffers")

    def slab_views(self):
        """(state buffer now as (nf, nz, ny, nx), running-maximum bits as int64[1], plane sums (nz, 11), plane extrema (nz, 3))."""
        torch = self._torch
        p = [C.c_void_p() for _ in range(4)]
        self._check(self.lib.mc_tvd_slab_pointers(self._h, *[C.byref(x) for x in p]))
        g = self.grid
        f = self._view(p[0].value, self.nf * self.N, torch.float64).view(self.nf, self.nz, int(g.get("ny", 1)), int(g["nx"]))
        return (f, self._view(p[1].value, 1, torch.int64), self._view(p[2].value, self.nz * 11, torch.float64).view(self.nz, 11),
                self._view(p[3].value, self.nz * 3, torch.float64).view(self.nz, 3))

    def slab_diag_partial(self, axis: int, lo: int, hi: int):
        self._check(self.lib.mc_tvd_slab_diag_partial(self._h, int(axis), int(lo), int(hi)))

    def slab_diag_finish(self, nplane_global: float):
        d = Diag()
        Tp, rp, pp = np.zeros(self.nz), np.zeros(self.nz), np.zeros(self.nz)
        self._check(self.lib.mc_tvd_slab_diag_finish(self._h, float(nplane_global), C.byref(d), Tp.ctypes.data_as(_DP),
                                                     rp.ctypes.data_as(_DP), pp.ctypes.data_as(_DP)))
        return {n: getattr(d, n) for n, _ in Diag._fields_}, Tp, rp, pp

    def launch_count(self) -> int:
        return int(self.lib.mc_tvd_launch_count(self._h))

    def timing_enable(self, enable: bool = True):
        self._check(self.lib.mc_tvd_timing_enable(self._h, int(bool(enable))))

    def timing_read(self):
        """{kernel name: (ms_sum, count)} of the operator launches recorded since the last read."""
        ms = (C.c_double * 6)()
        cnt = (C.c_longlong * 6)()
        self._check(self.lib.mc_tvd_timing_read(self._h, ms, cnt))
        names = ["Lx+", "Ly+", "Lz+", "Lx-", "Ly-", "Lz-"]
        return {names[k]: (ms[k], int(cnt[k])) for k in range(6) if cnt[k]}

    def state(self) -> np.ndarray:
        """Download the current state as numpy (nf, N).  Synchronises."""
        self.stream.synchronize()
        return self.fields.cpu().numpy().reshape(self.nf, self.N)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.mc_tvd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr(a) -> int:
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.device.type == "cpu" and a.is_contiguous()
    return a.data_ptr()
