"""CPU-side checks of the boundary: libmc_tvd.so builds (nvcc cross-compiles without a GPU), loads, and
exports every symbol include/mc_tvd.h declares; host-only calls validate their arguments.  No compute
call is made here."""
from __future__ import annotations

import ctypes as C
import os
import re

import pytest

from paper_2411_10372_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "mc_tvd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mc_tvd_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    return binding.load_library()


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = _declared_functions()
    assert len(names) >= 9
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.SYMBOLS) == names          # the Python binding mirrors the header one to one


def test_struct_layouts_match_header():
    assert C.sizeof(binding.Diag) == 19 * 8
    assert C.sizeof(binding.Grid) == 4 * 4 + 3 * 8 + 8
    assert C.sizeof(binding.Params) == 13 * 8 + 5 * 4 + 4           # 13 doubles, 5 ints (co_mode the last), padded to 8
    assert C.sizeof(binding.Forces) == 16 * 8


def test_workspace_bytes_and_validation(lib):
    p = binding.make_params(inputs.make_params())
    for name in ("C1", "C5"):
        grid, _, _ = inputs.config(name)
        g = binding.make_grid(grid)
        wb = lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(p))
        nf = inputs.num_fields(grid)
        state = nf * inputs.num_nodes(grid) * 8
        assert state <= wb <= state + (64 << 20)                  # second buffer + small reduction scratch
    bad = binding.make_grid(inputs.make_grid(2, 64, 3))           # nz < 5
    assert lib.mc_tvd_workspace_bytes(C.byref(bad), C.byref(p)) == 0
    assert b"nz" in lib.mc_tvd_last_error()
    bad = binding.make_grid(inputs.make_grid(2, 64, 16))
    bad.ndim = 4
    assert lib.mc_tvd_workspace_bytes(C.byref(bad), C.byref(p)) == 0
    pb = binding.make_params(inputs.make_params(gamma=1.0))
    g = binding.make_grid(inputs.make_grid(2, 64, 16))
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(pb)) == 0
    pb = binding.make_params(inputs.make_params(tvd_form=2))
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(pb)) == 0
    pb = binding.make_params(inputs.make_params(co_mode=2))
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(pb)) == 0 and b"co_mode" in lib.mc_tvd_last_error()
    huge = binding.make_grid(inputs.make_grid(3, 2048, 1024, 2048))   # 2^32 nodes per field: 32-bit node offsets
    assert lib.mc_tvd_workspace_bytes(C.byref(huge), C.byref(p)) == 0
    assert b"2^32" in lib.mc_tvd_last_error()


def test_init_rejects_bad_arguments_before_touching_the_device(lib):
    g = binding.make_grid(inputs.make_grid(2, 64, 16))
    p = binding.make_params(inputs.make_params())
    h = C.c_void_p()
    assert lib.mc_tvd_init(C.byref(g), C.byref(p), None, None, 0, None, C.byref(h)) == -1      # NULL buffers
    assert lib.mc_tvd_init(C.byref(g), C.byref(p), None, None, 0, None, None) == -1            # NULL out
    z = (C.c_double * 16)()                                                                    # node heights all zero:
    g.z_nodes = C.cast(z, C.POINTER(C.c_double))                                               # not increasing
    assert lib.mc_tvd_init(C.byref(g), C.byref(p), None, None, 0, None, C.byref(h)) == -1
    assert b"increasing" in lib.mc_tvd_last_error()
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(p)) == 0
    for k in range(16):
        z[k] = k / 15.0
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(p)) > 0                              # a valid non-uniform grid
    pz = binding.make_params(inputs.make_params(bc_z=1))
    assert lib.mc_tvd_workspace_bytes(C.byref(g), C.byref(pz)) == 0                            # node heights need plates
    assert lib.mc_tvd_step(None, 1) == -1
    assert lib.mc_tvd_debug_set_chunk(None, 4) == -1
    assert lib.mc_tvd_sweep(None, 0, 1, 0.1) == -1
    assert lib.mc_tvd_dt(None, None) == -1
    assert lib.mc_tvd_diagnostics(None, None, None, None, None) == -1
    assert lib.mc_tvd_step_host(None, None, None, 1) == -1
    assert lib.mc_tvd_destroy(None) == 0
    assert lib.mc_tvd_launch_count(None) == 0


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2411_10372_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "mc_tvd_oracle" not in text, f


def test_no_cpu_fallback_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    grid = inputs.make_grid(2, 64, 16)
    params = inputs.make_params()
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.MCTVD(grid, params, inputs.conduction_state(grid, params))


def test_build_refuses_kernels_with_a_large_stack_frame():
    """A sweep kernel whose lambdas were not all inlined keeps its register pipeline in local memory (6x slower,
    seen once).  build.py parses ptxas -v and refuses such a build; the committed build's log must be clean."""
    from paper_2411_10372_b200 import build
    bad = ("ptxas info    : Compiling entry function '_ZN2mc8k_march3ILi2EEEvNS_9SweepArgsE' for 'sm_100a'\n"
           "    1472 bytes stack frame, 0 bytes spill stores, 0 bytes spill loads\n")
    with pytest.raises(RuntimeError, match="1472-byte stack frame"):
        build._check_stack_frames(bad)
    ok = bad.replace("1472 bytes", "40 bytes")
    build._check_stack_frames(ok)
    log = os.path.join(os.path.dirname(build.LIB_PATH), "build.log")
    if os.path.exists(log):
        build._check_stack_frames(open(log).read())


def test_every_kernel_source_is_a_build_dependency():
    """An edit to any file under csrc/ (or to the public header) must make load_library() rebuild the .so:
    the staleness check hashes the contents of exactly these files."""
    from paper_2411_10372_b200 import build
    deps = {os.path.basename(d) for d in build._deps()}
    csrc = os.path.join(ROOT, "paper_2411_10372_b200", "csrc")
    for f in os.listdir(csrc):
        assert f in deps, f
    assert "mc_tvd.h" in deps
    assert not build._stale()                                    # load_library() above built it from these sources
