"""mc_tvd_cfl_noalloc (include/mc_tvd.h): the CFL reduction for callers that cannot allocate -- its scratch is a fixed
device array inside the library instead of a caller's workspace.  Checked against the existing path (the reduction a
handle runs at mc_tvd_init, read back with mc_tvd_dt) on calls in a row that share the scratch array, against the CPU
oracle, and for the size limit.  Collected last on purpose (the suite runs with pytest -x): it must pass alone in a
fresh process and after every other test."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_DT = 4e-16          # the dt tolerance of tests/test_gpu_stretched.py and tests/test_gpu_slab.py


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


def _cases():
    """(grid, params, state): a 3-D uniform box spanning many blocks, a 2-D stretched box (the tables in the scratch
    array), a small 3-D stretched box with other parameters."""
    out = []
    g = inputs.make_grid(3, 60, 33, 44)
    p = inputs.make_params(Ra=1e5)
    out.append((g, p, inputs.rough_random_state(g, p, seed=31)))
    g = inputs.make_grid(2, 300, 70, z_stretch=1.5)
    p = inputs.make_params(Ra=1e4, cfl=0.3)
    out.append((g, p, inputs.rough_random_state(g, p, seed=32)))
    g = inputs.make_grid(3, 10, 9, 6, z_stretch=2.5)
    p = inputs.make_params(Ra=1e6, gamma=1.4, D=0.5)
    out.append((g, p, inputs.conduction_state(g, p, amplitude=1e-2)))
    return out


def test_two_calls_in_a_row_match_the_handle_path(gpu, orc):
    import torch
    dev = torch.device("cuda:0")
    cases = _cases()
    want = []
    for g, p, X in cases:                                   # the existing path: the reduction of mc_tvd_init
        s = gpu.MCTVD(g, p, X)
        want.append(s.dt())
        s.close()
    outs = [torch.full((2,), -1.0, dtype=torch.float64, device=dev) for _ in range(2 * len(cases))]
    fields = [torch.from_numpy(np.ascontiguousarray(X).reshape(-1)).to(dev) for _, _, X in cases]
    keep = [f.clone() for f in fields]
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated(dev)
    # back to back on one stream, no synchronisation in between (the stretched cases synchronise in the binding, the
    # uniform one does not), then the whole sequence again: every call finds the scratch as the last one left it
    for rep in range(2):
        for i, (g, p, _) in enumerate(cases):
            gpu.cfl_noalloc(g, p, fields[i], outs[rep * len(cases) + i])
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == mem0         # nothing went through torch's allocator either
    for rep in range(2):
        for i, (g, p, X) in enumerate(cases):
            s_max, dt = outs[rep * len(cases) + i].tolist()
            assert dt == pytest.approx(want[i], rel=TOL_DT), (rep, i)
            assert s_max == pytest.approx(p["cfl"] / want[i], rel=1e-15), (rep, i)      # (dt = cfl / s, rounded twice)
            assert dt == pytest.approx(orc.dt(orc.Problem(g, p), X), rel=TOL_DT), (rep, i)
    for f, k in zip(fields, keep):
        assert torch.equal(f, k)                            # the state is read only


def test_a_smaller_maximum_follows_a_larger_one(gpu):
    """The running maximum in the shared array must not survive a call: a state at rest after a fast one."""
    import torch
    g = inputs.make_grid(2, 64, 17)
    p = inputs.make_params(Ra=1e4)
    fast = inputs.rough_random_state(g, p, seed=5, rough=0.2)
    rest = inputs.conduction_state(g, p, amplitude=0.0)
    dts = []
    for X in (fast, rest):
        s = gpu.MCTVD(g, p, X)
        dts.append(s.dt())
        s.close()
    assert dts[1] > dts[0]
    out = torch.zeros(2, 2, dtype=torch.float64, device="cuda:0")
    for i, X in enumerate((fast, rest)):
        gpu.cfl_noalloc(g, p, torch.from_numpy(X.reshape(-1)).cuda(), out[i])
    torch.cuda.synchronize()
    assert out[0, 1].item() == pytest.approx(dts[0], rel=TOL_DT) and out[1, 1].item() == pytest.approx(dts[1], rel=TOL_DT)
    # fixed_dt overrides, as in a handle
    gpu.cfl_noalloc(g, dict(p, fixed_dt=1e-3), torch.from_numpy(rest.reshape(-1)).cuda(), out[0])
    torch.cuda.synchronize()
    assert out[0, 1].item() == 1e-3 and out[0, 0].item() == pytest.approx(p["cfl"] / dts[1], rel=1e-15)


def test_non_positive_density_gives_nan_and_the_next_call_is_clean(gpu):
    import torch
    g = inputs.make_grid(2, 32, 9)
    p = inputs.make_params(Ra=1e4)
    X = inputs.conduction_state(g, p, amplitude=1e-3)
    bad = X.copy()
    bad[0, 77] = -1.0
    out = torch.zeros(2, 2, dtype=torch.float64, device="cuda:0")
    gpu.cfl_noalloc(g, p, torch.from_numpy(bad.reshape(-1)).cuda(), out[0])
    gpu.cfl_noalloc(g, p, torch.from_numpy(X.reshape(-1)).cuda(), out[1])
    torch.cuda.synchronize()
    assert np.isnan(out[0, 0].item()) and np.isnan(out[0, 1].item())
    s = gpu.MCTVD(g, p, X)
    assert out[1, 1].item() == pytest.approx(s.dt(), rel=TOL_DT)
    s.close()


def test_sizes_beyond_the_scratch_array_are_refused(gpu):
    import torch
    p = inputs.make_params(Ra=1e4)
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda:0")
    for nz, ok in ((gpu.NOALLOC_MAX_NZ, True), (gpu.NOALLOC_MAX_NZ + 1, False)):
        g = inputs.make_grid(2, 4, nz, z_stretch=1.5)        # the tables fill the array to its last level
        X = inputs.conduction_state(g, p, amplitude=0.0)
        f = torch.from_numpy(X.reshape(-1)).cuda()
        if ok:
            gpu.cfl_noalloc(g, p, f, out)
            torch.cuda.synchronize()
            s = gpu.MCTVD(g, p, X)
            assert out[1].item() == pytest.approx(s.dt(), rel=TOL_DT)
            s.close()
            out.fill_(-1.0)
        else:
            with pytest.raises(gpu.MCTVDError) as e:
                gpu.cfl_noalloc(g, p, f, out)
            assert e.value.code == -5 and "MC_TVD_NOALLOC_MAX_NZ" in str(e.value)
            torch.cuda.synchronize()
            assert out.tolist() == [-1.0, -1.0]             # nothing was enqueued
    g = inputs.make_grid(2, 16, 9)
    X = inputs.conduction_state(g, p)
    with pytest.raises(gpu.MCTVDError) as e:                # an invalid problem is refused as in mc_tvd_init
        gpu.cfl_noalloc(dict(g, z_nodes=np.linspace(1.0, 0.0, 9)), p, torch.from_numpy(X.reshape(-1)).cuda(), out)
    assert e.value.code == -1
