"""GPU: the slab decomposition (paper_2411_10372_b200/slab.py over the mc_tvd_slab_* hooks) against the
undivided box.  All slabs live on this one GPU and run one after the other (`LocalComm`: device copies instead of NCCL
send/recv; the driver and the kernels are the ones a multi-GPU run uses)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2411_10372_b200 import inputs, slab
from tests.helpers import parity_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2411_10372_b200 import binding
    binding.load_library()
    return binding


@pytest.mark.parametrize("ndim,nx,ny,nz,world,stretch", [
    (3, 64, 48, 33, 2, None), (3, 60, 84, 19, 4, None), (3, 45, 36, 17, 3, 1.5),
    (2, 480, 1, 65, 4, None), (2, 366, 1, 40, 3, 1.5)])
def test_slabs_match_the_undivided_box(gpu, orc, ndim, nx, ny, nz, world, stretch):
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=stretch)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.moving_state(grid, params, amplitude=1e-2, u_amp=0.1)
    one = gpu.MCTVD(grid, params, X0)
    drv = slab.make_local_driver(gpu, grid, params, X0, world)
    n = 4
    for _ in range(n):
        # the all-reduced maximum; bit for bit when the local box reproduces the spacing exactly (slab._length_with_spacing)
        assert drv.dt() == pytest.approx(one.dt(), rel=4e-16)
        one.step(1)
        drv.step(1)
    ref = one.state()
    got = slab.gather_state(drv.local_states(), grid)
    # the same kernels on the same numbers; only a tile's position relative to the seam differs (fast / general loop body)
    assert parity_err(grid, params, got, ref).max() <= 1e-13
    d1, T1, r1, p1 = one.diagnostics()
    d2, T2, r2, p2 = drv.diagnostics()
    for k in ("nu_bottom", "nu_top", "nu_bar", "nu_bulk", "re", "mass", "energy", "max_mach", "min_rho", "min_T"):
        assert d2[k] == pytest.approx(d1[k], rel=1e-10), k
    assert d2["time"] == pytest.approx(d1["time"], rel=1e-15) and d2["step"] == d1["step"] == n
    assert np.allclose(T2, T1, rtol=1e-12) and np.allclose(r2, r1, rtol=1e-12) and np.allclose(p2, p1, rtol=1e-12)
    # against the oracle too (the undivided box), so that the comparison above is not two wrongs agreeing
    want, _, _ = orc.step(orc.Problem(grid, params), X0, n)
    assert parity_err(grid, params, got, want).max() <= 4e-12
    one.close()
    for r in drv.ranks:
        r.close()


@pytest.mark.parametrize("nx,ny,nz,world", [(64, 48, 33, 2), (60, 84, 19, 4), (56, 8, 12, 1)])
def test_fused_halo_push_matches_the_undivided_box(gpu, orc, nx, ny, nz, world):
    """mc_tvd_slab_peers: the sweep kernels store their owned rows and push the boundary rows into the neighbours' halos
    themselves; no copies between the launches, the CFL maximum reduced inside the last operator over the owned rows."""
    grid = inputs.make_grid(3, nx, nz, ny)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.moving_state(grid, params, amplitude=1e-2, u_amp=0.1)
    one = gpu.MCTVD(grid, params, X0)
    drv = slab.make_local_driver(gpu, grid, params, X0, world, fused=True)
    assert drv.fused
    n = 4
    for _ in range(n):
        assert drv.dt() == pytest.approx(one.dt(), rel=4e-16)
        one.step(1)
        drv.step(1)
    got = slab.gather_state(drv.local_states(), grid)
    assert parity_err(grid, params, got, one.state()).max() <= 1e-13
    want, _, _ = orc.step(orc.Problem(grid, params), X0, n)
    assert parity_err(grid, params, got, want).max() <= 4e-12
    for r, st in enumerate(drv.local_states()):              # the halo rows hold the neighbours' rows (pushed by them)
        assert parity_err(slab.local_grid(grid, world)[0], params, st, slab.scatter_state(got, grid, r, world)).max() <= 1e-15
    d1, d2 = one.diagnostics()[0], drv.diagnostics()[0]
    for k in ("nu_bar", "nu_bulk", "re", "mass"):
        assert d2[k] == pytest.approx(d1[k], rel=1e-10), k
    one.close()
    for r in drv.ranks:
        r.close()


def test_fused_halo_push_is_refused_where_it_is_not_built(gpu):
    for grid in (inputs.make_grid(2, 64, 17), inputs.make_grid(3, 45, 17, 24), inputs.make_grid(3, 32, 17, 24, z_stretch=1.5)):
        params = inputs.make_params()
        X0 = inputs.conduction_state(grid, params)
        with pytest.raises(gpu.MCTVDError) as e:
            slab.make_local_driver(gpu, grid, params, X0, 2, fused=True)
        assert e.value.code == -5


def _ipc_worker(rank: int, world: int, port: int, out_dir: str, fused: bool):
    """One slab per PROCESS (both on cuda:0; host barriers only, no kernel waits on another process's kernel)."""
    import os
    import sys
    import torch
    import torch.distributed as dist
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    from paper_2411_10372_b200 import binding
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    grid = inputs.make_grid(3, 64, 33, 48)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.moving_state(grid, params, amplitude=1e-2, u_amp=0.1)
    drv = slab.make_dist_driver(binding, grid, params, X0, device="cuda:0", fused=fused)
    dts = []
    for _ in range(3):
        dts.append(drv.dt())
        drv.step(1)
    d = drv.diagnostics()[0]
    np.save(os.path.join(out_dir, f"state{rank}.npy"), drv.local_states()[0])
    np.save(os.path.join(out_dir, f"dts{rank}.npy"), np.array(dts + [d["nu_bar"], d["mass"]]))
    dist.barrier()
    for r in drv.ranks:
        r.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("fused", [False, True])
def test_one_slab_per_process(gpu, tmp_path, fused):
    """Two processes, one slab each, a gloo group between them: `DistComm` with send / recv of the halo rows (fused =
    False) and with the fused halo push into the neighbour PROCESS's buffers opened through CUDA IPC (fused = True).
    Both must reproduce the undivided box."""
    import torch.multiprocessing as mp
    import os
    port = 26000 + (os.getpid() * 3 + int(fused)) % 3000
    mp.spawn(_ipc_worker, args=(2, port, str(tmp_path), fused), nprocs=2, join=True)
    grid = inputs.make_grid(3, 64, 33, 48)
    params = inputs.make_params(Ra=1e5)
    X0 = inputs.moving_state(grid, params, amplitude=1e-2, u_amp=0.1)
    one = gpu.MCTVD(grid, params, X0)
    dts = []
    for _ in range(3):
        dts.append(one.dt())
        one.step(1)
    d = one.diagnostics()[0]
    parts = [np.load(tmp_path / f"state{r}.npy") for r in range(2)]
    got = slab.gather_state(parts, grid)
    assert parity_err(grid, params, got, one.state()).max() <= 1e-13
    for r in range(2):
        rec = np.load(tmp_path / f"dts{r}.npy")
        assert np.allclose(rec[:3], dts, rtol=4e-16, atol=0)
        assert rec[3] == pytest.approx(d["nu_bar"], rel=1e-10) and rec[4] == pytest.approx(d["mass"], rel=1e-12)
    one.close()


def test_bench_slabs_mode_runs_under_a_one_rank_nccl_group():
    """bench.py --slabs through torch.distributed with the NCCL backend and a world of one rank (this box has one GPU):
    the DistComm code path (process group, all_reduce of the CFL maximum, the local wrap of the halos) end to end."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(24000 + os.getpid() % 3000))
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--slabs", "--workload", "C1", "--steps", "5",
                          "--warmup", "3"], capture_output=True, text=True, timeout=600, cwd=root, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    rec = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert rec["scaling"] == "strong" and rec["n_gpus"] == 1 and rec["value"] > 0 and rec["state_check"]["dt"] > 0
    ref = subprocess.run([sys.executable, "-c",
                          "from paper_2411_10372_b200 import binding, inputs\n"
                          "g, p, _ = inputs.config('C1'); s = binding.MCTVD(g, p, inputs.conduction_state(g, p)); s.step(8); print(repr(s.dt()))"],
                         capture_output=True, text=True, timeout=600, cwd=root)
    assert ref.returncode == 0, ref.stderr[-2000:]
    assert rec["state_check"]["dt"] == pytest.approx(float(ref.stdout.strip().splitlines()[-1]), rel=1e-14)   # 3 + 5 steps


def test_slab_hooks_reject_misuse(gpu):
    grid = inputs.make_grid(3, 16, 9, 12)
    params = inputs.make_params()
    s = gpu.MCTVD(grid, params, inputs.conduction_state(grid, params))
    with pytest.raises(gpu.MCTVDError):
        s.slab_op(1)                                     # operators come in order
    s.slab_op(0)
    with pytest.raises(gpu.MCTVDError):
        s.slab_reduce()                                  # mid-step: the state is not in d_fields
    with pytest.raises(gpu.MCTVDError):
        s.slab_commit(True)
    for op in range(1, 6):
        s.slab_op(op)
    s.slab_reduce()
    s.slab_commit(True)
    assert s.diagnostics()[0]["step"] == 1
    s.close()
