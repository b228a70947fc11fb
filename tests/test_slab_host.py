"""Host logic of the slab decomposition (paper_2411_10372_b200/slab.py), no GPU:
  * cutting and re-assembling the state, the halo exchange and the all-reduces of both communicators -- `LocalComm` in
    process and `DistComm` over torch.distributed with the gloo backend, world size 2 and 3;
  * the decomposition itself -- halo width 2, one exchange after every operator, the global CFL maximum -- run with
    the CPU oracle standing in for the per-slab kernels: the slab driver must reproduce the undivided box bit for bit.
"""
from __future__ import annotations

import os
import sys

import numpy as np
import pytest
import torch

from paper_2411_10372_b200 import inputs, slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_local_grid_scatter_gather_round_trip():
    g = inputs.make_grid(3, 6, 5, 12)
    gl, own = slab.local_grid(g, 3)
    assert own == 4 and gl["ny"] == 8 and gl["ly"] == pytest.approx(g["ly"] * 8 / 12) and gl["nx"] == 6
    X = np.arange(5 * 6 * 5 * 12, dtype=np.float64).reshape(5, -1)
    parts = [slab.scatter_state(X, g, r, 3) for r in range(3)]
    assert parts[0].shape == (5, 5 * 8 * 6)
    p0 = parts[0].reshape(5, 5, 8, 6)
    full = X.reshape(5, 5, 12, 6)
    assert np.array_equal(p0[:, :, :2], full[:, :, 10:12]) and np.array_equal(p0[:, :, 2:6], full[:, :, 0:4])
    assert np.array_equal(slab.gather_state(parts, g), X)
    g2 = inputs.make_grid(2, 12, 5)
    assert slab.slab_axis(g2) == "x" and slab.local_grid(g2, 2)[0]["nx"] == 10
    X2 = np.arange(4 * 5 * 12, dtype=np.float64).reshape(4, -1)
    assert np.array_equal(slab.gather_state([slab.scatter_state(X2, g2, r, 2) for r in range(2)], g2), X2)
    with pytest.raises(ValueError):
        slab.local_grid(g, 5)
    with pytest.raises(ValueError):
        slab.local_grid(g, 6)                    # 2 owned rows < twice the halo


def _stale(parts, gl, dim):
    """local states with their halo rows overwritten by rubbish, as (nf, nz, ny, nx) tensors"""
    out = []
    for p in parts:
        t = torch.from_numpy(p.copy()).view(p.shape[0], gl["nz"], gl["ny"], gl["nx"])
        t.narrow(dim, 0, 2).fill_(-7.0)
        t.narrow(dim, t.shape[dim] - 2, 2).fill_(-9.0)
        out.append(t)
    return out


@pytest.mark.parametrize("ndim,world", [(3, 2), (3, 3), (2, 2), (2, 4)])
def test_local_comm_exchange_restores_the_halos(ndim, world):
    g = inputs.make_grid(ndim, 24, 5, 12)
    nf = 4 if ndim == 2 else 5
    X = np.random.default_rng(1).normal(size=(nf, inputs.num_nodes(g)))
    gl, own = slab.local_grid(g, world)
    dim = 2 if ndim == 3 else 3
    parts = [slab.scatter_state(X, g, r, world) for r in range(world)]
    t = _stale(parts, gl, dim)
    comm = slab.LocalComm(world)
    comm.exchange(t, dim, 2, own)
    for r in range(world):
        assert np.array_equal(t[r].numpy().reshape(nf, -1), parts[r])
    a = [torch.tensor([3 + r], dtype=torch.int64) for r in range(world)]
    comm.allreduce(a, "max")
    assert all(int(x) == 2 + world for x in a)
    b = [torch.full((4, 3), float(r + 1)) for r in range(world)]
    comm.allreduce([x[:, 0] for x in b], "sum")
    assert all(float(x[0, 0]) == world * (world + 1) / 2 and float(x[0, 1]) == r + 1 for r, x in enumerate(b))


def _dist_worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    g = inputs.make_grid(3, 8, 5, 12)
    X = np.random.default_rng(2).normal(size=(5, inputs.num_nodes(g)))
    gl, own = slab.local_grid(g, world)
    want = slab.scatter_state(X, g, rank, world)
    t = _stale([want], gl, 2)
    comm = slab.DistComm()
    comm.exchange(t, 2, 2, own)
    ok_halo = bool(np.array_equal(t[0].numpy().reshape(5, -1), want))
    bits = torch.tensor([np.float64(1.5 + rank).view(np.int64)], dtype=torch.int64)
    comm.allreduce([bits], "max")
    sums = torch.full((4, 3), float(rank + 1), dtype=torch.float64)
    comm.allreduce([sums[:, 0]], "sum")
    comm.allreduce([sums[:, 1:]], "min")
    ok = ok_halo and bits.numpy().view(np.float64)[0] == 1.5 + world - 1 and float(sums[2, 0]) == world * (world + 1) / 2 \
        and float(sums[1, 2]) == 1.0
    with open(os.path.join(out_dir, f"r{rank}.txt"), "w") as f:
        f.write("ok" if ok else f"bad halo={ok_halo} bits={bits} sums={sums}")
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_dist_comm_gloo(tmp_path, world):
    import torch.multiprocessing as mp
    port = 23000 + (os.getpid() * 7 + world) % 4000
    mp.spawn(_dist_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        assert open(tmp_path / f"r{r}.txt").read() == "ok"


class OracleRank:
    """The CPU oracle behind the slab_* interface of binding.MCTVD (tests only): one slab's local periodic box."""

    def __init__(self, orc, grid_local, params, X_local):
        self.orc, self.prob, self.g, self.p = orc, orc.Problem(grid_local, params), grid_local, params
        nf = X_local.shape[0]
        self.f = torch.from_numpy(X_local.copy()).view(nf, grid_local["nz"], grid_local["ny"], grid_local["nx"])
        self.bits = torch.zeros(1, dtype=torch.int64)
        self.dt_now, self.time = float("nan"), 0.0

    def slab_views(self):
        return self.f, self.bits, None, None

    def slab_op(self, op):
        nd = self.g["ndim"]
        alpha = (2 if op % 2 == 0 else 0) if nd == 2 else 2 - (op % 3)         # Eq. 30: L_z, [L_y,] L_x, twice
        direction = -1 if (op // nd == 1 and self.p["dir_mode"] == 1) else +1
        X = self.f.numpy().reshape(self.f.shape[0], -1)
        Y = self.orc.sweep(self.prob, X, alpha, 0.5 * self.dt_now, direction)
        self.f.copy_(torch.from_numpy(Y).view_as(self.f))

    def slab_reduce(self):
        s = self.orc.max_speed(self.prob, self.f.numpy().reshape(self.f.shape[0], -1))
        self.bits[0] = max(int(self.bits[0]), int(np.float64(s).view(np.int64)))

    def slab_commit(self, advance):
        if advance:
            self.time += self.dt_now
        self.dt_now = self.p["cfl"] / float(self.bits.numpy().view(np.float64)[0])
        self.bits[0] = 0

    def dt(self):
        return self.dt_now

    def state(self):
        return self.f.numpy().reshape(self.f.shape[0], -1).copy()


@pytest.mark.parametrize("ndim,nx,ny,nz,world,stretch", [(3, 10, 12, 7, 3, None), (3, 6, 8, 9, 2, 1.5), (2, 24, 1, 9, 3, None),
                                                         (2, 16, 1, 7, 2, 1.5)])
def test_slab_driver_reproduces_the_undivided_box(orc, ndim, nx, ny, nz, world, stretch):
    """Halo 2, one exchange per operator, global CFL maximum: with the oracle as the per-slab operator the owned rows
    after three steps equal the undivided oracle run bit for bit, and every dt is the global one."""
    grid = inputs.make_grid(ndim, nx, nz, ny, z_stretch=stretch)
    params = inputs.make_params(Ra=1e4)
    X0 = inputs.rough_random_state(grid, params, seed=3)
    ref, dts, t_ref = orc.step(orc.Problem(grid, params), X0, 3)
    gl, own = slab.local_grid(grid, world)
    ranks = [OracleRank(orc, gl, params, slab.scatter_state(X0, grid, r, world)) for r in range(world)]
    drv = slab.SlabDriver(ranks, slab.LocalComm(world), grid)
    used = []
    for _ in range(3):
        used.append(drv.dt())
        drv.step(1)
    assert np.array_equal(np.array(used), dts)
    assert all(r.dt_now == ranks[0].dt_now for r in ranks) and ranks[0].time == pytest.approx(t_ref, rel=1e-15)
    got = slab.gather_state(drv.local_states(), grid)
    assert np.array_equal(got, ref)
    # and the halo rows hold the neighbours' rows again
    for r, rk in enumerate(ranks):
        assert np.array_equal(rk.state(), slab.scatter_state(ref, grid, r, world))
