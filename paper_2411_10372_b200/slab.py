"""Slab decomposition of one box over several GPUs (the paper's multi-GPU runs, PAPER.md:313-315 and
App. A, which exchange halos with mpi4py).

Plumbing only: every operator, reduction and diagnostic runs in the kernels behind the C ABI (include/mc_tvd.h, "Slab
decomposition"); this module cuts the state into slabs, refreshes the halo rows after every operator and all-reduces
three small device buffers.

Decomposition: the box is cut along a periodic horizontal direction -- y in 3-D, x in 2-D; z stays whole, so plates,
the z-march and the plane sums stay local to a column.  A rank's local box holds the rows it owns plus H = 2 halo rows
on either side and is treated as periodic by its handle.  Every operator L_alpha reaches 2 nodes along and across the
slab axis (SURVEY 8a "stencil footprint"), so one operator spoils exactly the outermost 2 rows of the local box, i.e.
halo rows only; they are refreshed from the neighbours' owned rows after EVERY operator (6 exchanges per 3-D step, each
2 rows x nx x nz x nf doubles per side).  The step's CFL reduction runs after the last exchange over the whole local box
(halo copies included: harmless for a maximum) and is all-reduced (MAX) before the handles form dt, so every rank
holds the same dt bit for bit.  Diagnostics: per-plane sums over the owned rows, all-reduced (SUM / MAX / MIN), then
the usual finish kernel with the global node count.

Two communicators share the driver: `DistComm` (one slab per process, torch.distributed send/recv and all_reduce:
NCCL over NVLink on GPUs, gloo in the CPU tests) and `LocalComm` (all slabs in this process, device copies: the
single-GPU emulation the tests and a one-GPU box use; the slabs run one after the other, nothing waits on another kernel).
"""
from __future__ import annotations

import numpy as np

HALO = 2


def slab_axis(grid: dict) -> str:
    return "y" if int(grid["ndim"]) == 3 else "x"


def local_grid(grid: dict, world: int, halo: int = HALO):
    """(grid of one rank's local box, owned rows per rank).  The slab axis must divide evenly."""
    ax = slab_axis(grid)
    n = int(grid["n" + ax])
    if n % world:
        raise ValueError(f"n{ax} = {n} is not a multiple of the number of slabs {world}")
    own = n // world
    if own < 2 * halo:
        raise ValueError(f"{own} owned rows per slab are fewer than twice the halo")
    g = dict(grid)
    g["n" + ax] = own + 2 * halo
    g["l" + ax] = _length_with_spacing(float(grid["l" + ax]) / n, own + 2 * halo)
    return g, own


def _length_with_spacing(d: float, n: int) -> float:
    """A box length L with L / n == d in fp64 where one exists (it usually does): the library forms its spacing as
    length / nodes, and with the undivided box's spacing reproduced to the last bit the slabs return the undivided
    result bit for bit, dt included.  Otherwise d n, whose spacing is off by one ulp (results then agree to ~1e-16)."""
    L = d * n
    for _ in range(8):
        q = L / n
        if q == d:
            return L
        L = float(np.nextafter(L, np.inf if q < d else -np.inf))
    return d * n


def _as4(X, grid):
    nf = 4 if int(grid["ndim"]) == 2 else 5
    return X.reshape(nf, int(grid["nz"]), int(grid.get("ny", 1)), int(grid["nx"]))


def scatter_state(X: np.ndarray, grid: dict, rank: int, world: int, halo: int = HALO) -> np.ndarray:
    """Rows [rank own - halo, (rank + 1) own + halo) of the global state along the slab axis, periodic: (nf, N_local)."""
    gl, own = local_grid(grid, world, halo)
    dim = 2 if slab_axis(grid) == "y" else 3
    n = int(grid["n" + slab_axis(grid)])
    idx = (np.arange(rank * own - halo, (rank + 1) * own + halo)) % n
    return np.ascontiguousarray(np.take(_as4(X, grid), idx, axis=dim)).reshape(X.shape[0], -1)


def gather_state(parts, grid: dict, halo: int = HALO) -> np.ndarray:
    """The global state from the ranks' local states (their owned rows), in rank order."""
    world = len(parts)
    gl, own = local_grid(grid, world, halo)
    dim = 2 if slab_axis(grid) == "y" else 3
    owned = [np.take(_as4(p, gl), np.arange(halo, halo + own), axis=dim) for p in parts]
    return np.ascontiguousarray(np.concatenate(owned, axis=dim)).reshape(parts[0].shape[0], -1)


class LocalComm:
    """All slabs live in this process (one GPU, or the CPU in tests): neighbours are list neighbours."""

    def __init__(self, world: int):
        self.world, self.rank0 = world, 0

    def exchange(self, fields, dim: int, halo: int, own: int):
        """fields: one (nf, nz, ny, nx) tensor per slab.  Low halo <- left neighbour's last owned rows, high halo <- right
        neighbour's first owned rows (periodic in rank)."""
        w = self.world
        lo = [f.narrow(dim, halo, halo).clone() for f in fields]                 # first owned rows
        hi = [f.narrow(dim, own, halo).clone() for f in fields]                  # last owned rows
        for r, f in enumerate(fields):
            f.narrow(dim, 0, halo).copy_(hi[(r - 1) % w])
            f.narrow(dim, halo + own, halo).copy_(lo[(r + 1) % w])

    def neighbour_buffers(self, ranks):
        """Per slab: the (d_fields, second buffer) device addresses of the slab below and of the slab above."""
        bufs = [r.slab_buffers() for r in ranks]
        w = len(ranks)
        return [(bufs[(i - 1) % w], bufs[(i + 1) % w]) for i in range(w)]

    def barrier(self, tensors):
        """Every slab's queued work has finished (one device and one stream: stream order already says so)."""
        import torch
        devs = {t.device for t in tensors if t.is_cuda}
        if len(devs) > 1:
            for d in devs:
                torch.cuda.synchronize(d)

    def allreduce(self, tensors, op: str):
        import torch
        red = {"max": torch.maximum, "min": torch.minimum, "sum": torch.add}[op]
        tot = tensors[0].clone()
        for t in tensors[1:]:
            tot = red(tot, t.to(tot.device))
        for t in tensors:
            t.copy_(tot)


class DistComm:
    """One slab per process: torch.distributed point-to-point for the halos, all_reduce for the three small buffers."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world, self.rank0 = dist.get_world_size(group), dist.get_rank(group)

    def exchange(self, fields, dim: int, halo: int, own: int):
        import torch
        dist, (f,) = self.dist, fields
        left, right = (self.rank0 - 1) % self.world, (self.rank0 + 1) % self.world
        lo = f.narrow(dim, halo, halo).contiguous()
        hi = f.narrow(dim, own, halo).contiguous()
        if f.is_cuda and self.world > 1 and dist.get_backend(self.group) == "gloo":
            lo, hi = lo.cpu(), hi.cpu()          # gloo moves host memory only (tests; NCCL sends device memory)
        if self.world == 1:
            f.narrow(dim, 0, halo).copy_(hi)
            f.narrow(dim, halo + own, halo).copy_(lo)
            return
        if left == right:                       # two ranks: one message per direction carries both row blocks
            send = torch.stack([lo, hi])
            recv = torch.empty_like(send)
            ops = [dist.P2POp(dist.isend, send, left, self.group), dist.P2POp(dist.irecv, recv, left, self.group)]
            for r in dist.batch_isend_irecv(ops):
                r.wait()
            from_lo, from_hi = recv[0], recv[1]                # the neighbour's first and last owned rows
        else:
            from_hi, from_lo = torch.empty_like(hi), torch.empty_like(lo)
            ops = [dist.P2POp(dist.isend, lo, left, self.group), dist.P2POp(dist.isend, hi, right, self.group),
                   dist.P2POp(dist.irecv, from_hi, left, self.group), dist.P2POp(dist.irecv, from_lo, right, self.group)]
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        f.narrow(dim, 0, halo).copy_(from_hi)                  # left neighbour's last owned rows
        f.narrow(dim, halo + own, halo).copy_(from_lo)         # right neighbour's first owned rows

    def neighbour_buffers(self, ranks):
        """The neighbouring PROCESSES' state buffers, opened through CUDA IPC (torch's tensor sharing): each rank
        publishes its two tensors, opens those of the ranks below and above and returns their addresses in its own
        address space.  Same node only; on several GPUs the mapping is peer memory, the stores travel over NVLink."""
        from torch.multiprocessing.reductions import reduce_tensor
        (r,) = ranks
        X, Y = r.slab_buffers()
        if self.world == 1:
            return [((X, Y), (X, Y))]
        mine = (reduce_tensor(r.fields), reduce_tensor(r.workspace), X - r.fields.data_ptr(), Y - r.workspace.data_ptr())
        everyone = [None] * self.world
        self.dist.all_gather_object(everyone, mine, group=self.group)
        self._ipc = []                                       # keep the opened tensors alive as long as the driver
        out = []
        for nb in ((self.rank0 - 1) % self.world, (self.rank0 + 1) % self.world):
            (ff, fa), (wf, wa), offx, offy = everyone[nb]
            tf, tw = ff(*fa), wf(*wa)
            self._ipc += [tf, tw]
            out.append((tf.data_ptr() + offx, tw.data_ptr() + offy))
        return [(out[0], out[1])]

    def barrier(self, tensors):
        """Every rank's queued work has finished: the operator's pushes have landed before anyone reads them."""
        import torch
        for t in tensors:
            if t.is_cuda:
                torch.cuda.synchronize(t.device)
        self.dist.barrier(group=self.group)

    def allreduce(self, tensors, op: str):
        dist, (t,) = self.dist, tensors
        red = {"max": dist.ReduceOp.MAX, "min": dist.ReduceOp.MIN, "sum": dist.ReduceOp.SUM}[op]
        on_host = t.is_cuda and dist.get_backend(self.group) == "gloo"     # (the CPU tests' backend, and the two-process-one-GPU test)
        buf = t.detach().cpu().contiguous() if on_host else t.contiguous()
        dist.all_reduce(buf, op=red, group=self.group)
        if on_host or buf.data_ptr() != t.data_ptr():
            t.copy_(buf)


class SlabDriver:
    """Runs the local slabs `ranks` (objects with the slab_* methods of binding.MCTVD) as one box through `comm`."""

    def __init__(self, ranks, comm, grid: dict, halo: int = HALO, fused: bool = False):
        self.ranks, self.comm, self.grid, self.halo = list(ranks), comm, dict(grid), halo
        self.dim = 2 if slab_axis(grid) == "y" else 3
        _, self.own = local_grid(grid, comm.world, halo)
        self.nops = 2 * int(grid["ndim"])
        self.fused = False
        if fused:
            self.enable_fused()
        self._refresh_dt(advance=False)        # the initial dt must be the global one

    def enable_fused(self):
        """Fused halo push (include/mc_tvd.h): every operator writes its boundary rows straight into the neighbours' halo
        rows, so nothing is exchanged between the launches.  The neighbours' buffers are addressed directly: slabs of this
        process (`LocalComm`) or of neighbouring processes through CUDA IPC (`DistComm`); raises where the library does
        not support it (2-D, odd nx, non-uniform z)."""
        for r, (lo, hi) in zip(self.ranks, self.comm.neighbour_buffers(self.ranks)):
            r.slab_peers(lo, hi, self.halo, self.halo + self.own, self.halo)
        self.fused = True

    def _fields(self):
        return [r.slab_views()[0] for r in self.ranks]

    def _refresh_dt(self, advance: bool):
        for r in self.ranks:
            r.slab_reduce()
        # positive doubles order like their bit patterns (NaN, a bad state, orders above +inf)
        self.comm.allreduce([r.slab_views()[1] for r in self.ranks], "max")
        for r in self.ranks:
            r.slab_commit(advance)

    def step(self, n_steps: int = 1):
        for _ in range(n_steps):
            for op in range(self.nops):
                for r in self.ranks:
                    r.slab_op(op)
                if self.fused:
                    self.comm.barrier(self._fields())      # the kernels have pushed the halos themselves
                else:
                    self.comm.exchange(self._fields(), self.dim, self.halo, self.own)
            if self.fused:                                  # the last operator reduced the maximum over the owned rows
                self.comm.allreduce([r.slab_views()[1] for r in self.ranks], "max")
                for r in self.ranks:
                    r.slab_commit(True)
            else:
                self._refresh_dt(advance=True)

    def dt(self) -> float:
        return self.ranks[0].dt()

    def diagnostics(self):
        """Global diagnostics (dict, T, rho, p profiles): identical on every rank."""
        axis = 1 if self.dim == 2 else 0
        for r in self.ranks:
            r.slab_diag_partial(axis, self.halo, self.halo + self.own)
        views = [r.slab_views() for r in self.ranks]
        self.comm.allreduce([v[2] for v in views], "sum")
        self.comm.allreduce([v[3][:, 0] for v in views], "max")
        self.comm.allreduce([v[3][:, 1:] for v in views], "min")
        nplane = float(self.grid["nx"]) * float(self.grid.get("ny", 1))
        out = [r.slab_diag_finish(nplane) for r in self.ranks]
        return out[0]

    def local_states(self):
        return [r.state() for r in self.ranks]


def make_local_driver(binding, grid: dict, params: dict, X0: np.ndarray, n_slabs: int, device="cuda:0", devices=None,
                      fused: bool = False):
    """All slabs driven by this process.  One device (default): the slabs run one after the other, the single-GPU
    emulation of the multi-GPU path.  devices = ["cuda:0", "cuda:1", ...] (one per slab): a single process drives several
    GPUs and `LocalComm`'s copies become peer-to-peer copies over NVLink (never run here: this box has one GPU)."""
    gl, _ = local_grid(grid, n_slabs)
    devs = list(devices) if devices is not None else [device] * n_slabs
    assert len(devs) == n_slabs
    ranks = [binding.MCTVD(gl, params, scatter_state(X0, grid, r, n_slabs), device=devs[r]) for r in range(n_slabs)]
    return SlabDriver(ranks, LocalComm(n_slabs), grid, fused=fused)


def make_dist_driver(binding, grid: dict, params: dict, X0: np.ndarray, device, group=None, fused: bool = False):
    """One slab per process of an initialised torch.distributed group (NCCL: one process per GPU).  fused: the halo push
    inside the sweep kernels through CUDA-IPC-mapped neighbour buffers instead of send / recv between the launches."""
    comm = DistComm(group)
    gl, _ = local_grid(grid, comm.world)
    rank = binding.MCTVD(gl, params, scatter_state(X0, grid, comm.rank0, comm.world), device=device)
    return SlabDriver([rank], comm, grid, fused=fused)
