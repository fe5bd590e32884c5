"""Host-side plumbing of the z-slab decomposition (include/flutas.h, flutas_slab_*).

The data path is entirely in the library's kernels: the two all-to-all transposes of PAPER.md:169-183 are the store
stages of the y transform and of the z stage, written straight into the peers' memory.  What is left for the host is
  * the partition (which planes / which rows of ky a rank owns) -- `partition`,
  * making every rank's exchange buffer addressable by every other rank -- one process: plain device pointers
    (`SlabGroup`); one process per GPU under torchrun: torch symmetric memory (`SlabRank`),
  * a stream-ordered barrier between the three phases of a step (`SlabRank`: an NCCL all-reduce of one element),
  * refreshing the halo planes a step does not produce (plane 0 of w, both halo planes of phi) -- `exchange_halos`.
No arithmetic of the method happens here.
"""
import torch
import torch.distributed as dist

from .binding import SlabPlan


def partition(nz, ny, n_ranks, rank):
    """(planes, rows): the half-open ranges of z planes and of ky rows (storage order) that `rank` owns"""
    if nz % n_ranks or ny % n_ranks or not (0 <= rank < n_ranks):
        raise ValueError("n_ranks must divide nz and ny, 0 <= rank < n_ranks")
    nzl, rpp = nz // n_ranks, ny // n_ranks
    return (rank * nzl, (rank + 1) * nzl), (rank * rpp, (rank + 1) * rpp)


def forward_destination(k, j, nz, ny, n_ranks):
    """where the forward transpose puts element (plane k, row j): (rank, plane, local row) of the z-local spectra"""
    rpp = ny // n_ranks
    return j // rpp, k, j % rpp


def backward_destinations(k, j, nz, ny, n_ranks, periodic):
    """where the backward transpose puts element (plane k, row j): a list of (rank, local plane, row) of the slab spectra
    (local plane 1 .. nzl = the slab; 0 and nzl + 1 = the halo planes of the neighbours)"""
    nzl = nz // n_ranks
    r, loc = k // nzl, k % nzl
    out = [(r, loc + 1, j)]
    if loc == 0 and (r > 0 or periodic):
        out.append(((r - 1) % n_ranks, nzl + 1, j))
    if loc == nzl - 1 and (r + 1 < n_ranks or periodic):
        out.append(((r + 1) % n_ranks, 0, j))
    return out


def halo_neighbours(n_ranks, rank, periodic):
    """(below, above): the ranks that own the plane below / above `rank`'s slab; None beyond a wall"""
    below = rank - 1 if rank > 0 else (n_ranks - 1 if periodic else None)
    above = rank + 1 if rank + 1 < n_ranks else (0 if periodic else None)
    return below, above


def exchange_halos(w, phi, nzl, periodic, group=None):
    """Refresh the halo planes a step reads but does not produce (include/flutas.h, flutas_slab_*: "on entry the halo planes
    of phi (both) and of w (plane 0) must hold the neighbours' values") -- one rank per process, any backend, the local
    arrays of (nzl + 2) planes being CPU or CUDA tensors.  A step leaves p^(n+1) with its halos; u, v need none; w and phi
    are their producers' job, and in a time loop that applies steps back to back this is the producer.
    Every rank sends its top owned plane of w and of phi upwards and its bottom owned plane of phi downwards (pure data
    movement; point-to-point, two messages per neighbour pair).  Stream-ordered on NCCL like any collective."""
    grp = group if group is not None else dist.group.WORLD
    n_ranks, rank = dist.get_world_size(grp), dist.get_rank(grp)
    below, above = halo_neighbours(n_ranks, rank, periodic)
    wv, fv = w.view(nzl + 2, -1), phi.view(nzl + 2, -1)
    up = torch.stack((wv[nzl], fv[nzl]))                 # to the rank above: its plane 0 of w and of phi
    down = fv[1].clone()                                 # to the rank below: its plane nzl + 1 of phi
    if n_ranks == 1:
        if periodic:
            wv[0].copy_(up[0]); fv[0].copy_(up[1]); fv[nzl + 1].copy_(down)
        return
    from_below, from_above = torch.empty_like(up), torch.empty_like(down)
    peer = lambda r: dist.get_global_rank(grp, r)
    ops = []
    # upward messages first, on both sides, so that two messages between the same pair (n_ranks = 2) match in order
    if above is not None:
        ops.append(dist.P2POp(dist.isend, up, peer(above), grp, 0))
    if below is not None:
        ops.append(dist.P2POp(dist.irecv, from_below, peer(below), grp, 0))
        ops.append(dist.P2POp(dist.isend, down, peer(below), grp, 1))
    if above is not None:
        ops.append(dist.P2POp(dist.irecv, from_above, peer(above), grp, 1))
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    if below is not None:
        wv[0].copy_(from_below[0]); fv[0].copy_(from_below[1])
    if above is not None:
        fv[nzl + 1].copy_(from_above)


class SlabGroup:
    """All n_ranks of a decomposition driven by ONE process on the current device, phase by phase on one stream (what a
    single-GPU box can run: the ranks' kernels never wait for one another, stream order is the barrier)."""

    def __init__(self, nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, n_ranks):
        self.n_ranks = int(n_ranks)
        self.plans = [SlabPlan(nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, n_ranks, r) for r in range(n_ranks)]
        p0 = self.plans[0]
        self.nzl, self.npts_local = p0.nzl, p0.npts_local
        self.exchange = [torch.empty(p0.exchange_bytes, dtype=torch.uint8, device="cuda") for _ in range(n_ranks)]
        self.workspace = [torch.empty(p0.workspace_bytes, dtype=torch.uint8, device="cuda") for _ in range(n_ranks)]
        ptrs = [e.data_ptr() for e in self.exchange]
        for pl, ws in zip(self.plans, self.workspace):
            pl.attach(ws, ptrs, keep=self.exchange)
        torch.cuda.synchronize()

    def step(self, fields, dt, dt_ratio=1.0, p_out=None):
        """fields[r] = (u, v, w, phi, p, p_old) local tensors of rank r; p_out[r] defaults to p (in place)"""
        for phase in range(3):
            for r, pl in enumerate(self.plans):
                u, v, w, phi, p, po = fields[r]
                pl.step_phase(phase, u, v, w, phi, p, po, p if p_out is None else p_out[r], dt, dt_ratio)

    def exchange_halos(self, fields, periodic):
        """exchange_halos (above) for the one-process group: fields[r] = (u, v, w, phi, p, p_old); plane 0 of w and both halo
        planes of phi of every rank from the neighbours' owned planes, as copies on the current stream"""
        n, nzl = self.n_ranks, self.nzl
        for r in range(n):
            below, above = halo_neighbours(n, r, periodic)
            w, phi = fields[r][2].view(nzl + 2, -1), fields[r][3].view(nzl + 2, -1)
            if below is not None:
                w[0].copy_(fields[below][2].view(nzl + 2, -1)[nzl])
                phi[0].copy_(fields[below][3].view(nzl + 2, -1)[nzl])
            if above is not None:
                phi[nzl + 1].copy_(fields[above][3].view(nzl + 2, -1)[1])

    def destroy(self):
        for pl in self.plans:
            pl.destroy()
        self.plans = []


class SlabRank:
    """One rank per process (torchrun, NCCL): the exchange buffer comes from torch symmetric memory, so that every peer's
    buffer has an address in this process (NVLink peer mapping); the barrier between phases is an all-reduce of one
    element on the current stream."""

    def __init__(self, nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, group=None):
        if not (dist.is_available() and dist.is_initialized()):
            raise RuntimeError("SlabRank needs an initialised torch.distributed process group (torchrun)")
        import torch.distributed._symmetric_memory as symm
        self.group = group if group is not None else dist.group.WORLD
        self.n_ranks, self.rank = dist.get_world_size(self.group), dist.get_rank(self.group)
        self.plan = SlabPlan(nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, self.n_ranks, self.rank)
        self.nzl, self.npts_local = self.plan.nzl, self.plan.npts_local
        self.exchange = symm.empty(self.plan.exchange_bytes, dtype=torch.uint8, device="cuda")
        self._hdl = symm.rendezvous(self.exchange, self.group.group_name)
        self.workspace = torch.empty(self.plan.workspace_bytes, dtype=torch.uint8, device="cuda")
        self.plan.attach(self.workspace, list(self._hdl.buffer_ptrs), keep=(self.exchange, self._hdl))
        self._token = torch.zeros(1, device="cuda")
        torch.cuda.synchronize()
        dist.barrier(self.group)           # every rank has cleared its buffer before anyone writes into a peer's

    def barrier_on_stream(self):
        dist.all_reduce(self._token, group=self.group)

    def step(self, u, v, w, phi, p, p_old, dt, dt_ratio=1.0, p_out=None):
        for phase in range(3):
            self.plan.step_phase(phase, u, v, w, phi, p, p_old, p if p_out is None else p_out, dt, dt_ratio)
            if phase < 2:
                self.barrier_on_stream()

    def exchange_halos(self, w, phi):
        """refresh plane 0 of w and both halo planes of phi from the neighbours (see exchange_halos above); call between two
        steps of a loop that feeds a step's velocity back in"""
        exchange_halos(w, phi, self.nzl, self.plan.bc_z == 0, self.group)

    def destroy(self):
        self.plan.destroy()
