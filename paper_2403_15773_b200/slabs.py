"""z-slab decomposition of one TSLB domain over several contexts / GPUs (include/tslb.h "z-slabs",
SURVEY §8(e); the paper's stated next step).

Plumbing only: which planes a rank owns, which face is a halo face, who the neighbours are, the
exchange of workspace handles and the per-step barrier.  The halo data itself is moved by the step
kernel (peer stores into the neighbour's ghost planes); nothing here touches field values.

  LocalSlabs  all slabs driven from this process (one GPU or several): tests, single-process runs
  RankSlab    one slab per torch.distributed rank (one process per GPU), CUDA IPC between processes
"""
import numpy as np

from . import tslb


def slab_ranges(nz, n, jet=False):
    """Balanced contiguous split of planes 0..nz-1 into n slabs -> [(z0, z1), ...] (z1 exclusive).
    Two planes per slab at least (the halo is two planes deep); three where a slab carries the inflow or
    the outflow plane (that plane is imposed, not pushed to the neighbour)."""
    if n < 1 or nz < 2 * n or (jet and n > 1 and nz // n < 3):
        raise ValueError("too few planes per slab: nz=%d, slabs=%d" % (nz, n))
    base, rem = divmod(nz, n)
    out, z = [], 0
    for r in range(n):
        w = base + (1 if r < rem else 0)
        out.append((z, z + w))
        z += w
    return out


def neighbor_plan(rank, n, jet):
    """-> dict(bc_zlo, bc_zhi, lo, hi): face types of slab `rank` of n and the ranks behind its halo
    faces (None where the face is a physical boundary).  Periodic z wraps around (a single periodic
    slab is its own neighbour)."""
    lo = rank - 1 if rank > 0 else (None if jet else n - 1)
    hi = rank + 1 if rank < n - 1 else (None if jet else 0)
    return dict(bc_zlo=tslb.BC_JET_INFLOW if lo is None else tslb.BC_HALO,
                bc_zhi=tslb.BC_OUTFLOW if hi is None else tslb.BC_HALO, lo=lo, hi=hi)


def _slice(a, z0, z1):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return np.ascontiguousarray(a[z0:z1])
    return a[z0:z1].contiguous()


class LocalSlabs:
    """n slabs of one (nz, ny, nx) domain, all driven by this process.  `devices` gives one CUDA
    ordinal per slab (default: all on device 0); with several devices every step ends with a
    synchronise of each device (the barrier of the protocol)."""

    def __init__(self, nx, ny, nz, omega, n_slabs, precision=tslb.F32, devices=None, jet=False, **kw):
        self.shape = (nz, ny, nx)
        self.ranges = slab_ranges(nz, n_slabs, jet)
        self.devices = list(devices) if devices is not None else [0] * n_slabs
        self.plans = [neighbor_plan(r, n_slabs, jet) for r in range(n_slabs)]
        self.sims = []
        for r, (z0, z1) in enumerate(self.ranges):
            pl = self.plans[r]
            self.sims.append(tslb.Tslb(nx, ny, z1 - z0, omega, precision=precision, device=self.devices[r],
                                       bc_zlo=pl["bc_zlo"], bc_zhi=pl["bc_zhi"], **kw))
        for r, s in enumerate(self.sims):
            pl = self.plans[r]
            if pl["lo"] is not None:
                s.attach_neighbor(0, self.sims[pl["lo"]])
            if pl["hi"] is not None:
                s.attach_neighbor(1, self.sims[pl["hi"]])
        self._multi = len(set(self.devices)) > 1

    def _sync(self):
        if self._multi:
            import torch
            for d in set(self.devices):
                torch.cuda.synchronize(d)

    def init_fields(self, rho, ux, uy, uz, phi=None, pineq=None):
        """Global (nz, ny, nx) arrays; each slab takes its planes."""
        for s, (z0, z1) in zip(self.sims, self.ranges):
            pq = None if pineq is None else [_slice(a, z0, z1) for a in pineq]
            s.init_fields(*[_slice(a, z0, z1) for a in (rho, ux, uy, uz)], _slice(phi, z0, z1), pq)
        self._sync()
        for s in self.sims:
            s.halo_push()
        self._sync()

    def step(self, n=1):
        for _ in range(int(n)):
            for s in self.sims:
                s.step(1)
            self._sync()

    def get_moments(self, **kw):
        parts = [s.get_moments(**kw) for s in self.sims]
        out = {}
        for k in parts[0]:
            if parts[0][k] is None:
                out[k] = None
            elif isinstance(parts[0][k], np.ndarray):
                out[k] = np.concatenate([p[k] for p in parts], axis=1 if k == "pineq" else 0)
            else:
                import torch
                out[k] = torch.cat([p[k] for p in parts], dim=1 if k == "pineq" else 0)
        return out

    @property
    def kernel_names(self):
        return [s.kernel_name for s in self.sims]

    @property
    def launch_count(self):
        return sum(s.launch_count for s in self.sims)

    def close(self):
        for s in self.sims:
            s.close()
        self.sims = []


def gather_neighbors(info, plan, dist=None):
    """all-gather every rank's `info` (any picklable object) and return the entries of this rank's
    lo / hi neighbours (None for a physical boundary).  Works with any backend."""
    if dist is None:
        import torch.distributed as dist
    infos = [None] * dist.get_world_size()
    dist.all_gather_object(infos, info)
    return (None if plan["lo"] is None else infos[plan["lo"]],
            None if plan["hi"] is None else infos[plan["hi"]])


class RankSlab:
    """This rank's slab of a (nz, ny, nx) domain split over the torch.distributed world (one process
    per GPU).  Workspaces are exchanged as CUDA IPC handles; the per-step barrier is a one-element
    all-reduce on the library's stream with the nccl backend (stream-ordered, no host sync), and a
    stream synchronise + host barrier otherwise."""

    def __init__(self, nx, ny, nz, omega, precision=tslb.F32, jet=False, device=0, **kw):
        import torch
        import torch.distributed as dist
        self._torch, self._dist = torch, dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.ranges = slab_ranges(nz, self.world, jet)
        self.z0, self.z1 = self.ranges[self.rank]
        self.plan = neighbor_plan(self.rank, self.world, jet)
        self.device = device
        self.sim = tslb.Tslb(nx, ny, self.z1 - self.z0, omega, precision=precision, device=device,
                             torch_workspace=False, bc_zlo=self.plan["bc_zlo"], bc_zhi=self.plan["bc_zhi"], **kw)
        lo, hi = gather_neighbors((self.sim.ipc_handle(), self.z1 - self.z0), self.plan, dist)
        me = (self.sim, self.z1 - self.z0)
        for face, nb, nb_rank in ((0, lo, self.plan["lo"]), (1, hi, self.plan["hi"])):
            if nb is None:
                continue
            if nb_rank == self.rank:                    # single periodic slab: its own neighbour
                self.sim.attach_neighbor(face, me[0])
            else:
                self.sim.attach_neighbor_ipc(face, nb[0], nb[1])
        self._nccl = dist.get_backend() == "nccl"
        self._flag = torch.zeros(1, device=torch.device("cuda", device)) if self._nccl else None

    def barrier(self):
        if self.world == 1:
            return
        if self._nccl:
            self._dist.all_reduce(self._flag)          # on the current stream = the library's stream
        else:
            self._torch.cuda.synchronize(self.device)
            self._dist.barrier()

    def init_fields(self, rho, ux, uy, uz, phi=None, pineq=None):
        """This rank's planes only: arrays of shape (z1 - z0, ny, nx)."""
        self.sim.init_fields(rho, ux, uy, uz, phi, pineq)
        self.barrier()
        self.sim.halo_push()
        self.barrier()

    def step(self, n=1):
        for _ in range(int(n)):
            self.sim.step(1)
            self.barrier()

    def get_moments(self, **kw):
        return self.sim.get_moments(**kw)

    def close(self):
        """Two phases: every rank closes the handles it imported, a barrier, then every rank frees its own
        workspace (freeing exported memory that an importer still has open is undefined behaviour)."""
        self._torch.cuda.synchronize(self.device)
        self.sim.detach_neighbors()
        if self.world > 1:
            self._dist.barrier()
        self.sim.close()
