"""Multi-GPU slab decomposition of the pressure projection.

The paper splits the Cartesian domain into slabs with one halo layer and solves the implicit and the elliptic
problems across ranks with all-to-all transposes, staged through the host.  Here: one process per
GPU over `torch.distributed` (NCCL across NVLink / NVSwitch), device buffers only.  A rank owns

  * planes [k0, k1) of u, v, w, p, phi (a z-slab)  -> divergence, x and y transforms, correction are local (a1-a3, a5-a7);
    the divergence needs the neighbour's first w plane, the correction the neighbour's last phi plane (one halo layer);
  * x-slots [s0, s1) of the packed spectrum for every row and every plane -> the z tridiagonals are local (a4).

Between the two sits one exchange each way.  In the slab spectrum [nzl][ny][N] a destination's slots are a strided slice
(packed once); in the pencil [nz][ny][nsl] a source's planes are CONTIGUOUS, so received chunks land in place and the way
back sends views without packing.

This module holds only plumbing: index ranges, buffers, packing copies, send/recv lists.  Every arithmetic step runs in
the kernels of libfsei behind `binding.SlabPlan` (fsei_slab_forward / fsei_pencil_solve / fsei_slab_backward /
fsei_slab_project).  `DistComm` runs the exchanges over a process group; `LocalComm` delivers them by copies between
the ranks of ONE process that are stepped stage by stage (no kernel of one rank ever waits on another's) -- used to
check the decomposition against the single-plan projection on one GPU.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def split(n: int, world: int) -> List[Tuple[int, int]]:
    """Balanced contiguous ranges [lo, hi) of n items over `world` ranks (every rank non-empty needs n >= world)."""
    return [(n * r // world, n * (r + 1) // world) for r in range(world)]


class SlabExchange:
    """Buffers and send/recv lists of one rank.  Pure torch: usable on CPU tensors (gloo tests) and on the GPU."""

    def __init__(self, nx: int, ny: int, nz: int, rank: int, world: int, device, dtype=None):
        import torch
        if nz < world or nx // 2 < world:
            raise ValueError("every rank needs at least one plane and one x-slot")
        self.nx, self.ny, self.nz, self.N = nx, ny, nz, nx // 2
        self.rank, self.world = rank, world
        self.kr, self.sr = split(nz, world), split(self.N, world)
        self.k0, self.k1 = self.kr[rank]
        self.s0, self.s1 = self.sr[rank]
        self.nzl, self.nsl = self.k1 - self.k0, self.s1 - self.s0
        dt = dtype or torch.float64
        mk = lambda *shape: torch.zeros(shape, dtype=dt, device=device)
        self.spec = mk(self.nzl, ny, self.N, 2)                       # slab spectrum (also the rhs of the x transform)
        self.pencil = mk(nz, ny, self.nsl, 2)                         # full z columns of this rank's slots
        self.send = [mk(self.nzl, ny, s1 - s0, 2) for (s0, s1) in self.sr]          # slab -> pencil: packed slices
        self.recv = [mk(self.nzl, ny, s1 - s0, 2) for (s0, s1) in self.sr]          # pencil -> slab: chunks per source
        self.w_ext = mk(self.nzl + 1, ny, nx)                         # w with the plane above (zeros at the top wall)
        self.phi_ext = mk(self.nzl + 2, ny, nx)                       # phi with the planes below and above

    # ---- halo of w (before a1): my first plane goes down, the neighbour's first plane arrives on top ----------
    def w_halo(self):
        sends = [(self.w_ext[0], self.rank - 1)] if self.rank > 0 else []
        recvs = [(self.w_ext[self.nzl], self.rank + 1)] if self.rank + 1 < self.world else []
        return sends, recvs

    # ---- slab spectrum -> pencils (between a3 and a4) ----------------------------------------------------------
    def to_pencils(self, src=None):
        """src: a slab array [nzl][ny][N][2] other than the spectrum (a real field read as pairs: the viscous z sweep)."""
        src = self.spec if src is None else src
        sends, recvs = [], []
        for d, (s0, s1) in enumerate(self.sr):
            self.send[d].copy_(src[:, :, s0:s1, :])
            sends.append((self.send[d], d))
        for s, (k0, k1) in enumerate(self.kr):
            recvs.append((self.pencil[k0:k1], s))                     # contiguous: lands in place
        return sends, recvs

    # ---- pencils -> slab spectrum (between a4 and a5) ------------------------------------------------------------
    def to_slabs(self):
        sends = [(self.pencil[k0:k1], d) for d, (k0, k1) in enumerate(self.kr)]   # contiguous views, no packing
        recvs = [(self.recv[s], s) for s in range(self.world)]
        return sends, recvs

    def unpack_slabs(self, dst=None):
        dst = self.spec if dst is None else dst
        for s, (s0, s1) in enumerate(self.sr):
            dst[:, :, s0:s1, :].copy_(self.recv[s])

    # ---- one halo layer of whole fields (explicit terms): exts = arrays [nzl + 2][ny][nx], own planes at 1 .. nzl --------
    def field_halos(self, exts):
        sends, recvs = [], []
        for e in exts:
            if self.rank > 0:
                sends.append((e[1], self.rank - 1)); recvs.append((e[0], self.rank - 1))
            if self.rank + 1 < self.world:
                sends.append((e[self.nzl], self.rank + 1)); recvs.append((e[self.nzl + 1], self.rank + 1))
        return sends, recvs

    # ---- halo of phi (before a7): my last plane goes up; with beta != 0 my first plane also goes down ---------
    def phi_halo(self, both: bool):
        sends, recvs = [], []
        if self.rank + 1 < self.world:
            sends.append((self.phi_ext[self.nzl], self.rank + 1))
        if self.rank > 0:
            recvs.append((self.phi_ext[0], self.rank - 1))
        if both:
            if self.rank > 0:
                sends.append((self.phi_ext[1], self.rank - 1))
            if self.rank + 1 < self.world:
                recvs.append((self.phi_ext[self.nzl + 1], self.rank + 1))
        return sends, recvs


class DistComm:
    """Exchanges over a torch.distributed process group: grouped point-to-point operations (NCCL fuses a batch into one
    all-to-all-like launch over NVLink / NVSwitch; gloo runs them on CPU tensors in the tests)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def exchange(self, sends, recvs):
        # gloo moves host memory only: device tensors are staged through host copies (the paper's own transport, P:L202-204;
        # here only so that the multi-process path can be exercised on a box with one GPU).  NCCL takes device tensors as is.
        stage = self.dist.get_backend(self.group) == "gloo"
        ops, landed = [], []
        for t, src in recvs:
            if src == self.rank:
                continue
            buf = t
            if stage and t.is_cuda:
                buf = t.new_empty(t.shape, device="cpu")
                landed.append((t, buf))
            ops.append(self.dist.P2POp(self.dist.irecv, buf, src, self.group))
        for t, dst in sends:
            if dst == self.rank:                                        # my own share: a local copy
                mine = [r for r, src in recvs if src == self.rank]
                mine[0].copy_(t)
                continue
            ops.append(self.dist.P2POp(self.dist.isend, t.cpu() if (stage and t.is_cuda) else t, dst, self.group))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()
        for t, buf in landed:
            t.copy_(buf)

    def fence(self):
        """All kernels enqueued so far on every rank have completed (peer stores included)."""
        import torch
        if torch.cuda.is_available():
            torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier(self.group)

    def ipc_buffers(self, x: "SlabExchange"):
        """(pencil_ptrs, spec_ptrs) of all ranks of ONE NODE as mapped into this process through CUDA IPC handles (the
        handles travel as pickled objects over the process group; torch opens them with cudaIpcOpenMemHandle).  The mapped
        tensors are kept alive on `x`.  Arguments of SlabProjection.set_peers."""
        from torch.multiprocessing.reductions import reduce_tensor
        mine = [reduce_tensor(x.pencil), reduce_tensor(x.spec)]
        allh = [None] * self.world
        self.dist.all_gather_object(allh, mine, group=self.group)
        keep, pencils, specs = [], [], []
        for r, (hp, hs) in enumerate(allh):
            tp, ts = (x.pencil, x.spec) if r == self.rank else (hp[0](*hp[1]), hs[0](*hs[1]))
            keep += [tp, ts]
            pencils.append(tp.data_ptr()); specs.append(ts.data_ptr())
        x._ipc_keepalive = keep
        return pencils, specs

    @staticmethod
    def symmetric_buffers(x: "SlabExchange", group=None):
        """Re-allocate a rank's pencil and slab spectrum in torch symmetric memory and return (pencil_ptrs, spec_ptrs) of all
        ranks as mapped into this process -- the arguments of SlabProjection.set_peers on a multi-GPU node."""
        import torch
        import torch.distributed._symmetric_memory as symm
        name = group.group_name if group is not None else torch.distributed.group.WORLD.group_name
        ptrs = []
        for attr in ("pencil", "spec"):
            old = getattr(x, attr)
            t = symm.empty(old.shape, dtype=old.dtype, device=old.device)
            h = symm.rendezvous(t, name)
            setattr(x, attr, t)
            ptrs.append([int(p) for p in h.buffer_ptrs])
        return ptrs[0], ptrs[1]


class LocalComm:
    """All ranks live in this process and are stepped stage by stage; an exchange is a set of copies.  For checking the
    decomposition on one GPU -- not a way to run it: the ranks run one after the other."""

    @staticmethod
    def exchange_all(lists: Sequence[Tuple[list, list]]):
        """lists[r] = (sends, recvs) of rank r.  Message from s to d = the next unmatched send of s addressed to d."""
        world = len(lists)
        queues = {(s, d): [t for t, dst in lists[s][0] if dst == d] for s in range(world) for d in range(world)}
        for d in range(world):
            for t, src in lists[d][1]:
                t.copy_(queues[(src, d)].pop(0))
        assert all(len(q) == 0 for q in queues.values()), "unmatched send"


class SlabProjection:
    """One rank of the decomposed projection: fields of the local slab + the stages around the exchanges."""

    def __init__(self, grid, rank: int, world: int, device="cuda"):
        import torch
        from .binding import SlabPlan
        nx, ny, nz = grid[0], grid[1], grid[2]
        self.x = SlabExchange(nx, ny, nz, rank, world, device)
        self.plan = SlabPlan(grid, self.x.k0, self.x.k1, self.x.s0, self.x.s1)
        nzl = self.x.nzl
        self.u = torch.zeros((nzl, ny, nx), dtype=torch.float64, device=device)
        self.v = torch.zeros_like(self.u)
        self.p = torch.zeros_like(self.u)
        self.w = self.x.w_ext[:nzl]                                   # the halo plane follows it in memory
        self.phi = self.x.phi_ext[1:nzl + 1]                          # the halo planes surround it in memory
        self.launches = 0
        self.peers = False

    def set_peers(self, pencil_ptrs, spec_ptrs):
        """Peer-store exchange: device addresses of every rank's pencil and slab spectrum (own buffers included; peers'
        buffers as mapped into this process).  The two all-to-all exchanges then happen inside the kernels' epilogues."""
        x = self.x
        self.plan.set_peers(pencil_ptrs, spec_ptrs, [k for k, _ in x.kr] + [x.nz], [a for a, _ in x.sr] + [x.N])
        self.peers = True

    def load(self, u, v, w, p=None):
        """Local planes [k0, k1) of global (or already local) host / device arrays."""
        import torch
        k0, k1 = self.x.k0, self.x.k1
        for dst, src in ((self.u, u), (self.v, v), (self.w, w), (self.p, p)):
            if src is None:
                dst.zero_()
                continue
            t = torch.as_tensor(src)
            dst.copy_(t[k0:k1] if t.shape[0] == self.x.nz else t)

    # stages: each returns the (sends, recvs) that must be exchanged before the next one
    def stage_w_halo(self):
        return self.x.w_halo()

    def stage_forward(self, alpha_dt, stream=None):
        self.plan.slab_forward(self.u, self.v, self.w, alpha_dt, self.x.spec, stream)
        self.launches += self.plan.last_launch_count
        return ([], []) if self.peers else self.x.to_pencils()          # peers: the y-transform stored into the owners' pencils

    def stage_solve(self, stream=None):
        self.plan.pencil_solve(self.x.pencil, stream)
        self.launches += self.plan.last_launch_count
        return ([], []) if self.peers else self.x.to_slabs()            # peers: the back substitution stored into the owners' spectra

    def stage_backward(self, beta, stream=None):
        if not self.peers:
            self.x.unpack_slabs()
        self.plan.slab_backward(self.x.spec, self.phi, stream)
        self.launches += self.plan.last_launch_count
        return self.x.phi_halo(both=beta != 0.0)

    def stage_project(self, alpha_dt, beta, stream=None):
        self.plan.slab_project(self.u, self.v, self.w, self.p, self.phi, alpha_dt, beta, stream)
        self.launches += self.plan.last_launch_count

    def project(self, comm: DistComm, alpha_dt, beta=0.0, stream=None):
        """The whole projection of this rank, exchanges over `comm` (all ranks call it together)."""
        comm.exchange(*self.stage_w_halo())
        comm.exchange(*self.stage_forward(alpha_dt, stream))
        if self.peers:
            comm.fence()                                    # every rank's stores into my pencil have landed
        comm.exchange(*self.stage_solve(stream))
        if self.peers:
            comm.fence()                                    # ... and into my slab spectrum
        comm.exchange(*self.stage_backward(beta, stream))
        self.stage_project(alpha_dt, beta, stream)

    def destroy(self):
        self.plan.destroy()


class SlabFluid(SlabProjection):
    """One rank of the decomposed fluid substep: explicit terms (one halo layer of u, v, w, p), implicit viscous step (x and
    y sweeps on the slab, z sweep on pencils: P:L248) and the projection.  Plumbing only, as above."""

    def __init__(self, grid, rank: int, world: int, device="cuda"):
        import torch
        super().__init__(grid, rank, world, device)
        nx, ny, nzl = self.x.nx, self.x.ny, self.x.nzl
        mk = lambda: torch.zeros((nzl + 2, ny, nx), dtype=torch.float64, device=device)
        self.ext = [mk() for _ in range(4)]                            # u, v, w, p with the planes below and above
        self.u, self.v, self.w, self.p = (e[1:nzl + 1] for e in self.ext)
        self.h = [torch.zeros((nzl, ny, nx), dtype=torch.float64, device=device) for _ in range(3)]
        self.r = [torch.zeros_like(self.h[0]) for _ in range(3)]
        self.f = (None, None, None)

    def stage_w_halo(self):
        x = self.x
        sends = [(self.w[0], x.rank - 1)] if x.rank > 0 else []
        recvs = [(self.ext[2][x.nzl + 1], x.rank + 1)] if x.rank + 1 < x.world else []
        return sends, recvs

    def stage_halos(self):
        """One halo layer of u, v, w, p on each side."""
        return self.x.field_halos(self.ext)

    def stage_explicit(self, gamma_dt, rho_dt, alpha_dt, beta, stream=None):
        self.plan.explicit_terms(self.u, self.v, self.w, self.p, *self.h, *self.r, gamma_dt, rho_dt, alpha_dt, beta,
                                 f=self.f, stream=stream)
        self.launches += self.plan.last_launch_count
        self.plan.slab_viscous_xy(*self.r, beta, stream)
        self.launches += self.plan.last_launch_count

    def _pairs(self, c):
        return self.r[c].view(self.x.nzl, self.x.ny, self.x.N, 2)

    def stage_visc_to_pencils(self, c):
        return self.x.to_pencils(self._pairs(c))

    def stage_visc_z(self, c, beta, stream=None):
        self.plan.pencil_viscous_z(self.x.pencil, c, beta, stream)
        self.launches += self.plan.last_launch_count
        return self.x.to_slabs()

    def stage_visc_add(self, c, stream=None):
        self.x.unpack_slabs(self._pairs(c))
        self.plan.slab_field_add((self.u, self.v, self.w)[c], self.r[c], stream)
        self.launches += self.plan.last_launch_count

    def substep(self, comm: DistComm, gamma_dt, rho_dt, alpha_dt, beta, stream=None):
        """One substep of this rank, exchanges over `comm` (all ranks call it together).  The viscous z sweeps exchange by
        explicit send/recv lists also when the projection uses peer stores."""
        comm.exchange(*self.stage_halos())
        self.stage_explicit(gamma_dt, rho_dt, alpha_dt, beta, stream)
        for c in range(3):
            comm.exchange(*self.stage_visc_to_pencils(c))
            comm.exchange(*self.stage_visc_z(c, beta, stream))
            self.stage_visc_add(c, stream)
        self.project(comm, alpha_dt, beta, stream)


def substep_local(ranks: Sequence["SlabFluid"], gamma_dt, rho_dt, alpha_dt, beta):
    """All ranks in one process, stage by stage (LocalComm)."""
    LocalComm.exchange_all([r.stage_halos() for r in ranks])
    for r in ranks:
        r.stage_explicit(gamma_dt, rho_dt, alpha_dt, beta)
    for c in range(3):
        LocalComm.exchange_all([r.stage_visc_to_pencils(c) for r in ranks])
        LocalComm.exchange_all([r.stage_visc_z(c, beta) for r in ranks])
        for r in ranks:
            r.stage_visc_add(c)
    project_local(ranks, alpha_dt, beta)


def local_peers(ranks: Sequence[SlabProjection]):
    """All ranks in one process: every rank's buffers are ordinary device allocations of this process."""
    pencils = [r.x.pencil.data_ptr() for r in ranks]
    specs = [r.x.spec.data_ptr() for r in ranks]
    for r in ranks:
        r.set_peers(pencils, specs)


def project_local(ranks: Sequence[SlabProjection], alpha_dt, beta=0.0):
    """All ranks in one process, stage by stage (LocalComm).  With peers set, the forward and solve stages of ALL ranks store
    into each other's buffers and the stage order is the fence."""
    LocalComm.exchange_all([r.stage_w_halo() for r in ranks])
    LocalComm.exchange_all([r.stage_forward(alpha_dt) for r in ranks])
    LocalComm.exchange_all([r.stage_solve() for r in ranks])
    LocalComm.exchange_all([r.stage_backward(beta) for r in ranks])
    for r in ranks:
        r.stage_project(alpha_dt, beta)
