"""z-slab decomposition over several GPUs: the plumbing around the lb_slab_* calls of include/lb.h.

The paper distributes the fluid box equally over its ranks; collision is local and
streaming reaches first neighbours only.  Here every rank (one process per GPU)
owns a slab of z planes; per step and face it sends the 5 populations per component that cross the
face and H planes of the phase field (include/lb.h); with rigid particles ("replicated data",
PAPER.md:312-316) every rank holds all of them and two sums of 6 doubles per particle go over the
ranks per step.  This module holds NO lattice-Boltzmann
arithmetic and no kernels: it allocates the message buffers (torch device tensors), moves them
with torch.distributed point-to-point operations (NCCL send/recv over NVLink; gloo in the CPU test
of the schedule) and orders the phases of a step so that the population exchange runs on a side
stream while the fused kernel works on the interior bricks.

    Slab            one slab handle + its message buffers
    DistributedSlab one slab per rank of a torch.distributed group (ring along z)
    LocalRing       several slabs of one box in ONE process on one device (tests; no communicator)
"""
from __future__ import annotations

import numpy as np

from . import lb


# ------------------------------------------------------------------------------ schedule (no GPU needed)
def ring_neighbours(rank, world):
    """(rank below, rank above) on the periodic ring of slabs along z."""
    return (rank - 1) % world, (rank + 1) % world


def split_planes(nz_global, world):
    """Equal split of nz_global planes over `world` slabs ("equally distributed"):
    the first nz_global % world slabs hold one plane more.  Returns [(z0, nz), ...]."""
    base, extra = divmod(nz_global, world)
    out, z = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((z, n))
        z += n
    return out


def slab_mask(solid_global, z0, nz):
    """The (nz + 2) planes z0 - 1 .. z0 + nz of a global solid mask [nz_global, ny, nx], periodic in
    z: what lb_set_geometry wants of a slab (its own planes and the two ghost planes)."""
    if solid_global is None:
        return None
    idx = np.arange(z0 - 1, z0 + nz + 1) % solid_global.shape[0]
    return np.ascontiguousarray(solid_global[idx])


def exchange(send_lo, send_hi, recv_lo, recv_hi, rank=0, world=1, group=None):
    """One halo exchange on the ring: send_hi travels to the rank above and arrives there as its
    recv_lo; send_lo travels to the rank below and arrives as its recv_hi.  Tensors on the device
    (NCCL) or on the host (gloo).  With NCCL, point-to-point operations between one pair of ranks
    match in the order they were posted: upward message first, then the downward one, on both
    sides (world = 2 makes the rank above and the rank below the same peer)."""
    if world == 1:
        recv_lo.copy_(send_hi)
        recv_hi.copy_(send_lo)
        return
    import torch.distributed as dist
    below, above = ring_neighbours(rank, world)
    ops = [dist.P2POp(dist.isend, send_hi, above, group=group, tag=0),
           dist.P2POp(dist.irecv, recv_lo, below, group=group, tag=0),
           dist.P2POp(dist.isend, send_lo, below, group=group, tag=1),
           dist.P2POp(dist.irecv, recv_hi, above, group=group, tag=1)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


def reduce_sums(sums, world=1, group=None):
    """The sum over the ranks of a [np, 6] float64 tensor, in place (replicated particles: link sums,
    then the impulses of the node changes).  Every rank must end up with the same bits, or the
    replicated particle states drift apart: an all-reduce gives that."""
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=group)
    return sums


# ------------------------------------------------------------------------------ one slab
class Slab:
    """The planes [z0, z0 + nz) of an nx x ny x nz_global box, on the current CUDA device."""

    def __init__(self, nx, ny, nz, z0, nz_global, tau_r=1.0, tau_b=1.0, A=0.0, beta=0.0, A_nc=0.0,
                 storage="ab", solid_global=None, g=(0.0, 0.0, 0.0), phi_c=0.9, configure=None, zc=0):
        self.z0, self.nz, self.nz_global = int(z0), int(nz), int(nz_global)
        self.sim = lb.LB(nx, ny, nz, tau_r, tau_b, A, beta, A_nc)
        self.sim.set_storage(storage)
        self.sim.set_slab(z0, nz_global)
        m = slab_mask(solid_global, z0, nz)
        if m is not None:
            self.sim.set_geometry(np.ascontiguousarray(m, dtype=np.uint8))
        self.sim.set_body_force(*g)
        self.sim.set_nc_cutoff(phi_c)
        if configure is not None:
            configure(self.sim)
        if zc:
            self.sim.set_tuning(zc=zc)         # z planes per brick (0 = automatic)
        self.buf = None

    @classmethod
    def from_workload(cls, w, z0, nz, storage="ab", zc=0, nz_global=None):
        """The slab [z0, z0 + nz) of a workloads.Workload (its fields are sliced by init_from).
        nz_global > w.nz: the box is the workload repeated along z (weak scaling: every rank holds
        one period; the mask and the fields wrap with period w.nz)."""
        from . import workloads
        return cls(w.nx, w.ny, nz, z0, nz_global or w.nz, *w.params, storage=storage, solid_global=w.solid, g=w.g,
                   phi_c=w.phi_c, configure=lambda sim: workloads.configure_walls(sim, w), zc=zc)

    def init(self, rho_r, rho_b, u):
        """Fields of the slab's own planes: [nz, ny, nx], u [3, nz, ny, nx]."""
        import torch
        self.sim.init(rho_r, rho_b, u)
        pop, phi = self.sim.slab_halo_bytes()
        dev = torch.device("cuda", torch.cuda.current_device())
        mk = lambda nbytes: torch.empty(max(nbytes, 16) // 4, dtype=torch.float32, device=dev)
        self.buf = {k: mk(pop if k.startswith("p") else phi)
                    for k in ("p_send_lo", "p_send_hi", "p_recv_lo", "p_recv_hi", "f_send_lo", "f_send_hi", "f_recv_lo", "f_recv_hi")}
        self.halo_bytes = (pop, phi)
        self.np = getattr(self.sim, "npart", 0)
        # the slab's share of the particle sums [np, 6], and where the totals come back
        self.sums = torch.zeros((max(self.np, 1), 6), dtype=torch.float64, device=dev)

    def init_from(self, w):
        z0 = self.z0 % w.nz                      # a box taller than the workload repeats it along z
        assert z0 + self.nz <= w.nz
        sl = slice(z0, z0 + self.nz)
        self.init(np.ascontiguousarray(w.rho_r[sl]), None if w.rho_b is None else np.ascontiguousarray(w.rho_b[sl]),
                  np.ascontiguousarray(w.u[:, sl]))

    # phases (names of include/lb.h)
    def begin(self):
        self.sim.slab_begin(self.buf["p_send_lo"], self.buf["p_send_hi"])

    def interior(self):
        self.sim.slab_interior()

    def end(self):
        self.sim.slab_end(self.buf["p_recv_lo"], self.buf["p_recv_hi"])

    def pack_phi(self):
        self.sim.slab_pack_phi(self.buf["f_send_lo"], self.buf["f_send_hi"])

    def unpack_phi(self):
        self.sim.slab_unpack_phi(self.buf["f_recv_lo"], self.buf["f_recv_hi"])

    def part_get(self):
        self.sim.slab_part_get(self.sums)
        return self.sums

    def part_put(self, total):
        self.sim.slab_part_put(total)


# ------------------------------------------------------------------------------ one slab per rank
class DistributedSlab:
    """One slab per rank of a torch.distributed process group (backend nccl on GPUs)."""

    def __init__(self, slab, rank, world, group=None, overlap=True):
        import torch
        self.slab, self.rank, self.world, self.group = slab, rank, world, group
        self.side = torch.cuda.Stream() if overlap else None

    def _x(self, kind):
        b = self.slab.buf
        exchange(b[kind + "_send_lo"], b[kind + "_send_hi"], b[kind + "_recv_lo"], b[kind + "_recv_hi"],
                 self.rank, self.world, self.group)

    def init_from(self, w):
        self.slab.init_from(w)
        self.exchange_phi()

    def init(self, rho_r, rho_b, u):
        self.slab.init(rho_r, rho_b, u)
        self.exchange_phi()

    def exchange_phi(self):
        self.slab.pack_phi()
        if self.slab.halo_bytes[1]:
            self._x("f")
        self.slab.unpack_phi()

    def step(self, nsteps=1):
        """nsteps time steps.  Per step: boundary bricks and packing on the main stream; the
        population exchange on a side stream while the main stream works on the interior bricks;
        then the boundary planes of phi and the (small) phi exchange."""
        import torch
        main = torch.cuda.current_stream()
        for _ in range(int(nsteps)):
            self.slab.begin()
            if self.slab.np > 0:
                # replicated particles: link sums, then the impulses of the node changes, summed over
                # the ranks (every rank gets the same bits back); no overlap in this step
                for _stage in range(2):
                    self.slab.part_put(reduce_sums(self.slab.part_get(), self.world, self.group))
                self._x("p")
                self.slab.interior()
                self.slab.end()
                self.exchange_phi()
                continue
            if self.side is not None:
                ready = main.record_event()
                with torch.cuda.stream(self.side):
                    self.side.wait_event(ready)
                    self._x("p")
                    done = self.side.record_event()
                self.slab.interior()
                main.wait_event(done)
            else:
                self._x("p")
                self.slab.interior()
            self.slab.end()
            self.exchange_phi()


# ------------------------------------------------------------------------------ several slabs, one process
class LocalRing:
    """The slabs of one box in ONE process on one device, stepped phase by phase with device copies
    in place of the communicator: the test vehicle for the slab kernels, the packing and the order
    of the phases (bit-identical to the undivided box)."""

    def __init__(self, w, counts, storage="ab", zc=0):
        assert sum(counts) == w.nz
        self.w, self.slabs, z = w, [], 0
        for n in counts:
            self.slabs.append(Slab.from_workload(w, z, n, storage, zc))
            z += n

    def _x(self, kind):
        n = len(self.slabs)
        for i, s in enumerate(self.slabs):
            up, dn = self.slabs[(i + 1) % n], self.slabs[(i - 1) % n]
            up.buf[kind + "_recv_lo"].copy_(s.buf[kind + "_send_hi"])
            dn.buf[kind + "_recv_hi"].copy_(s.buf[kind + "_send_lo"])

    def _phi(self):
        for s in self.slabs:
            s.pack_phi()
        self._x("f")
        for s in self.slabs:
            s.unpack_phi()

    def init(self):
        for s in self.slabs:
            s.init_from(self.w)
        self._phi()

    def step(self, nsteps=1):
        for _ in range(int(nsteps)):
            for s in self.slabs:
                s.begin()
            if self.slabs[0].np > 0:
                for _stage in range(2):        # the two sums over the slabs, in slab order
                    total = None
                    for s in self.slabs:
                        part = s.part_get()
                        total = part.clone() if total is None else total + part
                    for s in self.slabs:
                        s.part_put(total)
            self._x("p")
            for s in self.slabs:
                s.interior()
            for s in self.slabs:
                s.end()
            self._phi()

    def gather(self, what, *args):
        """Concatenate a per-slab accessor along z: what = 'get_macros' | 'get_populations' | 'get_phi'."""
        parts = [getattr(s.sim, what)(*args) for s in self.slabs]
        if what == "get_macros":
            rr = np.concatenate([p[0] for p in parts], 0)
            rb = None if parts[0][1] is None else np.concatenate([p[1] for p in parts], 0)
            u = np.concatenate([p[2] for p in parts], 1)
            return rr, rb, u
        return np.concatenate(parts, 1 if what == "get_populations" else 0)
