"""z-slab decomposition over `torch.distributed` ranks: the caller side of `rflbm_set_slab` / `rflbm_halo_*`.

PAPER.md:292 ("the simulation box is extended along the z direction", L_z = 256 n_GPU) and :300 ("linear
decomposition"): every rank owns a contiguous range of z layers of ONE global lattice; after every step the nine
`c_z = -1` and the nine `c_z = +1` populations of its two boundary layers travel to the rank below / above
(9 nx ny sizeof(real) bytes per face: 4.7 MB at 256^2 fp64).  All arithmetic stays in the CUDA kernels of csrc/
(the step, pack and unpack kernels behind include/rflbm.h); this module only decides who owns what and moves the
packed faces: point-to-point send/recv (NCCL between GPUs; gloo through pinned host buffers where ranks share a GPU
or the backend is gloo), no reduction collective on the data path.  STATUS: the gloo transport is what every test runs
(2-3 ranks, CPU tensors and one shared GPU); the NCCL branches (FaceTransport.exchange, SlabLattice.diagnostics) are
UNTESTED ON HARDWARE - no box with two GPUs has been available to this repository.  Because walls and the Philox key use the GLOBAL
z, the ranks together compute, bit for bit, what one handle computes on the undivided lattice
(tests/test_gpu_slab.py on one process, tests/test_gpu_slab_dist.py on two).

BASELINE.json's headline (and `bench.py`'s default) is one GPU; `bench.py --decomp slab` times this path.
"""
from __future__ import annotations

from . import binding
from .binding import F64, SCHEME_AB, SIDE_HIGH, SIDE_LOW


def slab_extent(rank: int, world: int, nz_global: int):
    """(z0, nz) of the layers rank `rank` of `world` owns: contiguous, in rank order, sizes differing by at most one."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("rank / world")
    if nz_global < world:
        raise ValueError(f"{nz_global} layers cannot be cut into {world} non-empty slabs")
    base, rem = divmod(nz_global, world)
    return rank * base + min(rank, rem), base + (1 if rank < rem else 0)


def neighbours(rank: int, world: int):
    """(below, above): the ranks that own the layers under / over this rank's slab (periodic along z)."""
    return (rank - 1) % world, (rank + 1) % world


class FaceTransport:
    """Moves the two packed faces of every rank to its neighbours and returns the two it receives.

    exchange(low_face, high_face) -> (for_low_side, for_high_side): `low_face` (this rank's LOW pack) goes to the rank
    below, `high_face` to the rank above; `for_high_side` is the LOW pack of the rank above, `for_low_side` the HIGH pack
    of the rank below.  world 1: the rank is its own neighbour, nothing moves.  Tensors may live on the CPU (gloo) or on
    a CUDA device; with a gloo group, device tensors are staged through pinned host buffers.
    """

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        if dist.is_available() and dist.is_initialized():
            self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
            self.backend = dist.get_backend(group)
        else:
            self.rank, self.world, self.backend = 0, 1, "none"
        self.below, self.above = neighbours(self.rank, self.world)
        self._host = {}

    def _peer(self, r):
        return r if self.group is None else self.dist.get_global_rank(self.group, r)

    def _pinned(self, key, like):
        import torch
        t = self._host.get(key)
        if t is None or t.shape != like.shape or t.dtype != like.dtype:
            t = torch.empty(like.shape, dtype=like.dtype, pin_memory=torch.cuda.is_available())
            self._host[key] = t
        return t

    def exchange(self, low_face, high_face, recv_low=None, recv_high=None):
        import torch
        if self.world == 1:
            return high_face, low_face
        dist = self.dist
        recv_low = torch.empty_like(high_face) if recv_low is None else recv_low
        recv_high = torch.empty_like(low_face) if recv_high is None else recv_high
        if low_face.is_cuda and self.backend == "nccl":
            # matching order between one pair of ranks (world 2: below == above): sends LOW then HIGH; the first receive
            # from a rank is therefore its LOW pack (wanted at this rank's HIGH side), the second its HIGH pack
            ops = [dist.P2POp(dist.isend, low_face, self._peer(self.below), self.group),
                   dist.P2POp(dist.isend, high_face, self._peer(self.above), self.group),
                   dist.P2POp(dist.irecv, recv_high, self._peer(self.above), self.group),
                   dist.P2POp(dist.irecv, recv_low, self._peer(self.below), self.group)]
            for req in dist.batch_isend_irecv(ops):
                req.wait()
            return recv_low, recv_high
        # CPU transport (gloo): tags tell the two faces of one peer apart (tag = side the face was packed on)
        staged = low_face.is_cuda
        if staged:
            s_lo, s_hi = self._pinned("s_lo", low_face), self._pinned("s_hi", high_face)
            r_lo, r_hi = self._pinned("r_lo", recv_low), self._pinned("r_hi", recv_high)
            s_lo.copy_(low_face, non_blocking=True)
            s_hi.copy_(high_face, non_blocking=True)
            torch.cuda.current_stream(low_face.device).synchronize()
        else:
            s_lo, s_hi, r_lo, r_hi = low_face, high_face, recv_low, recv_high
        reqs = [dist.isend(s_lo, self._peer(self.below), group=self.group, tag=SIDE_LOW),
                dist.isend(s_hi, self._peer(self.above), group=self.group, tag=SIDE_HIGH),
                dist.irecv(r_hi, self._peer(self.above), group=self.group, tag=SIDE_LOW),
                dist.irecv(r_lo, self._peer(self.below), group=self.group, tag=SIDE_HIGH)]
        for req in reqs:
            req.wait()
        if staged:
            recv_low.copy_(r_lo, non_blocking=True)
            recv_high.copy_(r_hi, non_blocking=True)
        return recv_low, recv_high


class SlabLattice:
    """One global nx x ny x nz_global lattice cut into z slabs, one per rank of `group` (default: the world).

    Construct it on every rank with the same arguments (torch.distributed initialised, or not at all for one rank);
    `init`, `step` are collective.  `sim` is this rank's `binding.Rflbm` handle (layers [z0, z0+nz) of the global
    lattice); `moments`, `stress`, `get_populations` return this rank's layers; `gather` assembles a global array on
    every rank (a convenience for checks, through host memory), `diagnostics` combines the ten sums over all ranks.
    """

    def __init__(self, nx, ny, nz_global, tau, kT, rho0=1.0, seed=0, precision=F64, device="cuda:0", scheme=SCHEME_AB,
                 group=None, walls=False, force=None, stream=None):
        import torch
        self.torch = torch
        self.transport = FaceTransport(group)
        self.rank, self.world = self.transport.rank, self.transport.world
        self.nx, self.ny, self.nz_global = nx, ny, nz_global
        self.z0, self.nz = slab_extent(self.rank, self.world, nz_global)
        self.walls = bool(walls)
        self.sim = binding.Rflbm(nx, ny, self.nz, tau, kT, rho0, seed, precision, device=device, stream=stream,
                                 scheme=scheme, slab=(self.z0, nz_global))
        if walls:
            self.sim.set_walls_z(True)
        if force is not None:
            self.sim.set_force(*force)
        face = (9, ny, nx)
        with torch.cuda.device(self.sim.device):
            self._send = [torch.empty(face, dtype=self.sim.dtype, device=self.sim.device) for _ in range(2)]
            self._recv = [torch.empty(face, dtype=self.sim.dtype, device=self.sim.device) for _ in range(2)]
        self.face_bytes = self.sim.halo_bytes
        self.bytes_sent = 0

    def _ghosted(self, a):
        """layers z0-1 .. z0+nz (periodic) of a global field [..., nz_global, ny, nx] (numpy array or torch tensor)"""
        t = self.torch
        a = t.as_tensor(a)
        idx = t.tensor([(self.z0 - 1 + i) % self.nz_global for i in range(self.nz + 2)], device=a.device)
        return a.index_select(a.dim() - 3, idx).contiguous()

    def init(self, rho=None, u=None):
        """rho[nz_global, ny, nx], u[3, nz_global, ny, nx]: the GLOBAL fields (every rank passes the same), or None for rho0, u = 0"""
        if rho is None:
            self.sim.init()
        else:
            self.sim.init(self._ghosted(rho), self._ghosted(u))
        self.exchange()

    def set_populations(self, f, step=0):
        """f[27, nz_global, ny, nx]: the global pre-collision state at time `step` (checkpoint resume)"""
        self.sim.set_populations(self._ghosted(f), step)
        self.exchange()

    def exchange(self):
        """the face exchange the library asks for after init / set_populations / step (rflbm_halo_pending)"""
        sim = self.sim
        if not sim.halo_pending:
            return
        with sim._ctx():
            lo = sim.halo_pack(SIDE_LOW, self._send[0])
            hi = sim.halo_pack(SIDE_HIGH, self._send[1])
            for_low, for_high = self.transport.exchange(lo, hi, self._recv[0], self._recv[1])
            sim.halo_unpack(SIDE_LOW, for_low)
            sim.halo_unpack(SIDE_HIGH, for_high)
        if self.world > 1:
            self.bytes_sent += 2 * self.face_bytes

    def step(self, n=1):
        for _ in range(int(n)):
            self.sim.step(1)
            self.exchange()

    def moments(self):
        return self.sim.moments()

    def stress(self):
        return self.sim.stress()

    def get_populations(self):
        return self.sim.get_populations()

    def gather(self, local, zdim):
        """global array from every rank's local part (concatenated along `zdim` in rank order), on the CPU"""
        t = self.torch
        part = local.detach().cpu()
        if self.world == 1:
            return part
        parts = [None] * self.world
        self.transport.dist.all_gather_object(parts, part, group=self.transport.group)
        return t.cat(parts, dim=zdim)

    def fluid_sites(self):
        """fluid sites this rank owns (R12: with walls the global layers 0 and nz_global-1 are solid)"""
        layers = self.nz
        if self.walls:
            layers -= int(self.z0 == 0) + int(self.z0 + self.nz == self.nz_global)
        return self.nx * self.ny * layers

    def diagnostics(self):
        """the ten values of rflbm_diagnostics for the GLOBAL lattice: mass, momentum (sums), mean and variance of u over
        all fluid sites (combined from the per-rank values and site counts)"""
        t = self.torch
        n = float(self.fluid_sites())
        d = self.sim.diagnostics() if n > 0 else [0.0] * 10       # a slab that is only a wall layer owns no fluid site
        acc = t.tensor([n] + d[0:4] + [n * m for m in d[4:7]] + [n * (v + m * m) for m, v in zip(d[4:7], d[7:10])],
                       dtype=t.float64)
        if self.world > 1:
            dist = self.transport.dist
            if self.transport.backend == "nccl":
                acc = acc.to(self.sim.device)
            dist.all_reduce(acc, group=self.transport.group)
            acc = acc.cpu()
        acc = acc.tolist()
        ntot = acc[0]
        mean = [acc[5 + a] / ntot for a in range(3)]
        var = [acc[8 + a] / ntot - mean[a] ** 2 for a in range(3)]
        return acc[1:5] + mean + var

    def close(self):
        self.sim.close()
