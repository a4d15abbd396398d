"""Slab decomposition along x with a one-cell halo (the paper itself is single-device,
PAPER.md:L122).

Cells are coupled only through the one-cell stencil of Eq 2, so the lattice is cut
into slabs of x-layers (x is the slowest axis: a layer is ny*nz contiguous cells of every SoA plane).
Rank r owns the global layers [x0, x1) and runs an ordinary context of nx = (x1 - x0) + 2 layers whose
first and last layer stand for the neighbours' nearest layers: LBM_GHOST where that layer is fluid
(read like fluid, never updated, filled by the halo exchange), WALL / MOVING where it is solid (so
bounce-back at a wall owned by another rank needs no communication).  The ranks form a ring, which is
the periodic wrap of the library's index arithmetic; a cavity simply has walls at both ends of it.

Every time step each rank sends, per face, the populations that cross it (5 of 19 planes, 9 of 27)
and receives the ones that enter; what exactly a message holds depends on the scheme (two-population:
post-collision values pulled by the next step; AA: post-collision values after an even step, pushed
values merged on arrival after an odd step; swap: between pass 1 and pass 2) and is the library's
business (include/lbm.h).  The step runs in parts so that the transfer overlaps the interior update:
begin (outermost owned layers) -> pack -> end (interior) -> unpack -> finish.  That exchange is the
only data-path communication; the kinetic energy adds one scalar all-reduce.  SoA schemes only.

Two transports:
  * "peer": the library's own driver (`lbm_slab_step`): pack kernels store straight into the
    neighbouring slab's receive buffer (peer memory over NVLink) and publish a sequence number, unpack
    kernels wait for it; no host code and no communication library between the parts.  Slabs of one
    process are linked directly (`lbm_slab_link`), slabs of other processes through CUDA IPC handles
    exchanged once at start-up.
  * "p2p": pack -> torch.distributed isend / irecv (NCCL on GPUs; gloo with CPU buffers in the host
    tests) -> unpack, driven from Python once per step.

This module holds the decomposition arithmetic and the exchange plumbing, no arithmetic of the
method.
"""
import numpy as np

FLUID, WALL, MOVING, GHOST = 0, 1, 2, 3


def slab_range(NX, rank, world):
    """global x-range [x0, x1) owned by `rank`: layers dealt as evenly as possible, low ranks first"""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside [0, %d)" % (rank, world))
    if NX < world:
        raise ValueError("cannot cut %d layers into %d slabs" % (NX, world))
    base, rem = divmod(NX, world)
    x0 = rank * base + min(rank, rem)
    return x0, x0 + base + (1 if rank < rem else 0)


def neighbours(rank, world):
    """(rank owning the layers below x0, rank owning the layers above x1) on the periodic ring"""
    return (rank - 1) % world, (rank + 1) % world


def _ghost_layer(layer):
    return np.where(layer == FLUID, GHOST, layer).astype(np.uint8)


def local_flags(flags, x0, x1):
    """uint8 [x1-x0+2, ny, nz] from global flags [NX, ny, nz]: the owned layers between the two
    neighbouring layers, where fluid becomes GHOST and solid stays solid"""
    NX = flags.shape[0]
    lo, hi = flags[(x0 - 1) % NX], flags[x1 % NX]
    return np.concatenate([_ghost_layer(lo)[None], flags[x0:x1].astype(np.uint8), _ghost_layer(hi)[None]], axis=0)


def local_field(a, x0, x1, axis=0):
    """slice of a global field with one wrapped layer on either side along `axis` (the values in
    the ghost layers are never used by the owner: its first step is local)"""
    NX = a.shape[axis]
    idx = np.arange(x0 - 1, x1 + 1) % NX
    return np.ascontiguousarray(np.take(a, idx, axis=axis))


def cavity_slab(NX, NY, NZ, x0, x1, seed=0):
    """(flags_local, rho_local, u_local) of the slab [x0, x1) of an NX x NY x NZ lid-driven cavity with
    the seeded noise init of inputs.py, built layer by layer so that no rank ever holds the global
    arrays (weak-scaling runs); the values are those of the undivided lattice."""
    from . import inputs
    pattern = inputs.cavity_flags(3, NY, NZ)      # [0] = a wall layer, [1] = an inner layer
    xs = np.arange(x0 - 1, x1 + 1) % NX
    fl = np.stack([pattern[0] if (x == 0 or x == NX - 1) else pattern[1] for x in xs])
    fl[0], fl[-1] = _ghost_layer(fl[0]), _ghost_layer(fl[-1])
    cells = (xs.astype(np.int64)[:, None] * (NY * NZ) + np.arange(NY * NZ, dtype=np.int64)[None, :]).reshape(-1)
    rho, u = inputs.seeded_init(len(xs), NY, NZ, seed, index_offset=cells)
    return fl, rho, u


def interior(a, axis=0):
    """drop the two ghost layers of a local field"""
    sl = [slice(None)] * a.ndim
    sl[axis] = slice(1, -1)
    return a[tuple(sl)]


def exchange_local(engines):
    """halo exchange between slabs that live in this process, engines[r] owning slab r of the ring.
    An engine offers halo_pack(face) -> buffer and halo_unpack(face, buffer)."""
    W = len(engines)
    sent = [(e.halo_pack(0), e.halo_pack(1)) for e in engines]
    for r, e in enumerate(engines):
        left, right = neighbours(r, W)
        e.halo_unpack(0, sent[left][1])    # what left the left neighbour through its high face
        e.halo_unpack(1, sent[right][0])   # what left the right neighbour through its low face


def exchange_start(engine, dist, rank, world, group=None):
    """pack both faces and post the sends / receives; returns a handle for exchange_finish.  Over
    nccl the transfers run on the communicator's own stream, so whatever the caller launches next
    on the compute stream (step_end: the interior of the slab) overlaps them."""
    s0, s1 = engine.halo_pack(0), engine.halo_pack(1)
    r0, r1 = engine.halo_recv_buffer(0), engine.halo_recv_buffer(1)
    if world == 1:
        r0.copy_(s1)
        r1.copy_(s0)
        return (r0, r1, [])
    left, right = neighbours(rank, world)
    # the message tag is the face it LEFT through; nccl ignores tags and matches in order, so
    # with two ranks (left == right) the receives are posted in the peer's send order
    ops = [dist.P2POp(dist.isend, s0, left, group, 0), dist.P2POp(dist.isend, s1, right, group, 1),
           dist.P2POp(dist.irecv, r1, right, group, 0), dist.P2POp(dist.irecv, r0, left, group, 1)]
    return (r0, r1, dist.batch_isend_irecv(ops))


def exchange_finish(engine, handle):
    r0, r1, reqs = handle
    for req in reqs:
        req.wait()
    engine.halo_unpack(0, r0)
    engine.halo_unpack(1, r1)


def exchange_dist(engine, dist, rank, world, group=None):
    """the exchange over torch.distributed, one slab per process.  Buffers are torch tensors on the
    backend's device (CUDA for nccl, CPU for gloo); the engine offers halo_pack(face) -> tensor,
    halo_recv_buffer(face) -> tensor and halo_unpack(face, tensor)."""
    exchange_finish(engine, exchange_start(engine, dist, rank, world, group))


def step_dist(engine, dist, rank, world, group=None):
    """one time step of one slab per process over torch.distributed: the parts in the order every
    scheme needs (swap: the halo must arrive between pass 1 and pass 2)"""
    engine.step_begin()                                  # the two outermost owned layers
    h = exchange_start(engine, dist, rank, world, group)
    engine.step_end()                                    # the interior, while the halo travels
    exchange_finish(engine, h)
    engine.step_finish()


def link_ring(engines):
    """link the slabs of this process into the periodic ring (library transport, lbm_slab_link)"""
    W = len(engines)
    for r, e in enumerate(engines):
        left, right = neighbours(r, W)
        e.lbm.slab_link(0, engines[left].lbm)
        e.lbm.slab_link(1, engines[right].lbm)


def step_local(engines, mode="overlap"):
    """one time step of several GPU slabs living in this process (one stream).
    "overlap": outer layers, pack, interior, unpack, finish through the halo calls, buffers handed
    over directly; "plain": lbm_step(1) then the exchange (two-population and AA only); "peer": the
    library's driver after link_ring (post on all slabs, then complete on all)."""
    W = len(engines)
    if mode == "peer":
        for e in engines:
            e.lbm.slab_post()
        for e in engines:
            e.lbm.slab_complete()
    elif mode == "overlap":
        for e in engines:
            e.lbm.step_begin()
        sent = [(e.halo_pack(0), e.halo_pack(1)) for e in engines]
        for e in engines:
            e.lbm.step_end()
        for r, e in enumerate(engines):
            left, right = neighbours(r, W)
            e.halo_unpack(0, sent[left][1])
            e.halo_unpack(1, sent[right][0])
        for e in engines:
            e.lbm.step_finish()
    else:
        for e in engines:
            e.lbm.step(1)
        exchange_local(engines)


class GpuSlabEngine:
    """one slab on the current CUDA device: an Lbm context plus its four halo buffers.  Everything the
    engine launches or copies goes to the stream that was current when it was built (the context's)."""

    def __init__(self, flags_local, u_wall, lattice=19, collision="BGK_W2", omega=1.0, dtype="f64", scheme="2POP_SOA"):
        import torch
        from .binding import Lbm, NP_DTYPES
        nx, ny, nz = flags_local.shape
        self.shape = (nx, ny, nz)
        self._torch = torch
        self._stream = torch.cuda.current_stream()
        self.lbm = Lbm(nx, ny, nz, lattice=lattice, collision=collision, scheme=scheme, omega=omega, dtype=dtype)
        self.lbm.set_flags(flags_local, u_wall)
        tdt = torch.float64 if dtype == "f64" else torch.float32
        self.np_dtype = NP_DTYPES[dtype]
        cnt = self.lbm.halo_count
        self._send = [torch.empty(cnt, dtype=tdt, device="cuda") for _ in range(2)]
        self._recv = [torch.empty(cnt, dtype=tdt, device="cuda") for _ in range(2)]
        self.halo_bytes = 2 * cnt * self._send[0].element_size()  # sent per step (received: the same)

    def step_begin(self):
        self.lbm.step_begin()

    def step_end(self):
        self.lbm.step_end()

    def step_finish(self):
        self.lbm.step_finish()

    def halo_pack(self, face):
        self.lbm.halo_pack(face, self._send[face].data_ptr())
        return self._send[face]

    def halo_recv_buffer(self, face):
        return self._recv[face]

    def halo_unpack(self, face, buf):
        self.lbm.halo_unpack(face, buf.data_ptr())

    def on_stream(self):
        """context manager: torch work (copies, NCCL transfers) ordered on the context's stream"""
        return self._torch.cuda.stream(self._stream)

    def close(self):
        self.lbm.close()


class SlabLbm:
    """the user-facing multi-GPU object: one process per GPU, each owning one slab of an
    NX x NY x NZ lattice.  `flags` / `rho` / `u` are GLOBAL host arrays (every rank passes the same
    ones and keeps its slice); results come back per slab (macroscopic, populations) or global
    (kinetic energy)."""

    def __init__(self, NX, NY, NZ, flags=None, u_wall=(0.0, 0.0, 0.0), dist=None, rank=0, world=1, group=None,
                 lattice=19, collision="BGK_W2", omega=1.0, dtype="f64", flags_local=None, scheme="2POP_SOA",
                 transport=None):
        """flags: GLOBAL [NX, NY, NZ] (None = all fluid), or flags_local: this rank's [nxl+2, NY, NZ]
        with its ghost layers already in place (local_flags / cavity_slab).
        transport: "peer" (library driver over peer memory; default for one rank) or "p2p"
        (torch.distributed send / recv; default for several ranks)"""
        self.dist, self.rank, self.group = dist, rank, group
        self.world = world if dist is not None else 1
        self.transport = transport or ("peer" if self.world == 1 else "p2p")
        self.N = (NX, NY, NZ)
        self.x0, self.x1 = slab_range(NX, rank, world)
        if flags_local is not None:
            self.flags_local = np.ascontiguousarray(flags_local, dtype=np.uint8).reshape(self.x1 - self.x0 + 2, NY, NZ)
        else:
            if flags is None:
                flags = np.zeros((NX, NY, NZ), dtype=np.uint8)
            self.flags_local = local_flags(np.asarray(flags).reshape(NX, NY, NZ), self.x0, self.x1)
        self.engine = GpuSlabEngine(self.flags_local, u_wall, lattice=lattice, collision=collision, omega=omega,
                                    dtype=dtype, scheme=scheme)
        self.lbm = self.engine.lbm
        self.Q = self.lbm.Q
        if self.transport == "peer":
            self._connect_peers()

    def _connect_peers(self):
        """library transport: one slab = the ring closes on itself; several processes = every rank
        publishes the CUDA IPC handle of its receive block and opens its two neighbours' """
        if self.world == 1:
            self.lbm.slab_link(0, self.lbm)
            self.lbm.slab_link(1, self.lbm)
            return
        handles = [None] * self.world
        self.dist.all_gather_object(handles, self.lbm.slab_export(), group=self.group)
        left, right = neighbours(self.rank, self.world)
        self.lbm.slab_import(0, handles[left])
        self.lbm.slab_import(1, handles[right])
        self.dist.barrier(group=self.group)

    def _local(self, a, lead):
        NX, NY, NZ = self.N
        a = np.asarray(a).reshape(lead + (NX, NY, NZ))
        return local_field(a, self.x0, self.x1, axis=len(lead)).astype(self.engine.np_dtype)

    def init_equilibrium(self, rho, u):
        self.lbm.init_equilibrium(self._local(rho, ()), self._local(u, (3,)))

    def init_equilibrium_local(self, rho_local, u_local):
        """rho [nxl+2, NY, NZ], u [3, nxl+2, NY, NZ] of this rank's context, ghost layers included"""
        self.lbm.init_equilibrium(np.asarray(rho_local, dtype=self.engine.np_dtype), np.asarray(u_local, dtype=self.engine.np_dtype))

    def step(self, n=1):
        if self.transport == "peer":
            self.lbm.slab_step(n)       # the whole loop inside the library, nothing per step on the host
            return
        with self.engine.on_stream():
            for _ in range(n):
                step_dist(self.engine, self.dist, self.rank, self.world, self.group)

    def macroscopic(self):
        """(rho [nxl, NY, NZ], u [3, nxl, NY, NZ]) of the owned layers"""
        nx, ny, nz = self.engine.shape
        rho, u = self.lbm.macroscopic()
        return interior(rho.reshape(nx, ny, nz)).copy(), interior(u.reshape(3, nx, ny, nz), axis=1).copy()

    def get_populations(self):
        """f [Q, nxl, NY, NZ] of the owned layers, canonical order"""
        nx, ny, nz = self.engine.shape
        return interior(self.lbm.get_populations().reshape(self.Q, nx, ny, nz), axis=1).copy()

    def kinetic_energy(self):
        """global sum: the slab's partial stays in device memory for the one scalar all-reduce"""
        import torch
        with self.engine.on_stream():
            t = torch.zeros(1, dtype=torch.float64, device="cuda")
            self.lbm.kinetic_energy_device(t.data_ptr())
            if self.dist is not None and self.world > 1:
                self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
            return float(t.item())

    @property
    def num_fluid(self):
        return self.lbm.num_fluid

    def close(self):
        if self.transport == "peer":
            self.lbm.slab_status()
        self.engine.close()
