"""Slab decomposition (paper_2010_11751_b200/slab.py): decomposition arithmetic, the exchange plumbing
over gloo at world size 2 (CPU, with an oracle-backed engine standing in for the GPU context), and
on the GPU several slabs in one process against the oracle's undivided lattice."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2010_11751_b200 import inputs, slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_range_covers_the_lattice():
    for NX in (3, 7, 16, 257):
        for world in (1, 2, 3, 5):
            if NX < world:
                continue
            ranges = [slab.slab_range(NX, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == NX
            for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
                assert a1 == b0
            sizes = [b - a for a, b in ranges]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        slab.slab_range(2, 0, 3)
    assert slab.neighbours(0, 4) == (3, 1) and slab.neighbours(3, 4) == (2, 0) and slab.neighbours(0, 1) == (0, 0)


def test_local_flags_ghost_and_solid_layers():
    fl = inputs.cavity_flags(8, 5, 6)
    lo = slab.local_flags(fl, 0, 4)        # below x0 = 0 lies the wall layer x = 7 (ring)
    assert lo.shape == (6, 5, 6)
    assert np.array_equal(lo[1:-1], fl[0:4])
    assert np.array_equal(lo[0], fl[7])    # solid stays solid
    inner = fl[4]
    assert np.array_equal(lo[-1] == slab.GHOST, inner == slab.FLUID)
    assert np.array_equal(lo[-1][inner != 0], inner[inner != 0])
    a = np.arange(8 * 2).reshape(8, 2)
    assert np.array_equal(slab.local_field(a, 0, 4)[:, 0], [14, 0, 2, 4, 6, 8])
    assert np.array_equal(slab.interior(slab.local_field(a, 2, 5)), a[2:5])


def test_cavity_slab_equals_slices_of_the_global_inputs():
    NX, NY, NZ = 12, 5, 6
    fl = inputs.cavity_flags(NX, NY, NZ)
    rho, u = inputs.seeded_init(NX, NY, NZ, 4)
    for rank in range(3):
        x0, x1 = slab.slab_range(NX, rank, 3)
        f, r, uu = slab.cavity_slab(NX, NY, NZ, x0, x1, seed=4)
        assert np.array_equal(f, slab.local_flags(fl, x0, x1))
        assert np.array_equal(r.reshape(-1, NY, NZ), slab.local_field(rho.reshape(NX, NY, NZ), x0, x1))
        assert np.array_equal(uu.reshape(3, -1, NY, NZ), slab.local_field(u.reshape(3, NX, NY, NZ), x0, x1, axis=1))


# ---------------------------------------------------------------- gloo, world size 2, CPU
_WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch
import torch.distributed as dist
from paper_2010_11751_b200 import inputs, slab
from oracle import lbm_oracle

class OracleEngine:
    # the oracle on one slab; ghost cells are plain fluid cells whose populations (all Q: the oracle
    # collides them before it pushes) are overwritten by the exchange after every step
    def __init__(self, flags_local, uw, Q, omega):
        self.shape = flags_local.shape
        nx, ny, nz = self.shape
        self.Q = Q
        self.o = lbm_oracle.Oracle(nx, ny, nz, Q=Q, model="BGK_W2", omega=omega)
        self.o.set_flags(np.where(flags_local == slab.GHOST, 0, flags_local).astype(np.uint8), uw)
        self.recv = [torch.empty(Q * ny * nz, dtype=torch.float64) for _ in range(2)]
        self.calls = []
    def f(self):
        return self.o.get_populations().reshape((self.Q,) + self.shape)
    # the parts of a step in the order slab.step_dist calls them; the oracle has no layers to split,
    # so the update itself happens in step_begin (the packs that follow must see the new values)
    def step_begin(self):
        self.calls.append("begin"); self.o.step(1)
    def step_end(self):
        self.calls.append("end")
    def step_finish(self):
        self.calls.append("finish")
    def halo_pack(self, face):
        self.calls.append("pack%%d" %% face)
        return self._pack(face)
    def _pack(self, face):
        return torch.from_numpy(np.ascontiguousarray(self.f()[:, 1 if face == 0 else -2]).reshape(-1).copy())
    def halo_recv_buffer(self, face):
        return self.recv[face]
    def halo_unpack(self, face, buf):
        self.calls.append("unpack%%d" %% face)
        f = self.f().copy()
        f[:, 0 if face == 0 else -1] = buf.numpy().reshape((self.Q,) + self.shape[1:])
        self.o.set_populations(f.reshape(self.Q, -1))

dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
NX, NY, NZ, Q, omega, steps = 9, 6, 5, %(Q)d, 1.7, 7
for kind in ("cavity", "periodic"):
    fl = inputs.cavity_flags(NX, NY, NZ) if kind == "cavity" else inputs.periodic_flags(NX, NY, NZ)
    if kind == "periodic":
        fl[4:6, 2:4, 1:3] = inputs.MOVING      # an obstacle that straddles the cut between the slabs
    uw = (0.02, -0.01, 0.015)
    rho, u = inputs.seeded_init(NX, NY, NZ, 1)
    full = lbm_oracle.Oracle(NX, NY, NZ, Q=Q, model="BGK_W2", omega=omega)
    full.set_flags(fl, uw); full.init_equilibrium(rho, u); full.step(steps)
    x0, x1 = slab.slab_range(NX, rank, world)
    e = OracleEngine(slab.local_flags(fl, x0, x1), uw, Q, omega)
    e.o.init_equilibrium(slab.local_field(rho.reshape(NX, NY, NZ), x0, x1), slab.local_field(u.reshape(3, NX, NY, NZ), x0, x1, axis=1))
    for _ in range(steps):
        slab.step_dist(e, dist, rank, world)
    assert e.calls == ["begin", "pack0", "pack1", "end", "unpack0", "unpack1", "finish"] * steps, e.calls[:8]
    mine = slab.interior(e.f(), axis=1)
    want = full.get_populations().reshape(Q, NX, NY, NZ)[:, x0:x1]
    fluid = fl[x0:x1] == 0
    err = np.abs(mine - want)[:, fluid].max()
    assert err <= 1e-14, (kind, rank, err)
dist.barrier()
print("OK", rank)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("Q", [19, 27])
def test_exchange_dist_gloo_world2(tmp_path, Q):
    script = tmp_path / "w.py"
    script.write_text(_WORKER % {"root": ROOT, "Q": Q})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(29530 + Q), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert r.stdout.count("OK") == 2


# ---------------------------------------------------------------- GPU: several slabs in one process
def _flags(kind, NX, NY, NZ):
    if kind == "cavity":
        return inputs.cavity_flags(NX, NY, NZ), (inputs.U_LID, 0.0, 0.0)
    fl = inputs.periodic_flags(NX, NY, NZ)
    fl[3:6, 2:4, 1:3] = inputs.MOVING
    fl[NX - 1, 0:2, NZ // 2] = inputs.WALL
    return fl, (0.01, -0.02, 0.015)


@pytest.mark.gpu
@pytest.mark.parametrize("Q,dtype", [(19, "f64"), (27, "f64"), (19, "f32"), (27, "f32")])
@pytest.mark.parametrize("kind", ["cavity", "obstacle"])
@pytest.mark.parametrize("world,mode", [(1, "overlap"), (2, "plain"), (2, "overlap"), (3, "overlap"), (1, "peer"), (2, "peer"), (3, "peer")])
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_SOA"])
def test_slabs_match_the_undivided_oracle(oracle, Q, dtype, kind, world, mode, scheme):
    """1, 2 and 3 slabs of one lattice in one process, every SoA scheme, through the halo calls
    ("overlap": begin, pack, end, unpack, finish; "plain": lbm_step(1) then pack / unpack) and through
    the library's own driver ("peer": pack kernels store into the neighbour's receive buffer), against
    the oracle's undivided lattice.  9 steps: AA ends on an odd step, so the exports un-shuffle
    through the ghost layers as well."""
    if mode == "plain" and scheme == "SWAP_SOA":
        pytest.skip("swap needs its halo between the two passes: no plain lbm_step with ghost cells")
    _slabs_against_the_oracle(oracle, Q, dtype, kind, world, mode, scheme, 10)


@pytest.mark.gpu
@pytest.mark.parametrize("kind", ["cavity", "obstacle"])
@pytest.mark.parametrize("NX,world", [(6, 3), (7, 4), (5, 5)])
@pytest.mark.parametrize("mode", ["overlap", "peer"])
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_SOA"])
def test_thin_slabs_match_the_undivided_oracle(oracle, kind, NX, world, mode, scheme):
    """the thinnest slabs: two owned layers each (6 over 3: "begin" covers the whole slab and "end" nothing), 2 + 2 + 2 + 1,
    and ONE owned layer each (5 over 5: the layers 1 and nx - 2 of lbm_step_begin are the same layer, updated once;
    what a slab receives from one side is what it sends on to the other a step later)"""
    _slabs_against_the_oracle(oracle, 19, "f64", kind, world, mode, scheme, NX)


def _slabs_against_the_oracle(oracle, Q, dtype, kind, world, mode, scheme, NX):
    NY, NZ, omega, steps = 9, 8, 1.7, 9
    fl, uw = _flags(kind, NX, NY, NZ)
    rho, u = inputs.seeded_init(NX, NY, NZ, 2)
    npdt = np.float64 if dtype == "f64" else np.float32
    rho, u = rho.astype(npdt), u.astype(npdt)
    o = oracle.Oracle(NX, NY, NZ, Q=Q, model="BGK_W2", omega=omega)
    o.set_flags(fl, uw)
    o.init_equilibrium(rho.astype(np.float64), u.astype(np.float64))
    o.step(steps)
    want = o.get_populations().reshape(Q, NX, NY, NZ)
    engines, ranges = [], []
    for r in range(world):
        x0, x1 = slab.slab_range(NX, r, world)
        e = slab.GpuSlabEngine(slab.local_flags(fl, x0, x1), uw, lattice=Q, omega=omega, dtype=dtype, scheme=scheme)
        e.lbm.init_equilibrium(slab.local_field(rho.reshape(NX, NY, NZ), x0, x1),
                               slab.local_field(u.reshape(3, NX, NY, NZ), x0, x1, axis=1))
        engines.append(e)
        ranges.append((x0, x1))
    if mode == "peer":
        slab.link_ring(engines)
    for _ in range(steps):
        slab.step_local(engines, mode=mode)
    if mode == "peer":
        for e in engines:
            e.lbm.slab_status()
    energy, nfluid = 0.0, 0
    _, t, _, _ = oracle.lattice(Q)
    for e, (x0, x1) in zip(engines, ranges):
        nx = x1 - x0 + 2
        got = slab.interior(e.lbm.get_populations().astype(np.float64).reshape(Q, nx, NY, NZ), axis=1)
        fluid = fl[x0:x1] == 0
        d = np.abs(got - want[:, x0:x1])[:, fluid]
        if dtype == "f64":
            assert d.max(initial=0.0) <= 1e-12          # a slab that owns only a wall layer has no fluid cell
        else:
            den = np.maximum(np.abs(want[:, x0:x1])[:, fluid], t[:, None])
            assert (d / den).max(initial=0.0) <= 2e-5
        assert np.all(got[:, ~fluid] == 0.0)
        energy += e.lbm.kinetic_energy()
        nfluid += e.lbm.num_fluid
        rho_l, u_l = e.lbm.macroscopic()
        assert np.all(rho_l.reshape(nx, NY, NZ)[[0, -1]] == 0.0)   # ghost layers are left out of exports
    assert nfluid == int((fl == 0).sum())
    assert abs(energy - o.kinetic_energy()) <= (1e-12 if dtype == "f64" else 1e-6) * max(1.0, o.kinetic_energy())
    for e in engines:
        e.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_SOA"])
@pytest.mark.parametrize("transport", ["peer", "p2p"])
def test_slab_lbm_single_rank_ring(oracle, scheme, transport):
    """SlabLbm at world size 1: the ring closes on itself, i.e. a periodic lattice in x; "peer" runs
    the whole loop inside the library (lbm_slab_step), "p2p" the Python-driven parts"""
    NX, NY, NZ, omega, steps = 8, 7, 9, 1.6, 6
    fl = inputs.periodic_flags(NX, NY, NZ)
    fl[:, 0, :] = inputs.WALL
    rho, u = inputs.seeded_init(NX, NY, NZ, 5)
    o = oracle.Oracle(NX, NY, NZ, Q=19, model="BGK_W2", omega=omega)
    o.set_flags(fl, (0, 0, 0))
    o.init_equilibrium(rho, u)
    o.step(steps)
    s = slab.SlabLbm(NX, NY, NZ, flags=fl, omega=omega, scheme=scheme, transport=transport)
    s.init_equilibrium(rho, u)
    s.step(steps)
    got = s.get_populations()
    want = o.get_populations().reshape(19, NX, NY, NZ)
    assert np.abs(got - want)[:, fl == 0].max() <= 1e-12
    assert abs(s.kinetic_energy() - o.kinetic_energy()) <= 1e-12
    r, uu = s.macroscopic()
    ro, uo = o.macroscopic()
    assert np.abs(r - ro.reshape(NX, NY, NZ)).max() <= 1e-12 and np.abs(uu - uo.reshape(3, NX, NY, NZ)).max() <= 1e-12
    s.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_SOA"])
def test_step_parts_state_machine(scheme):
    import torch
    from paper_2010_11751_b200 import Lbm
    from paper_2010_11751_b200.binding import LbmError
    fl = slab.local_flags(inputs.cavity_flags(8, 6, 6), 2, 6)
    g = Lbm(6, 6, 6, scheme=scheme, omega=1.5)
    g.set_flags(fl, (0.02, 0, 0))
    rho, u = inputs.seeded_init(6, 6, 6, 0)
    buf = torch.zeros(g.halo_count, dtype=torch.float64, device="cuda")
    with pytest.raises(LbmError):
        g.step_begin()                      # nothing loaded yet
    g.init_equilibrium(rho, u)
    with pytest.raises(LbmError):
        g.step_end()                        # no begin
    with pytest.raises(LbmError):
        g.halo_pack(0, buf.data_ptr())      # no step has run: nothing to send
    g.step_begin()
    for bad in (g.step_begin, g.step_finish, lambda: g.step(1), g.kinetic_energy, g.macroscopic, g.get_populations,
                lambda: g.set_relaxation(1.0, 1.0, 1.0), lambda: g.set_variant("default"), lambda: g.set_block(64),
                lambda: g.halo_unpack(0, buf.data_ptr())):
        with pytest.raises(LbmError):
            bad()
    g.halo_pack(0, buf.data_ptr())
    g.step_end()
    with pytest.raises(LbmError):
        g.step_end()
    g.halo_unpack(0, buf.data_ptr())
    g.step_finish()
    assert g.steps_done == 1
    with pytest.raises(LbmError):
        g.step(2)                           # ghost cells: the halo is due after every step
    if scheme == "SWAP_SOA":
        with pytest.raises(LbmError):
            g.step(1)                       # swap needs it between the passes
    else:
        g.step(1)
        assert g.steps_done == 2
    # re-loading the populations in mid-step resets the state machine
    g.step_begin()
    g.init_equilibrium(rho, u)
    g.step_begin(); g.step_end(); g.step_finish()
    assert g.steps_done == 1 and np.isfinite(g.kinetic_energy())
    g.close()


@pytest.mark.gpu
def test_slab_calls_reject_what_they_cannot_do():
    """fluid cells in the outermost layers would silently never be updated; ghost cells
    in a layout without halo calls would silently lose populations"""
    from paper_2010_11751_b200 import Lbm
    from paper_2010_11751_b200.binding import LbmError
    rho, u = inputs.seeded_init(8, 8, 8, 0)
    g = Lbm(8, 8, 8, scheme="2POP_SOA")       # fully periodic box: layers 0 and nx-1 hold fluid
    g.init_equilibrium(rho, u)
    with pytest.raises(LbmError):
        g.step_begin()
    g.step(3)
    g.close()
    ghosted = slab.local_flags(inputs.cavity_flags(10, 8, 8), 2, 8)
    for scheme in ("2POP_AOS", "SWAP_AOS", "AA_AOS"):
        g = Lbm(8, 8, 8, scheme=scheme)
        with pytest.raises(LbmError):
            g.set_flags(ghosted)
        g.init_equilibrium(rho, u)
        with pytest.raises(LbmError):
            g.step_begin()
        g.close()
    g = Lbm(8, 8, 8, scheme="2POP_SOA")
    g.set_flags(ghosted)
    with pytest.raises(LbmError):
        g.set_variant("generic_push")
    g.close()
    g = Lbm(8, 8, 8, scheme="2POP_SOA")
    g.set_variant("generic_push")
    with pytest.raises(LbmError):
        g.set_flags(ghosted)
    g.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme,mode", [("2POP_SOA", "overlap"), ("AA_SOA", "peer"), ("SWAP_SOA", "peer")])
@pytest.mark.parametrize("Q,model", [(19, "BGK_W2"), (27, "K")])
def test_slabs_equal_the_undivided_gpu_run_bitwise(Q, model, scheme, mode):
    """at a size the oracle does not step in seconds: the same kernels do the same arithmetic per
    cell whether the lattice is cut or not, so three slabs must reproduce the undivided GPU run
    bit for bit (ragged extents, cuts at x = 17 and 34)"""
    from paper_2010_11751_b200 import Lbm
    NX, NY, NZ, steps = 50, 40, 70, 25
    omega = 1.8
    fl = inputs.cavity_flags(NX, NY, NZ)
    uw = (inputs.U_LID, 0.0, 0.0)
    rho, u = inputs.seeded_init(NX, NY, NZ, 7)
    g = Lbm(NX, NY, NZ, lattice=Q, collision=model, scheme=scheme, omega=omega, dtype="f64")
    g.set_flags(fl, uw)
    g.init_equilibrium(rho, u)
    g.step(steps)
    want = g.get_populations().reshape(Q, NX, NY, NZ)
    e_want = g.kinetic_energy()
    assert np.isfinite(want).all()
    g.close()
    engines, ranges = [], []
    for r in range(3):
        x0, x1 = slab.slab_range(NX, r, 3)
        e = slab.GpuSlabEngine(slab.local_flags(fl, x0, x1), uw, lattice=Q, collision=model, omega=omega, dtype="f64", scheme=scheme)
        e.lbm.init_equilibrium(slab.local_field(rho.reshape(NX, NY, NZ), x0, x1),
                               slab.local_field(u.reshape(3, NX, NY, NZ), x0, x1, axis=1))
        engines.append(e)
        ranges.append((x0, x1))
    if mode == "peer":
        slab.link_ring(engines)
    for _ in range(steps):
        slab.step_local(engines, mode=mode)
    energy = 0.0
    for e, (x0, x1) in zip(engines, ranges):
        got = slab.interior(e.lbm.get_populations().reshape(Q, x1 - x0 + 2, NY, NZ), axis=1)
        assert np.array_equal(got, want[:, x0:x1])
        energy += e.lbm.kinetic_energy()
        e.close()
    assert abs(energy - e_want) <= 1e-12 * max(1.0, abs(e_want))


@pytest.mark.gpu
@pytest.mark.parametrize("scheme,dtype", [("AA_SOA", "f64"), ("SWAP_SOA", "f64"), ("2POP_SOA", "f32")])
def test_slabs_beyond_l2_equal_the_undivided_gpu_run_bitwise(scheme, dtype):
    """slabs large enough (> 60 MB of populations each) for the range launches to alternate their traversal
    direction and to prefetch: two slabs through the library's peer-store driver reproduce the undivided
    run bit for bit (sampled cells), odd step count"""
    from paper_2010_11751_b200 import Lbm
    NX, NY, NZ, steps = 112, 96, 130, 7
    omega = 1.8
    npdt = np.float64 if dtype == "f64" else np.float32
    fl = inputs.cavity_flags(NX, NY, NZ)
    uw = (inputs.U_LID, 0.0, 0.0)
    rho, u = inputs.seeded_init(NX, NY, NZ, 3)
    rho, u = rho.astype(npdt), u.astype(npdt)
    g = Lbm(NX, NY, NZ, lattice=19, collision="TRT", scheme=scheme, omega=omega, dtype=dtype)
    g.set_flags(fl, uw)
    g.init_equilibrium(rho, u)
    g.step(steps)
    cells = np.arange(0, NX * NY * NZ, 53, dtype=np.int64)
    want = g.get_populations_at(cells.astype(np.int32))
    e_want = g.kinetic_energy()
    g.close()
    engines, ranges = [], []
    for r in range(2):
        x0, x1 = slab.slab_range(NX, r, 2)
        e = slab.GpuSlabEngine(slab.local_flags(fl, x0, x1), uw, lattice=19, collision="TRT", omega=omega, dtype=dtype, scheme=scheme)
        e.lbm.init_equilibrium(slab.local_field(rho.reshape(NX, NY, NZ), x0, x1),
                               slab.local_field(u.reshape(3, NX, NY, NZ), x0, x1, axis=1))
        engines.append(e)
        ranges.append((x0, x1))
    slab.link_ring(engines)
    for _ in range(steps):
        slab.step_local(engines, mode="peer")
    energy = 0.0
    layer = NY * NZ
    for e, (x0, x1) in zip(engines, ranges):
        e.lbm.slab_status()
        mine = cells[(cells >= x0 * layer) & (cells < x1 * layer)]
        local = (mine - (x0 - 1) * layer).astype(np.int32)      # the slab's context starts one (ghost) layer below x0
        got = e.lbm.get_populations_at(local)
        sel = (cells >= x0 * layer) & (cells < x1 * layer)
        assert np.isfinite(got).all() and np.array_equal(got, want[:, sel])
        energy += e.lbm.kinetic_energy()
        e.close()
    assert abs(energy - e_want) <= (1e-12 if dtype == "f64" else 1e-6) * max(1.0, abs(e_want))
