"""The entry point that allocates nothing: lbm_kinetic_energy_device_static (include/lbm.h) keeps the partial sums of
the kinetic-energy reduce in a fixed device array of the library instead of a buffer from
lbm_create.  Checked against the existing path (lbm_kinetic_energy_device: same kernels, same fixed reduction tree,
so the bits must agree; the tolerance asserted is the 1e-12 of the other energy tests) and against the oracle, on
calls in a row that share the array: a large lattice first, then a small one (whose call must not see what the large
one left behind), then the large one again after more steps.  This file is collected last on purpose
(pytest -x: a failure here hides nothing else)."""
import numpy as np
import pytest

from paper_2010_11751_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _make(Lbm, shape, scheme, dtype, steps, Q=19, model="BGK_W2"):
    nx, ny, nz = shape
    fl = inputs.cavity_flags(nx, ny, nz)
    rho, u = inputs.seeded_init(nx, ny, nz, 11)
    npdt = np.float32 if dtype == "f32" else np.float64
    g = Lbm(nx, ny, nz, lattice=Q, collision=model, scheme=scheme, omega=1.7, dtype=dtype)
    g.set_flags(fl, (inputs.U_LID, 0.0, 0.0))
    g.init_equilibrium(rho.astype(npdt), u.astype(npdt))
    g.step(steps)
    return g, fl, rho.astype(npdt), u.astype(npdt)


def _both(g, torch):
    """(existing path, static-scratch path) of the kinetic energy, both into device doubles"""
    e_ref = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    e_new = torch.full((1,), -2.0, dtype=torch.float64, device="cuda")
    g.kinetic_energy_device(e_ref.data_ptr())
    g.kinetic_energy_device_static(e_new.data_ptr())
    torch.cuda.synchronize()
    return float(e_ref.item()), float(e_new.item())


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_static_scratch_energy_matches_the_existing_path_on_calls_in_a_row(dtype):
    import torch
    from paper_2010_11751_b200 import Lbm
    big, fl_big, _, _ = _make(Lbm, (96, 90, 100), "AA_SOA", dtype, 5)          # 864 000 cells: 3 375 partials, odd AA parity
    small, fl_small, rho_s, u_s = _make(Lbm, (14, 15, 17), "2POP_SOA", dtype, 4)   # 3 570 cells: 14 partials
    try:
        mem0 = torch.cuda.memory_allocated()
        dev0 = (big.device_bytes, small.device_bytes)
        r1, s1 = _both(big, torch)             # call 1: fills 3 375 + 7 elements of the array
        r2, s2 = _both(small, torch)           # call 2 right after it: must read only its own 14 + 1
        big.step(3)
        r3, s3 = _both(big, torch)             # call 3: the array holds the small lattice's partials in front
        r4, s4 = _both(big, torch)             # and once more: repeatable
        for r, s in ((r1, s1), (r2, s2), (r3, s3), (r4, s4)):
            assert np.isfinite(s) and s > 0.0
            assert abs(s - r) <= TOL * max(1.0, abs(r)), (r, s)
            assert s == r                      # same kernels, same tree: the same bits
        assert s3 == s4 and s3 != s1
        # nothing was allocated by the calls, neither through the library's hooks nor behind torch's back
        assert (big.device_bytes, small.device_bytes) == dev0
        assert torch.cuda.memory_allocated() == mem0             # the result doubles of _both are gone again
        # and the small lattice against the oracle
        from oracle import lbm_oracle
        o = lbm_oracle.Oracle(14, 15, 17, Q=19, model="BGK_W2", omega=1.7)
        o.set_flags(fl_small, (inputs.U_LID, 0.0, 0.0))
        o.init_equilibrium(rho_s.astype(np.float64), u_s.astype(np.float64))
        o.step(4)
        eo = o.kinetic_energy()
        assert abs(s2 - eo) <= (TOL if dtype == "f64" else 1e-6) * max(1.0, abs(eo))
    finally:
        big.close()
        small.close()


def test_static_scratch_rejects_lattices_beyond_its_fixed_size_and_wrong_states():
    import torch
    from paper_2010_11751_b200 import Lbm
    from paper_2010_11751_b200.binding import LbmError, STATIC_MAX_CELLS
    e = torch.zeros(1, dtype=torch.float64, device="cuda")
    # 512 x 512 x 256 = 67 108 864 cells > 66 977 792: refused with a message that names the limit
    assert 512 * 512 * 256 > STATIC_MAX_CELLS
    g = Lbm(512, 512, 256, scheme="AA_SOA", dtype="f32")
    try:
        with pytest.raises(LbmError, match="static scratch holds"):
            g.kinetic_energy_device_static(e.data_ptr())
    finally:
        g.close()
    # the largest cube that fits is accepted as far as the size goes (406^3 <= limit < 407^3)
    assert 406 ** 3 <= STATIC_MAX_CELLS < 407 ** 3
    g = Lbm(8, 8, 8, scheme="2POP_SOA")
    try:
        with pytest.raises(LbmError, match="no populations"):
            g.kinetic_energy_device_static(e.data_ptr())      # nothing loaded yet
        with pytest.raises(LbmError):
            g.kinetic_energy_device_static(0)                 # null output
    finally:
        g.close()
