"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot step 256^3 or 512^3 lattices in seconds, but a lattice Boltzmann update has a
finite domain of dependence: after s steps the populations of a cell depend only on the initial
state within s cells of it (one cell per step, Eq 2).  So sampled outputs are
computed "one by one": for a small box of cells the oracle steps the sub-lattice that contains the
box plus a halo of s cells (same flags, same seeded initial values, cut faces left to the
sub-lattice's own periodic wrap, whose error cannot reach the box in s steps) and the CUDA path's
populations of those cells (lbm_get_populations_at) must match element by element.  Boxes sit at
the lid corner, on walls, across thread-block and row boundaries, and in the bulk.  On top of
that: properties that hold at any size (mass conservation, scheme independence PAPER.md:L141) at
the config's full step count, config 2 in full against the oracle, and the shear-wave decay.
"""
import numpy as np
import pytest

from paper_2010_11751_b200 import inputs

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 2e-5
MOMENT_SPACE = ("RM", "HM", "CM", "CHM", "K", "RR")
ALL_MODELS = ["BGK_W2", "BGK_NW4", "TRT", "RM", "HM", "CM", "CHM", "K", "RR", "REG"]
ALL_SCHEMES = ["2POP_SOA", "2POP_AOS", "SWAP_SOA", "SWAP_AOS", "AA_SOA", "AA_AOS"]


@pytest.fixture(scope="module")
def Lbm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_11751_b200 import Lbm as cls
    return cls


_case_cache = {}


def cavity(n, re):
    """flags, u_wall, rho, u (float64), omega of the n^3 cavity; cached (512^3 takes a while)"""
    if n not in _case_cache:
        _case_cache.clear()
        fl = inputs.cavity_flags(n, n, n)
        rho, u = inputs.seeded_init(n, n, n, 0)
        _case_cache[n] = (fl, rho, u)
    fl, rho, u = _case_cache[n]
    return fl, (inputs.U_LID, 0.0, 0.0), rho, u, inputs.omega_from_re(n, re)


def sample_boxes(n, b):
    """origins of b^3 boxes: lid corner, lid/wall edge, a wall, the far corner, bulk positions that
    straddle 128-cell block boundaries and row ends"""
    m = n // 2
    return [(1, 1, n - 1 - b), (m, 1, n - 1 - b), (1, m - 3, m - 3), (n - 1 - b, n - 1 - b, 1),
            (m - 3, m - 3, 128 - 3 if n > 140 else m - 3), (m + 5, n - 1 - b, n - 1 - b), (m, m, m)]


def make_gpu(Lbm, n, Q, model, scheme, dtype, omega, fl, uw, rho, u, bulk_one=True):
    npdt = np.float32 if dtype == "f32" else np.float64
    g = Lbm(n, n, n, lattice=Q, collision=model, scheme=scheme, omega=omega, dtype=dtype)
    g.set_flags(fl, uw)
    if bulk_one and model in MOMENT_SPACE:  # the harness setting (R25)
        hi = omega if model == "RR" else 1.0
        g.set_relaxation(1.0, hi, hi)
    g.init_equilibrium(rho.astype(npdt), u.astype(npdt))
    return g


def subbox_error(g, oracle, n, Q, model, dtype, omega, fl, uw, rho, u, steps, b=6, bulk_one=True, boxes=None):
    """max error of the CUDA path against the oracle over all sample boxes after `steps` steps
    (g must already have done them)"""
    npdt = np.float32 if dtype == "f32" else np.float64
    rho3 = rho.reshape(n, n, n)
    u3 = u.reshape(3, n, n, n)
    _, t, _, _ = oracle.lattice(Q)
    worst = 0.0
    for (x0, y0, z0) in (boxes or sample_boxes(n, b)):
        lo = [max(0, v - steps) for v in (x0, y0, z0)]
        hi = [min(n, v + b + steps) for v in (x0, y0, z0)]
        sl = tuple(slice(a, c) for a, c in zip(lo, hi))
        sfl = np.ascontiguousarray(fl[sl])
        sx, sy, sz = sfl.shape
        o = oracle.Oracle(sx, sy, sz, Q=Q, model=model, omega=omega)
        o.set_flags(sfl, uw)
        if bulk_one and model in MOMENT_SPACE:
            hi_rate = omega if model == "RR" else 1.0
            o.set_relaxation(1.0, hi_rate, hi_rate)
        srho = np.ascontiguousarray(rho3[sl]).astype(npdt).astype(np.float64)  # oracle fed the rounded inputs (R20)
        su = np.ascontiguousarray(u3[(slice(None),) + sl]).astype(npdt).astype(np.float64)
        o.init_equilibrium(srho.reshape(-1), su.reshape(3, -1))
        o.step(steps)
        fo = o.get_populations().reshape(Q, sx, sy, sz)
        bx = np.arange(x0, x0 + b)
        by = np.arange(y0, y0 + b)
        bz = np.arange(z0, z0 + b)
        X, Y, Z = np.meshgrid(bx, by, bz, indexing="ij")
        cells = ((X * n + Y) * n + Z).reshape(-1).astype(np.int32)
        fg = g.get_populations_at(cells).astype(np.float64)
        ref = fo[:, X - lo[0], Y - lo[1], Z - lo[2]].reshape(Q, -1)
        fluid = fl.reshape(-1)[cells] == 0
        assert fluid.any()
        assert np.isfinite(fg).all()
        assert np.all(fg[:, ~fluid] == 0.0)
        d = np.abs(fg - ref)[:, fluid]
        if dtype == "f32":
            d = d / np.maximum(np.abs(ref[:, fluid]), t[:, None])
        worst = max(worst, float(d.max()))
    return worst


def fluid_mass(g, fl):
    rho, _ = g.macroscopic()
    assert np.isfinite(rho).all()
    return float(rho.astype(np.float64)[fl.reshape(-1) == 0].sum(dtype=np.float64))


# ------------------------------------------------------------------ config 2 (128^3 AA, in full)
def test_config2_cavity128_aa_full_oracle(Lbm, oracle):
    """BASELINE.json config 2: every population of the 128^3 cavity against the oracle at the
    100-step gate, at an odd step count (AA un-shuffle) and at the config's 1000 steps."""
    n = 128
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 19, "BGK_W2", "AA_SOA", "f64", omega, fl, uw, rho, u)
    o = oracle.Oracle(n, n, n, Q=19, model="BGK_W2", omega=omega)
    o.set_flags(fl, uw)
    o.init_equilibrium(rho, u)
    fluid = fl.reshape(-1) == 0
    errs = {}
    done = 0
    for target in (100, 999, 1000):
        g.step(target - done)
        o.step(target - done)
        done = target
        fg, fo = g.get_populations(), o.get_populations()
        assert np.isfinite(fg).all()
        errs[target] = float(np.abs(fg - fo)[:, fluid].max())
    assert errs[100] <= TOL64, errs
    assert errs[999] <= TOL64 and errs[1000] <= TOL64, errs   # expected ~1e-15 (R23, R24)
    assert abs(g.kinetic_energy() - o.kinetic_energy()) <= 1e-12 * max(1.0, o.kinetic_energy())


@pytest.mark.parametrize("omega,tol", [(1.0, 1e-6), (1.9702104184, None)])
def test_config2_shear_wave_128(Lbm, oracle, omega, tol):
    """periodic 128^3, u_x = 0.01 sin(2 pi y/128), 1000 steps: decay exp(-nu k^2 t) (pin P3) and
    element-wise agreement with the oracle's 1 x 128 x 1 box (the field is uniform in x and z)."""
    n, steps = 128, 1000
    rho, u = inputs.shear_wave(n, n, n)
    g = Lbm(n, n, n, lattice=19, collision="BGK_W2", scheme="AA_SOA", omega=omega, dtype="f64")
    g.set_flags(inputs.periodic_flags(n, n, n))
    g.init_equilibrium(rho, u)
    g.step(steps)
    rg, ug = g.macroscopic()
    ux = ug[0].reshape(n, n, n)
    assert np.abs(ux - ux[0:1, :, 0:1]).max() <= 1e-13            # stays uniform in x and z
    r1, u1 = inputs.shear_wave(1, n, 1)
    o = oracle.Oracle(1, n, 1, Q=19, model="BGK_W2", omega=omega)
    o.set_flags(inputs.periodic_flags(1, n, 1))
    o.init_equilibrium(r1, u1)
    o.step(steps)
    ro, uo = o.macroscopic()
    assert np.abs(ux[3, :, 5] - uo[0]).max() <= 1e-13
    assert np.abs(rg.reshape(n, n, n)[3, :, 5] - ro).max() <= 1e-13
    y = np.arange(n)
    s = np.sin(2 * np.pi * y / n)
    amp = 2.0 * (ux[3, :, 5] * s).mean() / 0.01
    nu = (1.0 / omega - 0.5) / 3.0
    k = 2 * np.pi / n
    expect = np.exp(-nu * k * k * steps)
    if tol is not None:
        assert abs(np.log(amp) / np.log(expect) - 1.0) <= tol     # fitted viscosity
    else:
        assert abs(amp - expect) <= 5e-4                           # P3, loose form at config 2's omega


# ------------------------------------------------------------------ config 3 (256^3)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA"])
@pytest.mark.parametrize("model", ["TRT", "REG"])
def test_config3_256_sampled(Lbm, oracle, model, scheme, dtype):
    n, steps = 256, 7  # odd: AA exports through the un-shuffle, 2-pop through the lazy stream
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 19, model, scheme, dtype, omega, fl, uw, rho, u)
    g.step(steps)
    err = subbox_error(g, oracle, n, 19, model, dtype, omega, fl, uw, rho, u, steps)
    assert err <= (TOL32 if dtype == "f32" else TOL64), err


def test_config3_256_properties_500_steps(Lbm):
    """mass conservation over the config's 500 steps and scheme independence"""
    n = 256
    fl, uw, rho, u, omega = cavity(n, 1000)
    cells = np.concatenate([((np.arange(1, 9)[:, None, None] * n + np.arange(1, 9)[None, :, None]) * n
                             + np.arange(n - 9, n - 1)[None, None, :]).reshape(-1),
                            np.arange(n * n * 100 + n * 77 + 3, n * n * 100 + n * 77 + 250)]).astype(np.int32)
    pops = {}
    for scheme in ("2POP_SOA", "AA_SOA"):
        g = make_gpu(Lbm, n, 19, "TRT", scheme, "f64", omega, fl, uw, rho, u)
        m0 = fluid_mass(g, fl)
        g.step(500)
        m1 = fluid_mass(g, fl)
        assert abs(m1 - m0) <= 1e-13 * 500 * m0, (m0, m1)
        pops[scheme] = g.get_populations_at(cells)
        g.close()
    assert np.abs(pops["2POP_SOA"] - pops["AA_SOA"]).max() <= 1e-13


# ------------------------------------------------------------------ config 4 (192^3 D3Q27 swap)
@pytest.mark.parametrize("model", ALL_MODELS)
def test_config4_192_d3q27_swap_sampled(Lbm, oracle, model):
    n, steps = 192, 5
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 27, model, "SWAP_SOA", "f64", omega, fl, uw, rho, u)
    g.step(steps)
    err = subbox_error(g, oracle, n, 27, model, "f64", omega, fl, uw, rho, u, steps, b=5)
    assert err <= TOL64, err


def test_config4_192_mass_200_steps(Lbm):
    n = 192
    fl, uw, rho, u, omega = cavity(n, 1000)
    for model in ("K", "RR"):
        g = make_gpu(Lbm, n, 27, model, "SWAP_SOA", "f64", omega, fl, uw, rho, u)
        m0 = fluid_mass(g, fl)
        g.step(200)
        m1 = fluid_mass(g, fl)
        assert abs(m1 - m0) <= 1e-13 * 200 * m0, (model, m0, m1)
        g.close()


# ------------------------------------------------------------------ config 5 (512^3)
@pytest.mark.parametrize("scheme,dtype", [("AA_SOA", "f32"), ("2POP_SOA", "f64")] +
                         [(s, "f32") for s in ALL_SCHEMES if s != "AA_SOA"] + [("AA_SOA", "f64"), ("SWAP_SOA", "f64")])
def test_config5_512_sampled(Lbm, oracle, scheme, dtype):
    """134M cells: 64-bit slot arithmetic (19 * 512^3 > 2^31), all schemes"""
    n, steps = 512, 5
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 19, "BGK_W2", scheme, dtype, omega, fl, uw, rho, u)
    g.step(steps)
    err = subbox_error(g, oracle, n, 19, "BGK_W2", dtype, omega, fl, uw, rho, u, steps)
    assert err <= (TOL32 if dtype == "f32" else TOL64), err
    assert np.isfinite(g.kinetic_energy())
    g.close()


# ------------------------------------------------------------------ target (256^3 BGK fp64)
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA"])
def test_target_256_bgk_sampled(Lbm, oracle, scheme):
    n = 256
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 19, "BGK_W2", scheme, "f64", omega, fl, uw, rho, u)
    for steps in (6, 7):
        g.init_equilibrium(rho, u)
        g.step(steps)
        err = subbox_error(g, oracle, n, 19, "BGK_W2", "f64", omega, fl, uw, rho, u, steps)
        assert err <= TOL64, (steps, err)


# ------------------------------------------------------------------ the 100-step gate at full size
def _report(name, **kv):
    """append one line to gpurun_out/parity_report.jsonl (scratch; summarised under profiles/)"""
    import json
    import os
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    try:
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_report.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(test=name, **kv)) + "\n")
    except OSError:
        pass


_oracle_256 = {}


def oracle_target_256(oracle, steps):
    """every population of the 256^3 target (D3Q19 BGK-W2 fp64 cavity, Re = 1000, seeded init) after
    `steps` oracle steps; computed once per session (about 17 M cells x 100 steps on the host cores)"""
    if steps not in _oracle_256:
        n = 256
        fl, uw, rho, u, omega = cavity(n, 1000)
        o = oracle.Oracle(n, n, n, Q=19, model="BGK_W2", omega=omega)
        o.set_flags(fl, uw)
        o.init_equilibrium(rho, u)
        o.step(steps)
        _oracle_256.clear()
        _oracle_256[steps] = (o.get_populations(), o.kinetic_energy())
        del o
    return _oracle_256[steps]


@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA"])
def test_target_256_bgk_every_population_100_steps(Lbm, oracle, scheme):
    """north_star's gate on the target itself: max |f_gpu - f_oracle| <= 1e-12 over EVERY population of
    EVERY fluid cell of the 256^3 cavity after 100 steps, in the launch configuration bench.py times
    ("identical results"; readings R23, R24)."""
    n, steps = 256, 100
    fl, uw, rho, u, omega = cavity(n, 1000)
    fo, eo = oracle_target_256(oracle, steps)
    g = make_gpu(Lbm, n, 19, "BGK_W2", scheme, "f64", omega, fl, uw, rho, u)
    g.step(steps)
    fg = g.get_populations()
    eg = g.kinetic_energy()
    g.close()
    assert np.isfinite(fg).all()
    fluid = fl.reshape(-1) == 0
    err = 0.0
    for k in range(19):      # plane by plane: no 2.5 GB temporaries
        err = max(err, float(np.abs(fg[k] - fo[k])[fluid].max()))
        assert np.all(fg[k][~fluid] == 0.0)
    _report("target_256_100_steps", scheme=scheme, max_abs=err, energy_gpu=eg, energy_oracle=eo)
    assert err <= TOL64, err
    assert abs(eg - eo) <= 1e-12 * max(1.0, abs(eo))


@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA"])
@pytest.mark.parametrize("model", ["TRT", "REG"])
def test_config3_fp32_500_steps_beyond_l2(Lbm, oracle, model, scheme):
    """config 3's step count (500) in fp32 against the fp64 oracle on a lattice beyond L2 (112 x 96 x 130,
    1.4 M cells, 106 MB per array: the strided-prefetch path of the fp32 kernels), every population;
    the 100-step gate (<= 2e-5 relative, R20) and the 500-step error are reported separately (R24)."""
    nx, ny, nz = 112, 96, 130
    fl = inputs.cavity_flags(nx, ny, nz)
    uw = (inputs.U_LID, 0.0, 0.0)
    rho, u = inputs.seeded_init(nx, ny, nz, 0)
    omega = inputs.omega_from_re(256, 1000)            # config 3's relaxation rate
    rho32, u32 = rho.astype(np.float32), u.astype(np.float32)
    g = Lbm(nx, ny, nz, lattice=19, collision=model, scheme=scheme, omega=omega, dtype="f32")
    g.set_flags(fl, uw)
    g.init_equilibrium(rho32, u32)
    o = oracle.Oracle(nx, ny, nz, Q=19, model=model, omega=omega)
    o.set_flags(fl, uw)
    o.init_equilibrium(rho32.astype(np.float64), u32.astype(np.float64))   # the rounded inputs (R20)
    _, t, _, _ = oracle.lattice(19)
    fluid = fl.reshape(-1) == 0
    errs = {}
    done = 0
    for target in (100, 500):
        g.step(target - done)
        o.step(target - done)
        done = target
        fg = g.get_populations().astype(np.float64)
        fo = o.get_populations()
        assert np.isfinite(fg).all()
        d = np.abs(fg - fo)[:, fluid]
        errs[target] = (float((d / np.maximum(np.abs(fo[:, fluid]), t[:, None])).max()), float(d.max()))
    g.close()
    _report("config3_fp32_500_steps", model=model, scheme=scheme, rel_100=errs[100][0], abs_100=errs[100][1],
            rel_500=errs[500][0], abs_500=errs[500][1])
    assert errs[100][0] <= TOL32, errs
    assert errs[500][0] <= TOL32, errs


@pytest.mark.parametrize("scheme,steps", [("2POP_SOA", 100), ("AA_SOA", 100), ("AA_SOA", 101)])
def test_config3_256_sampled_100_steps(Lbm, oracle, scheme, steps):
    """config 3 (TRT, fp64) at the 100-step gate on the full 256^3 lattice: sampled boxes whose domain of
    dependence (100 cells each way) the oracle steps; the lid-corner box alone spans 106^3 cells."""
    n = 256
    fl, uw, rho, u, omega = cavity(n, 1000)
    g = make_gpu(Lbm, n, 19, "TRT", scheme, "f64", omega, fl, uw, rho, u)
    g.step(steps)
    err = subbox_error(g, oracle, n, 19, "TRT", "f64", omega, fl, uw, rho, u, steps, boxes=[(1, 1, n - 7), (n // 2, n // 2, n // 2)])
    g.close()
    _report("config3_256_sampled_100", scheme=scheme, steps=steps, max_abs=err)
    assert err <= TOL64, err
