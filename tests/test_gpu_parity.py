"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerances are BASELINE.json's: max-abs population difference <= 1e-12
after 100 steps in fp64; <= 2e-5 relative (to max(|f|, t_k), reading R20) in fp32."""
import numpy as np
import pytest

from paper_2010_11751_b200 import inputs

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 2e-5
ALL_MODELS = ["BGK_W2", "BGK_NW4", "TRT", "RM", "HM", "CM", "CHM", "K", "RR", "REG"]
ALL_SCHEMES = ["2POP_SOA", "2POP_AOS", "SWAP_SOA", "SWAP_AOS", "AA_SOA", "AA_AOS"]


@pytest.fixture(scope="module")
def Lbm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_11751_b200 import Lbm as cls
    return cls


def box_flags(nx, ny, nz, kind):
    if kind == "cavity":
        return inputs.cavity_flags(nx, ny, nz), (inputs.U_LID, 0.0, 0.0)
    if kind == "periodic":
        return inputs.periodic_flags(nx, ny, nz), (0.0, 0.0, 0.0)
    if kind == "obstacle":  # periodic box with a moving block and a resting block inside: walls + seam
        fl = inputs.periodic_flags(nx, ny, nz)
        fl[1:3, 2:4, 1:3] = inputs.MOVING
        fl[nx - 2:, 0:2, nz // 2] = inputs.WALL
        return fl, (0.01, -0.02, 0.015)
    raise ValueError(kind)


def run_pair(Lbm, oracle, shape, Q, model, scheme, dtype, steps, kind="cavity", omega=1.7, variant=None, seed=0,
             rates=None, chunks=None):
    nx, ny, nz = shape
    fl, uw = box_flags(nx, ny, nz, kind)
    rho, u = inputs.seeded_init(nx, ny, nz, seed)
    npdt = np.float32 if dtype == "f32" else np.float64
    rho_in, u_in = rho.astype(npdt), u.astype(npdt)
    g = Lbm(nx, ny, nz, lattice=Q, collision=model, scheme=scheme, omega=omega, dtype=dtype)
    o = oracle.Oracle(nx, ny, nz, Q=Q, model=model, omega=omega)
    g.set_flags(fl, uw)
    o.set_flags(fl, uw)
    if rates is not None:
        g.set_relaxation(*rates)
        o.set_relaxation(*rates)
    if variant is not None:
        g.set_variant(variant)
    g.init_equilibrium(rho_in, u_in)
    o.init_equilibrium(rho_in.astype(np.float64), u_in.astype(np.float64))  # oracle fed the rounded inputs (R20)
    for n in (chunks or [steps]):
        g.step(n)
    o.step(steps)
    assert g.steps_done == steps
    return g, o, fl


def pop_error(g, o, fl, Q, oracle, relative):
    fg = g.get_populations().astype(np.float64)
    fo = o.get_populations()
    assert np.isfinite(fg).all()
    fluid = (fl.reshape(-1) == 0)
    assert np.all(fg[:, ~fluid] == 0.0)
    d = np.abs(fg - fo)[:, fluid]
    if not relative:
        return d.max()
    _, t, _, _ = oracle.lattice(Q)
    den = np.maximum(np.abs(fo[:, fluid]), t[:, None])
    return (d / den).max()


def test_config1_cavity32_bgk_2pop_fp64(Lbm, oracle):
    """BASELINE.json config 1: 32^3 cavity, D3Q19 BGK-W2, 2-pop SoA, Re=100, 100 steps."""
    n = 32
    omega = inputs.omega_from_re(n, 100)
    g, o, fl = run_pair(Lbm, oracle, (n, n, n), 19, "BGK_W2", "2POP_SOA", "f64", 100, omega=omega)
    err = pop_error(g, o, fl, 19, oracle, False)
    assert err <= TOL64, err
    rg, ug = g.macroscopic()
    ro, uo = o.macroscopic()
    assert np.abs(rg - ro).max() <= 1e-12 and np.abs(ug - uo).max() <= 1e-12
    eg, eo = g.kinetic_energy(), o.kinetic_energy()
    assert abs(eg - eo) <= 1e-12 * max(1.0, abs(eo))
    assert eg == g.kinetic_energy()  # fixed reduction tree: bitwise repeatable
    import torch
    e_d = torch.zeros(1, dtype=torch.float64, device="cuda")
    g.kinetic_energy_device(e_d.data_ptr())
    assert float(e_d.item()) == eg


@pytest.mark.parametrize("variant", ["generic_push", "generic_pull"])
@pytest.mark.parametrize("kind", ["cavity", "periodic", "obstacle"])
def test_2pop_variants_ragged(Lbm, oracle, variant, kind):
    g, o, fl = run_pair(Lbm, oracle, (13, 10, 7), 19, "BGK_W2", "2POP_SOA", "f64", 25, kind=kind, variant=variant,
                        chunks=[1, 7, 17])
    assert pop_error(g, o, fl, 19, oracle, False) <= TOL64
    rg, ug = g.macroscopic()
    ro, uo = o.macroscopic()
    assert np.abs(rg - ro).max() <= 1e-12 and np.abs(ug - uo).max() <= 1e-12
    assert abs(g.kinetic_energy() - o.kinetic_energy()) <= 1e-13


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("scheme", ALL_SCHEMES)
@pytest.mark.parametrize("kind", ["cavity", "obstacle"])
def test_schemes_match_oracle(Lbm, oracle, Q, scheme, kind):
    """all six schemes give the oracle's populations, at even and odd step counts"""
    for steps in (6, 7):
        g, o, fl = run_pair(Lbm, oracle, (9, 11, 8), Q, "BGK_W2", scheme, "f64", steps, kind=kind)
        assert pop_error(g, o, fl, Q, oracle, False) <= TOL64
        rg, ug = g.macroscopic()
        ro, uo = o.macroscopic()
        assert np.abs(rg - ro).max() <= 1e-12 and np.abs(ug - uo).max() <= 1e-12
        assert abs(g.kinetic_energy() - o.kinetic_energy()) <= 1e-13


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("model", ALL_MODELS)
def test_models_match_oracle_100_steps(Lbm, oracle, Q, model):
    """every collision model, default rates (R14), 100 steps on a small lid cavity, AA scheme"""
    g, o, fl = run_pair(Lbm, oracle, (8, 9, 10), Q, model, "AA_SOA", "f64", 100, omega=1.6)
    assert pop_error(g, o, fl, Q, oracle, False) <= TOL64


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("model", ["RM", "HM", "CM", "CHM", "K", "RR"])
def test_models_custom_rates(Lbm, oracle, Q, model):
    """Eq 11 / Eq 13-15 with a bulk rate and distinct third- and higher-order rates"""
    g, o, fl = run_pair(Lbm, oracle, (7, 8, 9), Q, model, "SWAP_SOA", "f64", 21, kind="obstacle", omega=1.5,
                        rates=(1.1, 1.3, 0.9))
    assert pop_error(g, o, fl, Q, oracle, False) <= TOL64


@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_AOS"])
@pytest.mark.parametrize("model", ["BGK_W2", "TRT", "REG"])
@pytest.mark.parametrize("Q", [19, 27])
def test_fp32(Lbm, oracle, Q, model, scheme):
    n = 16
    omega = inputs.omega_from_re(n, 100)
    g, o, fl = run_pair(Lbm, oracle, (n, n, n), Q, model, scheme, "f32", 100, omega=omega)
    assert pop_error(g, o, fl, Q, oracle, True) <= TOL32


@pytest.mark.parametrize("model", ["BGK_NW4", "RM", "HM", "CM", "CHM", "K", "RR"])
@pytest.mark.parametrize("Q", [19, 27])
def test_fp32_moment_space_models(Lbm, oracle, Q, model):
    """the moment-space family in fp32 on shifted storage (R20), omega_bulk = 1 as in the paper's
    production run (R25), 100 steps, both parities of the AA scheme and two-population"""
    n = 14
    omega = inputs.omega_from_re(n, 100)
    hi = omega if model == "RR" else 1.0
    for scheme, steps in (("AA_SOA", 100), ("2POP_SOA", 99)):
        g, o, fl = run_pair(Lbm, oracle, (n, n + 1, n + 3), Q, model, scheme, "f32", steps, omega=omega, rates=(1.0, hi, hi))
        assert pop_error(g, o, fl, Q, oracle, True) <= TOL32
        assert abs(g.kinetic_energy() - o.kinetic_energy()) <= 1e-5 * max(1.0, o.kinetic_energy())


def test_set_get_roundtrip_and_restart(Lbm, oracle):
    """populations exported at an odd AA step and re-imported continue identically"""
    shape = (9, 8, 10)
    g, o, fl = run_pair(Lbm, oracle, shape, 19, "TRT", "AA_SOA", "f64", 5, kind="obstacle")
    f5 = g.get_populations()
    g2 = Lbm(*shape, lattice=19, collision="TRT", scheme="2POP_AOS", omega=1.7, dtype="f64")
    fl2, uw = box_flags(*shape, "obstacle")
    g2.set_flags(fl2, uw)
    g2.set_populations(f5)
    assert np.array_equal(g2.get_populations(), f5)
    g.step(4)
    g2.step(4)
    o.step(4)
    assert np.abs(g.get_populations() - g2.get_populations()).max() <= 1e-14
    assert pop_error(g2, o, fl, 19, oracle, False) <= TOL64


def test_state_errors(Lbm):
    from paper_2010_11751_b200.binding import LbmError
    g = Lbm(8, 8, 8)
    with pytest.raises(LbmError):
        g.step(1)
    with pytest.raises(LbmError):
        g.kinetic_energy()
    with pytest.raises(LbmError):
        Lbm(2, 8, 8)
    assert g.kernel_launches >= 1 and g.device_bytes > 0


@pytest.mark.parametrize("scheme", ALL_SCHEMES)
def test_graph_replay_is_bitwise_the_plain_path(Lbm, oracle, scheme):
    """lbm_step through the captured CUDA graph (launch-bound lattices) == plain launches, bit for bit,
    from even and odd starting parities, and both match the oracle"""
    shape = (12, 9, 10)
    chunks = [3, 40, 16, 1, 37, 3]          # graph blocks start at odd and even times
    steps = sum(chunks)
    g, o, fl = run_pair(Lbm, oracle, shape, 19, "BGK_W2", scheme, "f64", steps, kind="obstacle", chunks=chunks)
    assert g.graph_replays >= 4
    fg = g.get_populations()
    assert pop_error(g, o, fl, 19, oracle, False) <= TOL64
    h = Lbm(*shape, lattice=19, collision="BGK_W2", scheme=scheme, omega=1.7, dtype="f64")
    fl2, uw = box_flags(*shape, "obstacle")
    rho, u = inputs.seeded_init(*shape, 0)
    h.set_flags(fl2, uw)
    h.set_graph("off")
    h.init_equilibrium(rho, u)
    h.step(steps)
    assert h.graph_replays == 0
    assert np.array_equal(h.get_populations(), fg)
    assert h.kernel_launches - 1 <= g.kernel_launches  # the graph's launches are counted too


def test_graph_dropped_when_rates_change(Lbm, oracle):
    """a setter between two lbm_step calls must not leave a stale graph behind"""
    shape = (10, 10, 10)
    fl, uw = box_flags(*shape, "cavity")
    rho, u = inputs.seeded_init(*shape, 3)
    g = Lbm(*shape, lattice=19, collision="RM", scheme="AA_SOA", omega=1.6, dtype="f64")
    o = oracle.Oracle(*shape, Q=19, model="RM", omega=1.6)
    for s in (g, o):
        s.set_flags(fl, uw)
        s.init_equilibrium(rho, u)
        s.step(32)
        s.set_relaxation(1.0, 1.2, 0.8)
        s.step(33)
    assert g.graph_replays >= 3
    assert pop_error(g, o, fl, 19, oracle, False) <= TOL64


@pytest.mark.parametrize("scheme,dtype,Q,model", [
    ("AA_SOA", "f64", 19, "TRT"), ("AA_SOA", "f32", 19, "TRT"), ("2POP_SOA", "f32", 19, "TRT"), ("SWAP_SOA", "f64", 19, "TRT"),
    ("SWAP_SOA", "f32", 19, "TRT"), ("2POP_SOA", "f64", 19, "BGK_W2"), ("AA_SOA", "f32", 27, "K"), ("SWAP_SOA", "f32", 27, "K"),
    ("2POP_SOA", "f64", 27, "K"), ("SWAP_SOA", "f64", 27, "BGK_W2")])
def test_prefetch_and_dependent_launch_do_not_change_results(Lbm, scheme, dtype, Q, model):
    """the L2 prefetch (on beyond 100 MB of populations; per thread in fp64, one strided warp in 32 in fp32, also in
    swap pass 2), the alternating traversal direction (beyond 60 MB) and the programmatic dependent launch are
    pure scheduling: populations after 11 steps are bit for bit those of a run with all three off"""
    nx, ny, nz = 112, 96, 130          # 1.4 M cells: 212 MB (fp64) / 106 MB (fp32) per array
    fl = inputs.cavity_flags(nx, ny, nz)
    rho, u = inputs.seeded_init(nx, ny, nz, 9)
    npdt = np.float32 if dtype == "f32" else np.float64
    cells = np.arange(0, nx * ny * nz, 97, dtype=np.int32)

    def run(variant="default"):
        g = Lbm(nx, ny, nz, lattice=Q, collision=model, scheme=scheme, omega=1.8, dtype=dtype)
        g.set_flags(fl, (inputs.U_LID, 0.0, 0.0))
        g.set_variant(variant)
        g.set_graph("off")
        g.init_equilibrium(rho.astype(npdt), u.astype(npdt))
        g.step(11)
        f, e = g.get_populations_at(cells), g.kinetic_energy()
        g.close()
        return f, e

    f1, e1 = run()
    f0, e0 = run("plain")
    assert np.isfinite(f1).all() and np.array_equal(f0, f1) and e0 == e1


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("scheme", ALL_SCHEMES)
@pytest.mark.parametrize("model", ALL_MODELS)
def test_every_model_on_every_scheme(Lbm, oracle, Q, scheme, model):
    """the cross product scheme x layout x model x lattice in fp64 (the staged AoS kernels and the
    two-population pull form with the moment-space models included), 7 steps on a ragged box with
    walls, a moving block and the periodic seam"""
    g, o, fl = run_pair(Lbm, oracle, (7, 8, 9), Q, model, scheme, "f64", 7, kind="obstacle", omega=1.6)
    assert pop_error(g, o, fl, Q, oracle, False) <= TOL64


_LONG_ROWS_ORACLE = {}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("scheme", ALL_SCHEMES)
@pytest.mark.parametrize("model", ALL_MODELS)
def test_every_model_on_every_scheme_long_rows(Lbm, oracle, Q, scheme, model, dtype):
    """the same cross product, in both precisions, on a box whose z-rows (100 cells) hold whole warps of bulk cells:
    the unmasked access path, the cooperative warp gather / scatter / exchange of the AoS kernels and their patches of
    four rows run here, next to the masked path of the warps at the walls, the moving block and the periodic seam
    (on the 7 x 8 x 9 box above every warp has an edge cell).  7 steps in two calls (3 + 4: both AA parities)."""
    shape, steps = (5, 6, 100), 7
    key = (Q, model, dtype)
    fl, uw = box_flags(*shape, "obstacle")
    rho, u = inputs.seeded_init(*shape, 4)
    npdt = np.float32 if dtype == "f32" else np.float64
    rho_in, u_in = rho.astype(npdt), u.astype(npdt)
    if key not in _LONG_ROWS_ORACLE:          # the oracle's result does not depend on the scheme
        o = oracle.Oracle(*shape, Q=Q, model=model, omega=1.6)
        o.set_flags(fl, uw)
        o.init_equilibrium(rho_in.astype(np.float64), u_in.astype(np.float64))
        o.step(steps)
        _LONG_ROWS_ORACLE[key] = o.get_populations().copy()
    fo = _LONG_ROWS_ORACLE[key]
    g = Lbm(*shape, lattice=Q, collision=model, scheme=scheme, omega=1.6, dtype=dtype)
    try:
        g.set_flags(fl, uw)
        g.init_equilibrium(rho_in, u_in)
        g.step(3)
        g.step(4)
        fg = g.get_populations().astype(np.float64)
    finally:
        g.close()
    fluid = fl.reshape(-1) == 0
    assert np.isfinite(fg).all() and np.all(fg[:, ~fluid] == 0.0)
    d = np.abs(fg - fo)[:, fluid]
    if dtype == "f64":
        assert d.max() <= TOL64, d.max()
    else:
        _, t, _, _ = oracle.lattice(Q)
        assert (d / np.maximum(np.abs(fo[:, fluid]), t[:, None])).max() <= TOL32


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("model", ["RM", "HM", "CM", "CHM", "K"])
def test_equilibrated_high_orders_is_the_general_collision_at_rate_one(Lbm, oracle, Q, model, dtype):
    """with the rates of every order >= 3 exactly 1 the library runs
    the variant that never computes those pre-collision moments.  It must give what the general
    kernel gives at a rate one ulp below 1 (which dispatches the general kernel), and the oracle's
    result at rate 1, for a bulk rate equal to and different from omega."""
    below_one = float(np.nextafter(1.0, 0.0))
    for bulk in (1.6, 1.0):
        g1, o, fl = run_pair(Lbm, oracle, (8, 9, 10), Q, model, "AA_SOA", dtype, 21, kind="obstacle", omega=1.6,
                             rates=(bulk, 1.0, 1.0))
        err = pop_error(g1, o, fl, Q, oracle, dtype == "f32")
        assert err <= (TOL64 if dtype == "f64" else TOL32), err
        g2 = Lbm(8, 9, 10, lattice=Q, collision=model, scheme="AA_SOA", omega=1.6, dtype=dtype)
        fl2, uw = box_flags(8, 9, 10, "obstacle")
        g2.set_flags(fl2, uw)
        g2.set_relaxation(bulk, below_one, below_one)
        rho, u = inputs.seeded_init(8, 9, 10, 0)
        g2.init_equilibrium(rho, u)
        g2.step(21)
        d = np.abs(g1.get_populations().astype(np.float64) - g2.get_populations().astype(np.float64)).max()
        assert d <= (1e-13 if dtype == "f64" else 2e-6), d
        g1.close(); g2.close()


def test_side_arrays_are_small(Lbm):
    """in-place AA storage halves the footprint only if the side arrays stay small: one code byte and
    a quarter byte of group table per cell, link masks for the edge cells only, staging areas held
    only while a host-facing call runs"""
    n = 256
    fl, uw, rho, u, omega = inputs.cavity_case(n, 1000)
    g = Lbm(n, n, n, scheme="AA_SOA", omega=omega, dtype="f32")
    g.set_flags(fl, uw)
    g.init_equilibrium(rho.astype(np.float32), u.astype(np.float32))
    g.step(2)
    rg, ug = g.macroscopic()
    assert np.isfinite(rg).all()
    pop_bytes = 19 * n ** 3 * 4
    assert g.device_bytes <= 1.05 * pop_bytes, (g.device_bytes, pop_bytes)
    g.close()


def test_graph_cache_keeps_both_parities(Lbm, oracle):
    """lbm_step(17) called repeatedly flips the parity (pop[0] / AA storage) between calls: the graph of
    each parity is captured once and replayed, not re-captured every call"""
    for scheme in ("2POP_SOA", "AA_SOA"):
        nx, ny, nz = 8, 9, 10
        fl, uw = box_flags(nx, ny, nz, "cavity")
        rho, u = inputs.seeded_init(nx, ny, nz, 0)
        g = Lbm(nx, ny, nz, scheme=scheme, omega=1.7)
        o = oracle.Oracle(nx, ny, nz, Q=19, model="BGK_W2", omega=1.7)
        g.set_flags(fl, uw); o.set_flags(fl, uw)
        g.init_equilibrium(rho, u); o.init_equilibrium(rho, u)
        g.step(1); o.step(1)
        for _ in range(6):
            g.step(17); o.step(17)
        assert g.graph_replays == 6
        assert pop_error(g, o, fl, 19, oracle, False) <= TOL64
        g.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("Q,model", [(19, "BGK_W2"), (19, "TRT"), (27, "K"), (27, "BGK_W2")])
@pytest.mark.parametrize("scheme", ["2POP_SOA", "AA_SOA", "SWAP_SOA"])
def test_tma_staged_kernels(Lbm, oracle, Q, model, scheme, dtype):
    """the step kernels whose loads are staged through shared memory by TMA bulk copies (tma_step.cuh):
    against the oracle on a box with walls, a moving block and the periodic seam, at a size where a
    block walks several tiles (the stage ring wraps) and the first / last tiles are not staged; and
    bit for bit the one-cell-per-thread kernels (same arithmetic per cell)."""
    shape = (64, 88, 96)   # 540 672 cells: 4.7 (fp32) / 9.5 (fp64) tiles per block of a 444-block grid
    steps = 7
    g, o, fl = run_pair(Lbm, oracle, shape, Q, model, scheme, dtype, steps, kind="obstacle", omega=1.6, variant="tma")
    err = pop_error(g, o, fl, Q, oracle, dtype == "f32")
    assert err <= (TOL64 if dtype == "f64" else TOL32), err
    ref = Lbm(*shape, lattice=Q, collision=model, scheme=scheme, omega=1.6, dtype=dtype)
    fl2, uw = box_flags(*shape, "obstacle")
    ref.set_flags(fl2, uw)
    ref.set_variant("no_tma")
    rho, u = inputs.seeded_init(*shape, 0)
    ref.init_equilibrium(rho, u)
    ref.step(steps)
    assert np.array_equal(g.get_populations(), ref.get_populations())
    g.close(); ref.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("Q,model", [(19, "BGK_W2"), (19, "TRT"), (27, "BGK_W2"), (27, "K")])
def test_aos_marching_tile_kernel(Lbm, oracle, Q, model, dtype):
    """the marching-tile kernel of the two-population AoS scheme (aos_march.cuh, variant aos_march; needs
    the outermost x-layers solid): a cavity with an obstacle inside, ragged in y and z (partial tiles),
    two x-segments; against the oracle, and bit for bit the default AoS kernels (cooperative gather) and
    the plain ones (variant aos_plain)"""
    nx, ny, nz, steps = 36, 23, 70, 7
    fl = inputs.cavity_flags(nx, ny, nz)
    fl[10:14, 5:9, 30:40] = inputs.WALL
    fl[20:22, 12:20, 3:6] = inputs.MOVING
    uw = (0.02, -0.01, 0.015)
    rho, u = inputs.seeded_init(nx, ny, nz, 3)
    npdt = np.float32 if dtype == "f32" else np.float64
    rho_in, u_in = rho.astype(npdt), u.astype(npdt)
    o = oracle.Oracle(nx, ny, nz, Q=Q, model=model, omega=1.6)
    o.set_flags(fl, uw)
    o.init_equilibrium(rho_in.astype(np.float64), u_in.astype(np.float64))
    o.step(steps)
    got = {}
    for variant in ("aos_march", "default", "aos_plain"):
        g = Lbm(nx, ny, nz, lattice=Q, collision=model, scheme="2POP_AOS", omega=1.6, dtype=dtype)
        g.set_flags(fl, uw)
        g.set_variant(variant)
        g.init_equilibrium(rho_in, u_in)
        g.step(steps)
        if variant == "aos_march":
            err = pop_error(g, o, fl, Q, oracle, dtype == "f32")
            assert err <= (TOL64 if dtype == "f64" else TOL32), err
            assert abs(g.kinetic_energy() - o.kinetic_energy()) <= (1e-12 if dtype == "f64" else 1e-5) * max(1.0, o.kinetic_energy())
        got[variant] = g.get_populations()
        g.close()
    assert np.array_equal(got["aos_march"], got["aos_plain"])
    assert np.array_equal(got["default"], got["aos_plain"])
