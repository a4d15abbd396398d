"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no lattice tables, no equilibrium, no
collision, no streaming): it only builds flag fields and (rho, u) arrays, which are handed
unchanged to both the CUDA path and the oracle.  It imports neither of them.

Recipe (BASELINE.json configs):
  * cavity: N^3 box whose outermost layer is wall, the whole plane iz = nz-1
    flagged MOVING with u_wall = (0.02, 0, 0); nu = U (N-2) / Re, omega = 1/(3 nu + 1/2) (L352).
  * seeded noise: rho = 1 + 1e-3 U(-1,1), u_i = 0.01 U(-1,1), counter-based splitmix64 keyed by
    (seed, cell index, component), so the value of a cell never depends on traversal order.
  * shear wave: periodic box, rho = 1, u_x = amp sin(2 pi y / ny).
The paper's workload (lid-driven cavity, L391-397) is itself synthetic; no dataset stands behind it.
"""
import numpy as np

FLUID, WALL, MOVING = 0, 1, 2
U_LID = 0.02

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = x
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def uniform_pm1(seed, index, comp):
    """U(-1,1) for (seed, cell index array, component 0..3); pure function of its arguments."""
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        key = (np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15) + np.uint64(4) * idx + np.uint64(comp)) & _M64
        h = _splitmix64(key)
    return 2.0 * ((h >> np.uint64(11)).astype(np.float64) * 2.0 ** -53) - 1.0


def cavity_flags(nx, ny, nz):
    """uint8 [nx,ny,nz]: outer layer WALL, the whole plane iz = nz-1 MOVING (R9)."""
    fl = np.zeros((nx, ny, nz), dtype=np.uint8)
    fl[0, :, :] = WALL
    fl[-1, :, :] = WALL
    fl[:, 0, :] = WALL
    fl[:, -1, :] = WALL
    fl[:, :, 0] = WALL
    fl[:, :, -1] = MOVING
    return fl


def periodic_flags(nx, ny, nz):
    return np.zeros((nx, ny, nz), dtype=np.uint8)


def seeded_init(nx, ny, nz, seed=0, index_offset=None):
    """rho [N], u [3,N] float64 with the seeded noise of BASELINE.json (every cell gets a value;
    non-fluid cells are ignored by both sides).  index_offset lets a sub-box reuse the values of a
    larger box: pass the global cell indices of the sub-box cells."""
    n = nx * ny * nz
    idx = np.arange(n, dtype=np.uint64) if index_offset is None else np.asarray(index_offset, dtype=np.uint64).reshape(-1)
    rho = 1.0 + 1e-3 * uniform_pm1(seed, idx, 0)
    u = np.stack([0.01 * uniform_pm1(seed, idx, c) for c in (1, 2, 3)])
    return rho, u


def shear_wave(nx, ny, nz, amp=0.01):
    """rho = 1, u_x = amp sin(2 pi y / ny) (BASELINE.json config 2, pin P3)."""
    rho = np.ones(nx * ny * nz)
    y = np.arange(ny, dtype=np.float64)
    ux = np.broadcast_to((amp * np.sin(2.0 * np.pi * y / ny))[None, :, None], (nx, ny, nz)).reshape(-1)
    u = np.zeros((3, nx * ny * nz))
    u[0] = ux
    return rho, u


def omega_from_re(n, re, u_lid=U_LID):
    """nu = U (N-2)/Re (L391, L397); omega = 1/(3 nu + 1/2) (L352)."""
    nu = u_lid * (n - 2) / re
    return 1.0 / (3.0 * nu + 0.5)


# BASELINE.json configs, made concrete.  'schemes' / 'models' / 'dtypes' list what
# the config sweeps; bench.py and the parity tests pick from here.
CONFIGS = {
    1: dict(n=32, lattice=19, models=["BGK_W2"], dtypes=["f64"], schemes=["2POP_SOA"], re=100, steps=100),
    2: dict(n=128, lattice=19, models=["BGK_W2"], dtypes=["f64"], schemes=["AA_SOA"], re=1000, steps=1000),
    3: dict(n=256, lattice=19, models=["TRT", "REG"], dtypes=["f64", "f32"], schemes=["2POP_SOA", "AA_SOA"], re=1000, steps=500),
    4: dict(n=192, lattice=27, models=["BGK_W2", "BGK_NW4", "TRT", "RM", "HM", "CM", "CHM", "K", "RR", "REG"],
            dtypes=["f64"], schemes=["SWAP_SOA"], re=1000, steps=200),
    5: dict(n=512, lattice=19, models=["BGK_W2"], dtypes=["f32", "f64"],
            schemes=["2POP_SOA", "2POP_AOS", "SWAP_SOA", "SWAP_AOS", "AA_SOA", "AA_AOS"], re=1000, steps=200),
    # the north_star target: D3Q19 BGK fp64 at 256^3
    "target": dict(n=256, lattice=19, models=["BGK_W2"], dtypes=["f64"], schemes=["2POP_SOA", "AA_SOA"], re=1000, steps=200),
}


def cavity_case(n, re, seed=0):
    """(flags[n,n,n], u_wall, rho[N], u[3,N], omega) of one cavity config."""
    fl = cavity_flags(n, n, n)
    rho, u = seeded_init(n, n, n, seed)
    return fl, (U_LID, 0.0, 0.0), rho, u, omega_from_re(n, re)
