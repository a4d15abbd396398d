"""Steady lid-driven cavity at Re = 1000 and its centre-line velocity profiles (Fig 2 left).

    python -m paper_2010_11751_b200.cavity --n 128 [--re 1000] [--ulb 0.06] [--out profile.json]

The paper validates its code with the velocity profiles along the two centre lines of the cubic cavity
and compares them with the spectral data of its ref. [62], which is not available here; what can be
shown is self-consistency under grid refinement: the profiles at N = 128 and N = 256
agree (tests/test_gpu_cavity_profile.py).  Set-up as in the paper: N^3 nodes with a wall node on every
extremity (dx = L / (N - 2)), u_LB = 0.06 (L397), BGK-W2, start from rest.  The lid is the
plane iz = nz - 1 moving along +x (reading R9), so the paper's u_y(x) on y = z = 0 (the component along
the lid motion, on the line normal to the lid) is u_x(z) on the line x = y = centre here, and its
u_x(y) is u_z(x) on the line y = z = centre.

This module only drives the library (flags, rates, stepping, exports); it holds no arithmetic of the
method.  GPU only.
"""
import argparse
import json

import numpy as np

from . import inputs


def centre_line(field, axis):
    """values of a [n, n, n] field on the line through the centre of the cavity along `axis`.  For
    even n the centre falls between two nodes: the mean of the four lines around it."""
    n = field.shape[0]
    h = n // 2
    idx = [slice(h - 1, h + 1) if n % 2 == 0 else slice(h, h + 1)] * 3
    idx[axis] = slice(1, n - 1)          # fluid nodes only
    block = field[tuple(idx)]
    other = tuple(a for a in range(3) if a != axis)
    return block.mean(axis=other)


def node_positions(n):
    """positions of the fluid nodes 1 .. n-2 in units of L, walls half-way between nodes at 0 and 1"""
    return (np.arange(1, n - 1) - 0.5) / (n - 2)


def steady_cavity_profiles(n, re=1000.0, u_lb=0.06, max_turnovers=100.0, tol=1e-9, check_every=1000, scheme="AA_SOA",
                           dtype="f64", log=None):
    """Run the N^3 cavity from rest until the kinetic energy changes by less than `tol` (relative) over
    `check_every` steps, or for max_turnovers * (N - 2) / u_LB steps.  Returns a dict with the two
    centre-line profiles (in units of the lid velocity), the step count and the energy history."""
    from .binding import Lbm
    nu = u_lb * (n - 2) / re
    omega = 1.0 / (3.0 * nu + 0.5)
    fl = inputs.cavity_flags(n, n, n)
    g = Lbm(n, n, n, lattice=19, collision="BGK_W2", scheme=scheme, omega=omega, dtype=dtype)
    try:
        g.set_flags(fl, (u_lb, 0.0, 0.0))
        npdt = np.float64 if dtype == "f64" else np.float32
        g.init_equilibrium(np.ones(n ** 3, dtype=npdt), np.zeros((3, n ** 3), dtype=npdt))
        max_steps = int(max_turnovers * (n - 2) / u_lb)
        history, steps, e_prev, change = [], 0, None, None
        while steps < max_steps:
            chunk = min(check_every, max_steps - steps)
            g.step(chunk)
            steps += chunk
            e = g.kinetic_energy()
            if not np.isfinite(e):
                raise RuntimeError("cavity run blew up at step %d" % steps)
            change = None if e_prev is None else abs(e - e_prev) / max(abs(e), 1e-300)
            history.append((steps, e))
            if log and (steps // check_every) % 10 == 0:
                log("n=%d step %d E=%.12e change/%d=%s" % (n, steps, e, check_every, change))
            if change is not None and change < tol:
                break
            e_prev = e
        rho, u = g.macroscopic()
    finally:
        g.close()
    u = u.reshape(3, n, n, n).astype(np.float64)
    return {
        "n": n, "re": re, "u_lb": u_lb, "omega": omega, "steps": steps, "turnovers": steps * u_lb / (n - 2),
        "energy_change_per_check": change, "check_every": check_every, "converged": bool(change is not None and change < tol),
        "pos": node_positions(n).tolist(),
        "ux_along_z": (centre_line(u[0], 2) / u_lb).tolist(),   # the paper's u_y(x): along the lid motion, on the lid-normal line
        "uz_along_x": (centre_line(u[2], 0) / u_lb).tolist(),   # the paper's u_x(y): lid-normal component, on the line along the motion
        "energy_history": history,
    }


def profile_difference(coarse, fine, key):
    """max |fine - coarse interpolated to the fine nodes| of one profile, in units of the lid velocity"""
    c = np.interp(np.asarray(fine["pos"]), np.concatenate(([0.0], coarse["pos"], [1.0])),
                  np.concatenate(([_wall_value(key, 0)], coarse[key], [_wall_value(key, 1)])))
    return float(np.abs(np.asarray(fine[key]) - c).max())


def _wall_value(key, end):
    # no-slip walls; the line normal to the lid ends on the lid, where u_x = U
    return 1.0 if (key == "ux_along_z" and end == 1) else 0.0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, action="append", default=[])
    ap.add_argument("--re", type=float, default=1000.0)
    ap.add_argument("--ulb", type=float, default=0.06)
    ap.add_argument("--max-turnovers", type=float, default=100.0)
    ap.add_argument("--tol", type=float, default=1e-9)
    ap.add_argument("--dtype", default="f64")
    ap.add_argument("--out", default=None)
    args = ap.parse_args(argv)
    res = [steady_cavity_profiles(n, args.re, args.ulb, args.max_turnovers, args.tol, dtype=args.dtype, log=print)
           for n in (args.n or [128])]
    for r in res:
        print("n=%d: %d steps (%.1f turnovers), converged=%s, last relative energy change per %d steps %.3e, min u_x(z) = %.4f, "
              "min / max u_z(x) = %.4f / %.4f" % (r["n"], r["steps"], r["turnovers"], r["converged"], r["check_every"],
                                                 r["energy_change_per_check"], min(r["ux_along_z"]), min(r["uz_along_x"]),
                                                 max(r["uz_along_x"])))
    for a, b in zip(res, res[1:]):
        for key in ("ux_along_z", "uz_along_x"):
            print("max |%s(N=%d) - %s(N=%d)| = %.4f U" % (key, b["n"], key, a["n"], profile_difference(a, b, key)))
    if args.out:
        with open(args.out, "w") as fh:
            json.dump(res, fh)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
