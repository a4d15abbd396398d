"""Throughput sweep over lattices, collision models, schemes, precisions and sizes.

    python -m paper_2010_11751_b200.sweep --group schemes [--steps 200] [--md out.md] [--jsonl out.jsonl]

Groups mirror the paper's experiments on BASELINE.json's configs:
  schemes   six scheme x layout combinations, D3Q19 BGK-W2 fp64, 256^3      (Fig 4)
  fp32      the same six in fp32
  models19  ten collision models, D3Q19 fp64 AA-SoA, 128^3                  (Fig 6)
  models27  ten collision models, D3Q27 fp64 swap-SoA and AA-SoA, 192^3     (BASELINE.json config 4)
  config3   TRT / REG x fp64 / fp32 x 2-pop / AA at 256^3                   (BASELINE.json config 3)
  config5   512^3 BGK-W2: fp32 AA, fp64 2-pop and the scheme sweep          (BASELINE.json config 5)
  sizes     domain-size sweep, 2-pop and AA, BGK-W2 and RR                  (Fig 7)
  rr400     RR with omega_bulk = 1 at N = 400

Every case is the lid-driven cavity of inputs.py with the seeded noise init; timing is CUDA events
on the context's stream around `lbm_step(steps)`, median of `--repeat` runs after a warm-up.  The
roofline column divides the algorithmic bytes (2 Q s per fluid-cell update; swap 2(2Q-1) s;
PAPER.md Eq 16 generalised) by MEASURED_PEAKS.json's copy bandwidth.  Needs a GPU; no CPU fallback.
"""
import argparse
import json
import os
import sys

import numpy as np

from . import inputs
from .clocks import ClockSampler

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
ALL_MODELS = ["BGK_W2", "BGK_NW4", "TRT", "RM", "HM", "CM", "CHM", "K", "RR", "REG"]
ALL_SCHEMES = ["2POP_SOA", "2POP_AOS", "SWAP_SOA", "SWAP_AOS", "AA_SOA", "AA_AOS"]


MOMENT_SPACE = ("RM", "HM", "CM", "CHM", "K", "RR")


def case(n, Q=19, model="BGK_W2", scheme="2POP_SOA", dtype="f64", re=1000, variant=None, bulk="default", block=None, omega=None,
         general=False):
    """bulk: omega_bulk of the moment-space models.  The harness default is 1 (the paper's production
    setting): with omega_bulk = omega the seeded-noise cavity is linearly unstable for
    these models at the benchmark's omega ~ 1.95 (reading R25).  None = library default."""
    if bulk == "default":
        bulk = 1.0 if model in MOMENT_SPACE else None
    # general: rates of order >= 3 one ulp below 1, which dispatches the general collision kernel instead
    # of the variant with those orders equilibrated (same result to round-off)
    return dict(n=n, Q=Q, model=model, scheme=scheme, dtype=dtype, re=re, variant=variant, bulk=bulk, block=block, omega=omega,
                general=general)


def groups():
    g = {}
    g["schemes"] = [case(256, scheme=s) for s in ALL_SCHEMES] + [case(256, variant="generic_push")]
    g["fp32"] = [case(256, scheme=s, dtype="f32") for s in ALL_SCHEMES]
    g["models19"] = [case(128, model=m, scheme="AA_SOA") for m in ALL_MODELS] + \
                    [case(256, model=m, scheme="AA_SOA") for m in ALL_MODELS]
    g["models27"] = [case(192, Q=27, model=m, scheme=s) for s in ("SWAP_SOA", "AA_SOA") for m in ALL_MODELS]
    g["config3"] = [case(256, model=m, scheme=s, dtype=d) for m in ("TRT", "REG") for d in ("f64", "f32")
                    for s in ("2POP_SOA", "AA_SOA")]
    g["config5"] = [case(512, scheme="AA_SOA", dtype="f32"), case(512, scheme="2POP_SOA", dtype="f64")] + \
                   [case(512, scheme=s, dtype="f32") for s in ALL_SCHEMES if s != "AA_SOA"] + \
                   [case(512, scheme=s, dtype="f64") for s in ALL_SCHEMES if s != "2POP_SOA"]
    sizes = [16, 24, 32, 48, 64, 80, 90, 96, 100, 112, 128, 160, 192, 224, 256, 320, 384, 448, 512]
    # fixed omega (config 1's): Re = 1000 would push omega to 1.998 at N = 16, where the seeded noise blows BGK up
    g["sizes"] = [case(n, model=m, scheme=s, omega=inputs.omega_from_re(32, 100)) for m in ("BGK_W2", "RR")
                  for s in ("2POP_SOA", "AA_SOA") for n in sizes]
    # Fig 7 resolved where the L2 plateau and cliff are (PAPER.md:L484 steps N by 1): every 4th size from
    # 48 to 128 plus sizes that are not multiples of 4, 8 or 32
    fine = sorted(set(list(range(48, 129, 4)) + [50, 63, 65, 75, 81, 85, 90, 95, 99, 101, 110, 127, 129, 150, 200, 250, 255, 257, 300]))
    g["sizes_fine"] = [case(n, model="BGK_W2", scheme=s, omega=inputs.omega_from_re(32, 100)) for s in ("2POP_SOA", "AA_SOA")
                       for n in fine]
    g["rr400"] = [case(400, model="RR", scheme=s, re=10000, bulk=1.0) for s in ("2POP_SOA", "AA_SOA")]
    g["target"] = [case(256), case(256, scheme="AA_SOA")]
    g["blocks"] = [case(256, scheme=s, dtype=d, block=b) for d in ("f64", "f32") for s in ("2POP_SOA", "AA_SOA")
                   for b in (64, 128, 256)]
    g["misc27"] = [case(192, Q=27, model=m, scheme=s, dtype="f32") for m in ("BGK_W2", "TRT", "REG")
                   for s in ("2POP_SOA", "AA_SOA", "SWAP_SOA")] + [case(192, Q=27, scheme="2POP_SOA")]
    g["models_f32"] = [case(256, model=m, scheme="AA_SOA", dtype="f32") for m in ALL_MODELS] + \
                      [case(192, Q=27, model=m, scheme="AA_SOA", dtype="f32") for m in ALL_MODELS]
    # equilibrated high-order moments: the five models that have a variant, with it
    # and with the general kernel, against BGK on the same lattice
    g["f3"] = [case(n, Q=Q, model=m, scheme=s, dtype=d, general=gen)
               for (n, Q) in ((192, 27), (256, 19)) for d in ("f64", "f32") for s in ("AA_SOA", "SWAP_SOA")
               for m, gens in (("BGK_W2", (False,)), ("RM", (True, False)), ("HM", (True, False)), ("CM", (True, False)),
                               ("CHM", (True, False)), ("K", (True, False)))
               for gen in gens]
    g["small"] = [case(n, scheme=s, omega=inputs.omega_from_re(32, 100)) for s in ("2POP_SOA", "AA_SOA", "SWAP_SOA")
                  for n in (16, 32, 48, 64)]
    return g


def bytes_per_update(Q, dtype, scheme):
    s = 8 if dtype == "f64" else 4
    return (2 * Q + 2 * (Q - 1)) * s if scheme.startswith("SWAP") else 2 * Q * s


def peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"])
    return 6650.0


_init_cache = {}


def run_case(c, steps, repeat, warmup):
    import torch
    from .binding import Lbm
    n = c["n"]
    npdt = np.float64 if c["dtype"] == "f64" else np.float32
    key = (n, c["dtype"])
    if key not in _init_cache:
        _init_cache.clear()
        fl = inputs.cavity_flags(n, n, n)
        rho, u = inputs.seeded_init(n, n, n, 0)
        _init_cache[key] = (fl, torch.from_numpy(rho.astype(npdt)).cuda(), torch.from_numpy(u.astype(npdt)).cuda())
    fl, rho_d, u_d = _init_cache[key]
    omega = c.get("omega") or inputs.omega_from_re(n, c["re"])
    g = Lbm(n, n, n, lattice=c["Q"], collision=c["model"], scheme=c["scheme"], omega=omega, dtype=c["dtype"])
    try:
        g.set_flags(fl, (inputs.U_LID, 0.0, 0.0))
        if c["variant"]:
            g.set_variant(c["variant"])
        if c["block"]:
            g.set_block(c["block"])
        if c["bulk"] is not None and c["model"] in MOMENT_SPACE:
            hi = omega if c["model"] == "RR" else (float(np.nextafter(1.0, 0.0)) if c.get("general") else 1.0)
            g.set_relaxation(c["bulk"], hi, hi)
        g.init_equilibrium_device(rho_d.data_ptr(), u_d.data_ptr())
        g.step(warmup)
        torch.cuda.synchronize()
        sampler = ClockSampler(torch.cuda.current_device())
        sampler.start()
        times = []
        for _ in range(repeat):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            g.step(steps)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1) / steps)
        clocks = sampler.stop()
        energy = g.kinetic_energy()
        nfluid = g.num_fluid
        dev_bytes = g.device_bytes
    finally:
        g.close()
    ms = float(np.median(times))
    bpu = bytes_per_update(c["Q"], c["dtype"], c["scheme"])
    gbs = nfluid * bpu / (ms * 1e-3) / 1e9
    out = dict(c)
    out.update(ms_per_step=ms, mlups=nfluid / ms / 1e3, gbs=gbs, frac=gbs / peak_gbs(), bytes_per_update=bpu,
               fluid_cells=int(nfluid), steps=steps, finite=bool(np.isfinite(energy)), kinetic_energy=energy,
               clocks=clocks, device_bytes=int(dev_bytes))
    return out


def to_md(rows, title):
    lines = ["### %s" % title, "",
             "| N | lattice | model | scheme | dtype | variant | block | orders >= 3 | ms/step | MLUPS (fluid) | GB/s (algorithmic) | of measured copy | finite | SM MHz (median / max) | throttle reasons | clock samples |",
             "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for r in rows:
        ck = r.get("clocks") or {}
        lines.append("| %d | D3Q%d | %s | %s | %s | %s | %s | %s | %.4f | %.0f | %.0f | %.1f %% | %s | %s / %s | %s | %s |" % (
            r["n"], r["Q"], r["model"], r["scheme"], r["dtype"], r["variant"] or "default", r["block"] or "default",
            "-" if r["model"] not in ("RM", "HM", "CM", "CHM", "K") else "general kernel" if r.get("general") else "equilibrated", r["ms_per_step"], r["mlups"],
            r["gbs"], 100 * r["frac"], "yes" if r["finite"] else "NO", ck.get("sm_mhz"), ck.get("sm_max_mhz"),
            ",".join(ck.get("reasons") or []) or "none", ck.get("samples")))
    return "\n".join(lines) + "\n"


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--group", action="append", default=[], help="one of: " + ", ".join(sorted(groups())))
    ap.add_argument("--case", action="append", default=[],
                    help="one case N,Q,MODEL,SCHEME,DTYPE[,VARIANT], e.g. 256,19,BGK_W2,2POP_SOA,f32")
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--repeat", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--md", default=None)
    ap.add_argument("--jsonl", default=None)
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("sweep needs a CUDA device (no CPU fallback)")
    G = groups()
    if args.case:
        cs = []
        for spec in args.case:
            p = spec.split(",")
            cs.append(case(int(p[0]), Q=int(p[1]), model=p[2], scheme=p[3], dtype=p[4], variant=p[5] if len(p) > 5 else None))
        G["cases"] = cs
        args.group.append("cases")
    if not args.group:
        ap.error("give --group or --case")
    md = []
    for name in args.group:
        rows = []
        for c in G[name]:
            steps = args.steps if c["n"] >= 64 else args.steps * 10
            if c["n"] >= 448:
                steps = max(20, args.steps // 4)
            r = run_case(c, steps, args.repeat, args.warmup)
            rows.append(r)
            print(json.dumps(r), flush=True)
            if args.jsonl:
                with open(args.jsonl, "a") as fh:
                    fh.write(json.dumps(r) + "\n")
        md.append(to_md(rows, name))
    if args.md:
        with open(args.md, "w") as fh:
            fh.write("\n".join(md))
    return 0


if __name__ == "__main__":
    sys.exit(main())
