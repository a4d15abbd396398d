#!/usr/bin/env python
"""bench.py -- MLUPS and fraction of the HBM roofline of the lattice Boltzmann hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload target|1..5] [--impl reference]

One "step" is one collide-and-stream cycle over every cell of the
workload; the timed region runs exactly K of them and then, once, the macroscopic export (a9) and
the kinetic-energy reduce (a10), so that every row of the hot path is inside it.  Prints ONE JSON
line (rank 0).  `value` = fluid-cell updates of all ranks / time, populations resident in HBM;
`e2e` = the same metric through the C-ABI calls that take HOST buffers (lbm_init_equilibrium ->
lbm_step(K) -> lbm_macroscopic + lbm_kinetic_energy), copies inside the timed region.
`--impl reference` times the CPU oracle (oracle/) on the host cores instead, on a bounded sample.
The path does not shard ("replicas only"): with --gpus N every rank runs the same
workload on its own GPU and the values add up (weak scaling); there is no data-path collective.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2010_11751_b200 import inputs  # noqa: E402  (seeded inputs only; no arithmetic of the method)

MOMENT_SPACE = ("RM", "HM", "CM", "CHM", "K", "RR")
METRIC = "MLUPS"
UNIT = "million fluid-lattice-node updates per second"

# name -> (n, lattice, model, scheme, dtype, Re)   (BASELINE.json configs)
WORKLOADS = {
    "target": (256, 19, "BGK_W2", "AA_SOA", "f64", 1000),
    "target2pop": (256, 19, "BGK_W2", "2POP_SOA", "f64", 1000),
    "1": (32, 19, "BGK_W2", "2POP_SOA", "f64", 100),
    "2": (128, 19, "BGK_W2", "AA_SOA", "f64", 1000),
    "3": (256, 19, "TRT", "AA_SOA", "f64", 1000),
    "4": (192, 27, "K", "SWAP_SOA", "f64", 1000),
    "5": (512, 19, "BGK_W2", "AA_SOA", "f32", 1000),
}


def bytes_per_update(Q, dtype, scheme):
    """algorithmic bytes per fluid-cell update (Eq 16 of the paper generalised)"""
    s = 8 if dtype == "f64" else 4
    if scheme.startswith("SWAP"):
        return (2 * Q + 2 * (Q - 1)) * s
    return 2 * Q * s


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


from paper_2010_11751_b200.clocks import ClockSampler  # noqa: E402


def dist_setup(n_gpus):
    """(rank, world, dist or None).  Under torchrun the env carries RANK/WORLD_SIZE/LOCAL_RANK."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world == 1:
        return 0, 1, None
    import torch
    import torch.distributed as dist
    backend = "nccl" if torch.cuda.is_available() else "gloo"
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group(backend=backend)
    return rank, world, dist


def aggregate(dist, local_ms, local_units, device="cpu"):
    """max time over ranks and summed units (replicas: no data-path collective, only this)."""
    if dist is None:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def traffic_from_profiles(workload, kernel):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        parts = [p.strip() for p in line.split(",")]
        if len(parts) >= 3 and parts[0] == workload and parts[1] == kernel:
            try:
                return float(parts[2])
            except ValueError:
                return None
    return None


def set_oracle_threads(n):
    """OpenMP thread count of the oracle library (libgomp is already loaded by it); n <= 0 = all cores"""
    import ctypes
    from oracle import lbm_oracle
    lbm_oracle.lib()
    gomp = ctypes.CDLL("libgomp.so.1")
    gomp.omp_set_num_threads(int(n) if n > 0 else (os.cpu_count() or 1))


def oracle_sample_time(n, Q, model, re, steps, warm=1):
    """seconds per oracle step on an n^3 cavity of the workload's recipe (bounded sample)"""
    from oracle import lbm_oracle  # bench.py's cpu_baseline / --impl reference legs may use the oracle
    fl, uw, rho, u, omega = inputs.cavity_case(n, re)
    o = lbm_oracle.Oracle(n, n, n, Q=Q, model=model, omega=omega)
    o.set_flags(fl, uw)
    if model in MOMENT_SPACE:
        hi = omega if model == "RR" else 1.0
        o.set_relaxation(1.0, hi, hi)
    o.init_equilibrium(rho, u)
    o.step(warm)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    assert np.isfinite(o.kinetic_energy())
    return dt / steps, int((fl == 0).sum()), lbm_oracle.num_threads()


def oracle_sample_size(n, Q, model, re, budget_s, min_steps=3):
    """largest cavity edge <= min(n, 256) of which `min_steps` oracle steps fit into budget_s, from
    the rate of a 64^3 probe (from there on the oracle's rate per cell hardly depends on the size)"""
    probe = 64 if n >= 64 else 32
    t32, nf32, _ = oracle_sample_time(probe, Q, model, re, 2)
    per_cell = t32 / nf32
    for ns in (n, 256, 192, 128, 96, 64, 48, 32):
        if ns <= min(n, 256) and per_cell * (ns - 2) ** 3 * (min_steps + 1) <= budget_s:
            return ns
    return 32


def cpu_baseline(workload, budget_s=20.0):
    """the oracle as it stands on the host cores: all cores on a bounded sample of the workload (its own
    lattice when 3 steps of it fit the budget, else a smaller cavity of the same recipe), plus the
    single-thread rate at 32^3 and 128^3 that SURVEY 8(d) asks for"""
    n, Q, model, scheme, dtype, re = WORKLOADS[workload]
    set_oracle_threads(0)
    ns = oracle_sample_size(n, Q, model, re, budget_s)
    t1, nfluid, threads = oracle_sample_time(ns, Q, model, re, 1)
    steps = int(max(3, min(400, budget_s / max(t1, 1e-6))))
    t, nfluid, threads = oracle_sample_time(ns, Q, model, re, steps)
    out = {"value": nfluid / t / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": "%d^3 lid cavity of the same recipe (%s D3Q%d, fp64)%s, %d oracle steps, OpenMP over x"
                     % (ns, model, Q, "" if ns == n else " standing in for the %d^3 workload" % n, steps)}
    set_oracle_threads(1)
    single = {}
    for m in (32, 128):
        t32, nf32, _ = oracle_sample_time(32, Q, model, re, 1, warm=0)
        if m == 128 and t32 / nf32 * 126 ** 3 * 2 > 30.0:     # generic-matrix models: 128^3 on one thread takes minutes
            single["128^3"] = None
            continue
        ts, nf, _ = oracle_sample_time(m, Q, model, re, 10 if m == 32 else 1, warm=1 if m == 32 else 0)
        single["%d^3" % m] = nf / ts / 1e6
    set_oracle_threads(0)
    out["single_thread_mlups"] = single
    return out


def run_reference(args):
    """the oracle as it stands, timed on the host cores (rank 0 only)"""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    n, Q, model, scheme, dtype, re = WORKLOADS[args.workload]
    # every step = one oracle time step over the sample; the whole run must end within minutes
    ns = oracle_sample_size(n, Q, model, re, 150.0, min_steps=args.steps + args.warmup)
    t, nfluid, threads = oracle_sample_time(ns, Q, model, re, args.steps, warm=args.warmup)
    value = nfluid / t / 1e6
    sample = "%d^3 lid cavity of the same recipe%s, every step one oracle time step over it" % (
        ns, "" if ns == n else " (bounded sample of the %d^3 workload)" % n)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(name, world):
    n, Q, model, scheme, dtype, re = WORKLOADS[name]
    return {
        "workload": "%s: D3Q%d %s lid-driven cavity %d^3 %s, scheme %s, Re=%d, seeded noise init (seed 0)"
                    % (name, Q, model, n, dtype, scheme, re),
        "lattice": "D3Q%d" % Q, "collision": model, "scheme": scheme, "n": n, "re": re,
        "parallelism": "replicas x%d (no data-path collective)" % world,
        "l2": ("populations %.2f GB per array >> 126 MB L2, no flush needed" if n >= 128 else
               "populations %.3f GB per array fit the 126 MB L2: launch-bound lattice, MLUPS reported, no HBM roofline claim")
              % (n ** 3 * Q * (8 if dtype == "f64" else 4) / 1e9),
    }


def kernel_name(scheme, model, Q, dtype):
    fam = "pull-collide (LD_PULL->ST_LOCAL)" if scheme.startswith("2POP") else \
          "AA even/odd pair" if scheme.startswith("AA") else "swap pass 1 + pass 2"
    return "step_kernel<%s,D3Q%d,%s,%s> %s" % ("double" if dtype == "f64" else "float", Q, model,
                                                "SoA" if scheme.endswith("SOA") else "AoS", fam)


def run_gpu(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the lattice Boltzmann path has no CPU fallback")
    rank, world, dist = dist_setup(args.gpus)
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    from paper_2010_11751_b200 import Lbm

    n, Q, model, scheme, dtype, re = WORKLOADS[args.workload]
    K, W = args.steps, max(args.warmup, 3)
    npdt = np.float64 if dtype == "f64" else np.float32
    fl, uw, rho, u, omega = inputs.cavity_case(n, re)
    N = n ** 3
    # pinned host buffers for the end-to-end leg, device copies for the HBM-resident leg
    rho_h = torch.from_numpy(rho.astype(npdt)).pin_memory()
    u_h = torch.from_numpy(u.astype(npdt)).pin_memory()
    out_rho_h = torch.empty(N, dtype=rho_h.dtype).pin_memory()
    out_u_h = torch.empty((3, N), dtype=rho_h.dtype).pin_memory()
    rho_d, u_d = rho_h.to(dev), u_h.to(dev)
    out_rho_d, out_u_d = torch.empty_like(rho_d), torch.empty_like(u_d)

    g = Lbm(n, n, n, lattice=Q, collision=model, scheme=scheme, omega=omega, dtype=dtype)
    g.set_flags(fl, uw)
    if args.variant:
        g.set_variant(args.variant)
    if model in MOMENT_SPACE:  # DESIGN.md R25: omega_bulk = 1 keeps the seeded cavity stable
        hi = omega if model == "RR" else 1.0
        g.set_relaxation(1.0, hi, hi)
    nfluid = g.num_fluid

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- HBM-resident leg -------------------------------------------------------------------
    g.init_equilibrium_device(rho_d.data_ptr(), u_d.data_ptr())
    g.step(W)
    g.macroscopic_device(out_rho_d.data_ptr(), out_u_d.data_ptr())
    g.kinetic_energy()
    sampler = ClockSampler(local_rank)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
    e_d = torch.zeros(1, dtype=torch.float64, device=dev)
    barrier()
    sampler.start()
    l0 = g.kernel_launches
    ev[0].record()
    g.step(K)                                   # a1-a8, K times
    ev[1].record()
    g.macroscopic_device(out_rho_d.data_ptr(), out_u_d.data_ptr())   # a9
    ev[2].record()
    g.kinetic_energy_device(e_d.data_ptr())     # a10 on the device (three kernels)
    ev[4].record()
    energy = g.kinetic_energy()                 # a10 again through the host call (synchronises; 8 B to the host)
    ev[3].record()
    barrier()
    launches = g.kernel_launches - l0
    ms_total = ev[0].elapsed_time(ev[3])
    ms_steps = ev[0].elapsed_time(ev[1])
    ms_macro = ev[1].elapsed_time(ev[2])
    ms_energy = ev[2].elapsed_time(ev[4])
    assert np.isfinite(energy), "simulation blew up"
    assert abs(float(e_d.item()) - energy) == 0.0   # fixed reduction tree: bitwise repeatable

    # ---- end-to-end leg: host buffers in, host buffers out, copies inside the timed region ----
    rho_np, u_np = rho_h.numpy(), u_h.numpy()
    orho_np, ou_np = out_rho_h.numpy(), out_u_h.numpy()
    g.init_equilibrium(rho_np, u_np)
    g.step(3)
    g.macroscopic(orho_np, ou_np)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.init_equilibrium(rho_np, u_np)
    g.step(K)
    g.macroscopic(orho_np, ou_np)
    energy_e2e = g.kinetic_energy()
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    clocks = sampler.stop()
    assert np.isfinite(orho_np).all() and np.isfinite(energy_e2e)

    ms_total_g, units_g = aggregate(dist, ms_total, nfluid * K, dev)
    ms_e2e_g, _ = aggregate(dist, ms_e2e, nfluid * K, dev)
    ms_steps_g, _ = aggregate(dist, ms_steps, 0, dev)
    if rank != 0:
        return
    s = 8 if dtype == "f64" else 4
    bpu = bytes_per_update(Q, dtype, scheme)
    peak, peak_src = measured_peaks()
    step_ms = ms_steps / K
    achieved = nfluid * bpu / (step_ms * 1e-3) / 1e9
    kname = kernel_name(scheme, model, Q, dtype)
    traffic = traffic_from_profiles(args.workload, "step")
    line = {
        "metric": METRIC, "value": units_g / (ms_total_g * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": ms_total_g / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": dtype, "data": "synthetic", "config": workload_config(args.workload, world),
        "roofline": {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                     "bytes_per_update": bpu, "updates_per_launch": nfluid, "ms_per_launch": step_ms,
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "kernels": {
            "step": {"ms": step_ms, "mlups": nfluid / step_ms / 1e3, "gbs": achieved},
            "macroscopic": {"ms": ms_macro, "gbs": nfluid * (Q + 4) * s / (ms_macro * 1e-3) / 1e9},
            "kinetic_energy": {"ms": ms_energy, "gbs": nfluid * Q * s / (ms_energy * 1e-3) / 1e9,
                               "note": "lbm_kinetic_energy_device: reduce kernel + two summing stages"},
        },
        "e2e": {"value": units_g / (ms_e2e_g * 1e-3) / 1e6, "unit": UNIT,
                "h2d_bytes_per_step": 4 * N * s / K, "d2h_bytes_per_step": (4 * N * s + 8) / K,
                "ms": ms_e2e_g, "calls": "lbm_init_equilibrium(host) -> lbm_step(K) -> lbm_macroscopic(host) + lbm_kinetic_energy",
                "host_memory": "pinned"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "mlups_all_cells": N * K * world / (ms_total_g * 1e-3) / 1e6,
        "fluid_cells": int(nfluid), "kinetic_energy": energy,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.workload)
    print(json.dumps(line), flush=True)


def run_gpu_slab(args):
    """--decomp slab: ONE lattice of (N n) x n x n cells cut into N x-slabs, one per GPU, with a halo
    exchange after every step (paper_2010_11751_b200/slab.py).  Weak scaling: every rank
    owns n layers.  Two-population SoA workloads only."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the lattice Boltzmann path has no CPU fallback")
    rank, world, dist = dist_setup(args.gpus)
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    from paper_2010_11751_b200 import slab
    n, Q, model, scheme, dtype, re = WORKLOADS[args.workload]
    if not scheme.endswith("SOA"):
        raise SystemExit("--decomp slab needs an SoA workload")
    K, W = args.steps, max(args.warmup, 3)
    NX = world * n
    omega = inputs.omega_from_re(n, re)
    x0, x1 = slab.slab_range(NX, rank, world)
    fl, rho, u = slab.cavity_slab(NX, n, n, x0, x1, seed=0)
    g = slab.SlabLbm(NX, n, n, flags_local=fl, u_wall=(inputs.U_LID, 0.0, 0.0), dist=dist, rank=rank, world=world,
                     lattice=Q, collision=model, omega=omega, dtype=dtype, scheme=scheme, transport=args.transport)
    nfluid = g.num_fluid

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    g.init_equilibrium_local(rho, u)
    g.step(W)
    sampler = ClockSampler(local_rank)
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    barrier()
    sampler.start()
    l0 = g.lbm.kernel_launches
    e0.record()
    g.step(K)
    e1.record()
    energy = g.kinetic_energy()
    e2.record()
    barrier()
    launches = g.lbm.kernel_launches - l0
    ms_steps, ms_total = e0.elapsed_time(e1), e0.elapsed_time(e2)
    # end to end: host arrays in, K steps, host arrays out
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    g.init_equilibrium_local(rho, u)
    g.step(K)
    rho_out, u_out = g.macroscopic()
    g.kinetic_energy()
    t1.record()
    barrier()
    ms_e2e = t0.elapsed_time(t1)
    clocks = sampler.stop()
    assert np.isfinite(energy) and np.isfinite(rho_out).all()
    ms_total_g, units_g = aggregate(dist, ms_total, nfluid * K, dev)
    ms_e2e_g, _ = aggregate(dist, ms_e2e, 0, dev)
    if rank != 0:
        return
    s = 8 if dtype == "f64" else 4
    bpu = bytes_per_update(Q, dtype, scheme)
    peak, peak_src = measured_peaks()
    step_ms = ms_steps / K
    achieved = nfluid * bpu / (step_ms * 1e-3) / 1e9
    cfg = workload_config(args.workload, world)
    cfg["workload"] = "%s, as ONE %d x %d x %d cavity cut into %d x-slabs" % (cfg["workload"], NX, n, n, world)
    cfg["parallelism"] = "slab x%d along x, one-cell halo: %d of %d planes per face per step, transport %s" % (
        world, 5 if Q == 19 else 9, Q,
        "peer stores from the pack kernel into the neighbour's receive buffer (lbm_slab_step)" if g.transport == "peer"
        else "torch.distributed p2p")
    nloc = (x1 - x0 + 2) * n * n
    line = {
        "metric": METRIC, "value": units_g / (ms_total_g * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": ms_total_g / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": dtype, "data": "synthetic", "config": cfg,
        "roofline": {"bound": "hbm", "kernel": kernel_name(scheme, model, Q, dtype) + " + halo pack/unpack + exchange (rank 0)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic_from_profiles("target2pop", "step"), "peak_source": peak_src,
                     "bytes_per_update": bpu, "updates_per_launch": nfluid, "ms_per_launch": step_ms},
        "halo": {"bytes_sent_per_step_per_rank": g.engine.halo_bytes, "ms_per_step_incl_exchange": step_ms},
        "e2e": {"value": units_g / (ms_e2e_g * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": 4 * nloc * s / K,
                "d2h_bytes_per_step": (4 * nloc * s + 8) / K, "ms": ms_e2e_g,
                "calls": "SlabLbm.init_equilibrium_local(host) -> step(K) -> macroscopic(host) + kinetic_energy"},
        "gpu_launches": int(launches), "clocks": clocks, "fluid_cells": int(nfluid), "kinetic_energy": energy,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="target", choices=sorted(WORKLOADS) + ["case"])
    ap.add_argument("--case", default=None,
                    help="any other case N,Q,MODEL,SCHEME,DTYPE[,RE], e.g. 256,19,BGK_W2,2POP_AOS,f64 (overrides --workload)")
    ap.add_argument("--variant", default=None, help="step-kernel variant (binding.VARIANTS), default = library's choice")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--transport", default=None, choices=["peer", "p2p"],
                    help="--decomp slab: library driver over peer memory / torch.distributed send-recv (default: peer for one rank, p2p otherwise)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="replicas (default): N independent lattices; slab: one lattice cut along x with a halo exchange")
    args = ap.parse_args()
    if args.case:
        p = args.case.split(",")
        WORKLOADS["case"] = (int(p[0]), int(p[1]), p[2], p[3], p[4], int(p[5]) if len(p) > 5 else 1000)
        args.workload = "case"
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp == "slab":
        run_gpu_slab(args)
    else:
        run_gpu(args)
    try:
        import torch.distributed as dist
        if dist.is_available() and dist.is_initialized():
            dist.destroy_process_group()
    except Exception:
        pass


if __name__ == "__main__":
    main()
