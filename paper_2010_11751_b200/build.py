"""Build liblbm_b200.so (the C-ABI library of include/lbm.h) in-tree with nvcc for sm_100a.

    python -m paper_2010_11751_b200.build [--force]

csrc/inst.cu is compiled once per (lattice, collision model) pair; the objects land in
paper_2010_11751_b200/build/ and the library beside this file.  nvcc cross-compiles without a GPU.
"""
import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblbm_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", INCLUDE]
LATTICES = (19, 27)
MODELS = range(15)   # collision.cuh: the ten models + five variants with orders >= 3 equilibrated


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))) + \
        [os.path.join(INCLUDE, "lbm.h")]


def _stamp():
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for p in _sources():
        with open(p, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def jobs():
    out = []
    for q in LATTICES:
        for m in MODELS:
            out.append((os.path.join(CSRC, "inst.cu"), os.path.join(OBJ, "inst_q%d_m%d.o" % (q, m)),
                        ["-DLBM_INST_Q=%d" % q, "-DLBM_INST_MODEL=%d" % m]))
    for name in sorted(os.listdir(CSRC)):
        if name.endswith(".cu") and name != "inst.cu":
            out.append((os.path.join(CSRC, name), os.path.join(OBJ, name[:-3] + ".o"), []))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    stamp_file = os.path.join(OBJ, "stamp.txt")
    stamp = _stamp()
    if not force and os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    todo = jobs()
    extra = ["-Xptxas", "-v"] if verbose else []
    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        futs = {ex.submit(_run, ["nvcc"] + NVCC_FLAGS + extra + defs + ["-c", src, "-o", obj]): obj
                for src, obj, defs in todo}
        for f in cf.as_completed(futs):
            log = f.result()
            if verbose:
                with open(futs[f] + ".log", "w") as fh:
                    fh.write(log)
    _run(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + [obj for _, obj, _ in todo])
    with open(stamp_file, "w") as fh:
        fh.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
