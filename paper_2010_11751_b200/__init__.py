"""B200-native lattice Boltzmann stream-and-collide hot path (arxiv 2010.11751).

`Lbm` (binding.py) is the thin ctypes front end of the C-ABI library declared in include/lbm.h;
every step of the path runs in the hand-written sm_100a kernels under csrc/.  `inputs` holds the
seeded synthetic workloads only.  There is no CPU fallback: creating an `Lbm` without the built
CUDA library or without a GPU raises.
"""

__all__ = ["Lbm", "load_library", "inputs"]


def __getattr__(name):
    if name in ("Lbm", "load_library", "LbmError"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
