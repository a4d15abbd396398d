"""Thin ctypes binding of liblbm_b200.so (include/lbm.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory (its
caching allocator, through the lbm_set_hooks callbacks) and the stream (torch's current stream at
the time of `Lbm(...)`); nothing else.  There is no CPU fallback: a missing library or a missing
GPU raises LbmError.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblbm_b200.so")

LATTICES = {"D3Q19": 19, "D3Q27": 27, 19: 19, 27: 27}
MODELS = {"BGK_W2": 0, "BGK_NW4": 1, "TRT": 2, "RM": 3, "HM": 4, "CM": 5, "CHM": 6, "K": 7, "RR": 8, "REG": 9}
SCHEMES = {"2POP_SOA": 0, "2POP_AOS": 1, "SWAP_SOA": 2, "SWAP_AOS": 3, "AA_SOA": 4, "AA_AOS": 5}
DTYPES = {"f32": 0, "f64": 1}
NP_DTYPES = {"f32": np.float32, "f64": np.float64}
VARIANTS = {"default": 0, "generic_push": 1, "generic_pull": 2, "aos_plain": 3, "tma": 4, "no_tma": 5, "plain": 6, "aos_march": 7}
FLUID, WALL, MOVING, GHOST = 0, 1, 2, 3

# every symbol include/lbm.h declares (checked by tests/test_abi.py)
SYMBOLS = [
    "lbm_set_hooks", "lbm_create", "lbm_destroy", "lbm_set_flags", "lbm_set_relaxation", "lbm_set_trt_magic",
    "lbm_init_equilibrium", "lbm_init_equilibrium_device", "lbm_step", "lbm_macroscopic", "lbm_macroscopic_device", "lbm_kinetic_energy", "lbm_kinetic_energy_device", "lbm_kinetic_energy_device_static", "lbm_get_populations", "lbm_get_populations_at",
    "lbm_set_populations", "lbm_steps_done", "lbm_num_fluid", "lbm_device_bytes", "lbm_kernel_launches",
    "lbm_sync", "lbm_set_variant", "lbm_set_block", "lbm_set_graph", "lbm_graph_replays", "lbm_halo_count", "lbm_halo_pack", "lbm_halo_unpack", "lbm_step_begin", "lbm_step_end", "lbm_step_finish",
    "lbm_slab_link", "lbm_slab_export", "lbm_slab_import", "lbm_slab_post", "lbm_slab_complete", "lbm_slab_step", "lbm_slab_status",
    "lbm_last_error", "lbm_version",
]
GRAPH_MODES = {"auto": 0, "off": 1, "on": 2}
STATIC_SCRATCH_DOUBLES = 262144                      # include/lbm.h
STATIC_MAX_CELLS = (STATIC_SCRATCH_DOUBLES - 512) * 256


class LbmError(RuntimeError):
    pass


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p)

_lib = None
_hooks = None      # keeps the ctypes callbacks alive
_live = {}         # device pointer -> torch tensor backing it


def load_library(path=LIB_PATH):
    """dlopen the C-ABI library and declare its signatures.  Needs no GPU."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise LbmError("%s is missing: run `python -m paper_2010_11751_b200.build` (there is no CPU fallback)" % path)
    L = C.CDLL(path)
    vp, dp, i, d = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
    L.lbm_set_hooks.argtypes = [_ALLOC_FN, _FREE_FN, vp]
    L.lbm_create.restype = vp
    L.lbm_create.argtypes = [i, i, i, i, i, i, d, i]
    L.lbm_destroy.argtypes = [vp]
    L.lbm_set_flags.argtypes = [vp, vp, dp]
    L.lbm_set_relaxation.argtypes = [vp, d, d, d]
    L.lbm_set_trt_magic.argtypes = [vp, d]
    L.lbm_init_equilibrium.argtypes = [vp, vp, vp]
    L.lbm_init_equilibrium_device.argtypes = [vp, vp, vp]
    L.lbm_macroscopic_device.argtypes = [vp, vp, vp]
    L.lbm_step.argtypes = [vp, i]
    L.lbm_macroscopic.argtypes = [vp, vp, vp]
    L.lbm_kinetic_energy.argtypes = [vp, dp]
    L.lbm_kinetic_energy_device.argtypes = [vp, vp]
    L.lbm_kinetic_energy_device_static.argtypes = [vp, vp]
    L.lbm_get_populations.argtypes = [vp, vp]
    L.lbm_get_populations_at.argtypes = [vp, vp, i, vp]
    L.lbm_set_populations.argtypes = [vp, vp]
    L.lbm_set_graph.argtypes = [vp, i]
    L.lbm_step_begin.argtypes = [vp]
    L.lbm_step_end.argtypes = [vp]
    L.lbm_step_finish.argtypes = [vp]
    L.lbm_slab_link.argtypes = [vp, i, vp]
    L.lbm_slab_export.argtypes = [vp, vp]
    L.lbm_slab_import.argtypes = [vp, i, vp]
    L.lbm_slab_post.argtypes = [vp]
    L.lbm_slab_complete.argtypes = [vp]
    L.lbm_slab_step.argtypes = [vp, i]
    L.lbm_slab_status.argtypes = [vp]
    L.lbm_halo_count.restype = C.c_longlong
    L.lbm_halo_count.argtypes = [vp]
    L.lbm_halo_pack.argtypes = [vp, i, vp]
    L.lbm_halo_unpack.argtypes = [vp, i, vp]
    for name in ("lbm_steps_done", "lbm_num_fluid", "lbm_device_bytes", "lbm_kernel_launches", "lbm_graph_replays"):
        getattr(L, name).restype = C.c_longlong
        getattr(L, name).argtypes = [vp]
    L.lbm_sync.argtypes = [vp]
    L.lbm_set_variant.argtypes = [vp, i]
    L.lbm_set_block.argtypes = [vp, i]
    L.lbm_last_error.restype = C.c_char_p
    L.lbm_version.restype = C.c_char_p
    _lib = L
    return L


def _install_torch_hooks(L):
    """Point the library's allocator at torch's caching allocator and its stream at torch's current one."""
    global _hooks
    import torch
    if not torch.cuda.is_available():
        raise LbmError("no CUDA device: the lattice Boltzmann path runs on the GPU only (no CPU fallback)")

    if _hooks is None:  # the callbacks must outlive every context: create them once

        def _alloc(nbytes):
            try:
                t = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device="cuda")
            except Exception:  # out of memory: the C side reports LBM_E_ALLOC
                return None
            _live[t.data_ptr()] = t
            return t.data_ptr()

        def _free(ptr):
            _live.pop(ptr, None)

        _hooks = (_ALLOC_FN(_alloc), _FREE_FN(_free))
    stream = torch.cuda.current_stream().cuda_stream
    rc = L.lbm_set_hooks(_hooks[0], _hooks[1], C.c_void_p(stream))
    if rc != 0:
        raise LbmError(L.lbm_last_error().decode())


def _host_ptr(a):
    return C.c_void_p(a.ctypes.data)


class Lbm:
    """One lattice Boltzmann context (see include/lbm.h for the meaning of every call)."""

    def __init__(self, nx, ny, nz, lattice="D3Q19", collision="BGK_W2", scheme="2POP_SOA", omega=1.0, dtype="f64"):
        self._h = None
        L = load_library()
        _install_torch_hooks(L)
        self._L = L
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.N = self.nx * self.ny * self.nz
        self.Q = LATTICES[lattice]
        self.dtype = dtype
        self.np_dtype = NP_DTYPES[dtype]
        self.collision, self.scheme = collision, scheme
        h = L.lbm_create(self.nx, self.ny, self.nz, self.Q, MODELS[collision], SCHEMES[scheme], float(omega), DTYPES[dtype])
        if not h:
            raise LbmError(L.lbm_last_error().decode())
        self._h = C.c_void_p(h)

    def _ck(self, rc):
        if rc != 0:
            raise LbmError("%s (code %d)" % (self._L.lbm_last_error().decode(), rc))

    def close(self):
        if self._h is not None:
            self._L.lbm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _arr(self, a, n):
        a = np.ascontiguousarray(a, dtype=self.np_dtype).reshape(-1)
        if a.size != n:
            raise ValueError("expected %d elements, got %d" % (n, a.size))
        return a

    def set_flags(self, flags, u_wall=(0.0, 0.0, 0.0)):
        fl = np.ascontiguousarray(flags, dtype=np.uint8).reshape(-1)
        if fl.size != self.N:
            raise ValueError("flags must have nx*ny*nz entries")
        uw = (C.c_double * 3)(*[float(v) for v in u_wall])
        self._ck(self._L.lbm_set_flags(self._h, _host_ptr(fl), uw))

    def set_relaxation(self, omega_bulk, omega3, omega_hi):
        self._ck(self._L.lbm_set_relaxation(self._h, float(omega_bulk), float(omega3), float(omega_hi)))

    def set_trt_magic(self, lam):
        self._ck(self._L.lbm_set_trt_magic(self._h, float(lam)))

    def set_variant(self, variant):
        self._ck(self._L.lbm_set_variant(self._h, VARIANTS[variant] if isinstance(variant, str) else int(variant)))

    def set_block(self, threads):
        self._ck(self._L.lbm_set_block(self._h, int(threads)))

    def init_equilibrium(self, rho, u):
        r, uu = self._arr(rho, self.N), self._arr(u, 3 * self.N)
        self._ck(self._L.lbm_init_equilibrium(self._h, _host_ptr(r), _host_ptr(uu)))

    def step(self, n=1):
        self._ck(self._L.lbm_step(self._h, int(n)))

    def sync(self):
        self._ck(self._L.lbm_sync(self._h))

    def macroscopic(self, out_rho=None, out_u=None):
        rho = np.empty(self.N, dtype=self.np_dtype) if out_rho is None else out_rho
        u = np.empty((3, self.N), dtype=self.np_dtype) if out_u is None else out_u
        self._ck(self._L.lbm_macroscopic(self._h, _host_ptr(rho), _host_ptr(u)))
        return rho, u

    def init_equilibrium_device(self, rho_ptr, u_ptr):
        """rho_ptr, u_ptr: integer device addresses of [N] and [3][N] arrays of the context dtype."""
        self._ck(self._L.lbm_init_equilibrium_device(self._h, C.c_void_p(int(rho_ptr)), C.c_void_p(int(u_ptr))))

    def macroscopic_device(self, rho_ptr, u_ptr):
        self._ck(self._L.lbm_macroscopic_device(self._h, C.c_void_p(int(rho_ptr)), C.c_void_p(int(u_ptr))))

    def kinetic_energy(self):
        e = C.c_double(0.0)
        self._ck(self._L.lbm_kinetic_energy(self._h, C.byref(e)))
        return e.value

    def kinetic_energy_device(self, e_ptr):
        """e_ptr: integer device address of one double; asynchronous on the stream"""
        self._ck(self._L.lbm_kinetic_energy_device(self._h, C.c_void_p(int(e_ptr))))

    def kinetic_energy_device_static(self, e_ptr):
        """as kinetic_energy_device, with the partial sums in the library's fixed device array: allocates
        nothing; lattices of at most STATIC_MAX_CELLS cells (include/lbm.h)"""
        self._ck(self._L.lbm_kinetic_energy_device_static(self._h, C.c_void_p(int(e_ptr))))

    def get_populations(self):
        f = np.empty((self.Q, self.N), dtype=self.np_dtype)
        self._ck(self._L.lbm_get_populations(self._h, _host_ptr(f)))
        return f

    def get_populations_at(self, cells):
        """f[Q, m] of the listed cell indices (int32)."""
        cc = np.ascontiguousarray(cells, dtype=np.int32).reshape(-1)
        f = np.empty((self.Q, cc.size), dtype=self.np_dtype)
        self._ck(self._L.lbm_get_populations_at(self._h, _host_ptr(cc), int(cc.size), _host_ptr(f)))
        return f

    def set_populations(self, f):
        ff = self._arr(f, self.Q * self.N)
        self._ck(self._L.lbm_set_populations(self._h, _host_ptr(ff)))

    @property
    def steps_done(self):
        return self._L.lbm_steps_done(self._h)

    @property
    def num_fluid(self):
        return self._L.lbm_num_fluid(self._h)

    @property
    def device_bytes(self):
        return self._L.lbm_device_bytes(self._h)

    @property
    def kernel_launches(self):
        return self._L.lbm_kernel_launches(self._h)

    def step_begin(self):
        """outermost owned x-layers of the next step (slab overlap; see include/lbm.h)"""
        self._ck(self._L.lbm_step_begin(self._h))

    def step_end(self):
        self._ck(self._L.lbm_step_end(self._h))

    def step_finish(self):
        self._ck(self._L.lbm_step_finish(self._h))

    def slab_link(self, face, peer):
        """the slab beyond `face` is the context `peer` of this process (None = nothing beyond)"""
        self._ck(self._L.lbm_slab_link(self._h, int(face), peer._h if peer is not None else None))

    def slab_export(self):
        """64-byte CUDA IPC handle of this context's halo receive block"""
        h = C.create_string_buffer(64)
        self._ck(self._L.lbm_slab_export(self._h, h))
        return h.raw

    def slab_import(self, face, handle):
        self._ck(self._L.lbm_slab_import(self._h, int(face), C.create_string_buffer(bytes(handle), 64)))

    def slab_post(self):
        self._ck(self._L.lbm_slab_post(self._h))

    def slab_complete(self):
        self._ck(self._L.lbm_slab_complete(self._h))

    def slab_step(self, n=1):
        self._ck(self._L.lbm_slab_step(self._h, int(n)))

    def slab_status(self):
        self._ck(self._L.lbm_slab_status(self._h))

    @property
    def halo_count(self):
        """elements of one halo buffer (lbm_halo_pack / lbm_halo_unpack)"""
        return self._L.lbm_halo_count(self._h)

    def halo_pack(self, face, buf_ptr):
        self._ck(self._L.lbm_halo_pack(self._h, int(face), C.c_void_p(buf_ptr)))

    def halo_unpack(self, face, buf_ptr):
        self._ck(self._L.lbm_halo_unpack(self._h, int(face), C.c_void_p(buf_ptr)))

    @property
    def graph_replays(self):
        return self._L.lbm_graph_replays(self._h)

    def set_graph(self, mode):
        """CUDA-graph replay of step(): "auto" (small lattices only), "off", "on"."""
        self._ck(self._L.lbm_set_graph(self._h, GRAPH_MODES[mode]))
