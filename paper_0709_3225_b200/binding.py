"""Thin ctypes binding over libljmd_b200.so: same names as include/ljmd.h, argument
marshalling only.  Arrays may be torch tensors (CPU or CUDA), numpy arrays, or raw integer
addresses.  Importing this module fails loudly if the CUDA library is missing: there is no
CPU fallback (the oracle under oracle/ is test infrastructure and is never imported here).
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libljmd_b200.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libljmd_b200.so is not built; run `python -m paper_0709_3225_b200.build` "
        "(needs nvcc).  There is no CPU fallback.")

_lib = ctypes.CDLL(LIB_PATH)
_alloc_keepalive = []

MD_OK, MD_EINVAL, MD_EDOMAIN, MD_ESTATE, MD_ENOMEM, MD_ECUDA, MD_EUNSUPPORTED = 0, -1, -2, -3, -4, -5, -6
MD_ALLPAIRS, MD_CELL, MD_VERLET = 0, 1, 2
MD_TRUNCATED, MD_ENERGY_SHIFTED, MD_FORCE_SHIFTED = 0, 1, 2
MD_POT_LJ, MD_POT_YUKAWA = 0, 1
R48_U32_HI32, R48_U32_HI31, R48_F64, R48_U64_STATE = 0, 1, 2, 3
MD_STATIC_MAX_ATOMS = 16384        # include/ljmd.h; tests/test_abi.py keeps the two equal
R48_DTYPES = {0: np.uint32, 1: np.uint32, 2: np.float64, 3: np.uint64}

_vp, _i64, _i32, _d = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
_pd = ctypes.POINTER(ctypes.c_double)
ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p)
FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

_SIGS = {
    "md_create": ([ctypes.POINTER(_vp), _i64, _d, _d, _d, _d, _d, _i32], _i32),
    "md_destroy": ([_vp], _i32),
    "md_set_state": ([_vp, _vp, _vp], _i32),
    "md_get_state": ([_vp, _vp, _vp], _i32),
    "md_compute_forces": ([_vp, _i32], _i32),
    "md_step": ([_vp, _i64, _i32], _i32),
    "md_get_forces": ([_vp, _vp], _i32),
    "md_get_energies": ([_vp, _pd, _pd, _pd], _i32),
    "rand48_fill": ([_vp, _i64, _i64, _i32, _vp], _i32),
    "rand48_fill_on": ([_vp, _i64, _i64, _i32, _vp, _vp], _i32),
    "md_strerror": ([_i32], ctypes.c_char_p),
    "md_init_velocities": ([_vp, ctypes.c_double, ctypes.c_uint64], _i32),
    "md_set_stream": ([_vp, _vp], _i32),
    "md_set_potential": ([_vp, _i32, _d, _d], _i32),
    "rand48_set_stream": ([_vp], _i32),
    "md_set_allocator": ([ALLOC_FN, FREE_FN], _i32),
    "md_set_option": ([_vp, ctypes.c_char_p, _d], _i32),
    "md_get_stat": ([_vp, ctypes.c_char_p, _pd], _i32),
    "md_last_cuda_error": ([], ctypes.c_char_p),
    "rand48_kernel_launches": ([], _i64),
    "md_probe_fp32_peak": ([_pd, _pd, _vp], _i32),
    "md_forces_allpairs_static": ([_vp, _i64, _d, _d, _d, _d, _i32, _vp, _vp, _vp], _i32),
}
for _name, (_args, _res) in _SIGS.items():
    _fn = getattr(_lib, _name)          # AttributeError here = header/library mismatch
    _fn.argtypes, _fn.restype = _args, _res


class MDError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _lib.md_strerror(code).decode()
        if code == MD_ECUDA:
            msg += " -- " + _lib.md_last_cuda_error().decode()
        super().__init__("%s: %s" % (where, msg))


def _check(code, where):
    if code != MD_OK:
        raise MDError(code, where)


def _addr(a):
    """Address of a torch tensor / numpy array / int; None -> NULL.  The array must be
    contiguous; the caller keeps it alive for the duration of the call."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError("expected torch tensor, numpy array or address")


def md_strerror(code):
    return _lib.md_strerror(code).decode()


def md_last_cuda_error():
    return _lib.md_last_cuda_error().decode()


def _torch_cuda():
    """torch, if it is importable and sees a device; else None (the raw C ABI needs neither)."""
    try:
        import torch
    except ImportError:
        return None
    return torch if torch.cuda.is_available() else None


def current_stream():
    """Handle of PyTorch's current CUDA stream (0 = legacy default stream when torch is absent)."""
    t = _torch_cuda()
    return int(t.cuda.current_stream().cuda_stream) if t is not None else 0


def md_create(N, L, rc, eps, sigma, dt, shifted, torch_plumbing=True):
    """md_create; with torch_plumbing (default) the handle allocates through PyTorch's caching allocator
    and runs on PyTorch's current stream, as north_star prescribes ("PyTorch is used only for device memory
    and streams"); False leaves the library's own defaults (cudaMalloc, legacy default stream)."""
    t = _torch_cuda() if torch_plumbing else None
    if t is not None and not _alloc_keepalive:
        use_torch_allocator()
    h = _vp()
    _check(_lib.md_create(ctypes.byref(h), N, L, rc, eps, sigma, dt, shifted), "md_create")
    if t is not None:
        md_set_stream(h, current_stream())
    return h


def md_destroy(h):
    _check(_lib.md_destroy(h), "md_destroy")


def md_set_state(h, pos, vel):
    _check(_lib.md_set_state(h, _addr(pos), _addr(vel)), "md_set_state")


def md_get_state(h, pos, vel):
    _check(_lib.md_get_state(h, _addr(pos), _addr(vel)), "md_get_state")


def md_compute_forces(h, algo):
    _check(_lib.md_compute_forces(h, algo), "md_compute_forces")


def md_step(h, nsteps, algo):
    _check(_lib.md_step(h, nsteps, algo), "md_step")


def md_get_forces(h, f):
    _check(_lib.md_get_forces(h, _addr(f)), "md_get_forces")


def md_get_energies(h):
    ke, pe, w = _d(), _d(), _d()
    _check(_lib.md_get_energies(h, ctypes.byref(ke), ctypes.byref(pe), ctypes.byref(w)), "md_get_energies")
    return ke.value, pe.value, w.value


def rand48_fill(seeds, nstreams, ndraws, kind, out, stream=None):
    """rand48_fill on `stream` (default: PyTorch's current stream)."""
    st = current_stream() if stream is None else int(stream)
    _check(_lib.rand48_fill_on(_addr(seeds), nstreams, ndraws, kind, _addr(out), st), "rand48_fill")


def md_init_velocities(h, T, seed48):
    _check(_lib.md_init_velocities(h, float(T), int(seed48)), "md_init_velocities")


def md_set_potential(h, kind, a=0.0, b=0.0):
    _check(_lib.md_set_potential(h, int(kind), float(a), float(b)), "md_set_potential")


def md_set_stream(h, stream):
    _check(_lib.md_set_stream(h, stream), "md_set_stream")


def rand48_set_stream(stream):
    _check(_lib.rand48_set_stream(stream), "rand48_set_stream")


def md_set_option(h, key, value):
    _check(_lib.md_set_option(h, key.encode(), float(value)), "md_set_option(%s)" % key)


def md_get_stat(h, key):
    v = _d()
    _check(_lib.md_get_stat(h, key.encode(), ctypes.byref(v)), "md_get_stat(%s)" % key)
    return v.value


def rand48_kernel_launches():
    return _lib.rand48_kernel_launches()


def md_forces_allpairs_static(pos, N, L, rc, eps, sigma, shifted, forces, pe_virial, stream=None):
    """md_forces_allpairs_static: all-pairs forces, PE and virial for callers that cannot allocate device memory
    (their own pool owns the whole card, or cudaMalloc's device-wide stall is not allowed where they run).
    pos [N,3] float32, forces [N,3] float32 and pe_virial [2] float64 must all be DEVICE arrays of the
    caller; the library's scratch is a fixed 1.3 MB array inside the .so, hence N <= MD_STATIC_MAX_ATOMS.
    Calls share that array: do not let two of them overlap on the GPU.  Runs on `stream` (default:
    PyTorch's current stream) and returns when the results are complete."""
    if N > MD_STATIC_MAX_ATOMS:
        raise MDError(MD_EUNSUPPORTED, "md_forces_allpairs_static: N = %d exceeds MD_STATIC_MAX_ATOMS = %d, "
                      "the size its built-in scratch array is made for (use md_create + md_compute_forces)"
                      % (N, MD_STATIC_MAX_ATOMS))
    st = current_stream() if stream is None else int(stream)
    _check(_lib.md_forces_allpairs_static(_addr(pos), N, L, rc, eps, sigma, shifted, _addr(forces), _addr(pe_virial),
                                          st), "md_forces_allpairs_static")


def md_probe_fp32_peak(stream=None):
    """(TFLOP/s, ms) of the library's FFMA-chain calibration kernel on the current device."""
    tf, ms = _d(), _d()
    st = current_stream() if stream is None else int(stream)
    _check(_lib.md_probe_fp32_peak(ctypes.byref(tf), ctypes.byref(ms), st), "md_probe_fp32_peak")
    return tf.value, ms.value


def use_torch_allocator():
    """Route the library's device allocations through PyTorch's caching allocator."""
    import torch

    def _alloc(nbytes, stream):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr, stream):
        torch.cuda.caching_allocator_delete(int(ptr))

    a, f = ALLOC_FN(_alloc), FREE_FN(_free)
    _alloc_keepalive[:] = [a, f]
    _check(_lib.md_set_allocator(a, f), "md_set_allocator")


class Sim:
    """Convenience owner of an md_sim handle (numpy in / numpy out)."""

    def __init__(self, N, L, rc=2.5, eps=1.0, sigma=1.0, dt=0.005, shifted=MD_ENERGY_SHIFTED):
        self.N = int(N)
        self.h = md_create(self.N, L, rc, eps, sigma, dt, shifted)

    def close(self):
        if self.h is not None:
            md_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_state(self, pos, vel):
        pos = np.ascontiguousarray(pos, dtype=np.float32)
        vel = np.ascontiguousarray(vel, dtype=np.float32)
        assert pos.shape == (self.N, 3) and vel.shape == (self.N, 3)
        md_set_state(self.h, pos, vel)

    def init_velocities(self, T, seed48):
        md_init_velocities(self.h, T, seed48)

    def get_state(self):
        pos = np.empty((self.N, 3), dtype=np.float32)
        vel = np.empty((self.N, 3), dtype=np.float32)
        md_get_state(self.h, pos, vel)
        return pos, vel

    def compute_forces(self, algo):
        md_compute_forces(self.h, algo)

    def step(self, nsteps, algo):
        md_step(self.h, nsteps, algo)

    def forces(self):
        f = np.empty((self.N, 3), dtype=np.float32)
        md_get_forces(self.h, f)
        return f

    def energies(self):
        return md_get_energies(self.h)

    def potential(self, kind, a=0.0, b=0.0):
        md_set_potential(self.h, kind, a, b)

    def option(self, key, value):
        md_set_option(self.h, key, value)

    def stat(self, key):
        return md_get_stat(self.h, key)


def rand48(seeds, ndraws, kind=R48_U32_HI32):
    """numpy convenience: returns (out [nstreams, ndraws], final seeds)."""
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64).copy()
    out = np.empty((seeds.shape[0], ndraws), dtype=R48_DTYPES[kind])
    rand48_fill(seeds, seeds.shape[0], ndraws, kind, out)
    return out, seeds
