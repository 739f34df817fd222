"""ctypes wrapper around oracle/ljmd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_0709_3225_b200 and shares no
arithmetic with it.  See the header of ljmd_oracle.c for citations and pins.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ljmd_oracle.c")
_LIB = os.path.join(_HERE, "libljmd_oracle.so")


def build(force=False):
    """Compile ljmd_oracle.c with gcc (FP64, -O2, no fast-math, no FMA contraction)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        d, i64, i32 = ctypes.c_double, ctypes.c_int64, ctypes.c_int
        u64 = ctypes.c_uint64
        pd = ctypes.POINTER(ctypes.c_double)
        vp = ctypes.c_void_p
        L.lj_pair.argtypes = [i32, d, d, d, d, pd, pd]
        L.lj_pair.restype = i32
        L.forces_allpairs.argtypes = [i64, vp, d, d, d, d, i32, vp, pd, pd]
        L.forces_allpairs.restype = None
        L.forces_cell.argtypes = [i64, vp, d, d, d, d, i32, vp, pd, pd]
        L.forces_cell.restype = i32
        L.cell_grid.argtypes = [d, d, ctypes.POINTER(i32), pd]
        L.cell_grid.restype = i32
        L.yukawa_pair.argtypes = [ctypes.c_int, d, d, d, d, ctypes.POINTER(d), ctypes.POINTER(d)]
        L.yukawa_pair.restype = ctypes.c_int
        L.set_potential.argtypes = [ctypes.c_int, d, d]
        L.set_potential.restype = None
        L.near_cutoff_pairs.argtypes = [i64, vp, d, d, d, vp, i64]
        L.near_cutoff_pairs.restype = i64
        L.near_cutoff_pairs_cell.argtypes = [i64, vp, d, d, d, vp, i64]
        L.near_cutoff_pairs_cell.restype = i64
        L.kinetic_energy.argtypes = [i64, vp]
        L.kinetic_energy.restype = d
        L.verlet_step.argtypes = [i64, vp, vp, vp, d, d, d, d, d, i32, i32, pd, pd, pd]
        L.verlet_step.restype = i32
        L.verlet_run.argtypes = [i64, vp, vp, vp, d, d, d, d, d, i32, i32, i64, vp]
        L.verlet_run.restype = i32
        L.rand48_next.argtypes = [u64]
        L.rand48_next.restype = u64
        L.rand48_fill_seq.argtypes = [vp, i64, i64, i32, vp]
        L.rand48_fill_seq.restype = None
        L.rand48_skip_consts_linear.argtypes = [u64, ctypes.POINTER(u64), ctypes.POINTER(u64)]
        L.rand48_skip_consts_linear.restype = None
        L.rand48_skip_consts.argtypes = [u64, ctypes.POINTER(u64), ctypes.POINTER(u64)]
        L.rand48_skip_consts.restype = None
        L.rand48_skip.argtypes = [u64, u64]
        L.rand48_skip.restype = u64
        L.rand48_leapfrog.argtypes = [u64, i64, i64, vp]
        L.rand48_leapfrog.restype = None
        L.mb_velocities.argtypes = [i64, d, ctypes.POINTER(u64), vp]
        L.mb_velocities.restype = None
        L.andersen_collide.argtypes = [i64, vp, d, ctypes.c_uint32, u64, i64]
        L.andersen_collide.restype = i64
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def set_threads(n):
    """OpenMP thread count used by forces_cell (the only parallel loop)."""
    os.environ["OMP_NUM_THREADS"] = str(int(n))
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
    except OSError:
        pass


def lj_pair(mode, r2, eps=1.0, sigma=1.0, rc=2.5):
    """(inside, U, f/r) for one pair at squared distance r2.  PAPER.md:56-62."""
    u, fr = ctypes.c_double(), ctypes.c_double()
    inside = lib().lj_pair(mode, r2, eps, sigma, rc, ctypes.byref(u), ctypes.byref(fr))
    return bool(inside), u.value, fr.value


def yukawa_pair(mode, r2, A=1.0, kappa=1.0, rc=2.5):
    """(inside, U, f/r) of the screened Coulomb pair U = A exp(-kappa r)/r.  PAPER.md:184 (other pair
    potentials, "including the coulombic interaction"); SURVEY 8(f) item 4."""
    u, fr = ctypes.c_double(), ctypes.c_double()
    inside = lib().yukawa_pair(mode, r2, A, kappa, rc, ctypes.byref(u), ctypes.byref(fr))
    return bool(inside), u.value, fr.value


class potential:
    """with oracle.potential(1, A, kappa): ... -- the force loops (and verlet_*) evaluate the Yukawa pair inside
    the block, Lennard-Jones again after it."""

    def __init__(self, kind, A=1.0, kappa=1.0):
        self.args = (int(kind), float(A), float(kappa))

    def __enter__(self):
        lib().set_potential(*self.args)
        return self

    def __exit__(self, *a):
        lib().set_potential(0, 1.0, 1.0)


def forces(pos, L, rc=2.5, eps=1.0, sigma=1.0, mode=1, algo=0):
    """F [N,3], PE, W for positions pos [N,3] (FP64).  algo 0 all-pairs, 1 cell list."""
    pos = _f64(pos)
    N = pos.shape[0]
    F = np.zeros((N, 3), dtype=np.float64)
    pe, w = ctypes.c_double(), ctypes.c_double()
    if algo == 0:
        lib().forces_allpairs(N, _ptr(pos), L, rc, eps, sigma, mode, _ptr(F),
                              ctypes.byref(pe), ctypes.byref(w))
    else:
        rcode = lib().forces_cell(N, _ptr(pos), L, rc, eps, sigma, mode, _ptr(F),
                                  ctypes.byref(pe), ctypes.byref(w))
        if rcode != 0:
            raise ValueError("cell list needs at least 3 cells per dimension (PAPER.md:130)")
    return F, pe.value, w.value


def cell_grid(L, rc):
    """(ncell, side) with ncell = int[L/rc], side = L/ncell.  PAPER.md:134."""
    n, s = ctypes.c_int(), ctypes.c_double()
    ok = lib().cell_grid(L, rc, ctypes.byref(n), ctypes.byref(s))
    return n.value, s.value, ok == 0


def near_cutoff_pairs(pos, L, rc=2.5, tol=4e-7, cap=1 << 16):
    pos = _f64(pos)
    out = np.zeros((cap, 2), dtype=np.int64)
    n = lib().near_cutoff_pairs(pos.shape[0], _ptr(pos), L, rc, tol, _ptr(out), cap)
    return out[:min(n, cap)], n


def near_cutoff_pairs_cell(pos, L, rc=2.5, tol=4e-7, cap=1 << 16):
    """The same ordered pairs through the linked cells (large N).  PAPER.md:98, :108; R16."""
    pos = _f64(pos)
    out = np.zeros((cap, 2), dtype=np.int64)
    n = lib().near_cutoff_pairs_cell(pos.shape[0], _ptr(pos), L, rc, tol, _ptr(out), cap)
    if n < 0:
        raise ValueError("fewer than 3 cells per dimension")
    return out[:min(n, cap)], n


def kinetic_energy(vel):
    vel = _f64(vel)
    return lib().kinetic_energy(vel.shape[0], _ptr(vel))


def verlet_run(pos, vel, L, nsteps, rc=2.5, eps=1.0, sigma=1.0, dt=0.005, mode=1, algo=0):
    """Run nsteps velocity-Verlet steps.  Returns pos, vel, F (final) and the
    [nsteps+1, 3] trace of (KE, PE, W) at t = 0..nsteps.  PAPER.md:64."""
    pos = _f64(pos).copy()
    vel = _f64(vel).copy()
    N = pos.shape[0]
    F = np.zeros((N, 3), dtype=np.float64)
    trace = np.zeros((nsteps + 1, 3), dtype=np.float64)
    rcode = lib().verlet_run(N, _ptr(pos), _ptr(vel), _ptr(F), L, rc, eps, sigma, dt,
                             mode, algo, nsteps, _ptr(trace))
    if rcode != 0:
        raise ValueError("verlet_run failed (cell list needs >= 3 cells per dimension)")
    return pos, vel, F, trace


def rand48_next(x):
    return lib().rand48_next(x)


_KIND_DTYPE = {0: np.uint32, 1: np.uint32, 2: np.float64, 3: np.uint64}


def rand48_fill(seeds, ndraws, kind=0):
    """Sequential rand48.  seeds: array of 48-bit states.  Returns (out [nstreams, ndraws],
    final states).  PAPER.md:142-146."""
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64).copy()
    out = np.zeros((seeds.shape[0], ndraws), dtype=_KIND_DTYPE[kind])
    lib().rand48_fill_seq(_ptr(seeds), seeds.shape[0], ndraws, kind, _ptr(out))
    return out, seeds


def rand48_skip_consts(m, linear=False):
    A, C = ctypes.c_uint64(), ctypes.c_uint64()
    fn = lib().rand48_skip_consts_linear if linear else lib().rand48_skip_consts
    fn(m, ctypes.byref(A), ctypes.byref(C))
    return A.value, C.value


def rand48_skip(x, m):
    return lib().rand48_skip(x, m)


def rand48_leapfrog(seed, S, ndraws):
    out = np.zeros(ndraws, dtype=np.uint64)
    lib().rand48_leapfrog(seed, S, ndraws, _ptr(out))
    return out


def mb_velocities(N, T, seed48):
    """Maxwell-Boltzmann velocities [N,3] (FP64) from one rand48 stream started at state seed48, zero
    net momentum, sum v^2 = 3 N T; also returns the state after the 6 N draws.  SURVEY 8(d) recipe."""
    vel = np.zeros((N, 3), dtype=np.float64)
    st = ctypes.c_uint64(int(seed48))
    lib().mb_velocities(N, float(T), ctypes.byref(st), _ptr(vel))
    return vel, st.value


def andersen_collide(vel, T, thr, seed48, t):
    """Andersen thermostat collisions of step t on velocities vel [N,3] (FP64, copied): returns
    (new velocities, number of collisions).  thr / 2^32 is the collision probability per atom and step."""
    vel = _f64(vel).copy()
    n = lib().andersen_collide(vel.shape[0], _ptr(vel), float(T), int(thr), int(seed48), int(t))
    return vel, n


def verlet_step(pos, vel, F, L, rc=2.5, eps=1.0, sigma=1.0, dt=0.005, mode=1, algo=0):
    """One velocity-Verlet step in place on copies; returns pos, vel, F, (KE, PE, W).  PAPER.md:64."""
    pos, vel, F = _f64(pos).copy(), _f64(vel).copy(), _f64(F).copy()
    ke, pe, w = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    rcode = lib().verlet_step(pos.shape[0], _ptr(pos), _ptr(vel), _ptr(F), L, rc, eps, sigma, dt, mode, algo,
                              ctypes.byref(ke), ctypes.byref(pe), ctypes.byref(w))
    if rcode != 0:
        raise ValueError("verlet_step failed (cell list needs >= 3 cells per dimension)")
    return pos, vel, F, (ke.value, pe.value, w.value)
