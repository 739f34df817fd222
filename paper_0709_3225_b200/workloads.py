"""Seeded synthetic inputs shared by the CUDA path, the tests and the oracle harness.

This module holds NONE of the method's arithmetic: no pair force, no integrator,
no rand48.  Uniform random numbers are passed in by the caller (from the library's
rand48_fill on the product side, from oracle.rand48_fill in the tests), so the same
recipe serves both sides without sharing code between them.

Recipe: DESIGN.md section 4 (from SURVEY.md section 8(d) and BASELINE.json configs).
The paper itself gives no initial condition, temperature, density or time step
(PAPER.md:64 only names velocity Verlet); BASELINE.json's configs stand in.
"""
import numpy as np

MASTER_SEED = 20070920
MASK48 = (1 << 48) - 1
_M64 = (1 << 64) - 1

# name -> (n fcc cells per side, density, T*, steps, algo)   [BASELINE.json configs 1-4]
CONFIGS = {
    "c1_allpairs_500": dict(n=5, rho=0.8, T=1.0, steps=100, algo=0),
    "c2_allpairs_32k": dict(n=20, rho=0.8, T=1.0, steps=1000, algo=0),
    "c3_cell_256k": dict(n=40, rho=0.8, T=1.0, steps=1000, algo=1),
    "c4a_cell_2048k": dict(n=80, rho=0.8, T=1.2, steps=500, algo=1),
    "c4b_cell_2048k_rho03": dict(n=80, rho=0.3, T=1.2, steps=500, algo=1),
}
RC, EPS, SIGMA, DT, SHIFTED = 2.5, 1.0, 1.0, 0.005, 1
# config 5 [BASELINE.json]: 65536 streams x 4096 draws, then one stream of 2^28 draws
C5_NSTREAMS, C5_NDRAWS, C5_SINGLE_NDRAWS = 65536, 4096, 1 << 28


def splitmix64(state):
    """First output of the SplitMix64 generator whose state is `state` (R9)."""
    z = (state + 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_seeds(seed, nstreams):
    """48-bit start states: low 48 bits of splitmix64(seed + i), i < nstreams."""
    return np.array([splitmix64((seed + i) & _M64) & MASK48 for i in range(nstreams)],
                    dtype=np.uint64)


def box_length(N, rho):
    """L = (double)(float) cbrt(N / rho): the box is the FP32-rounded value (R13)."""
    return float(np.float32(np.cbrt(N / rho)))


def fcc_positions(n, rho):
    """4 n^3 atoms on an fcc lattice filling the cubic box; returns (pos float32 [N,3], L).

    Atom index t = ((ix*n + iy)*n + iz)*4 + b, basis b in {(0,0,0), (1/2,1/2,0),
    (1/2,0,1/2), (0,1/2,1/2)}, position = (cell + basis + 1/4) * a, a = L/n.
    """
    N = 4 * n ** 3
    L = box_length(N, rho)
    a = L / n
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], dtype=np.float64)
    g = np.arange(n, dtype=np.float64)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    pos = ((cells + basis[None, :, :] + 0.25) * a).reshape(N, 3)
    return pos.astype(np.float32), L


def md_system(name, velocity_source, seed=MASTER_SEED):
    """Build a named MD config.  velocity_source(N, T, seed48) -> float32 [N,3]: Maxwell-Boltzmann
    velocities at temperature T drawn from ONE rand48 stream started at state seed48 (the recipe of
    DESIGN.md section 4; the arithmetic lives with the caller: md_init_velocities on the product side,
    oracle.mb_velocities or the tests' NumPy generator on the test side)."""
    cfg = CONFIGS[name]
    pos, L = fcc_positions(cfg["n"], cfg["rho"])
    N = pos.shape[0]
    x0 = splitmix64(seed) & MASK48
    vel = np.ascontiguousarray(velocity_source(N, cfg["T"], x0), dtype=np.float32)
    assert vel.shape == (N, 3)
    return dict(name=name, N=N, L=L, pos=pos, vel=vel, rc=RC, eps=EPS, sigma=SIGMA, dt=DT,
                shifted=SHIFTED, steps=cfg["steps"], algo=cfg["algo"], rho=cfg["rho"], T=cfg["T"])


def perturbed_fcc(n, rho, amplitude, seed):
    """fcc lattice with every coordinate displaced by a uniform number in
    [-amplitude, amplitude) * a (numpy PCG stream), wrapped into [0,L), float32.
    Nearest neighbours sit at a/sqrt(2), so amplitude <= 0.12 keeps all pairs apart
    while giving forces of order 10-100.  Returns (pos float32 [N,3], L)."""
    pos, L = fcc_positions(n, rho)
    a = L / n
    rng = np.random.default_rng(seed)
    p = pos.astype(np.float64) + (rng.random(pos.shape) * 2.0 - 1.0) * amplitude * a
    p = np.float32(p - L * np.floor(p / L))
    p[p >= np.float32(L)] = 0.0
    return p, L
