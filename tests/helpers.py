"""Shared helpers for the parity tests (no arithmetic of the method lives here)."""
import numpy as np


def force_check(F_gpu, F_ref, rel=1e-4, floor=1e-5):
    """Strict per-component reading of BASELINE.json's tolerance (R15):
    |dF_c| <= max(rel |F_c|, floor).  Returns (#violations, worst err/tol)."""
    F_gpu = np.asarray(F_gpu, dtype=np.float64)
    tol = np.maximum(rel * np.abs(F_ref), floor)
    ratio = np.abs(F_gpu - F_ref) / tol
    return int(np.sum(ratio > 1.0)), float(np.max(ratio))


def melt(pos, vel, L, steps, oracle, **kw):
    """Advance with the oracle and return FP32-rounded (pos, vel) snapshot."""
    p, v, _, _ = oracle.verlet_run(pos, vel, L, steps, **kw)
    p = p.astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    return p, v.astype(np.float32)


def check_forces(F, Fo, pos, L, oracle, rc=2.5, max_atoms=200):
    """R15 on every component of a whole system.  A component may miss it only on an atom that has a partner
    inside the cutoff window of R16 (|r^2/rc^2 - 1| < 4e-7, listed by the oracle through its linked cells:
    either classification is correct there), and then by at most the force jump at the cutoff, 0.039.
    Returns the number of atoms excused that way."""
    F = np.asarray(F, dtype=np.float64)
    tol = np.maximum(1e-4 * np.abs(Fo), 1e-5)
    bad = np.argwhere(np.abs(F - Fo) > tol)
    atoms = sorted(set(int(a) for a in bad[:, 0]))
    assert len(atoms) <= max_atoms, "too many violations: %d components" % len(bad)
    if not atoms:
        return 0
    pairs, n = oracle.near_cutoff_pairs_cell(np.asarray(pos, dtype=np.float64), L, rc=rc, tol=4e-7, cap=1 << 20)
    assert n <= (1 << 20)
    flagged = set(int(i) for i in pairs[:, 0])
    for a in atoms:
        assert a in flagged, ("R15 violated on atom %d without a near-cutoff partner" % a, F[a], Fo[a])
        assert np.max(np.abs(F[a] - Fo[a])) < 0.04 + 1e-4, (a, F[a], Fo[a])
    return len(atoms)


def maxwell_boltzmann(uniforms, N, T):
    """The harness's own velocity generator (SURVEY 8(d) recipe, NumPy FP64, independent of both the oracle's
    C and the device kernel): float32 [N,3] from 6N uniform doubles in [0,1), Box-Muller cosine branch.
    For atom i, component c, in order: u1 = uniforms[6i+2c], u2 = uniforms[6i+2c+1];
    v = sqrt(T) sqrt(-2 ln(1-u1)) cos(2 pi u2).  Then the mean is subtracted and the set rescaled so that
    sum v^2 = 3 N T (R11), and cast to float32."""
    u = np.asarray(uniforms, dtype=np.float64).reshape(N, 3, 2)
    v = np.sqrt(T) * np.sqrt(-2.0 * np.log(1.0 - u[..., 0])) * np.cos(2.0 * np.pi * u[..., 1])
    v -= v.mean(axis=0, keepdims=True)
    v *= np.sqrt(3.0 * N * T / np.sum(v * v))
    return v.astype(np.float32)


def velocities_from(uniform_source):
    """velocity_source for workloads.md_system: the generator above fed by uniform_source(seed48, n)."""
    return lambda N, T, seed48: maxwell_boltzmann(uniform_source(seed48, 6 * N), N, T)
