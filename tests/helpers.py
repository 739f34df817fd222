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


def check_forces(F, Fo, pos, L, oracle, rc=2.5, max_atoms=200, eps=1.0, sigma=1.0):
    """R15 on every component of a whole system, with the excuse of R16 read per component:
    a pair with |r^2/rc^2 - 1| < 4e-7 (listed by the oracle through its linked cells) may be classified either
    way, so on an atom of such a pair the GPU force may differ from the oracle's by exactly that pair's own term
    at the cutoff, -(f_LJ(rc)/r) d: removed if the oracle counted the pair, added if it did not.  A component that
    misses R15 is accepted only if, for some choice of which flagged pairs of that atom were classified the other
    way, the residual is back inside R15 on all three components.  Modes 0 and 1 (mode 2 has no jump at rc).
    Returns the number of atoms excused that way."""
    F = np.asarray(F, dtype=np.float64)
    tol = np.maximum(1e-4 * np.abs(Fo), 1e-5)
    bad = np.argwhere(np.abs(F - Fo) > tol)
    atoms = sorted(set(int(a) for a in bad[:, 0]))
    assert len(atoms) <= max_atoms, "too many violations: %d components" % len(bad)
    if not atoms:
        return 0
    x = np.asarray(pos, dtype=np.float64)
    pairs, n = oracle.near_cutoff_pairs_cell(x, L, rc=rc, tol=4e-7, cap=1 << 20)
    assert n <= (1 << 20)
    for a in atoms:
        partners = [int(j) for j in pairs[pairs[:, 0] == a, 1]]
        assert partners, ("R15 violated on atom %d without a near-cutoff partner" % a, F[a], Fo[a])
        assert len(partners) <= 8
        terms = []
        for j in partners:
            d = x[j] - x[a]
            d -= L * np.rint(d / L)
            r2 = float(d @ d)
            _, _, fr = oracle.lj_pair(0, r2, eps, sigma, 1.01 * rc)      # the untruncated f/r at this distance
            sign = -1.0 if r2 < rc * rc else 1.0                         # oracle counted it: the GPU may have dropped it
            terms.append(sign * (-fr) * d)                               # Eq. 1: F_a -= (f/r) d
        ok = False
        for mask in range(1, 1 << len(terms)):
            resid = F[a] - Fo[a] - sum(t for k, t in enumerate(terms) if mask >> k & 1)
            if np.all(np.abs(resid) <= tol[a]):
                ok = True
                break
        assert ok, ("atom %d: deviation is not the cutoff term of its near-cutoff pairs" % a, F[a], Fo[a], terms)
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
