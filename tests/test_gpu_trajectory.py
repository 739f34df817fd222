"""The integrator compared element by element above N = 500 (gpu-marked): positions and velocities of whole
trajectories (50 and 40 steps) against oracle.verlet_run at N = 4,000 and 32,000 on all three force paths, and one step of the
N = 2,048,000 system (L = 137, the largest box: coarsest FP32 grid) against oracle.verlet_step.

What this covers that the force-parity tests do not (they read the GPU's own positions back): the drift and the
periodic wrap (common.cuh wrap_drift), the cell index of a drifted atom (cell_coord), the second half-kick folded
into the next step's first kernel, and the snap of seam-crossing atoms onto the local grid of the list path (R25).
PAPER.md:64 (velocity Verlet), step order per R4.

Tolerances.  A stored position is rounded to FP32 once per step: up to ulp(L)/2 = 2^-24 * 2^ceil(log2 L).  Over k
steps these roundings add up like a random walk.  The GPU then evaluates the force at the ROUNDED positions, the
oracle at its own FP64 ones, so the forces differ by (force constant) x (a few ulp(L)) -- up to ~1000 x 1e-5 on a
close pair -- and the velocities by hdt times that per step: the velocity bound scales with ulp(L) too.
Short trajectories: |dx| < max(2e-5, 12 ulp(L)), |dv| < max(2e-4, 250 ulp(L)) (the bounds of tests/test_gpu_mb.py at
N = 500, scaled with the box), rms |dx| < 2 ulp(L), rms |dv| < 40 ulp(L).  Single step at L = 137: |dx| <= ulp(L)/2 +
dt |dv| against the oracle (measured: exactly 0.500 ulp, 1.48 ulp after three steps); the velocity is checked to FP32 rounding against the velocity-Verlet formula applied to the GPU's own forces
of both ends of the step, and those forces against the oracle at the very same positions (R15/R16)."""
import os

import numpy as np
import pytest

import oracle
from helpers import maxwell_boltzmann, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


def ulp_of(L):
    return float(np.spacing(np.float32(np.nextafter(np.float32(L), np.float32(0)))))


def min_image(d, L):
    return d - L * np.rint(d / L)


def start_state(n, rho, T, oracle_uniforms, seed48=0x5EED5EED5EED):
    pos, L = wl.fcc_positions(n, rho)
    vel = maxwell_boltzmann(oracle_uniforms(seed48, 6 * pos.shape[0]), pos.shape[0], T)
    return pos, vel, L


@pytest.mark.parametrize("algo", [0, 1, 2], ids=["allpairs", "cell", "verlet"])
@pytest.mark.parametrize("n,steps,chunks", [(10, 50, (50,)), (10, 50, (1, 7, 42)), (20, 40, (40,))],
                         ids=["N4000", "N4000-chunked", "N32000"])
def test_trajectory_matches_the_oracle_element_by_element(b, oracle_uniforms, algo, n, steps, chunks):
    """T* = 2 so that atoms cross cell faces and the periodic seam within the run (checked)."""
    oracle.set_threads(os.cpu_count() or 1)
    pos, vel, L = start_state(n, 0.8, 2.0, oracle_uniforms)
    N = pos.shape[0]
    po, vo, Fo, tr = oracle.verlet_run(pos, vel, L, steps, algo=1)
    with b.Sim(N, L) as s:
        s.set_state(pos, vel)
        for c in chunks:
            s.step(c, algo)
        p, v = s.get_state()
        F = s.forces()
        ke, pe, w = s.energies()
    assert np.all(p >= 0) and np.all(p < np.float32(L))
    wrapped = np.sum(np.abs(p.astype(np.float64) - pos) > 0.5 * L)
    assert wrapped > 0                                       # some atoms went through the periodic seam
    dx = min_image(p.astype(np.float64) - po, L)
    dv = v.astype(np.float64) - vo
    tol_x = max(2e-5, 12 * ulp_of(L))
    assert np.max(np.abs(dx)) < tol_x, (np.max(np.abs(dx)), tol_x)
    assert np.sqrt(np.mean(dx * dx)) < 2 * ulp_of(L)
    tol_v = max(2e-4, 250 * ulp_of(L))
    assert np.max(np.abs(dv)) < tol_v, (np.max(np.abs(dv)), tol_v)
    assert np.sqrt(np.mean(dv * dv)) < 40 * ulp_of(L)
    assert np.max(np.abs(F.astype(np.float64) - Fo)) < 1e-3 * np.max(np.abs(Fo)) + 0.05    # forces at positions ~1e-5 apart
    print("max|dx| = %.2e (tol %.2e, ulp %.2e)  rms = %.2e  max|dv| = %.2e (tol %.2e)  rms = %.2e  seam crossings = %d"
          % (np.max(np.abs(dx)), tol_x, ulp_of(L), np.sqrt(np.mean(dx * dx)), np.max(np.abs(dv)), tol_v,
             np.sqrt(np.mean(dv * dv)), wrapped))
    assert ke + pe == pytest.approx(tr[steps, 0] + tr[steps, 1], rel=1e-5)


@pytest.fixture(scope="module")
def c4a_melted(b):
    """Config 4a (N = 2,048,000, L = 136.8) melted for 100 steps on the GPU, and the oracle's next three steps from
    that FP32 state (computed once for the module)."""
    oracle.set_threads(os.cpu_count() or 1)

    def src(seed48, m):
        out, _ = b.rand48([seed48], m, b.R48_F64)
        return out[0]
    sysd = wl.md_system("c4a_cell_2048k", velocities_from(src))
    N, L = sysd["N"], sysd["L"]
    with b.Sim(N, L) as s:
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(100, b.MD_CELL)
        p0, v0 = s.get_state()
    x, vv = p0.astype(np.float64), v0.astype(np.float64)
    Fo, _, _ = oracle.forces(x, L, algo=1)
    F0o = Fo.copy()
    ref = []
    for _ in range(3):
        x, vv, Fo, _ = oracle.verlet_step(x, vv, Fo, L, algo=1)
        ref.append((x.copy(), vv.copy(), Fo.copy()))
    return N, L, p0, v0, F0o, ref


@pytest.mark.parametrize("algo,opts", [(1, {}), (1, {"cell_kernel": 3, "fuse_integrator": 1}), (1, {"cell_skin": 0.3}), (2, {}),
                                       (2, {"vl_fuse": 0})],
                         ids=["cell", "cell3-fused", "skin-cells", "verlet", "verlet-unfused"])
def test_one_and_three_steps_of_the_largest_box(b, c4a_melted, algo, opts):
    """From the melted FP32 state of config 4a, md_step(1) and md_step(3) against the oracle's steps: every position
    within ulp(L) + dt |dv| per step; after one step every velocity equal, to FP32 rounding, to
    v0 + hdt F(x0) + hdt F(x1) with the GPU's own forces, which are the oracle's at those positions (R15/R16)."""
    from helpers import check_forces
    N, L, p0, v0, F0o, ref = c4a_melted
    dt, hdt = 0.005, 0.0025
    ulp = ulp_of(L)
    assert ulp == 2.0 ** -16
    for k in (1, 3):
        with b.Sim(N, L) as s:
            for key, val in opts.items():
                s.option(key, val)
            s.set_state(p0, v0)
            s.compute_forces(algo)
            F0 = s.forces().astype(np.float64)
            s.step(k, algo)
            p, v = s.get_state()
            F1 = s.forces().astype(np.float64)
        xo, vo, Fk = ref[k - 1]
        assert np.all(p >= 0) and np.all(p < np.float32(L))
        dv = np.abs(v.astype(np.float64) - vo)
        dx = np.abs(min_image(p.astype(np.float64) - xo, L))
        assert np.max(dv) < k * 1.5e-4, (k, float(np.max(dv)))     # hdt x force constant x position rounding (see above)
        # one step: the drift is correctly rounded (half an ulp of the largest coordinates); three: one ulp per step
        tol_x = (0.5 * ulp if k == 1 else k * ulp) + k * dt * (dv + 1e-5)
        assert np.all(dx <= tol_x), (k, float(np.max(dx / tol_x)), int(np.sum(dx > tol_x)))
        moved = int(np.sum(np.abs(p.astype(np.float64) - p0) > 0.5 * L))
        assert moved > 0                                     # atoms went through the periodic seam in these steps
        nflag = -1
        if k == 1:
            nflag = check_forces(F0, F0o, p0, L, oracle)
            F1o, _, _ = oracle.forces(p.astype(np.float64), L, algo=1)
            nflag += check_forces(F1, F1o, p, L, oracle)
            v_formula = v0.astype(np.float64) + hdt * F0 + hdt * F1
            kick = np.abs(v.astype(np.float64) - v_formula)
            assert np.all(kick <= 2e-6 * np.maximum(1.0, np.abs(v_formula))), float(np.max(kick))
        print("k=%d  max|dx|/ulp = %.3f  max|dv| = %.2e  R16 atoms = %d  seam crossings = %d"
              % (k, float(np.max(dx)) / ulp, float(np.max(dv)), nflag, moved))
