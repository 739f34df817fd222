"""Skin cells on the cell path (option "cell_skin"; cells wider than the
interaction range by a skin, "update the cell lists only every couple of time steps") against the FP64
oracle (gpu-marked).  Same forces and tolerances as the rebuild-every-step path (R15, R17)."""
import os

import numpy as np
import pytest

import oracle
from helpers import check_forces, force_check, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


@pytest.mark.parametrize("n,rho,amp", [(5, 0.8, 0.10), (7, 0.9, 0.08), (6, 0.3, 0.15), (10, 0.8, 0.1), (9, 0.05, 0.3)])
@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_forces_match_oracle(b, n, rho, amp, shifted):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=500 + n)
    with b.Sim(pos.shape[0], L, shifted=shifted) as s:
        s.option("cell_skin", 0.3)
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_CELL)
        F, (ke, pe, w) = s.forces(), s.energies()
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


def test_config1_energy_trace_while_cells_are_reused(b, oracle_uniforms):
    """Per-step total energy within 1e-5 of the oracle over 100 steps (R17); the cells are re-sorted only when
    an atom has strayed half the skin, and every force evaluation in between still matches the oracle."""
    c1 = wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))
    _, _, _, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 100, algo=0)
    with b.Sim(c1["N"], c1["L"]) as s:
        s.option("cell_skin", 0.3)
        s.set_state(c1["pos"], c1["vel"])
        s.compute_forces(b.MD_CELL)
        worst = 0.0
        for t in range(101):
            if t:
                s.step(1, b.MD_CELL)
            ke, pe, w = s.energies()
            Eo = tr[t, 0] + tr[t, 1]
            worst = max(worst, abs(ke + pe - Eo) / abs(Eo))
            if t % 10 == 7:                                # forces from cells that are several steps old
                p, v = s.get_state()
                Fo, _, _ = oracle.forces(p.astype(np.float64), c1["L"], algo=0)
                assert force_check(s.forces(), Fo)[0] == 0, t
        assert worst < 1e-5, worst
        builds, evals = s.stat("vl_builds"), s.stat("vl_steps")
        assert evals == 101 and 3 <= builds <= 40, (builds, evals)


def test_multi_step_calls_and_graph_replay_agree_with_single_steps(b, oracle_uniforms):
    c1 = wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))
    res = []
    for graph, chunks in ((1, [60]), (0, [60]), (1, [1] * 60)):
        with b.Sim(c1["N"], c1["L"]) as s:
            s.option("cell_skin", 0.3)
            s.option("graph", graph)
            s.set_state(c1["pos"], c1["vel"])
            for k in chunks:
                s.step(k, b.MD_CELL)
            res.append(s.get_state() + (s.energies(),))
    for r in res[1:]:
        # same physics; the order of atoms inside a cell comes from atomics, so FP32 sums differ in the last
        # bits and the trajectories part at rounding level
        d = r[0].astype(np.float64) - res[0][0]
        d -= c1["L"] * np.rint(d / c1["L"])
        assert np.max(np.abs(d)) < 2e-5 and np.max(np.abs(r[1] - res[0][1])) < 2e-4
        assert r[2][0] + r[2][1] == pytest.approx(res[0][2][0] + res[0][2][1], rel=1e-6)


def test_option_rules(b):
    pos, L = wl.perturbed_fcc(6, 0.8, 0.1, seed=3)
    with b.Sim(pos.shape[0], L) as s:
        s.option("cell_skin", 0.4)
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_CELL)
        with pytest.raises(b.MDError):
            s.option("cell_skin", 0.2)                 # the skin is in use
        s.option("cell_skin", 0.0)                     # back to rebuilding every step
        s.compute_forces(b.MD_CELL)
        Fo, _, _ = oracle.forces(pos.astype(np.float64), L, algo=0)
        assert force_check(s.forces(), Fo)[0] == 0
    with b.Sim(100, 8.0) as s:                         # int[8 / 2.8] = 2 cells: no skin cells
        s.option("cell_skin", 0.3)
        s.set_state(np.random.default_rng(1).random((100, 3)).astype(np.float32) * 8, np.zeros((100, 3), np.float32))
        with pytest.raises(b.MDError) as e:
            s.compute_forces(b.MD_CELL)
        assert e.value.code == b.MD_EDOMAIN


@pytest.mark.parametrize("name", ["c3_cell_256k", "c4b_cell_2048k_rho03"])
def test_full_size_parity(b, name):
    """The named number of steps at full size, forces from cells up to a dozen steps old, every atom."""
    oracle.set_threads(os.cpu_count() or 1)

    def src(seed48, n):
        out, _ = b.rand48([seed48], n, b.R48_F64)
        return out[0]
    sysd = wl.md_system(name, velocities_from(src))
    with b.Sim(sysd["N"], sysd["L"]) as s:
        s.option("cell_skin", 0.3)
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(sysd["steps"], b.MD_CELL)
        ke, pe, w = s.energies()
        F = s.forces()
        p, v = s.get_state()
        assert s.stat("vl_builds") < 0.3 * s.stat("vl_steps")
    Fo, peo, wo = oracle.forces(p.astype(np.float64), sysd["L"], algo=1)
    assert np.max(np.abs(Fo)) > 10
    check_forces(F, Fo, p, sysd["L"], oracle)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)
