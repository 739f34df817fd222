"""Pins for the oracle's velocity Verlet (O4) and the input recipe (O6).
PAPER.md:64; readings R4 (step order), R11, R13, R14, R17, R19."""
import numpy as np
import pytest

import oracle
from conftest import golden_lines
from helpers import maxwell_boltzmann, velocities_from
from paper_0709_3225_b200 import workloads as wl


def golden_c1():
    return {row[0]: row[1:] for row in golden_lines("config1_trajectory.txt")}


@pytest.fixture(scope="module")
def c1(oracle_uniforms):
    return wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))


def test_free_flight_closed_form():
    # two atoms that never come within rc move on straight lines, wrapped: x(t) = x0 + v t mod L
    L, dt, n = 12.0, 0.005, 400
    pos = np.array([[1.0, 1.0, 1.0], [7.0, 7.0, 7.0]])
    vel = np.array([[-0.9, 0.3, 0.0], [-0.9, 0.3, 0.0]])       # same velocity: distance stays 6 sqrt3
    p, v, F, tr = oracle.verlet_run(pos, vel, L, n, dt=dt)
    want = pos + vel * dt * n
    want -= L * np.floor(want / L)
    assert np.max(np.abs(p - want)) < 1e-12
    assert np.all((p >= 0) & (p < L))
    assert np.all(v == vel) and np.all(tr[:, 1] == 0) and tr[-1, 0] == pytest.approx(0.9, rel=1e-14)


def test_dimer_oscillation_conserves_energy_and_momentum():
    L = 12.0
    pos = np.array([[5.0, 5.0, 5.0], [6.05, 5.0, 5.0]])
    vel = np.array([[0.1, 0.0, 0.02], [-0.05, 0.03, 0.0]])
    p, v, F, tr = oracle.verlet_run(pos, vel, L, 4000, dt=0.002, mode=1)
    E = tr[:, 0] + tr[:, 1]
    assert np.ptp(tr[:, 1]) > 0.05                               # it does oscillate
    assert np.max(np.abs(E - E[0])) < 1e-4 * abs(E[0])                    # bounded fluctuation
    assert abs(E[2000:].mean() - E[:2000].mean()) < 5e-6 * abs(E[0])       # no secular drift
    assert np.max(np.abs(v.sum(axis=0) - vel.sum(axis=0))) < 1e-13


def test_energy_error_scales_as_dt_squared(c1):
    pos, L = wl.perturbed_fcc(4, 0.8, 0.05, seed=2)
    vel = c1["vel"][: pos.shape[0]].astype(np.float64) * 0.7
    vel -= vel.mean(axis=0)
    fl = []
    for dt, n in [(0.004, 250), (0.002, 500)]:
        _, _, _, tr = oracle.verlet_run(pos, vel, L, n, dt=dt)
        E = tr[:, 0] + tr[:, 1]
        fl.append(np.std(E))
    assert 3.0 < fl[0] / fl[1] < 5.5                             # halving dt quarters the fluctuation


def test_time_reversibility(c1):
    p0, v0 = c1["pos"].astype(np.float64), c1["vel"].astype(np.float64)
    p1, v1, _, _ = oracle.verlet_run(p0, v0, c1["L"], 100)
    p2, v2, _, _ = oracle.verlet_run(p1, -v1, c1["L"], 100)
    d = p2 - p0
    d -= c1["L"] * np.rint(d / c1["L"])
    assert np.max(np.abs(d)) < 1e-9 and np.max(np.abs(v2 + v0)) < 1e-8      # R19


def test_nve_no_drift_and_momentum(c1):
    p0, v0 = c1["pos"].astype(np.float64), c1["vel"].astype(np.float64)
    p, v, F, tr = oracle.verlet_run(p0, v0, c1["L"], 1500)
    E = tr[:, 0] + tr[:, 1]
    # R17 / SURVEY H8: transient excursion ~1.35e-4 around step 10, then fluctuation ~1e-5
    assert 1.0e-4 < np.max(np.abs(E[:30] - E[0])) / abs(E[0]) < 1.7e-4
    drift = abs(E[1000:1500].mean() - E[500:1000].mean()) / abs(E[0])
    assert drift < 1e-5
    assert np.max(np.abs(v.sum(axis=0) - v0.sum(axis=0))) < 1e-10      # momentum conserved
    assert np.all((p >= 0) & (p < c1["L"]))


def test_allpairs_and_cell_trajectories_agree(c1):
    p0, v0 = c1["pos"].astype(np.float64), c1["vel"].astype(np.float64)
    pa, va, _, ta = oracle.verlet_run(p0, v0, c1["L"], 50, algo=0)
    pc, vc, _, tc = oracle.verlet_run(p0, v0, c1["L"], 50, algo=1)
    assert np.max(np.abs(pa - pc)) < 1e-9 and np.max(np.abs(ta - tc)) < 1e-7


def test_config1_input_recipe(c1, oracle_uniforms):
    g = golden_c1()
    x0 = wl.splitmix64(wl.MASTER_SEED) & wl.MASK48
    assert x0 == int(g["rand48_start_state"][0], 16)
    _, st = oracle.rand48_fill([x0], 3000, kind=2)
    assert int(st[0]) == int(g["rand48_state_after_3000_draws"][0], 16)
    assert c1["N"] == 500 and c1["L"] == pytest.approx(8.549880027771, abs=1e-12)
    assert c1["vel"][0] == pytest.approx([float(x) for x in g["vel0"]], abs=2e-7)
    v = c1["vel"].astype(np.float64)
    assert np.sum(v * v) == pytest.approx(1500.0, rel=1e-7)      # sum v^2 = 3 N T (R11)
    assert np.max(np.abs(v.sum(axis=0))) < 1e-4


def test_config1_trajectory_matches_survey_probe(c1):
    g = golden_c1()
    p, v, F, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 100)

    def chk(step, key, col):
        row = g[key]
        want = float(row[row.index(col) + 1])
        have = {"KE": tr[step, 0], "PE": tr[step, 1], "W": tr[step, 2], "E": tr[step, 0] + tr[step, 1]}[col]
        assert have == pytest.approx(want, rel=2e-9), (key, col)

    for col in ("KE", "PE", "W"):
        chk(0, "step0", col)
        chk(100, "step100", col)
    chk(1, "step1", "KE"), chk(1, "step1", "PE"), chk(10, "step10", "E")
    assert F[0] == pytest.approx([float(x) for x in g["step100_F0"]], abs=2e-6)
