"""md_init_velocities (Maxwell-Boltzmann start velocities on the device, rand48 consumed in registers)
against the oracle's generator (gpu-marked)."""
import numpy as np
import pytest

import oracle
from conftest import golden_lines
from helpers import maxwell_boltzmann, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


@pytest.mark.parametrize("n,T,seed", [(5, 1.0, wl.MASTER_SEED), (10, 1.2, 77), (4, 0.3, 5), (40, 1.0, 9)])
def test_matches_the_oracle_generator(b, n, T, seed):
    pos, L = wl.fcc_positions(n, 0.8)
    N = pos.shape[0]
    x0 = wl.splitmix64(seed) & wl.MASK48
    vo, _ = oracle.mb_velocities(N, T, x0)
    with b.Sim(N, L) as s:
        s.set_state(pos, np.zeros_like(pos))
        s.init_velocities(T, x0)
        _, v = s.get_state()
        s.compute_forces(b.MD_CELL if n >= 5 else b.MD_ALLPAIRS)   # re-orders the slots: ids must survive
        s.init_velocities(T, x0)
        _, v2 = s.get_state()
        ke, _, _ = s.energies()
    # FP64 libm of the device and of the host may differ in the last place before the FP32 cast
    assert np.max(np.abs(v.astype(np.float64) - vo)) < 2.5e-7
    assert np.array_equal(v, v2)                         # caller's atom order whatever the slot order
    assert ke == pytest.approx(1.5 * N * T, rel=2e-7)
    assert np.max(np.abs(v.astype(np.float64).sum(axis=0))) < 2e-7 * N


def test_config1_pin_and_errors(b):
    g = {row[0]: row[1:] for row in golden_lines("config1_trajectory.txt")}
    pos, L = wl.fcc_positions(5, 0.8)
    with b.Sim(500, L) as s:
        with pytest.raises(b.MDError) as e:
            s.init_velocities(1.0, 1)                    # no state yet
        assert e.value.code == b.MD_ESTATE
        s.set_state(pos, np.zeros_like(pos))
        s.init_velocities(1.0, int(g["rand48_start_state"][0], 16))
        _, v = s.get_state()
        assert v[0].astype(np.float64) == pytest.approx([float(t) for t in g["vel0"]], abs=1e-7)
        for bad in ((0.0, 1), (-1.0, 1), (1.0, 1 << 48)):
            with pytest.raises(b.MDError) as e:
                s.init_velocities(*bad)
            assert e.value.code == b.MD_EINVAL


@pytest.mark.parametrize("graph", [1, 0])
@pytest.mark.parametrize("algo", [0, 1, 2])
def test_andersen_thermostat_matches_the_oracle(b, algo, graph, oracle_uniforms):
    """30 steps with collisions (nu dt = 0.05) on config 1 against the oracle's step + andersen_collide; the
    interior steps of a call are replayed from a CUDA graph (the step index lives in device memory) or launched
    directly."""
    c1 = wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))
    N, L, T, nu, seed = c1["N"], c1["L"], 1.5, 10.0, 0x0123456789AB
    with b.Sim(N, L) as s:
        s.option("andersen_T", T)
        s.option("andersen_seed", seed)
        s.option("andersen_nu", nu)
        s.option("graph", graph)
        thr = int(s.stat("andersen_threshold"))
        assert thr == int(np.floor(nu * 0.005 * 2.0 ** 32))
        s.set_state(c1["pos"], c1["vel"])
        s.step(12, algo)
        s.step(18, algo)                                   # the step index carries over between calls
        assert s.stat("andersen_steps") == 30
        assert (s.stat("graph_replays") > 0) == bool(graph)
        p, v = s.get_state()
        ke, pe, w = s.energies()
    po, vo = c1["pos"].astype(np.float64), c1["vel"].astype(np.float64)
    Fo, _, _ = oracle.forces(po, L, algo=0)
    ncoll = 0
    for t in range(30):
        po, vo, Fo, (_, peo, wo) = oracle.verlet_step(po, vo, Fo, L, algo=0)
        vo, n = oracle.andersen_collide(vo, T, thr, seed, t)
        ncoll += n
    assert 500 < ncoll < 1000                              # 30 x 500 x 0.05 = 750 expected
    d = p.astype(np.float64) - po
    d -= L * np.rint(d / L)
    assert np.max(np.abs(d)) < 2e-5 and np.max(np.abs(v.astype(np.float64) - vo)) < 2e-4
    assert ke == pytest.approx(oracle.kinetic_energy(vo), rel=1e-5) and pe == pytest.approx(peo, rel=1e-5)


def test_andersen_off_is_plain_nve(b, oracle_uniforms):
    c1 = wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))
    out = []
    for nu in (None, 0.0):
        with b.Sim(c1["N"], c1["L"]) as s:
            if nu is not None:
                s.option("andersen_T", 1.0)
                s.option("andersen_nu", nu)
            s.set_state(c1["pos"], c1["vel"])
            s.step(20, 0)
            out.append(s.get_state())
    assert np.max(np.abs(out[0][1] - out[1][1])) < 1e-4
