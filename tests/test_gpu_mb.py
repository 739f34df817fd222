"""md_init_velocities (Maxwell-Boltzmann start velocities on the device, rand48 consumed in registers)
against the oracle's generator (gpu-marked)."""
import numpy as np
import pytest

import oracle
from conftest import golden_lines
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
