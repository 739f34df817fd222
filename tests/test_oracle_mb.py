"""Pins of the oracle's Maxwell-Boltzmann generator (oracle.mb_velocities): the printed values of the
survey's independent NumPy probe (tests/golden/config1_trajectory.txt), the harness generator
(helpers.maxwell_boltzmann, the harness generator, fed with the oracle's sequential rand48), and the defining moments."""
import numpy as np
import pytest

import oracle
from conftest import golden_lines
from helpers import maxwell_boltzmann, velocities_from
from paper_0709_3225_b200 import workloads as wl


@pytest.fixture(scope="module")
def g():
    return {row[0]: row[1:] for row in golden_lines("config1_trajectory.txt")}


def test_config1_values_of_the_survey_probe(g):
    x0 = wl.splitmix64(wl.MASTER_SEED) & wl.MASK48
    assert x0 == int(g["rand48_start_state"][0], 16)
    v, x1 = oracle.mb_velocities(500, 1.0, x0)
    assert x1 == int(g["rand48_state_after_3000_draws"][0], 16)          # exactly 6 N draws, in order
    # the probe printed the FP32 state to 8 decimals
    assert v[0].astype(np.float32).astype(np.float64) == pytest.approx([float(t) for t in g["vel0"]], abs=1e-8)
    v32 = v.astype(np.float32).astype(np.float64)
    assert 0.5 * np.sum(v32 * v32) == pytest.approx(float(g["step0"][1]), rel=1e-9)   # KE of the FP32 state


@pytest.mark.parametrize("N,T,seed", [(500, 1.0, 1), (4000, 1.2, 77), (7, 0.3, 12345)])
def test_matches_the_harness_generator_and_the_moments(N, T, seed, oracle_uniforms):
    x0 = wl.splitmix64(seed) & wl.MASK48
    v, _ = oracle.mb_velocities(N, T, x0)
    ref = maxwell_boltzmann(oracle_uniforms(x0, 6 * N), N, T)        # float32
    assert np.max(np.abs(v - ref.astype(np.float64))) < 3e-7             # FP32 cast of the same numbers
    assert np.max(np.abs(v.sum(axis=0))) < 1e-10 * N                      # zero net momentum
    assert np.sum(v * v) == pytest.approx(3.0 * N * T, rel=1e-13)         # R11


def test_draw_order_is_atom_major_component_minor():
    """u1 of (atom 0, x) is the first draw: a state chosen so that 1 - u1 = 1 gives v_x = 0 before the
    mean is removed; checked through the second atom instead: velocities of a 2-atom system are
    antisymmetric after the mean is removed."""
    v, _ = oracle.mb_velocities(2, 1.0, 0x1234ABCD330E)
    assert np.allclose(v[0], -v[1], rtol=0, atol=1e-14)


# ---- Andersen thermostat (oracle.andersen_collide) ------------------------------------------
def test_andersen_never_and_always():
    rng = np.random.default_rng(3)
    v = rng.normal(size=(2000, 3))
    out, n = oracle.andersen_collide(v, 1.5, 0, 0x1234ABCD330E, 0)
    assert n == 0 and np.array_equal(out, v)                            # probability 0: untouched
    out, n = oracle.andersen_collide(v, 1.5, 0xFFFFFFFF, 0x1234ABCD330E, 0)
    assert n == 2000                                                    # probability 1 - 2^-32
    assert np.mean(out * out) == pytest.approx(1.5, rel=4.0 * np.sqrt(2.0 / 6000))   # <v_c^2> = T
    assert abs(np.mean(out)) < 4.0 * np.sqrt(1.5 / 6000)


def test_andersen_collision_rate_and_stream_ownership():
    """(t, i) owns draws 7 (t N + i) .. + 6 of ONE stream: the decisions of step t are the 32 high bits of
    every seventh draw of the sequential series (glibc-pinned rand48_fill), and steps do not overlap."""
    N, thr, seed = 5000, 1 << 29, 0x6ABB51034992                        # p = 1/8
    raw, _ = oracle.rand48_fill([seed], 7 * N * 3, kind=0)              # uint32 = x >> 16
    v = np.zeros((N, 3))
    for t in range(3):
        out, n = oracle.andersen_collide(v, 1.0, thr, seed, t)
        decide = raw[0][7 * N * t:7 * N * (t + 1):7] < thr
        assert n == int(decide.sum())
        assert np.array_equal(np.any(out != 0.0, axis=1), decide)       # exactly those atoms got new velocities
        assert abs(n - N / 8) < 4.0 * np.sqrt(N * (1 / 8) * (7 / 8))


def test_andersen_new_velocity_is_the_mb_formula_of_draws_1_to_6():
    """A colliding atom's new velocity equals what mb_velocities' formula gives for the same six uniforms;
    checked through mb_velocities itself on a 2-atom system built from that atom's draws is not possible
    (it removes the mean), so the doubles x * 2^-48 of the stream are fed to the harness formula."""
    N, seed = 64, 0x99D4809E0FCA
    u, _ = oracle.rand48_fill([seed], 7 * N, kind=2)
    out, n = oracle.andersen_collide(np.zeros((N, 3)), 0.7, 0xFFFFFFFF, seed, 0)
    u = u[0].reshape(N, 7)[:, 1:].reshape(N, 3, 2)
    ref = np.sqrt(0.7) * np.sqrt(-2.0 * np.log(1.0 - u[..., 0])) * np.cos(2.0 * np.pi * u[..., 1])
    assert n == N and np.max(np.abs(out - ref)) < 1e-14
