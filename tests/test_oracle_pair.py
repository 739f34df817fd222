"""Pins for oracle lj_pair (O1): closed forms, hand constants, finite differences.
PAPER.md:56-62 (Eq. 2-3); readings R1 (1/sigma factor), R2 (which shift)."""
import math

import numpy as np
import pytest

import oracle
from conftest import golden_lines

RMIN2 = 2.0 ** (1.0 / 3.0)          # (2^(1/6))^2


def consts():
    return {k: float(v) for k, v in golden_lines("lj_constants_rc25.txt")}


def test_closed_forms_at_rmin():
    inside, u, fr = oracle.lj_pair(0, RMIN2)
    assert inside
    assert abs(u + 1.0) < 1e-14                 # U_LJ(2^(1/6) sigma) = -eps
    assert abs(fr) < 1e-13                      # f_LJ(2^(1/6) sigma) = 0
    # with eps, sigma != 1
    eps, sig = 1.7, 0.9
    inside, u, fr = oracle.lj_pair(0, RMIN2 * sig * sig, eps, sig, 2.5 * sig)
    assert abs(u + eps) < 1e-13 and abs(fr) < 1e-12


def test_values_at_r_equal_sigma():
    # U_LJ(sigma) = 0 and f_LJ(sigma) = 24 eps / sigma (Eq. 2 with the 1/sigma factor, R1)
    eps, sig = 2.5, 1.3
    _, u, fr = oracle.lj_pair(0, sig * sig, eps, sig, 2.5 * sig)
    assert abs(u) < 1e-13
    assert abs(fr * sig - 24.0 * eps / sig) < 1e-11


def test_hand_constants_rc25():
    c = consts()
    rc2 = 6.25
    below = rc2 * (1 - 1e-15)
    _, u0, fr0 = oracle.lj_pair(0, below)
    assert abs(u0 - c["U_LJ_rc"]) < 1e-13
    assert abs(fr0 * 2.5 - c["f_LJ_rc"]) < 1e-13
    assert abs((1 / 2.5) ** 6 - c["rc_pow_minus6"]) < 1e-17
    _, u1, _ = oracle.lj_pair(1, RMIN2)
    assert abs(u1 - c["mode1_U_rmin"]) < 1e-12
    _, u2, fr2 = oracle.lj_pair(2, RMIN2)
    assert abs(u2 - c["mode2_U_rmin"]) < 1e-11
    assert abs(fr2 * math.sqrt(RMIN2) - c["mode2_f_rmin"]) < 1e-12


def test_shift_makes_energy_zero_at_cutoff():
    below = 6.25 * (1 - 1e-15)
    for mode in (1, 2):
        _, u, _ = oracle.lj_pair(mode, below)
        assert abs(u) < 1e-13                    # U(rc) = 0
    _, _, fr = oracle.lj_pair(2, below)
    assert abs(fr) < 1e-13                       # mode 2: f(rc) = 0


def test_strict_cutoff():
    # r < rc inside, r >= rc zero
    for mode in (0, 1, 2):
        inside, u, fr = oracle.lj_pair(mode, 6.25)
        assert (inside, u, fr) == (False, 0.0, 0.0)
        inside, _, _ = oracle.lj_pair(mode, np.nextafter(6.25, 0.0))
        assert inside
        inside, u, fr = oracle.lj_pair(mode, 7.0)
        assert (inside, u, fr) == (False, 0.0, 0.0)


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("eps,sig", [(1.0, 1.0), (0.7, 1.4)])
def test_force_is_minus_dU_dr(mode, eps, sig):
    rc = 2.5 * sig
    for r in np.linspace(0.9 * sig, 2.45 * sig, 23):
        h = 1e-5 * sig
        _, up, _ = oracle.lj_pair(mode, (r + h) ** 2, eps, sig, rc)
        _, um, _ = oracle.lj_pair(mode, (r - h) ** 2, eps, sig, rc)
        _, _, fr = oracle.lj_pair(mode, r * r, eps, sig, rc)
        f = fr * r
        assert abs(-(up - um) / (2 * h) - f) < 2e-7 * max(1.0, abs(f))


def test_sign_repulsive_inside_rmin():
    _, _, fr = oracle.lj_pair(1, 1.0)
    assert fr > 0                                # f > 0 is repulsive (R6)
    _, _, fr = oracle.lj_pair(1, 1.5 ** 2)
    assert fr < 0


# ---- second pair potential: screened Coulomb / Yukawa --------------------
def test_yukawa_coulomb_limit_by_hand():
    """kappa = 0 is the bare Coulomb pair: U = A/r, f = A/r^2 (two unit charges 2 apart: U = 1/2, f = 1/4)."""
    inside, u, fr = oracle.yukawa_pair(0, 4.0, A=1.0, kappa=0.0, rc=2.5)
    assert inside and u == pytest.approx(0.5, rel=1e-15) and fr * 2.0 == pytest.approx(0.25, rel=1e-15)
    inside, u, fr = oracle.yukawa_pair(0, 1.5 ** 2, A=3.0, kappa=0.0, rc=2.5)
    assert u == pytest.approx(2.0, rel=1e-15) and fr * 1.5 == pytest.approx(3.0 / 2.25, rel=1e-15)


def test_yukawa_closed_forms():
    A, kappa, rc = 5.0, 1.25, 2.5
    r = 1.0 / kappa                                         # U(1/kappa) = A kappa / e, f(1/kappa) = 2 A kappa^2 / e
    inside, u, fr = oracle.yukawa_pair(0, r * r, A, kappa, rc)
    assert u == pytest.approx(A * kappa / np.e, rel=1e-14)
    assert fr * r == pytest.approx(2.0 * A * kappa ** 2 / np.e, rel=1e-14)
    # cutoff: strict, zero beyond; mode 1 and 2 vanish at rc, mode 2 also in force
    assert oracle.yukawa_pair(0, rc * rc, A, kappa, rc) == (False, 0.0, 0.0)
    eps = 1e-9
    _, u1, _ = oracle.yukawa_pair(1, (rc - eps) ** 2, A, kappa, rc)
    _, u2, f2 = oracle.yukawa_pair(2, (rc - eps) ** 2, A, kappa, rc)
    assert abs(u1) < 1e-8 and abs(u2) < 1e-8 and abs(f2 * rc) < 1e-8
    # the shift of mode 1 is U_Y(rc)
    _, u0, _ = oracle.yukawa_pair(0, 1.7 ** 2, A, kappa, rc)
    _, u1, _ = oracle.yukawa_pair(1, 1.7 ** 2, A, kappa, rc)
    assert u0 - u1 == pytest.approx(A * np.exp(-kappa * rc) / rc, rel=1e-13)


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_yukawa_force_is_minus_dU_dr(mode):
    A, kappa, rc = 2.0, 0.8, 2.5
    for r in (0.6, 1.0, 1.9, 2.45):
        h = 1e-5
        _, up, _ = oracle.yukawa_pair(mode, (r + h) ** 2, A, kappa, rc)
        _, um, _ = oracle.yukawa_pair(mode, (r - h) ** 2, A, kappa, rc)
        _, _, fr = oracle.yukawa_pair(mode, r * r, A, kappa, rc)
        assert fr * r == pytest.approx(-(up - um) / (2 * h), rel=1e-8)


def test_yukawa_through_the_force_loops():
    """Two equal charges repel along their axis with f_Y(r) (Eq. 1 sign, R6); both loops agree on a random
    system; total force vanishes; the selector goes back to Lennard-Jones after the block."""
    A, kappa, L = 4.0, 1.1, 12.0
    pos = np.array([[1.0, 1.0, 1.0], [2.5, 1.0, 1.0]])
    with oracle.potential(1, A, kappa):
        F, pe, w = oracle.forces(pos, L, mode=0, algo=0)
    f = A * np.exp(-kappa * 1.5) * (1 / 1.5 ** 2 + kappa / 1.5)
    assert F[0] == pytest.approx([-f, 0, 0], abs=1e-14) and F[1] == pytest.approx([f, 0, 0], abs=1e-14)
    assert pe == pytest.approx(A * np.exp(-kappa * 1.5) / 1.5, rel=1e-14) and w == pytest.approx(1.5 * f, rel=1e-14)
    rng = np.random.default_rng(11)
    pos = rng.random((400, 3)) * L
    with oracle.potential(1, A, kappa):
        Fa, pea, wa = oracle.forces(pos, L, mode=2, algo=0)
        Fc, pec, wc = oracle.forces(pos, L, mode=2, algo=1)
    assert np.max(np.abs(Fa - Fc)) < 1e-11 and pec == pytest.approx(pea, rel=1e-12) and wc == pytest.approx(wa, rel=1e-12)
    assert np.max(np.abs(Fa.sum(axis=0))) < 1e-10 and np.all(Fa != 0)
    Flj, _, _ = oracle.forces(np.array([[1.0, 1.0, 1.0], [2.5, 1.0, 1.0]]), L, mode=0, algo=0)
    assert Flj[0, 0] == pytest.approx(-24 * (2 / 1.5 ** 13 - 1 / 1.5 ** 7), rel=1e-13)     # Lennard-Jones again: attracted
