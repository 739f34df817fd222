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
