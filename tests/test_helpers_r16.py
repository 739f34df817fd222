"""The R16 excuse of tests/helpers.py:check_forces, pinned on a dimer whose distance sits inside the cutoff window
(SURVEY 8(c) item 16): the only accepted deviation is that pair's own term at the cutoff, with the sign that goes
with the oracle's classification.  CPU only."""
import numpy as np
import pytest

import oracle
from helpers import check_forces

RC, L = 2.5, 10.0
F_RC = 24.0 * (2.0 / RC ** 13 - 1.0 / RC ** 7)            # f_LJ(rc) = -0.0390, attractive (Eq. 2)


def dimer(rel):
    """Two atoms along x at r = rc sqrt(1 + rel), plus a far bystander."""
    r = RC * np.sqrt(1.0 + rel)
    return np.array([[1.0, 1.0, 1.0], [1.0 + r, 1.0, 1.0], [6.0, 6.0, 6.0]])


@pytest.mark.parametrize("rel", [1e-7, -1e-7])
def test_only_the_pairs_own_cutoff_term_is_excused(rel):
    pos = dimer(rel)
    Fo, _, _ = oracle.forces(pos, L, algo=0)
    inside = rel < 0
    assert (abs(Fo[0, 0]) > 0.03) == inside
    # what a GPU path that classified the pair the other way returns: f < 0 pulls atom 0 towards +x
    flip = np.zeros_like(Fo)
    flip[0, 0], flip[1, 0] = -F_RC, F_RC
    other = Fo - flip if inside else Fo + flip
    assert check_forces(Fo.copy(), Fo, pos, L, oracle) == 0
    assert check_forces(other, Fo, pos, L, oracle) == 2
    with pytest.raises(AssertionError):                    # right size, wrong sign
        check_forces(Fo + flip if inside else Fo - flip, Fo, pos, L, oracle)
    with pytest.raises(AssertionError):                    # inside the old flat 0.04 allowance, not the pair's term
        bad = Fo.copy()
        bad[0, 1] += 0.02
        check_forces(bad, Fo, pos, L, oracle)
    with pytest.raises(AssertionError):                    # an atom with no near-cutoff partner
        bad = Fo.copy()
        bad[2, 0] += 1e-3
        check_forces(bad, Fo, pos, L, oracle)


def test_a_pair_outside_the_window_is_not_excused():
    pos = dimer(-1e-5)
    Fo, _, _ = oracle.forces(pos, L, algo=0)
    flip = np.zeros_like(Fo)
    flip[0, 0], flip[1, 0] = -F_RC, F_RC
    with pytest.raises(AssertionError):
        check_forces(Fo - flip, Fo, pos, L, oracle)
