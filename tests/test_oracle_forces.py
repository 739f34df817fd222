"""Pins for oracle forces_allpairs (O2) and forces_cell (O3).
PAPER.md:49-52 (Eq. 1), :98, :108, :130, :134; readings R3, R6, R12, R14."""
import math

import numpy as np
import pytest

import oracle
from conftest import golden_lines
from paper_0709_3225_b200 import workloads as wl


def fcc_f64(n, rho):
    """Perfect fcc lattice in FP64 (no FP32 rounding of box or positions)."""
    N = 4 * n ** 3
    L = (N / rho) ** (1.0 / 3.0)
    pos, _ = wl.fcc_positions(n, rho)
    a32 = wl.box_length(N, rho) / n
    return (pos.astype(np.float64) / a32 * 4).round() / 4 * (L / n), L   # exact multiples of a/4


def test_dimer_by_hand():
    L = 20.0
    for r, mode in [(1.0, 1), (1.3, 0), (2.0, 2), (2.49, 1)]:
        pos = np.array([[5.0, 5.0, 5.0], [5.0 + r, 5.0, 5.0]])
        F, pe, w = oracle.forces(pos, L, mode=mode)
        _, u, fr = oracle.lj_pair(mode, r * r)
        f = fr * r
        # Eq. 1: F_i = -f (r_j - r_i)/r; f > 0 pushes atom 0 towards -x
        assert F[0] == pytest.approx([-f, 0, 0], abs=1e-12)
        assert F[1] == pytest.approx([+f, 0, 0], abs=1e-12)
        assert pe == pytest.approx(u, abs=1e-13)
        assert w == pytest.approx(r * f, abs=1e-12)
    F, pe, w = oracle.forces(np.array([[1.0, 1, 1], [3.5, 1, 1]]), L)
    assert np.all(F == 0) and pe == 0 and w == 0          # r = rc exactly: outside


def test_dimer_across_the_seam():
    L = 10.0
    pos = np.array([[0.2, 5.0, 9.9], [9.5, 5.0, 0.3]])      # image distance (-0.7, 0, 0.4)
    F, pe, _ = oracle.forces(pos, L, mode=0)
    r2 = 0.7 ** 2 + 0.4 ** 2
    _, u, fr = oracle.lj_pair(0, r2)
    assert F[0] == pytest.approx([-fr * -0.7, 0.0, -fr * 0.4], rel=1e-11)
    assert pe == pytest.approx(u, rel=1e-12)


def test_equilateral_trimer_by_hand():
    r = 1.05
    pos = np.array([[4.0, 4.0, 4.0], [4.0 + r, 4.0, 4.0], [4.0 + r / 2, 4.0 + r * math.sqrt(3) / 2, 4.0]])
    F, pe, w = oracle.forces(pos, 12.0, mode=1)
    _, u, fr = oracle.lj_pair(1, r * r)
    f = fr * r
    # atom 2 is pushed along +y by both neighbours: 2 f cos(30 deg)
    assert F[2] == pytest.approx([0.0, 2 * f * math.cos(math.pi / 6), 0.0], abs=1e-10)
    assert pe == pytest.approx(3 * u, rel=1e-12)
    assert w == pytest.approx(3 * r * f, rel=1e-12)


def brute_numpy(pos, L, rc, eps, sigma, mode):
    """Independent N x N matrix formulation (different loop structure from the C code)."""
    d = pos[None, :, :] - pos[:, None, :]                  # d[i,j] = r_j - r_i
    d -= L * np.rint(d / L)
    r2 = np.sum(d * d, axis=-1)
    np.fill_diagonal(r2, np.inf)
    r = np.sqrt(r2)
    flj = lambda x: 24 * eps / sigma * (2 * (sigma / x) ** 13 - (sigma / x) ** 7)
    ulj = lambda x: 4 * eps * ((sigma / x) ** 12 - (sigma / x) ** 6)
    inside = r < rc
    f = np.where(inside, flj(r), 0.0)
    u = np.where(inside, ulj(r), 0.0)
    if mode >= 1:
        u = np.where(inside, u - ulj(rc), 0.0)
    if mode == 2:
        f = np.where(inside, f - flj(rc), 0.0)
        u = np.where(inside, u + (r - rc) * flj(rc), 0.0)
    with np.errstate(invalid="ignore"):
        F = -np.sum(np.where(inside[..., None], f[..., None] * d / r[..., None], 0.0), axis=1)
        w = 0.5 * np.sum(np.where(inside, f * r, 0.0))
    return F, 0.5 * np.sum(u), w


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("eps,sig", [(1.0, 1.0), (1.3, 0.8)])
def test_brute_force_small(mode, eps, sig):
    pos, L = wl.perturbed_fcc(3, 0.8, 0.08, seed=11)        # N = 108, L = 5.13 > 2 rc
    pos = pos.astype(np.float64) * sig
    L, rc = L * sig, 2.5 * sig
    Fb, peb, wb = brute_numpy(pos, L, rc, eps, sig, mode)
    F, pe, w = oracle.forces(pos, L, rc, eps, sig, mode, 0)
    assert np.max(np.abs(F - Fb)) < 1e-10 * max(1.0, np.max(np.abs(Fb)))
    assert pe == pytest.approx(peb, rel=1e-12)
    assert w == pytest.approx(wb, rel=1e-12)


def test_newton_third_law_and_translation():
    pos, L = wl.perturbed_fcc(5, 0.8, 0.1, seed=3)
    pos = pos.astype(np.float64)
    F, pe, w = oracle.forces(pos, L)
    assert np.max(np.abs(F)) > 10
    assert np.max(np.abs(F.sum(axis=0))) < 1e-10            # sum F = 0
    shift = np.array([0.37 * L, -1.91 * L, 5.123])
    p2 = pos + shift
    p2 -= L * np.floor(p2 / L)
    F2, pe2, w2 = oracle.forces(p2, L)
    assert np.max(np.abs(F2 - F)) < 1e-8
    assert pe2 == pytest.approx(pe, rel=1e-11) and w2 == pytest.approx(w, rel=1e-11)


def test_scale_invariance():
    # F(eps, sigma; x) = (eps/sigma) F(1, 1; x/sigma) with L, rc scaled by sigma (R1)
    pos, L = wl.perturbed_fcc(4, 0.8, 0.1, seed=5)
    pos = pos.astype(np.float64)
    eps, sig = 1.9, 1.35
    for mode in (0, 1, 2):
        F1, pe1, w1 = oracle.forces(pos, L, 2.5, 1.0, 1.0, mode)
        F2, pe2, w2 = oracle.forces(pos * sig, L * sig, 2.5 * sig, eps, sig, mode)
        assert np.max(np.abs(F2 - (eps / sig) * F1)) < 1e-9 * np.max(np.abs(F1))
        assert pe2 == pytest.approx(eps * pe1, rel=1e-11)
        assert w2 == pytest.approx(eps * w1, rel=1e-11)


def shell_sum(rho, mode):
    """Textbook fcc coordination shells: n_k neighbours at a*sqrt(k/2), k = 1.."""
    a = (4.0 / rho) ** (1.0 / 3.0)
    shells = [(12, 1), (6, 2), (24, 3), (12, 4), (24, 5), (8, 6), (48, 7), (6, 8)]
    pe = w = 0.0
    for n_k, k in shells:
        r = a * math.sqrt(k / 2.0)
        inside, u, fr = oracle.lj_pair(mode, r * r)
        pe += 0.5 * n_k * u
        w += 0.5 * n_k * fr * r * r
    return pe, w


@pytest.mark.parametrize("row", golden_lines("fcc_lattice_sums.txt"))
def test_fcc_lattice_sums(row):
    rho, mode, pe_ref, w_ref = float(row[0]), int(row[1]), float(row[2]), float(row[3])
    pe_s, w_s = shell_sum(rho, mode)
    assert pe_s == pytest.approx(pe_ref, abs=1e-11)
    assert w_s == pytest.approx(w_ref, abs=1e-11)
    n = 5 if rho == 0.8 else 4                              # L = 8.55 / 9.48: >= 3 cells
    pos, L = fcc_f64(n, rho)
    N = pos.shape[0]
    for algo in (0, 1):
        F, pe, w = oracle.forces(pos, L, mode=mode, algo=algo)
        assert np.max(np.abs(F)) < 1e-11                    # zero by symmetry
        assert pe / N == pytest.approx(pe_ref, abs=1e-11)
        assert w / N == pytest.approx(w_ref, abs=1e-10)


def test_fcc_neighbour_count():
    # 54 neighbours within rc at rho = 0.8, 18 at rho = 0.3
    for rho, n, want in [(0.8, 5, 54), (0.3, 4, 18)]:
        pos, L = fcc_f64(n, rho)
        d = pos[1:] - pos[0]
        d -= L * np.rint(d / L)
        assert int(np.sum(np.sum(d * d, axis=1) < 6.25)) == want


@pytest.mark.parametrize("n,rho,amp", [(5, 0.8, 0.1), (6, 0.8, 0.1), (4, 0.3, 0.2), (7, 0.3, 0.2), (9, 1.0, 0.08)])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_cell_list_agrees_with_allpairs(n, rho, amp, mode):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=17 + n)
    pos = pos.astype(np.float64)
    ncell, side, ok = oracle.cell_grid(L, 2.5)
    assert ok and ncell >= 3
    Fa, pea, wa = oracle.forces(pos, L, mode=mode, algo=0)
    Fc, pec, wc = oracle.forces(pos, L, mode=mode, algo=1)
    assert np.max(np.abs(Fa - Fc)) < 1e-12 * max(1.0, np.max(np.abs(Fa)))
    assert pec == pytest.approx(pea, rel=1e-12) and wc == pytest.approx(wa, rel=1e-12)


def test_cell_grid_paper_example():
    # L_x = 11, rc = 2.5 -> n_x = int[4.4] = 4, side 2.75
    ncell, side, ok = oracle.cell_grid(11.0, 2.5)
    assert (ncell, ok) == (4, True) and side == pytest.approx(2.75, abs=1e-15)
    # +10 % side -> +33 % atoms per cell -> +77 % interactions
    assert (side / 2.5) ** 3 == pytest.approx(1.331) and (side / 2.5) ** 6 == pytest.approx(1.77, abs=2e-3)
    # at least 3 cells per dimension
    assert oracle.cell_grid(7.4, 2.5)[2] is False
    assert oracle.cell_grid(7.5, 2.5)[0] == 3
    with pytest.raises(ValueError):
        oracle.forces(np.array([[1.0, 1, 1], [2.2, 1, 1]]), 7.4, algo=1)


def test_cell_list_atoms_on_cell_faces_and_box_edge():
    # atoms exactly on cell faces / at 0 / just below L must not be lost or double counted (R14)
    L = 10.0
    pos = np.array([[0.0, 0.0, 0.0], [2.5, 2.5, 2.5], [np.nextafter(10.0, 0), 0.5, 9.2],
                    [5.0, 7.5, 0.9], [1.0, 0.6, 0.1], [9.3, 9.9, 9.4], [3.4, 2.6, 2.0]])
    Fa, pea, wa = oracle.forces(pos, L, mode=1, algo=0)
    Fc, pec, wc = oracle.forces(pos, L, mode=1, algo=1)
    assert np.max(np.abs(Fa - Fc)) < 1e-12 and pec == pytest.approx(pea, rel=1e-13)


def test_near_cutoff_pairs():
    pos = np.array([[1.0, 1.0, 1.0], [3.5 - 1e-7, 1.0, 1.0], [1.0, 3.0, 1.0]])
    pairs, n = oracle.near_cutoff_pairs(pos, 12.0, tol=4e-7)
    assert n == 2 and sorted(map(tuple, pairs)) == [(0, 1), (1, 0)]


def test_near_cutoff_pairs_cell_lists_the_same_pairs():
    """The linked-cell lister against the O(N^2) one: a fluid-like system with a wide window (so that the
    lists are long), a pair planted across the periodic seam exactly in the window, and the 3-cell box."""
    rng = np.random.default_rng(5)
    for L, N, tol in ((12.0, 900, 2e-3), (7.6, 300, 5e-3)):
        pos = rng.random((N, 3)) * L
        pos[0] = (0.05, 3.0, 3.0)
        pos[1] = (L - 2.45 + 1e-7, 3.0, 3.0)             # r = 2.5 - 1e-7 through the seam
        a, na = oracle.near_cutoff_pairs(pos, L, tol=tol)
        c, nc = oracle.near_cutoff_pairs_cell(pos, L, tol=tol)
        assert na == nc and na > 20
        assert sorted(map(tuple, a)) == sorted(map(tuple, c))
        assert (0, 1) in set(map(tuple, c)) and (1, 0) in set(map(tuple, c))
    with pytest.raises(ValueError):
        oracle.near_cutoff_pairs_cell(rng.random((10, 3)) * 6.0, 6.0)
