"""Degenerate and extreme inputs through the C ABI against the oracle (gpu-marked): one atom, a dimer
across the periodic seam, every atom in one cell (hundreds of filter-row passes, empty cells
elsewhere), atoms on cell faces and on the box boundary, zero-length rand48 requests."""
import numpy as np
import pytest

import oracle
from helpers import force_check
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


def both_paths(b, pos, L, shifted=1, opts=()):
    pos = np.asarray(pos, dtype=np.float32)
    vel = np.zeros_like(pos)
    res = []
    for algo in (b.MD_ALLPAIRS, b.MD_CELL):
        with b.Sim(pos.shape[0], L, shifted=shifted) as s:
            for k, v in opts:
                s.option(k, v)
            s.set_state(pos, vel)
            s.compute_forces(algo)
            res.append((s.forces(), s.energies()))
    return res


def test_single_atom_has_no_force(b):
    for F, (ke, pe, w) in both_paths(b, [[1.0, 2.0, 3.0]], 10.0):
        assert np.all(F == 0) and ke == 0 and pe == 0 and w == 0


@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_dimer_across_the_seam(b, shifted):
    L = 20.0
    pos = np.array([[0.3, 10.0, 19.9], [19.6, 10.2, 0.4]], dtype=np.float32)      # r ~ 0.88: strongly repulsive
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    assert abs(Fo[0, 0]) > 10
    for F, (ke, pe, w) in both_paths(b, pos, L, shifted):
        assert force_check(F, Fo)[0] == 0
        assert pe == pytest.approx(peo, rel=1e-9) and w == pytest.approx(wo, rel=1e-9)
        assert np.allclose(F[0], -F[1], rtol=0, atol=1e-5)                       # Newton's third law


@pytest.mark.parametrize("kz", [0, 1, 3])
def test_all_atoms_in_one_cell(b, kz):
    """600 atoms on a jittered lattice inside one cell of a 12-cell box: 38 row passes, 2 candidate
    passes, every other cell empty."""
    rng = np.random.default_rng(11)
    g = np.stack(np.meshgrid(np.arange(10), np.arange(10), np.arange(6), indexing="ij"), -1).reshape(-1, 3)
    pos = (15.2 + 0.24 * g + 0.02 * rng.random(g.shape)).astype(np.float32)       # spacing 0.24: huge forces
    pos = 15.2 + (pos - 15.2) * 4.0                                                # spacing 0.96 sigma
    pos = pos.astype(np.float32)
    L = 30.5
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=0)
    for F, (ke, pe, w) in both_paths(b, pos, L, opts=(("cell_group", kz),)):
        assert force_check(F, Fo)[0] == 0
        assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


def test_atoms_on_cell_faces_and_box_boundary(b):
    """Coordinates exactly 0, exactly on multiples of the cell side, and the largest float below L."""
    L = 25.0
    with b.Sim(7, L) as s:
        side = s.stat("side")
    top = np.nextafter(np.float32(L), np.float32(0))
    pos = np.array([[0, 0, 0], [top, 1.0, 0.5], [side, 2 * side, 3 * side], [side - 1.0, 2 * side, 3 * side],
                    [side, 2 * side + 1.05, 3 * side], [0.0, top, 1.1], [1.0, 0.0, top]], dtype=np.float32)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), float(np.float32(L)), algo=0)
    for F, (ke, pe, w) in both_paths(b, pos, L):
        assert force_check(F, Fo)[0] == 0
        assert pe == pytest.approx(peo, rel=1e-6)


def test_rand48_zero_sized_requests(b):
    out, seeds = b.rand48([0x1234ABCD330E], 0, b.R48_U32_HI32)
    assert out.shape == (1, 0) and int(seeds[0]) == 0x1234ABCD330E


def test_morton_numbering_survives_a_later_grid_option(b):
    """"skin" / "cell_skin" rebuild the cell grids; the numbering chosen with "cell_order" must stay in force
    (a bench line labelled Morton would otherwise measure the linear numbering), with the oracle's forces."""
    pos, L = wl.perturbed_fcc(8, 0.8, 0.1, seed=31)
    Fo, _, _ = oracle.forces(pos.astype(np.float64), L, algo=0)
    with b.Sim(pos.shape[0], L) as s:
        n = int(s.stat("ncell"))
        s.option("cell_order", 1)
        assert s.stat("cell_order") == 1 and s.stat("cell_ids") == 8 ** 3 and n ** 3 < 8 ** 3
        s.option("skin", 0.4)
        assert s.stat("cell_order") == 1 and s.stat("cell_ids") == 8 ** 3
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_CELL)
        assert force_check(s.forces(), Fo)[0] == 0
        s.step(4, b.MD_CELL)
        s.option("cell_order", 0)
        assert s.stat("cell_order") == 0 and s.stat("cell_ids") == n ** 3
        s.compute_forces(b.MD_CELL)
        p, _ = s.get_state()
        Fo2, _, _ = oracle.forces(p.astype(np.float64), L, algo=0)
        assert force_check(s.forces(), Fo2)[0] == 0


def test_md_create_sizes_the_cell_arrays_for_the_linear_numbering(b):
    """A sparse box of 260 cells per side: 2 x 70 MB of cell arrays (plus 430 MB of per-row energy partials), not
    the 2 x 537 MB of the padded Morton cube (512^3 ids), which is allocated only when "cell_order" = 1 asks for it."""
    import torch
    L = 2.5 * 260 + 1.0
    pos = (np.random.default_rng(5).random((1000, 3)) * L).astype(np.float32)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    with b.Sim(pos.shape[0], L) as s:
        assert s.stat("ncell") == 260
        used = torch.cuda.memory_allocated() - before
        assert used < 700e6, used
        s.option("cell_order", 1)
        assert torch.cuda.memory_allocated() - before > 1400e6
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_CELL)
        F3 = s.forces()
    Fo, _, _ = oracle.forces(pos.astype(np.float64), L, algo=0)
    assert force_check(F3, Fo)[0] == 0
