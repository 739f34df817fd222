"""Parity of the CUDA MD path against the FP64 oracle, through the C ABI (gpu-marked).
Tolerances are BASELINE.json north_star's, read per DESIGN.md R15-R19."""
import numpy as np
import pytest

import oracle
from helpers import force_check, maxwell_boltzmann, melt, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# PE and W: every term FP64 on the all-pairs path; FP32 far-pair sums on the cell path (R23)
E_REL = {0: 1e-9, 1: 1e-6}


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


def gpu_forces(b, pos, vel, L, algo, shifted=1, eps=1.0, sigma=1.0, rc=2.5, opts=()):
    with b.Sim(pos.shape[0], L, rc=rc, eps=eps, sigma=sigma, shifted=shifted) as s:
        for k, v in opts:
            s.option(k, v)
        s.set_state(pos, vel)
        s.compute_forces(algo)
        return s.forces(), s.energies()


# (n fcc cells, rho, perturbation): several i/j tiles with ragged tails, several box sizes
CASES = [(3, 0.8, 0.08), (5, 0.8, 0.10), (6, 0.8, 0.10), (7, 0.9, 0.08), (4, 0.3, 0.15), (10, 0.8, 0.1)]


@pytest.mark.parametrize("n,rho,amp", CASES)
@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_forces_allpairs_match_oracle(b, n, rho, amp, shifted):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=100 + n)
    vel = np.zeros_like(pos)
    F, (ke, pe, w) = gpu_forces(b, pos, vel, L, b.MD_ALLPAIRS, shifted)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=1e-9, abs=1e-9)
    assert w == pytest.approx(wo, rel=1e-9, abs=1e-9)
    assert ke == 0.0


@pytest.mark.parametrize("n,rho,amp", [c for c in CASES if c[0] >= 4])
@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_forces_cell_match_oracle(b, n, rho, amp, shifted):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=100 + n)
    vel = np.zeros_like(pos)
    F, (ke, pe, w) = gpu_forces(b, pos, vel, L, b.MD_CELL, shifted)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=1)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=E_REL[1], abs=1e-9)
    assert w == pytest.approx(wo, rel=E_REL[1], abs=1e-9)


@pytest.mark.parametrize("n,rho,amp", [(6, 2.0, 0.04), (6, 1.3, 0.06), (8, 0.05, 0.3), (7, 0.8, 0.1)])
@pytest.mark.parametrize("precise_r2", [None, 0.0, 1e30])
def test_forces_cell_tiling_and_precision_modes(b, n, rho, amp, precise_r2):
    """Occupancies from < 1 to > 32 atoms per cell (several atom passes, > 512 candidates = several
    candidate passes, empty cells), with the default FP32/FP64 split, all-FP64 (precise_r2 huge,
    which also overflows the close-pair queue) and all-FP32 (precise_r2 = 0: energies only)."""
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=500 + n)
    vel = np.zeros_like(pos)
    opts = () if precise_r2 is None else (("precise_r2", precise_r2),)
    F, (ke, pe, w) = gpu_forces(b, pos, vel, L, b.MD_CELL, 1, opts=opts)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=1)
    nviol, worst = force_check(F, Fo)
    if precise_r2 == 0.0:
        assert worst < 50, worst                 # FP32 pair terms: close to, not inside, R15
    else:
        assert nviol == 0, (nviol, worst)
    rel = 1e-9 if precise_r2 == 1e30 else (1e-5 if precise_r2 == 0.0 else E_REL[1])
    assert pe == pytest.approx(peo, rel=rel, abs=1e-9)
    assert w == pytest.approx(wo, rel=rel, abs=1e-9)


@pytest.mark.parametrize("n,rho,amp", [(16, 0.3, 0.15), (14, 0.1, 0.3), (13, 0.8, 0.1)])
@pytest.mark.parametrize("kz", [1, 2, 3, 4, 5])
def test_forces_cell_row_groups(b, n, rho, amp, kz):
    """Row groups of kz cells per warp (option "cell_group"): same forces for every kz, including
    groups that touch the periodic seam in z and the ragged last group of a column."""
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=900 + n)
    vel = np.zeros_like(pos)
    F, (ke, pe, w) = gpu_forces(b, pos, vel, L, b.MD_CELL, 1, opts=(("cell_group", kz),))
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=1)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


@pytest.mark.parametrize("n,rho,amp", [(7, 0.9, 0.08), (10, 0.8, 0.1), (12, 0.8, 0.1), (16, 0.5, 0.12)])
@pytest.mark.parametrize("R", [1, 2, 4, 8])
def test_allpairs_sorted_kernel_matches_general_and_oracle(b, n, rho, amp, R):
    """The Hilbert-sorted, pre-shifted 3-FFMA filter kernel (R atoms per thread) against the
    unsorted per-pair minimum-image kernel and the oracle: ragged last block, several j
    splits, and (large R in a small box) blocks too wide to pre-shift, which must fall back
    to per-pair minimum images inside the kernel."""
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=300 + n)
    vel = np.zeros_like(pos)
    with b.Sim(pos.shape[0], L) as s:
        s.option("ap_R", R)
        assert s.stat("ap_tiled") == 1 and s.stat("ap_R") == R
        s.set_state(pos, vel)
        s.compute_forces(b.MD_ALLPAIRS)
        Ft, et = s.forces(), s.energies()
        s.option("ap_general", 1)
        s.set_state(pos, vel)
        s.compute_forces(b.MD_ALLPAIRS)
        Fg, eg = s.forces(), s.energies()
    assert np.max(np.abs(Ft.astype(np.float64) - Fg)) <= 1e-6 * max(1.0, np.max(np.abs(Fg)))
    assert et[1] == pytest.approx(eg[1], rel=1e-12) and et[2] == pytest.approx(eg[2], rel=1e-12)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=1)
    assert force_check(Ft, Fo)[0] == 0
    assert et[1] == pytest.approx(peo, rel=1e-9) and et[2] == pytest.approx(wo, rel=1e-9)


def test_allpairs_default_plan_uses_sorted_kernel_when_box_allows(b):
    for n, want in ((5, 0), (10, 1), (20, 1)):
        pos, L = wl.fcc_positions(n, 0.8)
        with b.Sim(pos.shape[0], L) as s:
            assert s.stat("ap_tiled") == want, n
            if n == 20:
                assert s.stat("ap_R") == 8


def test_allpairs_tiled_after_drift_without_resort(b, oracle_uniforms):
    """Between re-sorts atoms leave their tile (and cross the periodic seam): the per-block
    bounding box check must keep the result exact."""
    pos, L = wl.fcc_positions(10, 0.8)
    vel = maxwell_boltzmann(oracle_uniforms(wl.splitmix64(5) & wl.MASK48, 6 * 4000), 4000, 2.0)
    with b.Sim(4000, L) as s:
        s.option("ap_R", 2)
        s.option("sort_every", 1000)
        s.set_state(pos, vel)
        s.step(300, b.MD_ALLPAIRS)
        F = s.forces()
        p, v = s.get_state()
    Fo, _, _ = oracle.forces(p.astype(np.float64), L, algo=1)
    assert force_check(F, Fo)[0] == 0


def test_eps_sigma_not_one(b):
    pos, L = wl.perturbed_fcc(5, 0.8, 0.1, seed=9)
    sig, eps = 1.3, 0.7
    p2 = (pos.astype(np.float64) * sig).astype(np.float32)
    L2 = float(np.float32(L * sig))
    p2[p2 >= np.float32(L2)] = 0
    for algo in (0, 1):
        F, (_, pe, w) = gpu_forces(b, p2, np.zeros_like(p2), L2, algo, 1, eps, sig, 2.5 * sig)
        Fo, peo, wo = oracle.forces(p2.astype(np.float64), L2, 2.5 * sig, eps, sig, 1, algo)
        assert force_check(F, Fo)[0] == 0
        assert pe == pytest.approx(peo, rel=E_REL[algo]) and w == pytest.approx(wo, rel=E_REL[algo])


def test_perfect_lattice_forces_vanish(b):
    pos, L = wl.fcc_positions(5, 0.8)
    for algo in (0, 1):
        F, (_, pe, w) = gpu_forces(b, pos, np.zeros_like(pos), L, algo)
        assert np.max(np.abs(F)) < 2e-5
        assert pe / 500 == pytest.approx(-5.924190441386, abs=2e-6)


def test_state_roundtrip_and_atom_order(b):
    pos, L = wl.perturbed_fcc(6, 0.8, 0.1, seed=4)
    rng = np.random.default_rng(0)
    vel = rng.standard_normal(pos.shape).astype(np.float32)
    with b.Sim(pos.shape[0], L) as s:
        s.set_state(pos, vel)
        p, v = s.get_state()
        assert np.array_equal(p, pos) and np.array_equal(v, vel)
        s.compute_forces(b.MD_CELL)                     # reorders internally
        p, v = s.get_state()
        assert np.array_equal(p, pos) and np.array_equal(v, vel)
        Fc = s.forces()
        s.compute_forces(b.MD_ALLPAIRS)
        Fa = s.forces()
        assert np.max(np.abs(Fc.astype(np.float64) - Fa)) < 1e-5 * max(1.0, np.max(np.abs(Fa)))
        assert s.stat("ncell") == 3 or s.stat("ncell") == int(L / 2.5)


def test_set_state_wraps_positions(b):
    pos, L = wl.perturbed_fcc(4, 0.8, 0.1, seed=4)
    shifted = pos.astype(np.float64) + np.array([L, -2 * L, 3 * L])
    with b.Sim(pos.shape[0], L) as s:
        s.set_state(shifted.astype(np.float32), np.zeros_like(pos))
        p, _ = s.get_state()
        assert np.all((p >= 0) & (p < np.float32(L)))


def test_error_codes(b):
    pos, L = wl.perturbed_fcc(3, 0.8, 0.05, seed=4)     # L = 5.13: int[L/rc] = 2
    with b.Sim(pos.shape[0], L) as s:
        for fn in (lambda: s.step(1, 0), lambda: s.forces(), lambda: s.energies(), lambda: s.compute_forces(0)):
            with pytest.raises(b.MDError) as e:
                fn()
            assert e.value.code == b.MD_ESTATE
        s.set_state(pos, np.zeros_like(pos))
        with pytest.raises(b.MDError) as e:
            s.forces()
        assert e.value.code == b.MD_ESTATE               # stale
        with pytest.raises(b.MDError) as e:
            s.compute_forces(b.MD_CELL)
        assert e.value.code == b.MD_EDOMAIN
        with pytest.raises(b.MDError) as e:
            s.step(1, 5)
        assert e.value.code == b.MD_EINVAL
        s.step(0, 0)
        s.forces()


@pytest.fixture(scope="module")
def c1(oracle_uniforms):
    return wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))


@pytest.mark.parametrize("algo", [0, 1])
def test_config1_energy_trace_100_steps(b, c1, algo):
    """Per-step total energy within 1e-5 relative of the oracle over 100 steps (R17)."""
    _, _, _, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 100, algo=algo)
    with b.Sim(c1["N"], c1["L"]) as s:
        s.set_state(c1["pos"], c1["vel"])
        s.compute_forces(algo)
        worst = 0.0
        for t in range(101):
            if t:
                s.step(1, algo)
            ke, pe, w = s.energies()
            Eo = tr[t, 0] + tr[t, 1]
            worst = max(worst, abs(ke + pe - Eo) / abs(Eo))
            assert ke == pytest.approx(tr[t, 0], rel=2e-4) and pe == pytest.approx(tr[t, 1], rel=2e-4)
        assert worst < 1e-5, worst
        # forces on the melted state, from the identical FP32 snapshot
        p, v = s.get_state()
        s.set_state(p, v)
        s.compute_forces(algo)
        Fo, _, _ = oracle.forces(p.astype(np.float64), c1["L"], algo=algo)
        assert force_check(s.forces(), Fo)[0] == 0


def test_multi_step_equals_single_steps(b, c1):
    out = []
    for chunks in ([20], [1] * 20, [7, 13]):
        with b.Sim(c1["N"], c1["L"]) as s:
            s.set_state(c1["pos"], c1["vel"])
            for c in chunks:
                s.step(c, 0)
            out.append((s.get_state(), s.energies()))
    # the counting sort's atomic ranks make the summation order run-dependent: equal up to rounding
    for (p, v), e in out[1:]:
        assert np.max(np.abs(p - out[0][0][0])) < 1e-5 and np.max(np.abs(v - out[0][0][1])) < 1e-4
        assert e == pytest.approx(out[0][1], rel=1e-7)


def test_time_reversibility(b, c1):
    with b.Sim(c1["N"], c1["L"]) as s:
        s.set_state(c1["pos"], c1["vel"])
        s.step(100, 0)
        p, v = s.get_state()
        s.set_state(p, -v)
        s.step(100, 0)
        p2, v2 = s.get_state()
    d = p2.astype(np.float64) - c1["pos"]
    d -= c1["L"] * np.rint(d / c1["L"])
    assert np.max(np.abs(d)) < 1e-3                      # R19: FP32 returns to ~1e-4


def test_melted_snapshot_n4000(b, oracle_uniforms):
    """Forces on a melted N = 4000 snapshot (pair forces up to ~70), both algos."""
    pos, L = wl.fcc_positions(10, 0.8)
    x0 = wl.splitmix64(77) & wl.MASK48
    vel = maxwell_boltzmann(oracle_uniforms(x0, 6 * 4000), 4000, 1.0)
    with b.Sim(4000, L) as s:
        s.set_state(pos, vel)
        s.step(400, b.MD_CELL)
        p, v = s.get_state()
        Fo, peo, wo = oracle.forces(p.astype(np.float64), L, algo=1)
        assert np.max(np.abs(Fo)) > 30
        for algo in (0, 1):
            s.set_state(p, v)
            s.compute_forces(algo)
            nviol, worst = force_check(s.forces(), Fo)
            assert nviol == 0, (algo, nviol, worst)
            ke, pe, w = s.energies()
            assert pe == pytest.approx(peo, rel=E_REL[algo]) and w == pytest.approx(wo, rel=E_REL[algo])
            assert ke == pytest.approx(oracle.kinetic_energy(v.astype(np.float64)), rel=1e-9)


@pytest.mark.parametrize("algo,opts,nsteps", [(1, (), 25), (0, (("sort_every", 2),), 31), (0, (), 64)])
def test_graph_replay_equals_direct_launches(b, c1, algo, opts, nsteps):
    """Interior steps replayed from a CUDA graph ("graph" = 1, default) against direct launches."""
    out = []
    for graph in (1, 0):
        with b.Sim(c1["N"], c1["L"]) as s:
            for k, v in opts + (("graph", graph),):
                s.option(k, v)
            s.set_state(c1["pos"], c1["vel"])
            s.step(nsteps, algo)
            s.step(nsteps, algo)                         # second call: cached graph, other buffer parity
            assert (s.stat("graph_replays") > 0) == bool(graph)
            out.append((s.get_state(), s.energies(), s.stat("kernel_launches")))
    (p1, v1), e1, l1 = out[0]
    (p0, v0), e0, l0 = out[1]
    assert l1 == l0                                      # same kernels, launched or replayed
    # the counting sort's atomic ranks make the summation order run-dependent: equal up to rounding
    assert np.max(np.abs(p1 - p0)) < 1e-5 and np.max(np.abs(v1 - v0)) < 1e-4
    assert e1 == pytest.approx(e0, rel=2e-6)             # the virial is the most sensitive of the three


@pytest.mark.parametrize("algo", [0, 1, 2])
def test_user_stream_with_graph_replay(b, c1, algo):
    """md_set_stream with a non-default (non-blocking) stream: graphs are captured on that stream itself."""
    import torch
    ref = None
    for use_stream in (False, True):
        with b.Sim(c1["N"], c1["L"]) as s:
            if use_stream:
                st = torch.cuda.Stream()
                b.md_set_stream(s.h, st.cuda_stream)
            s.set_state(c1["pos"], c1["vel"])
            s.step(40, algo)
            s.step(40, algo)
            assert s.stat("graph_replays") > 0
            res = (s.get_state(), s.energies())
            if use_stream:
                b.md_set_stream(s.h, 0)
        if ref is None:
            ref = res
    d = res[0][0] - ref[0][0]
    d -= c1["L"] * np.rint(d / c1["L"])
    assert np.max(np.abs(d)) < 5e-5 and res[1][0] + res[1][1] == pytest.approx(ref[1][0] + ref[1][1], rel=1e-6)


@pytest.mark.parametrize("kernel", [2, 3])
def test_deterministic_option_gives_bit_identical_reruns(b, kernel, oracle_uniforms):
    """Option "deterministic": cells re-ordered by atom id after every build, so that two runs of the cell path sum
    every force in the same order.  60 steps at N = 4,000 from a hot lattice, twice: positions, velocities, forces and
    energies equal bit for bit (the steps in between go through the CUDA graph), and the forces are the oracle's."""
    pos, L = wl.fcc_positions(10, 0.8)
    vel = maxwell_boltzmann(oracle_uniforms(0xD37E12A1, 6 * pos.shape[0]), pos.shape[0], 2.0)
    runs = []
    for _ in range(2):
        with b.Sim(pos.shape[0], L) as s:
            s.option("cell_kernel", kernel)
            s.option("deterministic", 1)
            s.set_state(pos, vel)
            s.step(60, b.MD_CELL)
            runs.append((s.get_state(), s.forces(), s.energies()))
    (p0, v0), F0, e0 = runs[0]
    (p1, v1), F1, e1 = runs[1]
    assert np.array_equal(p0, p1) and np.array_equal(v0, v1) and np.array_equal(F0, F1) and e0 == e1
    Fo, peo, wo = oracle.forces(p0.astype(np.float64), L, algo=1)
    assert force_check(F0, Fo)[0] == 0
    assert e0[1] == pytest.approx(peo, rel=E_REL[1]) and e0[2] == pytest.approx(wo, rel=E_REL[1])
