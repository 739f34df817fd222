"""The neighbour-list path (algo = MD_VERLET) against the FP64 oracle and against
the cell path (gpu-marked).  Same tolerances as the other two force paths (R15, R17)."""
import numpy as np
import pytest

import oracle
from helpers import check_forces, force_check, maxwell_boltzmann, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


@pytest.fixture(scope="module")
def c1(oracle_uniforms):
    return wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))


@pytest.mark.parametrize("n,rho,amp", [(5, 0.8, 0.10), (6, 0.8, 0.10), (7, 0.9, 0.08), (5, 0.3, 0.15), (10, 0.8, 0.1),
                                       (8, 0.05, 0.3), (6, 1.3, 0.06)])
@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_forces_match_oracle(b, n, rho, amp, shifted):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=300 + n)
    vel = np.zeros_like(pos)
    with b.Sim(pos.shape[0], L, shifted=shifted) as s:
        s.set_state(pos, vel)
        s.compute_forces(b.MD_VERLET)
        F, (ke, pe, w) = s.forces(), s.energies()
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


def test_config1_energy_trace_and_list_reuse(b, c1):
    """Per-step total energy within 1e-5 of the oracle over 100 steps (R17) while the lists are reused."""
    _, _, _, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 100, algo=0)
    with b.Sim(c1["N"], c1["L"]) as s:
        s.set_state(c1["pos"], c1["vel"])
        s.compute_forces(b.MD_VERLET)
        worst = 0.0
        for t in range(101):
            if t:
                s.step(1, b.MD_VERLET)
            ke, pe, w = s.energies()
            Eo = tr[t, 0] + tr[t, 1]
            worst = max(worst, abs(ke + pe - Eo) / abs(Eo))
        assert worst < 1e-5, worst
        builds, evals = s.stat("vl_builds"), s.stat("vl_steps")
        assert evals == 101 and 3 <= builds <= 40, (builds, evals)       # reused, and rebuilt when atoms moved
        p, v = s.get_state()
        F = s.forces()
        Fo, _, _ = oracle.forces(p.astype(np.float64), c1["L"], algo=0)
        assert force_check(F, Fo)[0] == 0                                 # forces from a list several steps old


def test_multi_step_and_graph_equal_single_steps_and_cell_path(b, c1):
    out = []
    for algo, chunks, graph in ((b.MD_VERLET, [60], 1), (b.MD_VERLET, [1] * 60, 1), (b.MD_VERLET, [60], 0), (b.MD_CELL, [60], 1)):
        with b.Sim(c1["N"], c1["L"]) as s:
            s.option("graph", graph)
            s.set_state(c1["pos"], c1["vel"])
            for c in chunks:
                s.step(c, algo)
            out.append((s.get_state(), s.energies()))
    for (p, v), e in out[1:]:
        d = p - out[0][0][0]
        d -= c1["L"] * np.rint(d / c1["L"])
        assert np.max(np.abs(d)) < 2e-5 and np.max(np.abs(v - out[0][0][1])) < 2e-4
        assert e[0] + e[1] == pytest.approx(out[0][1][0] + out[0][1][1], rel=1e-6)


def test_switching_paths_between_calls(b, c1):
    with b.Sim(c1["N"], c1["L"]) as s:
        s.set_state(c1["pos"], c1["vel"])
        s.step(15, b.MD_VERLET)
        s.step(7, b.MD_CELL)
        s.step(9, b.MD_ALLPAIRS)
        s.step(15, b.MD_VERLET)
        p, v = s.get_state()
        F = s.forces()
        ke, pe, w = s.energies()
    Fo, peo, wo = oracle.forces(p.astype(np.float64), c1["L"], algo=0)
    assert force_check(F, Fo)[0] == 0 and pe == pytest.approx(peo, rel=1e-6)


def test_skin_option_and_domain_errors(b):
    pos, L = wl.perturbed_fcc(6, 0.8, 0.1, seed=3)
    Fo, _, _ = oracle.forces(pos.astype(np.float64), L, algo=0)
    for skin in (0.1, 0.6):
        with b.Sim(pos.shape[0], L) as s:
            s.option("skin", skin)
            s.set_state(pos, np.zeros_like(pos))
            s.compute_forces(b.MD_VERLET)
            assert force_check(s.forces(), Fo)[0] == 0
            with pytest.raises(b.MDError):
                s.option("skin", 0.2)                  # lists exist
    with b.Sim(100, 8.0) as s:                         # int[8 / 2.8] = 2 cells: no neighbour-list path
        s.set_state(np.random.default_rng(1).random((100, 3)).astype(np.float32) * 8, np.zeros((100, 3), np.float32))
        with pytest.raises(b.MDError) as e:
            s.compute_forces(b.MD_VERLET)
        assert e.value.code == b.MD_EDOMAIN


def test_list_overflow_grows_the_lists(b):
    """600 atoms inside one cell of a sparse box: lists far longer than the initial capacity.  They are never
    truncated: the evaluation reallocates them for the length the build asked for and
    rebuilds, and the forces are the oracle's."""
    g = np.stack(np.meshgrid(np.arange(10), np.arange(10), np.arange(6), indexing="ij"), -1).reshape(-1, 3)
    pos = (15.2 + 0.9 * g).astype(np.float32)
    L = 45.5
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=0)
    with b.Sim(pos.shape[0], L) as s:
        s.set_state(pos, np.zeros_like(pos))
        cap0 = None
        s.compute_forces(b.MD_VERLET)
        assert s.stat("vl_overflow") == 0 and s.stat("vl_cap") >= 80
        assert force_check(s.forces(), Fo)[0] == 0
        _, pe, w = s.energies()
        assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)
        s.step(3, b.MD_VERLET)                          # and the step loop runs on the enlarged lists
        assert s.stat("vl_overflow") == 0
    # the same through md_step's own first evaluation (stale forces)
    with b.Sim(pos.shape[0], L) as s:
        s.set_state(pos, np.zeros_like(pos))
        s.step(0, b.MD_VERLET)
        assert force_check(s.forces(), Fo)[0] == 0


@pytest.mark.parametrize("name,steps", [("c3_cell_256k", 1000), ("c4a_cell_2048k", 500), ("c4b_cell_2048k_rho03", 500)])
def test_full_size_parity(b, name, steps):
    import os
    oracle.set_threads(os.cpu_count() or 1)

    def src(seed48, n):
        out, _ = b.rand48([seed48], n, b.R48_F64)
        return out[0]
    sysd = wl.md_system(name, velocities_from(src))
    with b.Sim(sysd["N"], sysd["L"]) as s:
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(steps, b.MD_VERLET)
        ke, pe, w = s.energies()
        F = s.forces()
        p, v = s.get_state()
        assert s.stat("vl_builds") < s.stat("vl_steps")
    Fo, peo, wo = oracle.forces(p.astype(np.float64), sysd["L"], algo=1)
    # forces from lists that are up to a dozen steps old: every component within R15, except on atoms with a
    # partner inside the cutoff window of R16 (a pair dropped by a stale list fails this)
    check_forces(F, Fo, p, sysd["L"], oracle)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


@pytest.mark.parametrize("n,rho", [(8, 0.8), (10, 0.3), (9, 0.05)])
def test_both_list_builders_give_the_same_lists(b, n, rho):
    """Lists written by the cell kernel's filter (default) and by the plain thread-per-atom kernel
    ("vl_naive_build"): same forces to rounding, same energies, both within R15 of the oracle."""
    pos, L = wl.perturbed_fcc(n, rho, 0.12, seed=40 + n)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, algo=0)
    res = []
    for naive in (0, 1):
        with b.Sim(pos.shape[0], L) as s:
            s.option("vl_naive_build", naive)
            s.set_state(pos, np.zeros_like(pos))
            s.compute_forces(b.MD_VERLET)
            res.append((s.forces(), s.energies()))
            assert force_check(res[-1][0], Fo)[0] == 0
    # the two kernels write the entries in different orders: FP32 sums agree to rounding
    assert np.all(np.abs(res[0][0] - res[1][0]) <= 1e-5 + 2e-6 * np.abs(res[1][0]))
    assert res[0][1][1] == pytest.approx(res[1][1][1], rel=1e-7) and res[0][1][1] == pytest.approx(peo, rel=1e-6)


def test_eps_sigma_not_one(b):
    """Scaled units (R1): sigma = 1.7, eps = 0.4, rc = 2.5 sigma; skin defaults to 0.3 sigma."""
    sigma, eps = 1.7, 0.4
    pos, L = wl.perturbed_fcc(6, 0.8, 0.1, seed=21)
    pos = (pos.astype(np.float64) * sigma).astype(np.float32)
    L = float(np.float32(L * sigma))
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, rc=2.5 * sigma, eps=eps, sigma=sigma, algo=0)
    with b.Sim(pos.shape[0], L, rc=2.5 * sigma, eps=eps, sigma=sigma) as s:
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_VERLET)
        F = s.forces().astype(np.float64)
        ke, pe, w = s.energies()
    # the tolerance of R15 is stated in units of eps / sigma
    tol = np.maximum(1e-4 * np.abs(Fo), 1e-5 * eps / sigma)
    assert np.all(np.abs(F - Fo) <= tol)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


@pytest.mark.parametrize("shifted", [0, 1, 2])
@pytest.mark.parametrize("n,rho,amp", [(6, 0.8, 0.10), (7, 0.9, 0.08), (8, 0.3, 0.12), (10, 0.8, 0.1)])
def test_half_lists_with_reaction_forces(b, n, rho, amp, shifted):
    """Option "vl_half" (Newton's third law on this path: every pair once, the reaction through vector
    reductions): same forces and energies as the oracle, from fresh lists and after steps on reused ones."""
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=900 + n)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    with b.Sim(pos.shape[0], L, shifted=shifted) as s:
        s.option("vl_half", 1)
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_VERLET)
        assert force_check(s.forces(), Fo)[0] == 0
        _, pe, w = s.energies()
        assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)
        s.step(15, b.MD_VERLET)
        p, v = s.get_state()
        assert np.all(np.isfinite(p))
        Fo2, peo2, _ = oracle.forces(p.astype(np.float64), L, mode=shifted, algo=0)
        assert force_check(s.forces(), Fo2)[0] == 0
        assert s.energies()[1] == pytest.approx(peo2, rel=1e-6)


def test_half_lists_full_size_c3(b):
    import os
    oracle.set_threads(os.cpu_count() or 1)

    def src(seed48, n):
        out, _ = b.rand48([seed48], n, b.R48_F64)
        return out[0]
    sysd = wl.md_system("c3_cell_256k", velocities_from(src))
    with b.Sim(sysd["N"], sysd["L"]) as s:
        s.option("vl_half", 1)
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(1000, b.MD_VERLET)
        ke, pe, w = s.energies()
        F = s.forces()
        p, v = s.get_state()
    Fo, peo, wo = oracle.forces(p.astype(np.float64), sysd["L"], algo=1)
    check_forces(F, Fo, p, sysd["L"], oracle)
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


@pytest.mark.parametrize("fuse", [1, 0])
@pytest.mark.parametrize("graph,chunks", [(1, [100]), (0, [100]), (1, [7, 1, 30, 2, 60])])
def test_fused_integrator_of_the_list_path(b, c1, fuse, graph, chunks):
    """Option "vl_fuse" (default 1): interior steps integrate in the epilogue of the list force kernel (slots are
    stable between rebuilds: one kernel per step plus the conditional build launches).  Same energies as the oracle
    after 100 steps however the steps are split over calls, graph-replayed or not, fused or not."""
    _, _, _, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 100, algo=0)
    with b.Sim(c1["N"], c1["L"]) as s:
        s.option("vl_fuse", fuse)
        s.option("graph", graph)
        s.set_state(c1["pos"], c1["vel"])
        for k in chunks:
            s.step(k, b.MD_VERLET)
        ke, pe, w = s.energies()
        Eo = tr[100, 0] + tr[100, 1]
        assert abs(ke + pe - Eo) <= 1e-5 * abs(Eo)
        p, v = s.get_state()
        Fo, _, _ = oracle.forces(p.astype(np.float64), c1["L"], algo=0)
        assert force_check(s.forces(), Fo)[0] == 0
        assert s.stat("vl_steps") == 101 and 3 <= s.stat("vl_builds") <= 40
        assert ke == pytest.approx(oracle.kinetic_energy(v.astype(np.float64)), rel=1e-9)


def test_lists_grown_after_graphs_were_captured(b):
    """A handle that has already replayed CUDA graphs of the list path, then receives a denser state whose lists
    outgrow the capacity: the reallocation must also forget those graphs (their nodes hold the old list pointer
    and capacity).  Uniform state, 10 steps; clustered state (600 atoms in one cell), 10 steps; oracle forces."""
    g = np.stack(np.meshgrid(np.arange(10), np.arange(10), np.arange(6), indexing="ij"), -1).reshape(-1, 3)
    L = 45.5
    uniform = (2.0 + 4.3 * g).astype(np.float32)                  # every pair beyond rc: nothing moves
    clustered = (15.2 + 0.95 * g).astype(np.float32)
    with b.Sim(g.shape[0], L) as s:
        s.set_state(uniform, np.zeros_like(uniform))
        s.step(10, b.MD_VERLET)
        assert s.stat("graph_replays") > 0
        cap0 = s.stat("vl_cap")
        s.set_state(clustered, np.zeros_like(clustered))
        s.step(10, b.MD_VERLET)
        assert s.stat("vl_cap") > cap0 and s.stat("vl_overflow") == 0
        p, _ = s.get_state()
        F = s.forces()
        _, pe, w = s.energies()
    Fo, peo, wo = oracle.forces(p.astype(np.float64), L, algo=0)
    assert force_check(F, Fo)[0] == 0
    assert pe == pytest.approx(peo, rel=1e-6) and w == pytest.approx(wo, rel=1e-6)


def test_overflow_in_the_middle_of_a_run_is_reported(b):
    """A block of 1000 atoms contracting onto its centre and bouncing back: the builds around step 100 need lists
    of ~100 entries (capacity 40), the builds at the end of the 400 steps fit again.  md_step reads the flag once,
    at its end: it must still answer MD_ENOMEM (lists "are never truncated silently"), and the run repeated on the
    enlarged lists must succeed and give the oracle's forces."""
    n, a, alpha, L = 10, 1.3, 0.5, 45.5
    g = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"), -1).reshape(-1, 3)
    pos = (L / 2 + a * (g - (n - 1) / 2)).astype(np.float32)
    vel = (-alpha * (pos - np.float32(L / 2))).astype(np.float32)
    with b.Sim(pos.shape[0], L) as s:
        s.set_state(pos, vel)
        s.compute_forces(b.MD_VERLET)
        cap0 = s.stat("vl_cap")
        assert s.stat("vl_overflow") == 0 and cap0 < 60            # the start fits
        with pytest.raises(b.MDError) as e:
            s.step(400, b.MD_VERLET)
        assert e.value.code == b.MD_ENOMEM
        assert s.stat("vl_cap") > 80                                 # enlarged for the longest list any build asked for
        s.set_state(pos, vel)
        s.step(400, b.MD_VERLET)
        assert s.stat("vl_overflow") == 0
        p, _ = s.get_state()
        F = s.forces()
    Fo, _, _ = oracle.forces(p.astype(np.float64), L, algo=0)
    assert force_check(F, Fo)[0] == 0
