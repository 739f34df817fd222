"""A second pair potential through the same machinery ("trivial to replace
this potential by other pair-potentials, including the coulombic interaction"): screened Coulomb (Yukawa),
md_set_potential, on all three force paths against the FP64 oracle (gpu-marked)."""
import numpy as np
import pytest

import oracle
from helpers import force_check, velocities_from
from paper_0709_3225_b200 import workloads as wl

pytestmark = pytest.mark.gpu
A, KAPPA = 6.0, 1.2


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_0709_3225_b200 import binding
    return binding


PATHS = [("allpairs", 0, {}), ("cell", 1, {}), ("cell kernel 1", 1, {"cell_kernel": 1}),
         ("cell kernel 3", 1, {"cell_kernel": 3}), ("skin cells", 1, {"cell_skin": 0.3}), ("verlet", 2, {})]


@pytest.mark.parametrize("label,algo,opts", PATHS, ids=[p[0] for p in PATHS])
@pytest.mark.parametrize("shifted", [0, 1, 2])
@pytest.mark.parametrize("n,rho,amp,kappa", [(6, 0.8, 0.10, KAPPA), (8, 0.3, 0.2, KAPPA), (7, 0.9, 0.08, 0.0)])
def test_yukawa_forces_match_oracle(b, label, algo, opts, shifted, n, rho, amp, kappa):
    pos, L = wl.perturbed_fcc(n, rho, amp, seed=700 + n)
    with oracle.potential(1, A, kappa):
        Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
    with b.Sim(pos.shape[0], L, shifted=shifted) as s:
        for k, v in opts.items():
            s.option(k, v)
        s.potential(b.MD_POT_YUKAWA, A, kappa)
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(algo)
        F, (ke, pe, w) = s.forces(), s.energies()
        nviol, worst = force_check(F, Fo)
        assert nviol == 0, (nviol, worst)
        assert pe == pytest.approx(peo, rel=1e-9) and w == pytest.approx(wo, rel=1e-9)     # every term in FP64
        # and back to Lennard-Jones on the same handle
        s.potential(b.MD_POT_LJ)
        with pytest.raises(b.MDError):
            s.forces()                                     # stale
        s.compute_forces(algo)
        Flj, _, _ = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0)
        assert force_check(s.forces(), Flj)[0] == 0


@pytest.mark.parametrize("algo", [0, 1, 2])
def test_yukawa_energy_trace_matches_oracle(b, algo, oracle_uniforms):
    """60 velocity-Verlet steps of the config-1 system with the Yukawa pair: per-step total energy within 1e-5
    of the oracle (R17), and the energy itself conserved."""
    c1 = wl.md_system("c1_allpairs_500", velocities_from(oracle_uniforms))
    with oracle.potential(1, A, KAPPA):
        _, _, _, tr = oracle.verlet_run(c1["pos"], c1["vel"], c1["L"], 60, algo=0)
    with b.Sim(c1["N"], c1["L"]) as s:
        s.potential(b.MD_POT_YUKAWA, A, KAPPA)
        s.set_state(c1["pos"], c1["vel"])
        s.compute_forces(algo)
        E = []
        for t in range(61):
            if t:
                s.step(1, algo)
            ke, pe, _ = s.energies()
            E.append(ke + pe)
            Eo = tr[t, 0] + tr[t, 1]
            assert abs(E[-1] - Eo) <= 1e-5 * abs(Eo), (t, E[-1], Eo)
    assert abs(E[-1] - E[0]) < 2e-4 * abs(E[0])


def test_md_set_potential_arguments(b):
    with b.Sim(500, 9.0) as s:
        for bad in ((7, 1.0, 1.0), (b.MD_POT_YUKAWA, float("nan"), 1.0), (b.MD_POT_YUKAWA, 1.0, -0.5),
                    (b.MD_POT_YUKAWA, 1.0, float("inf"))):
            with pytest.raises(b.MDError) as e:
                s.potential(*bad)
            assert e.value.code == b.MD_EINVAL
    assert b._lib.md_set_potential(None, 0, 0.0, 0.0) == b.MD_EINVAL


def test_fp32_window_cannot_be_reopened_under_another_potential(b):
    """"precise_r2" opens the FP32 branch of the cell and list kernels, which is Lennard-Jones arithmetic: with the
    Yukawa pair set it is refused, so in-range pairs can never silently get LJ forces; back on LJ it is accepted."""
    pos, L = wl.perturbed_fcc(6, 0.8, 0.10, seed=706)
    with oracle.potential(1, A, KAPPA):
        Fo, _, _ = oracle.forces(pos.astype(np.float64), L, mode=1, algo=0)
    with b.Sim(pos.shape[0], L) as s:
        s.potential(b.MD_POT_YUKAWA, A, KAPPA)
        with pytest.raises(b.MDError) as e:
            s.option("precise_r2", 1.3)
        assert e.value.code == b.MD_EINVAL
        assert s.stat("precise_r2") > 1e100
        s.set_state(pos, np.zeros_like(pos))
        for algo in (b.MD_CELL, b.MD_VERLET):
            s.compute_forces(algo)
            assert force_check(s.forces(), Fo)[0] == 0
        s.potential(b.MD_POT_LJ)
        s.option("precise_r2", 1.3)
        assert s.stat("precise_r2") == 1.3
