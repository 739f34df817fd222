"""md_forces_allpairs_static: the all-pairs evaluation for callers that cannot allocate device memory.

Who needs it: a process whose own memory pool was given the whole card at start-up (a cudaMalloc made on its
behalf by a library fails there), and code inside a latency-bound loop, where cudaMalloc and cudaFree are not
allowed because they stall the whole device.  Every other way into this library goes through md_create, which
allocates.  This entry point takes its scratch from a fixed 1.3 MB array compiled into the .so, so it works
for N <= MD_STATIC_MAX_ATOMS only, and all calls share that array.

The GPU tests compare it with the existing path (md_create + md_compute_forces(MD_ALLPAIRS)) on the same
coordinates, at the tolerances the other parity tests use, and on two calls in a row: the second call finds the
array as the first one left it, so anything that should have been cleared and was not shows up there.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import os
import re

import numpy as np
import pytest

import oracle
from helpers import force_check
from paper_0709_3225_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def b():
    from paper_0709_3225_b200 import build
    build.build()
    from paper_0709_3225_b200 import binding
    return binding


# ---- without a device ---------------------------------------------------------------------------------

def test_limit_is_the_same_in_header_and_binding(b):
    src = open(os.path.join(ROOT, "include", "ljmd.h")).read()
    m = re.search(r"#define\s+MD_STATIC_MAX_ATOMS\s+(\d+)", src)
    assert m and int(m.group(1)) == b.MD_STATIC_MAX_ATOMS


def test_sizes_beyond_the_limit_are_refused_before_the_device_is_touched(b):
    """The raw C call answers MD_EUNSUPPORTED for N above the limit (checked before any CUDA call, so also on a
    machine without a GPU); the binding says why."""
    big = b.MD_STATIC_MAX_ATOMS + 1
    dummy = np.zeros(4, dtype=np.float64)          # never dereferenced: the size check comes first
    rc_ = b._lib.md_forces_allpairs_static(dummy.ctypes.data, big, 40.0, 2.5, 1.0, 1.0, 1, dummy.ctypes.data,
                                           dummy.ctypes.data, None)
    assert rc_ == b.MD_EUNSUPPORTED
    with pytest.raises(b.MDError) as e:
        b.md_forces_allpairs_static(dummy, big, 40.0, 2.5, 1.0, 1.0, 1, dummy, dummy, stream=0)
    assert e.value.code == b.MD_EUNSUPPORTED and "MD_STATIC_MAX_ATOMS" in str(e.value)


@pytest.mark.parametrize("args", [
    (0, 10.0, 2.5, 1.0, 1.0, 1), (100, 0.0, 2.5, 1.0, 1.0, 1), (100, 10.0, -1.0, 1.0, 1.0, 1),
    (100, 10.0, 2.5, -1.0, 1.0, 1), (100, 10.0, 2.5, 1.0, 0.0, 1), (100, 10.0, 2.5, 1.0, 1.0, 3),
    (100, 4.9, 2.5, 1.0, 1.0, 1), (100, float("nan"), 2.5, 1.0, 1.0, 1),
])
def test_bad_arguments_are_refused_as_by_md_create(b, args):
    N, L, rc, eps, sigma, shifted = args
    dummy = np.zeros(4, dtype=np.float64)
    p = dummy.ctypes.data
    assert b._lib.md_forces_allpairs_static(p, N, L, rc, eps, sigma, shifted, p, p, None) == b.MD_EINVAL
    assert b._lib.md_forces_allpairs_static(None, 100, 10.0, 2.5, 1.0, 1.0, 1, p, p, None) == b.MD_EINVAL
    assert b._lib.md_forces_allpairs_static(p, 100, 10.0, 2.5, 1.0, 1.0, 1, None, p, None) == b.MD_EINVAL
    assert b._lib.md_forces_allpairs_static(p, 100, 10.0, 2.5, 1.0, 1.0, 1, p, None, None) == b.MD_EINVAL


# ---- on the GPU ---------------------------------------------------------------------------------------

def existing_path(b, pos, L, shifted, eps=1.0, sigma=1.0, rc=2.5):
    with b.Sim(pos.shape[0], L, rc=rc, eps=eps, sigma=sigma, shifted=shifted) as s:
        s.set_state(pos, np.zeros_like(pos))
        s.compute_forces(b.MD_ALLPAIRS)
        _, pe, w = s.energies()
        return s.forces(), pe, w


def static_path(b, torch, pos, L, shifted, eps=1.0, sigma=1.0, rc=2.5, bufs=None):
    """One call of the new entry point.  The caller's arrays are made here, by the caller's allocator (PyTorch's);
    the outputs start as NaN so that an element the kernel did not write cannot pass."""
    N = pos.shape[0]
    if bufs is None:
        bufs = (torch.empty((N, 3), dtype=torch.float32, device="cuda"),
                torch.empty(2, dtype=torch.float64, device="cuda"))
    F, ew = bufs
    F.fill_(float("nan"))
    ew.fill_(float("nan"))
    dpos = torch.from_numpy(pos).cuda()
    b.md_forces_allpairs_static(dpos, N, L, rc, eps, sigma, shifted, F, ew)
    e = ew.cpu().numpy()
    return F.cpu().numpy(), float(e[0]), float(e[1])


def assert_same(b, got, ref, pos, L, shifted, **kw):
    F, pe, w = got
    Fe, pee, we = ref
    assert np.all(np.isfinite(F))
    nviol, worst = force_check(F, Fe.astype(np.float64))         # R15, the tolerance of every force parity test
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(pee, rel=1e-9, abs=1e-9) and w == pytest.approx(we, rel=1e-9, abs=1e-9)
    # and the oracle itself, as for the existing all-pairs path (tests/test_gpu_md.py)
    Fo, peo, wo = oracle.forces(pos.astype(np.float64), L, mode=shifted, algo=0, **kw)
    nviol, worst = force_check(F, Fo)
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(peo, rel=1e-9, abs=1e-9) and w == pytest.approx(wo, rel=1e-9, abs=1e-9)


@pytest.mark.gpu
@pytest.mark.parametrize("shifted", [0, 1, 2])
def test_two_calls_in_a_row_match_the_existing_path(b, shifted):
    """N = 4000 (32 tiles of 128 atoms with a ragged last one, 10 j splits): two calls in a row into the same
    output arrays, each compared with md_compute_forces(MD_ALLPAIRS) and with the oracle."""
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    pos, L = wl.perturbed_fcc(10, 0.8, 0.1, seed=4242)
    ref = existing_path(b, pos, L, shifted)
    N = pos.shape[0]
    bufs = (torch.empty((N, 3), dtype=torch.float32, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda"))
    first = static_path(b, torch, pos, L, shifted, bufs=bufs)
    second = static_path(b, torch, pos, L, shifted, bufs=bufs)
    assert_same(b, first, ref, pos, L, shifted)
    assert_same(b, second, ref, pos, L, shifted)
    # the sums are taken in a fixed order: the two calls agree to the last bit
    assert np.array_equal(first[0], second[0]) and first[1:] == second[1:]


@pytest.mark.gpu
def test_a_call_after_a_different_system_sees_no_leftovers(b):
    """The shared array keeps the previous call's partial sums and counters: a large system, then a small one in
    another box with other units (fewer tiles, fewer splits), then the large one again, each against the existing path."""
    import torch
    big, Lb = wl.perturbed_fcc(10, 0.8, 0.1, seed=7)
    small, Ls = wl.perturbed_fcc(4, 0.3, 0.15, seed=8)
    small = (small * np.float32(1.7)).astype(np.float32)          # sigma = 1.7: the same system in scaled units
    Ls = float(np.float32(Ls * 1.7))
    small[small >= np.float32(Ls)] = 0.0
    kw = dict(eps=2.5, sigma=1.7, rc=2.5 * 1.7)
    ref_big = existing_path(b, big, Lb, 1)
    ref_small = existing_path(b, small, Ls, 2, **kw)
    assert_same(b, static_path(b, torch, big, Lb, 1), ref_big, big, Lb, 1)
    assert_same(b, static_path(b, torch, small, Ls, 2, **kw), ref_small, small, Ls, 2, **kw)
    assert_same(b, static_path(b, torch, big, Lb, 1), ref_big, big, Lb, 1)


@pytest.mark.gpu
@pytest.mark.parametrize("n_atoms", [1, 2, 33, 500])
def test_small_and_ragged_sizes(b, n_atoms):
    """Fewer atoms than a tile, than a j chunk, one atom alone (zero force, zero energies)."""
    import torch
    pos, L = wl.perturbed_fcc(5, 0.8, 0.1, seed=11)
    pos = np.ascontiguousarray(pos[:n_atoms])
    assert_same(b, static_path(b, torch, pos, L, 1), existing_path(b, pos, L, 1), pos, L, 1)


@pytest.mark.gpu
def test_largest_size_and_what_is_refused_on_the_device(b):
    """N = MD_STATIC_MAX_ATOMS exactly (16 x 16 x 16 x 4 fcc sites: 128 tiles, 3 splits) against the existing path;
    host arrays are refused, since staging them would take an allocation."""
    import torch
    pos, L = wl.perturbed_fcc(16, 0.8, 0.1, seed=12)
    assert pos.shape[0] == b.MD_STATIC_MAX_ATOMS
    got = static_path(b, torch, pos, L, 1)
    F, pe, w = got
    Fe, pee, we = existing_path(b, pos, L, 1)
    nviol, worst = force_check(F, Fe.astype(np.float64))
    assert nviol == 0, (nviol, worst)
    assert pe == pytest.approx(pee, rel=1e-9) and w == pytest.approx(we, rel=1e-9)
    host_F = np.zeros((4, 3), dtype=np.float32)
    dev = torch.zeros((4, 3), dtype=torch.float32, device="cuda")
    ew = torch.zeros(2, dtype=torch.float64, device="cuda")
    with pytest.raises(b.MDError) as e:
        b.md_forces_allpairs_static(dev, 4, 10.0, 2.5, 1.0, 1.0, 1, host_F, ew)
    assert e.value.code == b.MD_EINVAL
