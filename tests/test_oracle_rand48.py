"""Pins for the oracle's rand48 (O5): glibc, skip-ahead constants, composition laws.
PAPER.md:142-164 (Eq. 5-7), :172; readings R5, R7, R8, R9, R10."""
import ctypes

import numpy as np
import pytest

import oracle
from conftest import golden_lines
from paper_0709_3225_b200 import workloads as wl

MASK = (1 << 48) - 1


def glibc_golden():
    return {row[0]: row[1:] for row in golden_lines("rand48_glibc.txt")}


def test_against_golden_glibc_series():
    g = glibc_golden()
    x0 = int(g["x0"][0], 16)
    raw, st = oracle.rand48_fill([x0], 5, kind=3)
    assert [int(x) for x in raw[0]] == [int(s, 16) for s in g["states"]]
    assert int(st[0]) == int(g["states"][-1], 16)
    assert list(oracle.rand48_fill([x0], 5, kind=1)[0][0]) == [int(s) for s in g["shift17"]]
    assert list(oracle.rand48_fill([x0], 5, kind=0)[0][0]) == [int(s) for s in g["shift16"]]
    assert oracle.rand48_fill([x0], 1, kind=2)[0][0, 0] == float.fromhex(g["first_double"][0])
    assert list(oracle.rand48_fill([int(g["srand48_0_x0"][0], 16)], 3, kind=1)[0][0]) == \
        [int(s) for s in g["srand48_0_lrand48"]]


def test_against_live_glibc():
    """'the first N random numbers of the lrand48 series' -- re-derived from libc."""
    try:
        libc = ctypes.CDLL("libc.so.6")
        libc.seed48, libc.lrand48, libc.mrand48, libc.drand48
    except (OSError, AttributeError):
        pytest.skip("no glibc rand48 on this machine")
    libc.lrand48.restype = ctypes.c_long
    libc.mrand48.restype = ctypes.c_long
    libc.drand48.restype = ctypes.c_double
    libc.seed48.restype = ctypes.c_void_p

    def seed(x):
        libc.seed48((ctypes.c_ushort * 3)(x & 0xFFFF, (x >> 16) & 0xFFFF, (x >> 32) & 0xFFFF))

    n = 2000
    for x0 in (0x1234ABCD330E, 0x330E, 0xFFFFFFFFFFFF, 0):
        seed(x0)
        assert [libc.lrand48() for _ in range(n)] == [int(v) for v in oracle.rand48_fill([x0], n, kind=1)[0][0]]
        seed(x0)
        assert [libc.mrand48() & 0xFFFFFFFF for _ in range(n)] == \
            [int(v) for v in oracle.rand48_fill([x0], n, kind=0)[0][0]]
        seed(x0)
        assert [libc.drand48() for _ in range(n)] == list(oracle.rand48_fill([x0], n, kind=2)[0][0])
    libc.srand48(0)
    assert libc.lrand48() == int(oracle.rand48_fill([0x330E], 1, kind=1)[0][0, 0])


def test_doubles_are_exact_and_in_unit_interval():
    raw, _ = oracle.rand48_fill([0xDEADBEEF1234], 5000, kind=3)
    dbl, _ = oracle.rand48_fill([0xDEADBEEF1234], 5000, kind=2)
    assert np.all(dbl >= 0) and np.all(dbl < 1)
    assert np.all((dbl * 2.0 ** 48).astype(np.uint64) == raw)          # x * 2^-48 exactly (R10)
    assert oracle.rand48_fill([0], 1, kind=3)[0][0, 0] == 0xB          # a*0 + c


def test_skip_constants_golden():
    rows = golden_lines("rand48_skip_consts.txt")
    for row in rows:
        if row[0].isdigit():
            k, A, C = int(row[0]), int(row[1], 16), int(row[2], 16)
            assert oracle.rand48_skip_consts(k) == (A, C), k
    g = {r[0]: r[1] for r in rows if not r[0].isdigit()}
    assert oracle.rand48_skip(0x1234ABCD330E, 1 << 28) == int(g["after_2p28"], 16)
    # Eq. 7 as printed (sum to m instead of m-1) is off by one (R5): for m = 1 it would give
    # a*c + c, not c
    assert oracle.rand48_skip_consts(1) == (0x5DEECE66D, 0xB)
    assert (0x5DEECE66D * 0xB + 0xB) & MASK == int(g["eq7_as_printed_m1"], 16)


def test_skip_constants_log_equals_linear_recurrence():
    for m in (0, 1, 2, 3, 31, 32, 33, 1000, 4096, 6144, 65537):
        assert oracle.rand48_skip_consts(m) == oracle.rand48_skip_consts(m, linear=True), m
    assert oracle.rand48_skip_consts(0) == (1, 0)


def test_skip_equals_stepping_and_composes():
    x = 0x0123456789AB
    seq, _ = oracle.rand48_fill([x], 3000, kind=3)
    for k in (1, 2, 31, 32, 33, 1024, 2999, 3000):
        assert oracle.rand48_skip(x, k) == int(seq[0, k - 1])
    assert oracle.rand48_skip(x, 0) == x
    for j, k in [(5, 7), (4096, 123), (1 << 27, 1 << 27), ((1 << 47) + 3, (1 << 47) - 3)]:
        assert oracle.rand48_skip(oracle.rand48_skip(x, j), k) == oracle.rand48_skip(x, (j + k) & MASK)
    assert oracle.rand48_skip(x, 1 << 48) == x                          # full period


def test_fill_concatenates():
    s = wl.stream_seeds(7, 5)
    a, st1 = oracle.rand48_fill(s, 100, kind=0)
    b, st2 = oracle.rand48_fill(st1, 57, kind=0)
    ab, st = oracle.rand48_fill(s, 157, kind=0)
    assert np.array_equal(np.concatenate([a, b], axis=1), ab) and np.array_equal(st, st2)


@pytest.mark.parametrize("S,n", [(1, 10), (32, 1000), (6144, 20000), (192, 191), (7, 50)])
def test_leapfrog_interleaves_to_sequential(S, n):
    # S lanes with stride-S constants reproduce the serial series
    x0 = 0x00C0FFEE0001
    assert np.array_equal(oracle.rand48_leapfrog(x0, S, n), oracle.rand48_fill([x0], n, kind=3)[0][0])


def test_splitmix64_golden():
    for state, out in golden_lines("splitmix64.txt"):
        assert wl.splitmix64(int(state)) == int(out, 16)
    assert wl.splitmix64(12345) & MASK == 0x8258A9D111A0
    s = wl.stream_seeds(wl.MASTER_SEED, 4)
    assert int(s[0]) == 0x6ABB51034992 and np.all(s <= MASK) and len(set(map(int, s))) == 4
