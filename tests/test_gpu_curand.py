"""The oracle's Philox4x32-10 against an independent LIBRARY implementation: cuRAND's device API
(curand_Philox4x32_10 and the public curandStatePhilox4_32_10_t generator), on the GPU box.  SURVEY 8(c) P-RNG: the
Random123 known-answer file is not in the container, so the three vectors of tests/golden/philox4x32_10_kat.txt were
computed from the SC'11 definition; this is the cross-check against code neither side wrote."""
import ctypes as C
import os

import numpy as np
import pytest

import oracle
from curand_helper import build_helper

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def curand_blocks(rows: np.ndarray) -> np.ndarray:
    L = C.CDLL(build_helper())
    L.curand_philox_blocks.restype = C.c_int
    L.curand_philox_blocks.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    rows = np.ascontiguousarray(rows, dtype=np.uint32)
    out = np.zeros((rows.shape[0], 8), dtype=np.uint32)
    assert L.curand_philox_blocks(rows.shape[0], rows.ctypes.data, out.ctypes.data) == 0
    return out


def test_oracle_philox_matches_curand():
    rng = np.random.Generator(np.random.Philox(5481))
    rows = [[int(x, 16) for x in line.split()[:6]]
            for line in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if line.strip() and line[0] != "#"]
    kat_out = [[int(x, 16) for x in line.split()[6:10]]
               for line in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if line.strip() and line[0] != "#"]
    # the counters the method draws: (index, chromosome, generation, tag) under key = seed
    for seed in (0, 3, 20121123, 2**63 + 5, 2**64 - 1):
        for tag in range(5):
            for _ in range(40):
                rows.append([int(rng.integers(0, 2**20)), int(rng.integers(0, 2**24)), int(rng.integers(0, 2**32)), tag,
                             seed & 0xFFFFFFFF, seed >> 32])
    rows += [[int(v) for v in rng.integers(0, 2**32, 6)] for _ in range(500)]           # arbitrary 32-bit words
    rows = np.asarray(rows, dtype=np.uint64).astype(np.uint32)
    got = curand_blocks(rows)
    for i, r in enumerate(rows):
        ref = oracle.philox4x32_10([int(v) for v in r[:4]], [int(v) for v in r[4:6]])
        assert np.array_equal(got[i, :4], ref), f"curand_Philox4x32_10 differs at row {i}: {r}"
        if r[1] < 2**30:
            assert np.array_equal(got[i, 4:], ref), f"curand_init + curand4 differs at row {i}: {r}"
    for i, out in enumerate(kat_out):                                                   # the golden vectors themselves
        assert [int(v) for v in got[i, :4]] == out
