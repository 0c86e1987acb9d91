"""Pins P1 and P9 for the oracle's random numbers (R1-R3).

P1: Philox4x32-10 blocks against a third-party engine (ATen host Philox, tests/golden/philox_aten.txt).
P9: the normals are N(0,1), uncorrelated across sites / steps / components, and the uniforms they are
    built from lie strictly inside (0,1) and are exactly representable in fp32.
"""
import os

import numpy as np
import pytest
from scipy import stats

from oracle import asd_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox_aten.txt")


def _cases():
    out = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        out.append((int(f[0], 16), int(f[1], 16), int(f[2], 16), [int(x, 16) for x in f[3:7]]))
    return out


def test_golden_file_has_cases():
    assert len(_cases()) >= 12


@pytest.mark.parametrize("seed,subseq,offset,expect", _cases())
def test_philox_raw_matches_aten(seed, subseq, offset, expect):
    key = (seed & 0xFFFFFFFF, seed >> 32)
    ctr = (offset & 0xFFFFFFFF, offset >> 32, subseq & 0xFFFFFFFF, subseq >> 32)
    got = orc.philox4x32_10(key, ctr)
    assert [int(x) for x in got] == expect


@pytest.mark.parametrize("seed,subseq,offset,expect", _cases())
def test_philox_keying_matches_aten(seed, subseq, offset, expect):
    """R1: block(seed, n, g, stream) == ATen Philox(seed, subsequence = g | stream<<60, offset = n)."""
    stream, g = subseq >> 60, subseq & ((1 << 60) - 1)
    got = orc.philox_block(seed, offset, g, stream)
    assert [int(x) for x in got] == expect


def test_uniform_mapping_endpoints_and_fp32_exact():
    # R2: u in (0,1), 24 significant bits => exact in fp32
    assert orc.uniform(0) == 2.0 ** -24
    assert orc.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert orc.uniform(0x1FF) == 2.0 ** -24            # low 9 bits are dropped
    assert orc.uniform(0x200) == 3 * 2.0 ** -24
    for r in (0, 1, 0x200, 0x7FFFFFFF, 0x80000000, 0xDEADBEEF, 0xFFFFFFFF):
        u = orc.uniform(r)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u


def test_normals_moments_and_independence():
    n = 200_000
    a = orc.normals3_bulk(1, 0, 0, n)               # step 0, sites 0..n-1
    b = orc.normals3_bulk(1, 1, 0, n)               # step 1, same sites
    c = orc.normals3_bulk(2, 0, 0, n)               # other seed
    tol = 5.0 / np.sqrt(n)
    for x in (a, b, c):
        assert np.all(np.abs(x.mean(axis=0)) < tol)
        assert np.all(np.abs(x.var(axis=0) - 1.0) < 2.0 * tol)
        assert np.all(np.abs(stats.kurtosis(x, axis=0)) < 0.06)
        assert np.all(np.abs(stats.skew(x, axis=0)) < 0.03)
        for comp in range(3):                        # Kolmogorov-Smirnov against the exact normal CDF
            assert stats.kstest(x[:, comp], "norm").pvalue > 1e-4
        cc = np.corrcoef(x.T)
        assert np.all(np.abs(cc - np.eye(3)) < tol)  # components uncorrelated
        for comp in range(3):                        # neighbouring sites uncorrelated
            assert abs(np.corrcoef(x[:-1, comp], x[1:, comp])[0, 1]) < tol
    for comp in range(3):
        assert abs(np.corrcoef(a[:, comp], b[:, comp])[0, 1]) < tol   # steps uncorrelated
        assert abs(np.corrcoef(a[:, comp], c[:, comp])[0, 1]) < tol   # seeds uncorrelated
    assert np.abs(a).max() < 5.78                    # R2 tail cut sqrt(2*24*ln2) = 5.768


def test_normals_are_a_pure_function_of_seed_step_site():
    x = orc.normals3_bulk(5, 17, 1000, 64)
    for a in (0, 13, 63):
        assert np.array_equal(orc.normals3(5, 17, 1000 + a), x[a])
    assert not np.array_equal(orc.normals3(5, 18, 1000), x[0])
