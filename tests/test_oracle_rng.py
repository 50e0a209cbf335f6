"""Pins for the oracle's random-number stream and uniform maps (R13, R14, R6b).

Nothing here retypes the oracle's formulas as the expected value: the Philox output is checked
against published known-answer vectors, the maps against exact rational arithmetic and their
stated ranges/symmetries, ln u against an 80-bit evaluation, the stream against its moments.
"""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

import oracle

GOLDEN = Path(__file__).parent / "golden" / "philox_kat.txt"


def _kat_rows():
    rows = []
    for line in GOLDEN.read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answer_vectors():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, want in rows:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(g) for g in got] == want


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # A keyed Philox is a permutation of counter space: distinct counters -> distinct outputs,
    # and each counter word must matter (a dropped word would collide here).
    key = (12345, 678)
    seen = set()
    for i in range(8):
        for c in range(8):
            for t in range(4):
                for p in range(2):
                    out = tuple(int(v) for v in oracle.philox4x32_10((i, c, t, p), key))
                    assert out not in seen
                    seen.add(out)
    assert tuple(oracle.philox4x32_10((1, 2, 3, 0), (1, 0))) != tuple(oracle.philox4x32_10((1, 2, 3, 0), (0, 1)))


def test_tmap_exact_symmetric_never_zero():
    rng = np.random.default_rng(7)
    words = list(rng.integers(0, 2**32, size=4000, dtype=np.uint64)) + [0, 2**32 - 1, 1 << 9, (1 << 9) - 1, 1 << 31]
    for w in words:
        w = int(w)
        k = w >> 9
        exact = Fraction(2 * k + 1, 2**23) - 1             # the real number R14 names
        got = oracle.tmap(w)
        assert Fraction(got) == exact                     # exactly representable in fp32
        assert got != 0.0 and -1.0 < got < 1.0
        assert oracle.tmap((~w) & 0xFFFFFFFF) == -got     # symmetric about 0
    assert oracle.tmap(0) == -1.0 + 2.0**-23
    assert oracle.tmap(0xFFFFFFFF) == 1.0 - 2.0**-23


def test_umap_exact_in_half_open_unit_interval():
    rng = np.random.default_rng(8)
    words = list(rng.integers(0, 2**32, size=4000, dtype=np.uint64)) + [0, 2**32 - 1, 255, 256]
    for w in words:
        w = int(w)
        exact = Fraction((w >> 8) + 1, 2**24)
        got = oracle.umap(w)
        assert Fraction(got) == exact
        assert 0.0 < got <= 1.0
    assert oracle.umap(0) == 2.0**-24
    assert oracle.umap(0xFFFFFFFF) == 1.0


def test_lnu_is_the_correctly_rounded_fp32_logarithm_for_every_u():
    # All 2^24 values u = k * 2^-24.  Reference: 80-bit logl rounded once to fp32.  (A result
    # within ~2^-63 of an fp32 rounding midpoint could fool the reference; with 2^24 inputs the
    # expected number of such cases is ~1e-5, and any case would show up as a mismatch here.)
    if np.finfo(np.longdouble).nmant < 63:
        pytest.skip("no 80-bit long double on this host")
    k = np.arange(1, 2**24 + 1, dtype=np.uint32)
    u = (k.astype(np.float64) * 2.0**-24).astype(np.float32)
    assert np.all(u.astype(np.float64) * 2.0**24 == k)     # u itself is exact
    got = oracle.lnu(u)
    ref = np.log(u.astype(np.longdouble)).astype(np.float32)
    bad = np.nonzero(got != ref)[0]
    assert bad.size == 0, f"{bad.size} values of u where lnu is not correctly rounded, first k={k[bad[:5]]}"
    assert got[-1] == 0.0 and np.all(got[:-1] < 0.0)


def test_move_stream_moments():
    # Displacement components are uniform on (-1, 1): mean 0, variance 1/3; u uniform on (0, 1].
    n = 200_000
    t = np.empty((n, 3))
    u = np.empty(n)
    key = (2024, 0)
    for j in range(n):
        w = oracle.philox4x32_10((j & 63, j >> 6, 5, 1), key)
        t[j] = [oracle.tmap(int(w[0])), oracle.tmap(int(w[1])), oracle.tmap(int(w[2]))]
        u[j] = oracle.umap(int(w[3]))
    se_mean = np.sqrt(1.0 / 3.0 / n)
    assert np.all(np.abs(t.mean(axis=0)) < 4 * se_mean)
    # var of t^2 for U(-1,1): E t^4 - (E t^2)^2 = 1/5 - 1/9
    se_var = np.sqrt((1 / 5 - 1 / 9) / n)
    assert np.all(np.abs((t**2).mean(axis=0) - 1 / 3) < 4 * se_var)
    assert abs(u.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
    c = np.corrcoef(np.column_stack([t, u]).T)
    assert np.all(np.abs(c - np.eye(4)) < 4 / np.sqrt(n))  # the four words are uncorrelated
