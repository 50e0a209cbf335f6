"""GPU unit parity: the pieces of one trial move (DESIGN.md section 2 steps 1, 5.1, 5.2, 5.6) evaluated
by the library's kernels through the C ABI, against the oracle, bit for bit."""
from pathlib import Path

import numpy as np
import pytest

import oracle
import scmf_inputs as si

pytestmark = pytest.mark.gpu

GOLDEN = Path(__file__).resolve().parent / "golden" / "philox_kat.txt"


@pytest.fixture(scope="module")
def soma():
    import __graft_entry__ as entry
    entry.build()
    import paper_2606_09356_b200 as soma
    return soma


def _kat():
    rows = []
    for line in GOLDEN.read_text().splitlines():
        line = line.split("#")[0].strip()
        if not line:
            continue
        v = [int(t, 16) for t in line.replace(";", " ").replace("->", " ").split()]
        assert len(v) == 10
        rows.append((v[0:4], v[4:6], v[6:10]))
    assert len(rows) == 3
    return rows


def test_philox_known_answers_on_device(soma):
    for ctr, key, want in _kat():
        got = soma.soma_debug_philox(np.array([ctr], dtype=np.uint32), key)
        assert [int(v) for v in got[0]] == want


def test_philox_random_counters_match_oracle(soma):
    rng = np.random.default_rng(11)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    ctr[:8] = [[0, 0, 0, 0], [1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1], [31, 255, 9, 1],
               [0xFFFFFFFF] * 4, [63, 0xFFFFFFFE, 0xFFFFFFFF, 0x00010001]]
    key = np.array([0x12345678, 0x9ABCDEF0], dtype=np.uint32)
    got = soma.soma_debug_philox(ctr, key)
    want = np.stack([oracle.philox4x32_10(c, key) for c in ctr])
    assert np.array_equal(got, want)


def test_uniform_maps_and_lnu_all_2_24_values(soma):
    """tmap over every 23-bit pattern (twice: low bits must not matter), u and the slow-path ln u over
    every one of the 2^24 values of u -- the kernel's near-threshold logarithm is the correctly
    rounded one (R6b), i.e. the oracle's bits."""
    k = np.arange(1 << 24, dtype=np.uint32)
    words = (k << np.uint32(8)) | np.uint32(0xA5)
    t, u, l, lf = soma.soma_debug_maps(words)
    u_want = ((k.astype(np.float64) + 1.0) * 2.0 ** -24).astype(np.float32)
    assert np.array_equal(u, u_want)
    k23 = (words >> np.uint32(9)).astype(np.float64)
    t_want = ((2.0 * k23 + 1.0) * 2.0 ** -23 - 1.0).astype(np.float32)      # exact in double
    assert np.array_equal(t, t_want)
    assert np.array_equal(l.view(np.uint32), oracle.lnu(u_want).view(np.uint32))
    # the hardware logarithm that decides every move outside the +-1e-4 band is far inside that band
    err = np.abs(lf.astype(np.float64) - np.log(u_want.astype(np.float64)))
    assert err.max() < 1e-4 / 16, err.max()
    # spot check against the oracle's own scalar maps
    for w in (0, 1, 0x1FF, 0x200, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 0xFFFFFE00, 0xDEADBEEF):
        tt, uu, _, _ = soma.soma_debug_maps(np.array([w], dtype=np.uint32))
        assert float(tt[0]) == oracle.tmap(w) and float(uu[0]) == oracle.umap(w)


def _threshold_sample(rng, n):
    """(dE, words, lnu): a sample concentrated on the acceptance threshold dE = -lnu."""
    words = rng.integers(0, 2 ** 32, size=n, dtype=np.uint64).astype(np.uint32)
    u = ((words >> np.uint32(8)).astype(np.float64) + 1.0) * 2.0 ** -24
    lnu = oracle.lnu(u.astype(np.float32))
    dE = np.empty(n, dtype=np.float32)
    q = n // 4
    dE[:q] = rng.normal(0.0, 3.0, q).astype(np.float32)                       # generic
    base = (-lnu[q:3 * q]).astype(np.float32)                                 # on the threshold
    ulps = rng.integers(-3, 4, size=2 * q)
    near = base.copy()
    for s in range(1, 4):
        near = np.where(ulps >= s, np.nextafter(near, np.float32(np.inf)), near)
        near = np.where(ulps <= -s, np.nextafter(near, np.float32(-np.inf)), near)
    dE[q:3 * q] = near
    dE[3 * q:] = (-lnu[3 * q:] + rng.uniform(-3e-4, 3e-4, n - 3 * q)).astype(np.float32)   # in/around the band
    dE[:20] = [0.0, -0.0, 1e-30, -1e-30, 1e-8, 17.0, 16.635532, 16.64, 100.0, np.inf, -np.inf, 5e-8, 6e-8, 1.1920929e-07, 2e-7, 3e-7,
               np.nan, -np.nan, 3.4e38, -3.4e38]
    return dE, words, lnu


def test_fused_kernels_accept_routine_matches_the_definition(soma):
    """metropolis_accept_fma -- the decision routine of the fused kernels, i.e. of the path bench.py times:
    one FFMA on the hardware logarithm, a +-1e-4 guard band, the exact logarithm inside it -- against the
    rule accept iff fl32(dE + lnu) <= 0 (DESIGN.md section 2 step 5.6) on the threshold-concentrated sample,
    and for EVERY one of the 2^24 values of u at dE = -lnu moved by 0, +-1, +-2, +-3 ulps."""
    dE, words, lnu = _threshold_sample(np.random.default_rng(6), 1 << 21)
    got = soma.soma_debug_accept_fma(dE, words)
    with np.errstate(invalid="ignore"):
        want = ((dE + lnu).astype(np.float32) <= 0).astype(np.uint8)
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, (bad[:10], dE[bad[:10]], lnu[bad[:10]])
    k = np.arange(1 << 24, dtype=np.uint32)
    words = (k << np.uint32(8)) | np.uint32(0x5A)
    u = ((k.astype(np.float64) + 1.0) * 2.0 ** -24).astype(np.float32)
    lnu = oracle.lnu(u)
    n_acc = 0
    for shift in (0, 1, -1, 2, -2, 3, -3):
        dE = (-lnu).astype(np.float32)
        for _ in range(abs(shift)):
            dE = np.nextafter(dE, np.float32(np.inf if shift > 0 else -np.inf))
        got = soma.soma_debug_accept_fma(dE, words)
        want = ((dE + lnu).astype(np.float32) <= 0).astype(np.uint8)
        bad = np.nonzero(got != want)[0]
        assert bad.size == 0, (shift, bad[:10], dE[bad[:10]], lnu[bad[:10]])
        n_acc += int(want.sum())
    assert 0.3 < n_acc / (7 * (1 << 24)) < 0.7                                # the shifts straddle the threshold


def test_accept_decisions_match_the_definition(soma):
    """accept iff fl32(dE + lnu) <= 0 (DESIGN.md section 2 step 5.6), lnu the oracle's.  The sample
    is concentrated on the threshold: dE = -lnu +- a few ulps, where the kernel's fast logarithm
    cannot decide and its double-precision path must."""
    rng = np.random.default_rng(5)
    n = 1 << 21
    words = rng.integers(0, 2 ** 32, size=n, dtype=np.uint64).astype(np.uint32)
    u = ((words >> np.uint32(8)).astype(np.float64) + 1.0) * 2.0 ** -24
    lnu = oracle.lnu(u.astype(np.float32))
    dE = np.empty(n, dtype=np.float32)
    q = n // 4
    dE[:q] = rng.normal(0.0, 3.0, q).astype(np.float32)                       # generic
    base = (-lnu[q:3 * q]).astype(np.float32)                                 # on the threshold
    ulps = rng.integers(-3, 4, size=2 * q)
    near = base.copy()
    for s in range(1, 4):
        near = np.where(ulps >= s, np.nextafter(near, np.float32(np.inf)), near)
        near = np.where(ulps <= -s, np.nextafter(near, np.float32(-np.inf)), near)
    dE[q:3 * q] = near
    dE[3 * q:] = (-lnu[3 * q:] + rng.uniform(-3e-4, 3e-4, n - 3 * q)).astype(np.float32)   # in/around the band
    dE[:16] = [0.0, -0.0, 1e-30, -1e-30, 1e-8, 17.0, 16.635532, 16.64, 100.0, np.inf, -np.inf, 5e-8, 6e-8, 1.1920929e-07, 2e-7, 3e-7]
    got = soma.soma_debug_accept(dE, words)
    want = ((dE + lnu).astype(np.float32) <= 0).astype(np.uint8)              # numpy fp32 add: round-to-nearest-even
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, (bad[:10], dE[bad[:10]], lnu[bad[:10]])
    assert 0.2 < want[q:3 * q].mean() < 0.8                                   # the sample really straddles the threshold


@pytest.mark.parametrize("grid,box", [((16, 16, 16), (8.0, 8.0, 8.0)), ((12, 10, 7), (6.0, 5.0, 3.5)),
                                      ((256, 256, 128), (128.0, 128.0, 64.0)), ((5, 3, 2), (1.7, 2.9, 0.3))])
def test_cell_index_matches_oracle_including_edges(soma, grid, box):
    s = si.custom_system(4, 4, 1, [[0, 0, 0, 0]], None, [[0.0]], 0.0, grid, box, seed=3)
    o = oracle.Oracle.from_system(s)
    rng = np.random.default_rng(7)
    n = 20000
    pts = [rng.uniform(-3.0 * box[d], 4.0 * box[d], n).astype(np.float32) for d in range(3)]
    L = np.array(box, dtype=np.float32)
    h = (L / np.array(grid, dtype=np.float32)).astype(np.float32)
    edges = []
    for d in range(3):
        e = [0.0, -0.0, -1e-7, 1e-7, L[d], np.nextafter(L[d], np.float32(0)), np.nextafter(L[d], np.float32(np.inf)), 2 * L[d], -L[d],
             np.nextafter(-L[d], np.float32(0)), h[d], np.nextafter(h[d], np.float32(0)), -h[d], 3 * h[d], 1000.0 * L[d], -1000.0 * L[d],
             1e-45, -1e-45]
        edges.append(np.array(e, dtype=np.float32))
    m = len(edges[0])
    for d in range(3):
        pts[d][:m] = edges[d]
        pts[d][m:2 * m] = edges[d][::-1]
    pts[1][m:2 * m] = edges[1]
    with soma.Soma.from_system(s) as g:
        got = g.debug_cell_index(*pts)
    want = np.array([o.cell_index(pts[0][k], pts[1][k], pts[2][k]) for k in range(n)], dtype=np.uint32)
    assert np.array_equal(got, want)


def test_red_throughput_hook_measures_the_three_increment_modes():
    """soma_debug_red_throughput (north_star: "the atomic throughput of the histogram"): runs, rejects bad
    arguments, and the rates are in a sane range for a B200 (10 G/s ... 10 T/s)."""
    import paper_2606_09356_b200 as soma
    n_ops = 1 << 26
    for mode in (0, 1, 2):
        ms = soma.soma_debug_red_throughput(1 << 24, n_ops, mode)
        rate = n_ops / (ms * 1e-3)
        assert 1e10 < rate < 1e13, (mode, rate)
    for mode in (3, 4, 5, 6):                            # the window in distributed shared memory (clusters of 8 / 16 CTAs)
        ms = soma.soma_debug_red_throughput(1 << 10, n_ops, mode)
        rate = n_ops / (ms * 1e-3)
        assert 1e10 < rate < 2e13, (mode, rate)
    for bad in ((0, 100, 0), (100, 0, 0), (100, 100, 7)):
        with pytest.raises(soma.SomaError):
            soma.soma_debug_red_throughput(*bad)
