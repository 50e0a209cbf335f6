"""Pins of the oracle's initial-state generator (R22): what the configs
demand of an initial state -- first bead uniform in the box, bond components N(0, b^2/3), hence
<R_ee^2> = (N-1) b^2 -- plus determinism and independence from the Monte-Carlo stream."""
import math

import numpy as np
from scipy import stats

import oracle
import scmf_inputs as si


def _gen(n=20000, N=32, seed=11, gen_seed=1234):
    s = si.custom_system(n, N, 2, [[0] * (N // 2) + [1] * (N - N // 2)], None, [[0, 20], [20, 0]], 50.0,
                         (16, 32, 8), (8.0, 16.0, 4.0), seed=seed, b=0.8)
    o = oracle.Oracle.from_system(s)
    o.generate_state(gen_seed)
    x, y, z = o.positions()
    return s, o, x.reshape(n, N).astype(np.float64), y.reshape(n, N).astype(np.float64), z.reshape(n, N).astype(np.float64)


def test_generated_state_first_bead_uniform_and_bonds_gaussian():
    s, o, x, y, z = _gen()
    n, N, b = x.shape[0], x.shape[1], 0.8
    for v, L in ((x, 8.0), (y, 16.0), (z, 4.0)):
        u = v[:, 0] / L
        assert 0.0 <= u.min() and u.max() < 1.0
        assert stats.kstest(u, "uniform").pvalue > 1e-4
        d = np.diff(v, axis=1).reshape(-1) / (b / math.sqrt(3.0))
        m = d.size
        assert abs(d.mean()) < 4 / math.sqrt(m)
        assert abs((d * d).mean() - 1.0) < 4 * math.sqrt(2.0 / m)
        assert abs((d ** 4).mean() - 3.0) < 4 * math.sqrt(96.0 / m)
        assert stats.kstest(d[:200000], "norm").pvalue > 1e-4
    # the three components of a bond and consecutive bonds are uncorrelated
    dx, dy, dz = (np.diff(v, axis=1).reshape(-1) for v in (x, y, z))
    for a_, b_ in ((dx, dy), (dx, dz), (dy, dz), (dx[:-1], dx[1:])):
        assert abs(np.corrcoef(a_, b_)[0, 1]) < 4 / math.sqrt(a_.size)
    r2 = (x[:, -1] - x[:, 0]) ** 2 + (y[:, -1] - y[:, 0]) ** 2 + (z[:, -1] - z[:, 0]) ** 2
    want = (N - 1) * b * b
    assert abs(r2.mean() - want) < 3 * want * math.sqrt(2.0 / (3.0 * n))          # north_star check 1 on the start state
    assert int(o.density().sum()) == n * N                                       # it was binned (step 4)


def test_generated_state_is_deterministic_keyed_and_off_the_move_stream():
    s, o, x, y, z = _gen(n=500, gen_seed=7)
    _, _, x2, _, _ = _gen(n=500, gen_seed=7)
    _, _, x3, _, _ = _gen(n=500, gen_seed=8)
    _, _, x4, _, _ = _gen(n=500, seed=12, gen_seed=7)          # the Monte-Carlo seed does not enter
    assert np.array_equal(x, x2) and not np.array_equal(x, x3) and np.array_equal(x, x4)
    # chain c of a larger system equals chain c of a smaller one (counter = (bead, chain))
    _, _, xl, _, _ = _gen(n=800, gen_seed=7)
    assert np.array_equal(xl[:500], x)
    # domain 1: the first-bead draw is not the Monte-Carlo draw of (chain 0, bead 0, step 0, parity 0)
    w_gen = oracle.philox4x32_10([0, 0, 0, 1 << 8], [7, 0])
    w_mc = oracle.philox4x32_10([0, 0, 0, 0], [7, 0])
    assert not np.array_equal(w_gen, w_mc)
    assert x[0, 0] == np.float32(8.0 * ((float(w_gen[0]) + 0.5) * 2.0 ** -32))


def test_validate_reports_what_it_should():
    """Pins of the validation report: hand-made states with known answers."""
    s = si.custom_system(3, 4, 2, [[0, 0, 1, 1]], None, [[0, 5], [5, 0]], 10.0, (4, 4, 4), (2.0, 2.0, 2.0), seed=3)
    o = oracle.Oracle.from_system(s)
    x = np.array([0, 1, 1, 1,   0, 0, 0, 0,   0.5, 0.5, 0.5, 2.5], dtype=np.float32)   # bonds: 1,0,0 | 0,0,0 | 0,0,2
    y = np.zeros(12, dtype=np.float32)
    z = np.zeros(12, dtype=np.float32)
    y[7] = 1.5                                                                          # chain 1: last bond = 1.5
    o.load_state(x, y, z)
    v = o.validate()
    assert v["nonfinite"] == 0 and v["density_total"] == 12 and v["density_per_type"] == [6, 6]
    assert v["max_bond_sq"] == 4.0
    assert v["mean_bond_sq"] == pytest_approx((1.0 + 2.25 + 4.0) / 9.0)
    x[5] = np.nan
    z[0] = np.inf
    o.set_beads([5, 0], x[[5, 0]], y[[5, 0]], z[[5, 0]])
    assert o.validate()["nonfinite"] == 2


def pytest_approx(v):
    import pytest
    return pytest.approx(v, rel=1e-12)
