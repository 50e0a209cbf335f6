"""Pins of the oracle's bond-force-biased ("smart Monte Carlo") move, R24:
the library-free normal deviates, the proposal-ratio algebra against its definition in double, the
stationary distribution in a frozen field, and the ideal-chain closed forms."""
import math

import numpy as np
from scipy import stats

import oracle
import scmf_inputs as si
from test_oracle_moves import _axis_kernel, _energy64, _frozen_field_system

A = 0.05


def test_library_free_log_and_sincos_agree_with_libm():
    """The fp32 routines behind the deviates against libm in double, at fp32 accuracy, for EVERY argument
    they can be given: U = (k + 0.5) 2^-23, k = 0 .. 2^23 - 1 (a slip in the exponent split, the quarter-turn
    rotation or a polynomial coefficient at any single k fails here)."""
    k = np.arange(1 << 23, dtype=np.float64)
    x = ((k + 0.5) * 2.0 ** -23).astype(np.float32)
    assert np.array_equal(x.astype(np.float64), (k + 0.5) * 2.0 ** -23)          # the arguments are exact in fp32
    lg, sn, cs = oracle.det_functions_n(x)
    xd = x.astype(np.float64)
    ref = np.log(xd)
    err = np.abs(lg.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref))
    assert err.max() <= 3e-7, (err.max(), x[err.argmax()])
    es = np.abs(sn.astype(np.float64) - np.sin(2 * np.pi * xd))
    ec = np.abs(cs.astype(np.float64) - np.cos(2 * np.pi * xd))
    assert es.max() < 4e-7 and ec.max() < 4e-7, (es.max(), x[es.argmax()], ec.max(), x[ec.argmax()])
    # the scalar entry point used elsewhere is the same routine
    for kk in (0, 1, 2, (1 << 23) - 1, 1 << 21, 1 << 22, 3 << 21, 12345):
        a = oracle.det_functions(float(x[kk]))
        assert (np.float32(a[0]), np.float32(a[1]), np.float32(a[2])) == (lg[kk], sn[kk], cs[kk])


def test_normal_deviates_are_standard_normal_and_independent():
    s = si.custom_system(40000, 4, 1, [[0, 0, 0, 0]], None, [[0.0]], 0.0, (4, 4, 4), (2.0, 2.0, 2.0), seed=5)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_smc(A)
    d = np.array([o.smc_draws(c, i, i & 1) for c in range(40000) for i in (1, 2)])
    xi, u = d[:, :3], d[:, 3]
    m = xi.shape[0]
    for k in range(3):
        v = xi[:, k]
        assert abs(v.mean()) < 4 / math.sqrt(m) and abs((v * v).mean() - 1) < 4 * math.sqrt(2 / m)
        assert abs((v ** 4).mean() - 3) < 4 * math.sqrt(96 / m)
        assert stats.kstest(v, "norm").pvalue > 1e-4
    c = np.corrcoef(np.column_stack([xi, u]).T)
    assert np.all(np.abs(c - np.eye(4)) < 5 / math.sqrt(m))
    assert stats.kstest(u, "uniform").pvalue > 1e-4


def _ln_T(x_from, x_to, nbs, kb):
    """ln of the proposal density (up to its constant): Gaussian of variance 2A around x + A F(x)."""
    F = -2.0 * kb * sum((x_from - nb for nb in nbs), np.zeros(3))
    return -float(((x_to - x_from - A * F) ** 2).sum()) / (4.0 * A)


def test_margin_is_dE_minus_log_proposal_ratio_and_antisymmetric():
    s, o, omega = _frozen_field_system(6, 5, 2, (2, 2, 2), (1.0, 1.0, 1.0), seed=31)
    o.set_smc(A)
    rng = np.random.default_rng(2)
    types = s.bead_types()
    x, y, z = (v.astype(np.float64) for v in o.positions())
    kb = 1.5
    for _ in range(300):
        j = int(rng.integers(0, 30))
        i = j % 5
        new = np.array([x[j], y[j], z[j]]) + rng.normal(0, 0.3, 3)
        new = new.astype(np.float32).astype(np.float64)
        nbs = [np.array([x[k], y[k], z[k]]) for k in ((j - 1) if i > 0 else None, (j + 1) if i < 4 else None) if k is not None]
        old = np.array([x[j], y[j], z[j]])
        e0 = _energy64(x, y, z, types, omega, 5, 1.0, (2, 2, 2), (1.0, 1.0, 1.0))
        x2, y2, z2 = x.copy(), y.copy(), z.copy()
        x2[j], y2[j], z2[j] = new
        e1 = _energy64(x2, y2, z2, types, omega, 5, 1.0, (2, 2, 2), (1.0, 1.0, 1.0))
        want = (e1 - e0) - (_ln_T(new, old, nbs, kb) - _ln_T(old, new, nbs, kb))      # dE - ln(T_rev / T_fwd)
        got = o.smc_margin(j, *new)
        assert abs(got - want) < 2e-4 * max(1.0, abs(want)), (got, want)
        # antisymmetry: the margin of the reverse move from the moved state
        o2 = oracle.Oracle.from_system(s)
        o2.load_state(x2.astype(np.float32), y2.astype(np.float32), z2.astype(np.float32))
        o2.set_omega(omega)
        o2.set_smc(A)
        assert abs(o2.smc_margin(j, *old) + got) < 4e-4 * max(1.0, abs(want))


def test_smc_sampler_reaches_the_boltzmann_occupancy_in_a_frozen_field():
    n_chains, grid, box = 120_000, (2, 2, 2), (1.0, 1.0, 1.0)
    pats = np.array([[0, 1]], dtype=np.uint8)
    s, o, omega = _frozen_field_system(n_chains, 2, 2, grid, box, seed=22, pats=pats)
    o.set_smc(A)
    for step in range(60):
        o.half_sweep(0); o.half_sweep(1)
        o.step = o.step + 1
    x, y, z = o.positions()
    g = [np.floor(v.astype(np.float64) * 2.0).astype(np.int64) % 2 for v in (x, y, z)]
    cell = ((g[0] * 2 + g[1]) * 2 + g[2]).reshape(n_chains, 2)
    obs = np.zeros((8, 8))
    np.add.at(obs, (cell[:, 0], cell[:, 1]), 1.0)
    k = _axis_kernel(1.5, 0.5, 1.0)
    want = np.zeros((8, 8))
    for c0 in range(8):
        a = ((c0 >> 2) & 1, (c0 >> 1) & 1, c0 & 1)
        for c1 in range(8):
            b = ((c1 >> 2) & 1, (c1 >> 1) & 1, c1 & 1)
            want[c0, c1] = math.exp(-float(omega[0, c0]) - float(omega[1, c1])) * k[a[0], b[0]] * k[a[1], b[1]] * k[a[2], b[2]]
    want *= n_chains / want.sum()
    chi2 = float(((obs - want) ** 2 / want).sum())
    assert chi2 < 63 + 3.5 * math.sqrt(2 * 63), chi2


def test_smc_keeps_ideal_chain_statistics_and_accepts_more_than_uniform_moves():
    w = si.scaled(si.config(1), 8192, (32, 32, 32))
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_smc(A)
    acc = o.mc_steps(12)
    x, y, z = (v.astype(np.float64).reshape(w.n_chains, w.N) for v in o.positions())
    r2 = ((x[:, -1] - x[:, 0]) ** 2 + (y[:, -1] - y[:, 0]) ** 2 + (z[:, -1] - z[:, 0]) ** 2).mean()
    want = (w.N - 1) * w.b ** 2
    assert abs(r2 - want) < 3 * want * math.sqrt(2.0 / (3.0 * w.n_chains))
    d = np.diff(x, axis=1).reshape(-1)
    assert abs((d * d).mean() - w.b ** 2 / 3) < 4 * math.sqrt(2.0 / d.size) * w.b ** 2 / 3
    rate = acc / (12 * w.n_beads)
    assert 0.75 < rate < 0.999, rate                      # force-biased proposals with a small step are mostly accepted
