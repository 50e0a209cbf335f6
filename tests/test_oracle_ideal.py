"""Closed-form pins on ideal chains (chiN = kappaN = 0, omega == 0): north_star oracle checks 1 and 3.

The Gaussian random-walk start is already the stationary distribution of the bonded Hamiltonian
H_b/kT = (3/(2 b^2)) sum |r_i - r_{i+1}|^2 (R1), so every closed form below must hold
after any number of Monte-Carlo steps -- and would drift if the bond constant, a sign in dE, a
neighbour index or the acceptance rule were wrong.
"""
import math

import numpy as np
from scipy import special, stats

import oracle
import scmf_inputs as si


def _ideal(n_chains=8192, N=64, steps=12, seed=2):
    w = si.scaled(si.config(1), n_chains, (16, 16, 16))
    w = w.__class__(**{**w.__dict__, "seed": seed})
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc = o.mc_steps(steps)
    return w, s, o, acc


def test_ideal_chain_end_to_end_distance_and_bond_statistics():
    w, s, o, _ = _ideal()
    n, N, b = w.n_chains, w.N, w.b
    assert np.all(o.omega() == 0.0)                                  # cfg 1: omega == 0 exactly
    x, y, z = (v.astype(np.float64).reshape(n, N) for v in o.positions())
    x0 = s.x.astype(np.float64).reshape(n, N)
    assert np.mean(np.abs(x - x0)) > 0.3                             # the chains really moved
    # check 1: <R_ee^2> = (N-1) b^2, single-time standard error (N-1) b^2 sqrt(2/(3n))
    r2 = (x[:, -1] - x[:, 0]) ** 2 + (y[:, -1] - y[:, 0]) ** 2 + (z[:, -1] - z[:, 0]) ** 2
    want = (N - 1) * b * b
    se = want * math.sqrt(2.0 / (3.0 * n))
    assert abs(r2.mean() - want) < 3 * se, (r2.mean(), want, se)
    # check 3: bond components ~ N(0, b^2/3): <l^2> = b^2, <l^4> = 5/3 b^4, <l> = b sqrt(8/(3 pi))
    l2 = np.diff(x, axis=1) ** 2 + np.diff(y, axis=1) ** 2 + np.diff(z, axis=1) ** 2
    m = l2.size
    assert abs(l2.mean() - b * b) < 4 * math.sqrt(2.0 / 3.0 / m) * b * b
    var_l4 = (35.0 / 3.0 - 25.0 / 9.0)                               # Var(l^4) = <l^8> - <l^4>^2 for chi_3 scaled
    assert abs((l2 ** 2).mean() - 5.0 / 3.0) < 4 * math.sqrt(var_l4 / m)
    l = np.sqrt(l2)
    assert abs(l.mean() - math.sqrt(8.0 / (3.0 * math.pi))) < 4 * math.sqrt((1 - 8 / (3 * math.pi)) / m)
    # Maxwell distribution of the bond length: chi-square on 40 equiprobable bins
    sample = l.reshape(-1)[:: 7][:60000]                             # thinned: neighbouring bonds correlate weakly
    edges = stats.maxwell.ppf(np.linspace(0, 1, 41), scale=b / math.sqrt(3.0))
    obs, _ = np.histogram(sample, bins=edges)
    chi2 = float(((obs - sample.size / 40) ** 2 / (sample.size / 40)).sum())
    assert chi2 < 39 + 4 * math.sqrt(2 * 39), chi2
    # each Cartesian bond component is Gaussian with variance b^2/3 and zero mean
    for v in (x, y, z):
        d = np.diff(v, axis=1)
        assert abs(d.mean()) < 4 * math.sqrt(1 / 3 / m)
        assert abs((d * d).mean() - 1 / 3) < 4 * math.sqrt(2 / 9 / m)


def _cube_average(f, a, n=48):
    xs, ws = np.polynomial.legendre.leggauss(n)
    X, Y, Z = np.meshgrid(a * xs, a * xs, a * xs, indexing="ij")
    W = ws[:, None, None] * ws[None, :, None] * ws[None, None, :]
    return float((W * f(np.sqrt(X * X + Y * Y + Z * Z))).sum() / 8.0)


def test_ideal_chain_acceptance_rate_closed_form():
    # For a uniform cube proposal of half-width a on an equilibrated ideal chain, dE given the
    # displacement d is Gaussian with variance = 2 x mean (interior bead: mean 3|d|^2/b^2; end bead:
    # mean 1.5|d|^2/b^2), hence <min(1, e^-dE)> = erfc(sqrt(mean)/2... ) exactly:
    #   interior: erfc( (sqrt 3 / 2) |d|/b ),   end: erfc( sqrt(3/8) |d|/b ),
    # averaged over the cube by Gauss-Legendre quadrature.
    w, s, o, acc = _ideal(n_chains=4096, N=64, steps=10, seed=12)
    a, b, N = w.move_halfwidth, w.b, w.N
    p_int = _cube_average(lambda r: special.erfc(math.sqrt(3.0) / 2.0 * r / b), a)
    p_end = _cube_average(lambda r: special.erfc(math.sqrt(3.0 / 8.0) * r / b), a)
    assert 0.55 < p_int < 0.58 and 0.67 < p_end < 0.70                # SURVEY 8(c)-C estimates 0.562 / 0.680
    want = ((N - 2) * p_int + 2 * p_end) / N
    moves = 10 * w.n_beads
    rate = acc / moves
    se = math.sqrt(want * (1 - want) / moves)
    assert abs(rate - want) < 4 * se, (rate, want, se)
