"""1000-step statistics (BASELINE.json `north_star`, last comparison bullet): acceptance
rate, mean squared end-to-end distance and the AB structure factor at the first three |q| shells of
the GPU run agree with the oracle's within 3 sigma; and the GPU's ideal-chain run (configs[1], full
size) reproduces the closed forms that pin the oracle itself (R_ee^2 = (N-1) b^2, acceptance rate)."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
import scmf_inputs as si
from helpers import gpu_system, mean_sq_end_to_end, structure_factor_AB

pytestmark = pytest.mark.gpu


def test_cfg0_1000_steps_statistics_within_3_sigma():
    w = si.config(0)
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(1000)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        acc_g = g.mc_steps(1000, want_accepted=True)
        gx, gy, gz = g.positions()
    ox, oy, oz = o.positions()
    moves = 1000 * w.n_beads
    p = acc_o / moves
    assert abs(acc_g / moves - p) <= 3 * math.sqrt(p * (1 - p) / moves)
    r2_g, se_g = mean_sq_end_to_end(gx, gy, gz, w.n_chains, w.N)
    r2_o, se_o = mean_sq_end_to_end(ox, oy, oz, w.n_chains, w.N)
    assert abs(r2_g - r2_o) <= 3 * math.hypot(se_g, se_o)
    types = s.bead_types()
    for (q1, s1, e1), (q2, s2, e2) in zip(structure_factor_AB(gx, gy, gz, types, w.box),
                                          structure_factor_AB(ox, oy, oz, types, w.box)):
        assert q1 == q2 and abs(s1 - s2) <= 3 * math.hypot(e1, e2) + 1e-12
    # with reading R6b the decisions are implementation-independent, so the runs are in fact identical
    assert acc_g == acc_o
    assert np.array_equal(gx, ox) and np.array_equal(gy, oy) and np.array_equal(gz, oz)


def _cube_average(f, a, n=48):
    xs, ws = np.polynomial.legendre.leggauss(n)
    X, Y, Z = np.meshgrid(a * xs, a * xs, a * xs, indexing="ij")
    W = ws[:, None, None] * ws[None, :, None] * ws[None, None, :]
    return float((W * f(np.sqrt(X * X + Y * Y + Z * Z))).sum() / 8.0)


def test_cfg1_ideal_chains_full_size_1000_steps_closed_forms():
    """configs[1]: 65,536 ideal chains of 64 beads, 1000 MC steps on the GPU alone (4.2 G moves)."""
    w = si.config(1)
    s = si.make_system(w)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        acc = g.mc_steps(1000, want_accepted=True)
        x, y, z = g.positions()
        dens = g.density()
    n, N, b, a = w.n_chains, w.N, w.b, w.move_halfwidth
    r2, _ = mean_sq_end_to_end(x, y, z, n, N)
    want = (N - 1) * b * b
    assert abs(r2 - want) <= 3 * want * math.sqrt(2.0 / (3.0 * n)), (r2, want)          # north_star check 1
    p_int = _cube_average(lambda r: special.erfc(math.sqrt(3.0) / 2.0 * r / b), a)
    p_end = _cube_average(lambda r: special.erfc(math.sqrt(3.0 / 8.0) * r / b), a)
    p = ((N - 2) * p_int + 2 * p_end) / N
    moves = 1000 * w.n_beads
    # moves of one chain are correlated in time; allow the binomial error of the chains, not of the moves
    assert abs(acc / moves - p) <= 4 * math.sqrt(p * (1 - p) / (n * N)), (acc / moves, p)
    assert int(dens.sum()) == w.n_beads                                                  # north_star check 2
    bx = np.diff(np.asarray(x, np.float64).reshape(n, N), axis=1)
    assert abs((bx * bx).mean() - b * b / 3) <= 4 * math.sqrt(2.0 / 9.0 / bx.size) * b * b   # bond components N(0, b^2/3)
