"""Pins of the oracle's target-density initialisation and umbrella potential (R25; SURVEY 8(f) row
f4; "generating particle positions that reproduce the supplied concentration fields ... placed
within half a mean end-to-end distance of their target positions and equilibrated using an umbrella
potential").  What the passage and the mathematics fix: the placed density follows the target (multinomial),
every chain's centre of mass sits at its target point so that all beads are within about R_e/2 of it, the chain
shape is the configs' Gaussian random walk, the umbrella term is k (phi - phi*) added to omega -- the derivative
of (k/2)(B/C) sum (phi - phi*)^2 -- and it pulls the density toward the target."""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats

import oracle
import scmf_inputs as si


def _target(grid, T, rng, kind="lamellae"):
    nx, ny, nz = grid
    ix = np.arange(nx)[:, None, None] + np.zeros((nx, ny, nz))
    if kind == "lamellae":                       # A-rich and B-rich slabs along x, an empty stripe in A
        a = 0.5 + 0.45 * np.cos(2 * np.pi * ix / nx)
        phi = np.stack([a, 1.0 - a][:T] + [np.full((nx, ny, nz), 0.3)] * max(0, T - 2))
        phi[0, 1] = 0.0
    else:
        phi = rng.uniform(0.0, 2.0, size=(T, nx, ny, nz))
    return phi.reshape(T, -1).astype(np.float32)


def test_single_bead_species_follow_the_target_multinomially():
    """N = 1 'chains' of type 0 and single-bead molecules of type 1: every molecule sits exactly at its target
    point, so the cell occupancies are one multinomial draw with p(c) = Q_t(c) / sum Q_t (chi-square), and the
    empty stripe of the target stays empty."""
    grid, box = (8, 4, 4), (4.0, 2.0, 2.0)
    n0, n1 = 60000, 40000
    s = si.custom_system(n0, 1, 2, [[0]], None, [[0, 0], [0, 0]], 0.0, grid, box, seed=5, n_single=[0, n1])
    o = oracle.Oracle.from_system(s)
    phi = _target(grid, 2, np.random.default_rng(1))
    o.init_from_density(phi, gen_seed=99)
    dens = o.density().reshape(2, -1).astype(np.int64)
    assert dens[0].sum() == n0 and dens[1].sum() == n1
    for t, n in ((0, n0), (1, n1)):
        q = np.rint(phi[t].astype(np.float64) * 65536.0)
        p = q / q.sum()
        assert np.all(dens[t][p == 0] == 0)
        keep = p > 0
        chi2 = (((dens[t][keep] - n * p[keep]) ** 2) / (n * p[keep])).sum()
        assert stats.chi2.sf(chi2, keep.sum() - 1) > 1e-4
        # and every cell within 5 sigma on its own
        assert np.all(np.abs(dens[t][keep] - n * p[keep]) < 5 * np.sqrt(n * p[keep] * (1 - p[keep])) + 1)


def test_target_cell_is_the_inverse_cdf_of_the_integer_weights():
    """The cell of every molecule recomputed with exact rational arithmetic from the Philox words (the
    generator itself is pinned by its known-answer vectors): k = floor(u64 S / 2^64), first prefix > k."""
    grid, box = (4, 2, 4), (2.0, 1.0, 2.0)
    n = 300
    rng = np.random.default_rng(3)
    phi = _target(grid, 2, rng, "random")
    phi[1, 5] = 0.0
    s = si.custom_system(n, 1, 2, [[0], [1]], np.arange(n) % 2, [[0, 0], [0, 0]], 0.0, grid, box, seed=6)
    o = oracle.Oracle.from_system(s)
    o.init_from_density(phi, gen_seed=0xABCDEF0123)
    x, y, z = o.positions()
    key = [0xABCDEF0123 & 0xFFFFFFFF, 0xABCDEF0123 >> 32]
    for c in range(n):
        t = c % 2
        q = [int(v) for v in np.rint(phi[t].astype(np.float64) * 65536.0)]
        prefix = np.cumsum(q).tolist()
        w = oracle.philox4x32_10([0, c, 0, 3 << 8], key)
        v = oracle.philox4x32_10([1, c, 0, 3 << 8], key)
        k = ((int(w[0]) << 32 | int(w[1])) * prefix[-1]) >> 64
        cell = next(i for i, pv in enumerate(prefix) if pv > k)
        ix, iy, iz = cell // (grid[1] * grid[2]), (cell // grid[2]) % grid[1], cell % grid[2]
        U = lambda a: (Fraction(int(a)) + Fraction(1, 2)) / 2 ** 32
        want = [float((ix + U(w[2])) * Fraction(1, 2)), float((iy + U(w[3])) * Fraction(1, 2)), float((iz + U(v[0])) * Fraction(1, 2))]
        got = [float(x[c]), float(y[c]), float(z[c])]
        assert got == [float(np.float32(a)) for a in want], (c, got, want)
        assert o.cell_index(*got) == cell


def test_chains_are_centred_on_their_target_and_keep_the_random_walk_shape():
    n, N, b = 20000, 16, 0.9
    grid, box = (8, 8, 4), (8.0, 8.0, 4.0)
    s = si.custom_system(n, N, 2, [[0] * 8 + [1] * 8, [1] * 16], (np.arange(n) % 4 == 0).astype(np.uint8), [[0, 10], [10, 0]], 30.0,
                         grid, box, seed=8, b=b)
    o = oracle.Oracle.from_system(s)
    phi = _target(grid, 2, np.random.default_rng(2))
    o.init_from_density(phi, gen_seed=4242)
    x, y, z = (v.reshape(n, N).astype(np.float64) for v in o.positions())
    com = np.stack([x.mean(1), y.mean(1), z.mean(1)], axis=1)
    assert np.all(com >= -1e-5) and np.all(com < np.array(box) + 1e-5)            # target points lie in the box
    # centre-of-mass cells follow the pattern's weights: pattern 0 (diblock) ~ 8 Q_A + 8 Q_B, pattern 1 ~ 16 Q_B
    q = np.rint(phi.astype(np.float64) * 65536.0)
    h = np.array(box) / np.array(grid)
    cells = ((np.floor(com[:, 0] / h[0]).astype(int) % grid[0]) * grid[1] + np.floor(com[:, 1] / h[1]).astype(int) % grid[1]) * grid[2] \
        + np.floor(com[:, 2] / h[2]).astype(int) % grid[2]
    for pat, wgt in ((0, 8 * q[0] + 8 * q[1]), (1, 16 * q[1])):
        sel = (np.arange(n) % 4 == 0) == bool(pat)
        cnt = np.bincount(cells[sel], minlength=q.shape[1])
        p = wgt / wgt.sum()
        keep = p > 0
        assert np.all(cnt[~keep] == 0)
        chi2 = (((cnt[keep] - sel.sum() * p[keep]) ** 2) / (sel.sum() * p[keep])).sum()
        assert stats.chi2.sf(chi2, keep.sum() - 1) > 1e-4
    # "within half a mean end-to-end distance of their target positions": rms distance of a bead from the
    # centre of mass is R_g = R_e / sqrt 6 < R_e / 2, R_e^2 = (N - 1) b^2 (<R_g^2> of an ideal chain of N beads
    # = b^2 (N^2 - 1) / (6 N))
    rg2 = ((x - com[:, :1]) ** 2 + (y - com[:, 1:2]) ** 2 + (z - com[:, 2:]) ** 2).mean()
    want = b * b * (N * N - 1) / (6.0 * N)
    assert abs(rg2 - want) < 0.02 * want
    assert math.sqrt(rg2) < 0.5 * math.sqrt((N - 1) * b * b)
    # the shape is the configs' Gaussian random walk: bond components N(0, b^2/3), <R_ee^2> = (N-1) b^2
    for v in (x, y, z):
        d = np.diff(v, axis=1).reshape(-1) / (b / math.sqrt(3.0))
        assert abs(d.mean()) < 4 / math.sqrt(d.size) and abs((d * d).mean() - 1.0) < 4 * math.sqrt(2.0 / d.size)
        assert stats.kstest(d[:100000], "norm").pvalue > 1e-4
    r2 = (x[:, -1] - x[:, 0]) ** 2 + (y[:, -1] - y[:, 0]) ** 2 + (z[:, -1] - z[:, 0]) ** 2
    assert abs(r2.mean() - (N - 1) * b * b) < 3 * (N - 1) * b * b * math.sqrt(2.0 / (3.0 * n))
    # the same walk as the plain generator's (same domain-1 draws): bond vectors are identical up to the fp32
    # rounding of the shifted coordinates
    o2 = oracle.Oracle.from_system(s)
    o2.generate_state(4242)
    x2 = o2.positions()[0].reshape(n, N).astype(np.float64)
    assert np.abs(np.diff(x, axis=1) - np.diff(x2, axis=1)).max() < 4e-6
    assert int(o.density().sum()) == n * N and o.step == 0


def test_bad_targets_are_refused_and_the_call_is_deterministic():
    grid, box = (4, 4, 4), (2.0, 2.0, 2.0)
    s = si.custom_system(50, 4, 2, [[0, 0, 1, 1]], None, [[0, 5], [5, 0]], 10.0, grid, box, seed=3)
    o = oracle.Oracle.from_system(s)
    phi = np.ones((2, 64), dtype=np.float32)
    for bad in (-0.1, np.nan, 65536.0):
        p = phi.copy()
        p[1, 7] = bad
        with pytest.raises(ValueError):
            o.init_from_density(p, 1)
    with pytest.raises(ValueError):
        o.init_from_density(np.zeros((2, 64), dtype=np.float32), 1)         # nothing to place the chains by
    o.init_from_density(phi, 17, step0=5)
    a = [v.copy() for v in o.positions()]
    o2 = oracle.Oracle.from_system(s)
    o2.init_from_density(phi, 17, step0=5)
    assert all(np.array_equal(u, v) for u, v in zip(a, o2.positions())) and o.step == 5
    o2.init_from_density(phi, 18)
    assert not np.array_equal(a[0], o2.positions()[0])


def test_umbrella_term_is_the_derivative_of_its_quadratic_potential():
    """omega with the umbrella = omega without + k (phi - phi*), checked against a finite difference of
    H_umb = (k/2)(B/C) sum (phi - phi*)^2 in double; k = 0 or no target changes nothing, bit for bit."""
    grid, box = (2, 2, 2), (1.0, 1.0, 1.0)
    s = si.custom_system(40, 4, 2, [[0, 0, 1, 1]], None, [[0, 7], [7, 0]], 12.0, grid, box, seed=4)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    w0 = o.omega().copy()
    rng = np.random.default_rng(5)
    tgt = rng.uniform(0.2, 1.8, size=(2, 8)).astype(np.float32)
    k = 3.5
    o.set_umbrella(tgt, k)
    w1 = o.omega().copy()
    n = o.density().reshape(2, 8).astype(np.float64)
    B, Cn = 160.0, 8.0

    def H(nn):
        return 0.5 * k * (B / Cn) * (((nn * Cn / B) - tgt.astype(np.float64)) ** 2).sum()

    for t in range(2):
        for c in range(8):
            up, dn = n.copy(), n.copy()
            up[t, c] += 0.5
            dn[t, c] -= 0.5
            assert (w1 - w0).reshape(2, 8)[t, c] == pytest.approx(H(up) - H(dn), abs=2e-5)
    o.set_umbrella(tgt, 0.0)
    assert np.array_equal(o.omega().view(np.uint32), w0.view(np.uint32))
    o.set_umbrella(tgt, k)
    o.set_umbrella(None, 0.0)
    assert np.array_equal(o.omega().view(np.uint32), w0.view(np.uint32))
    # with an external field as well: the umbrella term is added last
    ext = rng.normal(0, 1, size=(2, 8)).astype(np.float32)
    o.set_external_field(ext)
    we = o.omega().copy()
    o.set_umbrella(tgt, k)
    phi = (o.density().reshape(2, 8).astype(np.float32) * np.float32(o.constants()["dens_scale"]))
    assert np.array_equal(o.omega().reshape(2, 8), we.reshape(2, 8) + np.float32(k) * (phi - tgt))


def test_umbrella_equilibration_pulls_the_density_toward_the_target():
    """Non-interacting beads (chiN = kappaN = 0) started uniformly under the umbrella potential toward a
    modulated target: the stationary density is the self-consistent Boltzmann distribution
    phi(c) = exp(-k (phi(c) - phi*(c))) / Z (mean-field is exact for an ideal gas at ~300 beads per cell), far
    closer to the target than free diffusion leaves it; afterwards the umbrella is gone (omega = 0 again)."""
    grid, box = (8, 4, 4), (4.0, 2.0, 2.0)
    n, k = 40000, 0.5        # small k: the fluctuation corrections to mean field (~k^2 / beads per cell) stay below the tolerance
    s = si.custom_system(n, 1, 1, [[0]], None, [[0]], 0.0, grid, box, seed=9)
    tgt = _target(grid, 2, np.random.default_rng(1))[:1].copy()
    tgt[0] = np.where(tgt[0] == 0, 0.05, tgt[0])
    tgt *= 128.0 / tgt.sum()                                  # mean concentration 1
    uni = np.ones((1, 128), dtype=np.float32)

    def phi_of(o):
        return o.density().reshape(-1) * 128.0 / n

    def err(o):
        return float(((phi_of(o) - tgt[0]) ** 2).mean())

    o = oracle.Oracle.from_system(s)
    o.init_from_density(uni, 7)                               # uniform start
    e_start = err(o)
    o.set_umbrella(tgt, k)
    o.mc_steps(300)
    acc = np.zeros(128)
    for _ in range(100):                                      # time average over the stationary state
        o.mc_steps(1)
        acc += phi_of(o)
    acc /= 100
    o.set_umbrella(tgt, 2.0)                                  # a stiffer umbrella pulls closer
    o.mc_steps(100)
    o.set_umbrella(None, 0.0)
    e_umb = err(o)
    assert np.all(o.omega() == 0.0)                           # chiN = kappaN = 0 and no umbrella left
    fp = np.ones(128)
    for _ in range(2000):                                     # damped fixed-point iteration of the self-consistent equation
        new = np.exp(-k * (fp - tgt[0].astype(np.float64)))
        fp = 0.9 * fp + 0.1 * new * 128.0 / new.sum()
    slab = lambda v: v.reshape(8, 16).mean(1)
    assert np.abs(slab(acc) - slab(fp)).max() < 0.01, (slab(acc), slab(fp))
    assert np.abs(slab(fp) - 1.0).max() > 0.25                # and that is far from the uniform start
    o2 = oracle.Oracle.from_system(s)
    o2.init_from_density(uni, 7)
    o2.mc_steps(100)
    e_free = err(o2)
    assert e_umb < 0.5 * e_start and e_umb < 0.5 * e_free
    # the one-call form is placement + set_umbrella + mc_steps + umbrella off
    o3 = oracle.Oracle.from_system(s)
    o3.init_from_density(uni, 7, n_equil_steps=100, umbrella_k=0.0)
    assert np.array_equal(o3.positions()[0], o2.positions()[0]) and o3.step == 100
    o4 = oracle.Oracle.from_system(s)
    o4.init_from_density(tgt, 7, n_equil_steps=30, umbrella_k=k)
    o5 = oracle.Oracle.from_system(s)
    o5.init_from_density(tgt, 7)
    o5.set_umbrella(tgt, k)
    o5.mc_steps(30)
    o5.set_umbrella(None, 0.0)
    assert np.array_equal(o4.positions()[0], o5.positions()[0])
    assert np.array_equal(o4.omega(), o5.omega()) and o4.step == 30
