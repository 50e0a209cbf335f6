"""Pins for the oracle's cell index, binning and omega (DESIGN.md section 2 steps 1-3; R2, R8-R10, R12).

Expected values come from hand placement, conservation laws, special cases and an independent
double-precision evaluation of the grid Hamiltonian of R2 -- never from the oracle's own formula.
"""
import itertools

import numpy as np
import pytest

import oracle
import scmf_inputs as si


def _tiny(n_chains=1, N=4, T=2, grid=(4, 4, 4), box=(2.0, 2.0, 2.0), chiN=None, kappaN=50.0, pats=None,
          chain_pattern=None, seed=11):
    if pats is None:
        pats = np.array([[i * T // N for i in range(N)]], dtype=np.uint8)
    if chiN is None:
        chiN = np.full((T, T), 20.0, dtype=np.float32)
        np.fill_diagonal(chiN, 0)
    return oracle.Oracle(n_chains, N, T, pats, chain_pattern, 1.0, chiN, kappaN, grid, box, 0.5, seed)


def test_cell_index_layout_and_boundaries():
    # R12: cell = (ix*ny + iy)*nz + iz.  R8: floor (not truncation), face belongs to the upper
    # cell, periodic wrap by a non-negative modulo.  Non-cubic grid so a swapped axis shows up.
    o = _tiny(grid=(2, 3, 4), box=(1.0, 1.5, 2.0))        # h = 0.5 on every axis
    ny, nz = 3, 4
    idx = lambda ix, iy, iz: (ix * ny + iy) * nz + iz
    assert o.cell_index(0.25, 0.25, 0.25) == idx(0, 0, 0)
    assert o.cell_index(0.75, 0.25, 0.25) == idx(1, 0, 0)
    assert o.cell_index(0.25, 1.25, 0.25) == idx(0, 2, 0)
    assert o.cell_index(0.25, 0.25, 1.75) == idx(0, 0, 3)
    assert o.cell_index(0.5, 0.5, 0.5) == idx(1, 1, 1)            # on a face: upper cell
    assert o.cell_index(-0.0, 0.0, 0.0) == idx(0, 0, 0)
    assert o.cell_index(-1e-7, 0.0, 0.0) == idx(1, 0, 0)          # just below 0 wraps to the top
    assert o.cell_index(0.0, -1e-7, 0.0) == idx(0, 2, 0)
    assert o.cell_index(0.0, 0.0, -0.25) == idx(0, 0, 3)
    assert o.cell_index(1.0, 1.5, 2.0) == idx(0, 0, 0)            # r = L wraps to 0
    assert o.cell_index(np.nextafter(np.float32(1.0), np.float32(0)), 0.0, 0.0) == idx(1, 0, 0)
    assert o.cell_index(2.0, 3.0, 4.0) == idx(0, 0, 0)            # r = 2L
    assert o.cell_index(-1.0 - 0.25, -1.5 - 0.25, -2.0 - 0.25) == idx(1, 2, 3)
    assert o.cell_index(7.25, -7.25, 101.3) == idx(14 % 2, (-15) % 3, 202 % 4)


def test_bin_hand_placed_beads():
    # 2 chains of 3 beads, pattern A A B; beads placed by hand, some outside the box.
    pats = np.array([[0, 0, 1]], dtype=np.uint8)
    o = _tiny(n_chains=2, N=3, T=2, grid=(2, 2, 2), box=(1.0, 1.0, 1.0), pats=pats)
    x = np.array([0.1, 0.6, 0.6, -0.1, 1.1, 0.25], dtype=np.float32)
    y = np.array([0.1, 0.1, 0.6, 0.1, 0.1, 0.25], dtype=np.float32)
    z = np.array([0.1, 0.1, 0.6, 0.1, 0.1, 2.75], dtype=np.float32)
    o.load_state(x, y, z)
    want = np.zeros((2, 8), dtype=np.uint32)
    cell = lambda ix, iy, iz: (ix * 2 + iy) * 2 + iz
    want[0, cell(0, 0, 0)] += 1      # chain 0 bead 0 (A)
    want[0, cell(1, 0, 0)] += 1      # chain 0 bead 1 (A)
    want[1, cell(1, 1, 1)] += 1      # chain 0 bead 2 (B)
    want[0, cell(1, 0, 0)] += 1      # chain 1 bead 0 (A) at x=-0.1 -> wraps to ix=1
    want[0, cell(0, 0, 0)] += 1      # chain 1 bead 1 (A) at x=1.1 -> ix=0
    want[1, cell(0, 0, 1)] += 1      # chain 1 bead 2 (B) at z=2.75 -> iz=1
    assert np.array_equal(o.density(), want)


@pytest.mark.parametrize("cfg", [0])
def test_density_sums_to_bead_counts_exactly(cfg):
    # north_star oracle check 2: "the density grids sum to the total bead count exactly".
    s = si.make_system(si.config(cfg))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    types = s.bead_types()
    for step in range(3):
        d = o.density()
        assert int(d.sum()) == s.workload.n_beads
        for t in range(s.workload.n_types):
            assert int(d[t].sum()) == int((types == t).sum())
        o.mc_steps(1)


def test_density_matches_numpy_histogram_of_float64_cells():
    # Independent route: cell coordinates by float64 floor + Python modulo, counted by bincount.
    # (positions of this workload are far from cell faces in fp32 terms except by chance; the
    # fp32 product r*inv_h is exact here because inv_h = 2.)
    w = si.scaled(si.config(3), 512, (8, 8, 8))
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(2)
    x, y, z = o.positions()
    g = [np.floor(v.astype(np.float64) * 2.0).astype(np.int64) % 8 for v in (x, y, z)]
    cell = (g[0] * 8 + g[1]) * 8 + g[2]
    types = s.bead_types()
    want = np.stack([np.bincount(cell[types == t], minlength=512) for t in range(2)])
    assert np.array_equal(o.density().astype(np.int64), want)


def test_omega_special_cases():
    # R2/R10 special cases: homogeneous n_A = n_B = nbar/2 -> omega = chiN/(2N);
    # empty cell -> omega = -kappaN/N; chiN = kappaN = 0 -> omega == 0 exactly.
    N, n_chains, grid = 8, 16, (2, 2, 2)                          # B = 128, C = 8, nbar = 16
    o = _tiny(n_chains=n_chains, N=N, T=2, grid=grid, box=(1.0, 1.0, 1.0), kappaN=50.0)
    counts = np.full((2, 8), 8, dtype=np.uint32)
    counts[:, 3] = 0                                              # one empty cell
    o.set_density(counts)
    o.compute_omega()
    om = o.omega()
    assert np.allclose(np.delete(om, 3, axis=1), 20.0 / (2 * N), rtol=0, atol=1e-6)
    assert np.allclose(om[:, 3], -50.0 / N, rtol=0, atol=1e-6)
    z = _tiny(n_chains=n_chains, N=N, T=2, grid=grid, box=(1.0, 1.0, 1.0), kappaN=0.0,
              chiN=np.zeros((2, 2), dtype=np.float32))
    z.set_density(np.arange(16, dtype=np.uint32).reshape(2, 8))
    z.compute_omega()
    assert np.all(z.omega() == 0.0)


def _H_nb(counts, chiN, kappaN, N, nbar):
    """Grid Hamiltonian of DESIGN.md R2 in double:
    H/kT = (nbar/N) * sum_c [ kappaN/2 (sum_s phi_s - 1)^2 + sum_{s<t} chiN_st phi_s phi_t ]."""
    phi = counts.astype(np.float64) / nbar
    T = counts.shape[0]
    tot = phi.sum(axis=0)
    h = 0.5 * kappaN * (tot - 1.0) ** 2
    for s in range(T):
        for t in range(s + 1, T):
            h = h + chiN[s, t] * phi[s] * phi[t]
    return nbar / N * h.sum()


@pytest.mark.parametrize("T", [1, 2, 3])
def test_omega_is_the_derivative_of_the_grid_hamiltonian(T):
    # Brute force on a 2x2x2 grid: omega_t(c) = [H(n_t(c)+1) - H(n_t(c)-1)]/2 exactly, because H
    # is quadratic in the counts.  Asymmetric chiN-free check of the index order chiN[t][s].
    rng = np.random.default_rng(100 + T)
    N, n_chains = 6, 20
    B, Cn = N * n_chains, 8
    nbar = B / Cn
    chi = rng.uniform(1.0, 30.0, size=(T, T))
    chi = np.triu(chi, 1)
    chi = (chi + chi.T).astype(np.float32)
    kappaN = 37.0
    pats = np.array([[i % T for i in range(N)]], dtype=np.uint8)
    o = _tiny(n_chains=n_chains, N=N, T=T, grid=(2, 2, 2), box=(1.0, 1.0, 1.0), chiN=chi, kappaN=kappaN, pats=pats)
    counts = rng.integers(1, 30, size=(T, Cn)).astype(np.uint32)
    o.set_density(counts)
    o.compute_omega()
    om = o.omega()
    for t, c in itertools.product(range(T), range(Cn)):
        up, dn = counts.astype(np.int64).copy(), counts.astype(np.int64).copy()
        up[t, c] += 1
        dn[t, c] -= 1
        want = 0.5 * (_H_nb(up, chi.astype(np.float64), kappaN, N, nbar) - _H_nb(dn, chi.astype(np.float64), kappaN, N, nbar))
        assert abs(om[t, c] - want) < 2e-5 * max(1.0, abs(want)), (t, c, om[t, c], want)


def test_load_state_bins_and_computes_omega():
    s = si.make_system(si.config(0))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z, step0=17)
    assert o.step == 17
    d = o.density()
    assert d.sum() == s.workload.n_beads
    # omega of the loaded state, by the route of the previous test (double, from the counts)
    N, nbar = s.workload.N, s.workload.n_beads / s.workload.n_cells
    phi = d.astype(np.float64) / nbar
    want0 = (s.workload.kappaN * (phi.sum(axis=0) - 1.0) + s.workload.chiN * phi[1]) / N
    want1 = (s.workload.kappaN * (phi.sum(axis=0) - 1.0) + s.workload.chiN * phi[0]) / N
    om = o.omega()
    assert np.allclose(om[0], want0, rtol=0, atol=5e-6)
    assert np.allclose(om[1], want1, rtol=0, atol=5e-6)


# ---- external field (R21) ------------------------------------------

def test_external_field_boltzmann_occupancy_of_single_bead_molecules():
    """Single-bead molecules (N = 1) without interactions in a cell-wise constant external field are
    independent Metropolis walkers with stationary density proportional to exp(-ext(cell)): after a
    burn-in the cell occupancies are one multinomial draw from those weights (chi^2, 63 dof)."""
    from scipy import stats
    n, grid, box = 200_000, (4, 4, 4), (2.0, 2.0, 2.0)
    s = si.custom_system(n, 1, 1, [[0]], None, [[0.0]], 0.0, grid, box, seed=77)
    rng = np.random.default_rng(5)
    ext = rng.uniform(0.0, 2.0, size=(1, 64)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_external_field(ext)
    assert np.array_equal(o.omega(), ext)                       # no interactions: omega is the field itself
    o.mc_steps(120)
    counts = o.density().reshape(-1).astype(np.float64)
    p = np.exp(-ext.astype(np.float64).reshape(-1))
    p /= p.sum()
    chi2 = float(((counts - n * p) ** 2 / (n * p)).sum())
    assert chi2 < stats.chi2.ppf(1 - 1e-4, df=63), chi2
    # the field matters: against uniform weights the same counts are wildly off
    assert float(((counts - n / 64) ** 2 / (n / 64)).sum()) > 50 * 63


def test_external_field_adds_to_omega_in_fp32_and_can_be_removed():
    s = si.make_system(si.config(0))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    base = o.omega().copy()
    ext = np.random.default_rng(9).normal(0.0, 0.7, size=base.shape).astype(np.float32)
    o.set_external_field(ext)
    assert np.array_equal(o.omega().view(np.uint32), (base + ext).view(np.uint32))   # one fp32 add per cell
    o.mc_steps(2)                                                # the field persists across steps
    o2 = oracle.Oracle.from_system(s)
    o2.load_state(*o.positions(), step0=2)
    assert np.array_equal(o.omega() - o2.omega(), (o2.omega() + ext) - o2.omega())
    o.set_external_field(None)
    assert np.array_equal(o.omega().view(np.uint32), o2.omega().view(np.uint32))
    o.set_external_field(np.zeros_like(ext))                     # a zero field changes nothing, bit for bit
    assert np.array_equal(o.omega().view(np.uint32), o2.omega().view(np.uint32))


# ---- single-bead molecules next to chains (R23) --------------------

def _mixture(n_chains=300, n_single=(500, 0, 1200), seed=21, chi=None, kappaN=0.0, grid=(4, 4, 4), box=(2.0, 2.0, 2.0)):
    chi = np.zeros((3, 3)) if chi is None else chi
    return si.custom_system(n_chains, 8, 3, [[0, 0, 0, 0, 1, 1, 1, 1]], None, chi, kappaN, grid, box, seed=seed, n_single=n_single)


def test_single_bead_molecules_are_counted_by_type_and_normalise_the_density():
    s = _mixture()
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    d = o.density()
    assert d[0].sum() == 300 * 4 + 500 and d[1].sum() == 300 * 4 and d[2].sum() == 1200
    B = 300 * 8 + 1700
    assert o.constants()["dens_scale"] == np.float32(64 / B)              # phi normalised by ALL beads (R10)
    # histogram of the returned positions, type by type
    x, y, z = o.positions()
    cells = [o.cell_index(a, b_, c) for a, b_, c in zip(x, y, z)]
    types = s.bead_types()
    for t in range(3):
        assert np.array_equal(np.bincount(np.asarray(cells)[types == t], minlength=64), d[t])
    o.mc_steps(3)
    assert o.density().sum() == B


def test_single_bead_molecules_follow_the_boltzmann_weights_of_their_own_field():
    """Non-interacting mixture in an external field that differs by type: the solvent species (type 2)
    equilibrates to exp(-ext_2), untouched by the chains and by the other species' field."""
    from scipy import stats
    s = _mixture(n_chains=50, n_single=(20000, 0, 150000), seed=22)
    ext = np.random.default_rng(8).uniform(0.0, 1.5, size=(3, 64)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_external_field(ext)
    o.mc_steps(120)
    x, y, z = o.positions()
    types = s.bead_types()
    nN = 50 * 8
    for t, n in ((0, 20000), (2, 150000)):
        sel = np.flatnonzero(types == t)
        sel = sel[sel >= nN]                                              # the single-bead molecules of that type
        cells = np.array([o.cell_index(x[j], y[j], z[j]) for j in sel])
        counts = np.bincount(cells, minlength=64).astype(np.float64)
        p = np.exp(-ext[t].astype(np.float64)); p /= p.sum()
        chi2 = float(((counts - n * p) ** 2 / (n * p)).sum())
        assert chi2 < stats.chi2.ppf(1 - 1e-4, df=63), (t, chi2)


def test_single_bead_moves_are_order_independent_and_use_their_own_stream():
    s = _mixture(chi=np.array([[0, 8, 3], [8, 0, 5], [3, 5, 0.0]]), kappaN=20.0, seed=23)
    a = oracle.Oracle.from_system(s); a.load_state(s.x, s.y, s.z)
    b = oracle.Oracle.from_system(s); b.load_state(s.x, s.y, s.z)
    a.half_sweep(0, order=0); b.half_sweep(0, order=1)
    assert all(np.array_equal(u, v) for u, v in zip(a.positions(), b.positions()))
    # molecule m draws the stream of (bead 0, chain n_chains + m): check one trial position by hand
    c = oracle.Oracle.from_system(s); c.load_state(s.x, s.y, s.z)
    j = 300 * 8 + 7
    w = oracle.philox4x32_10([0, 300 + 7, 0, 0], [s.workload.seed & 0xffffffff, s.workload.seed >> 32])
    want = np.float32(s.x[j]) + np.float32(0.5) * np.float32(oracle.tmap(int(w[0])))
    c.set_omega(np.zeros((3, 64), np.float32))                            # dE = 0: every move is accepted
    c.half_sweep(0)
    assert c.positions()[0][j] == want
