"""Pins of the oracle's polymer species of different chain lengths (R26; SURVEY 8(f) row f2 "mixed chain
lengths"; the paper's systems hold polymer, solvent and non-solvent): the layout, the closed
forms per species, conservation, the reference length in omega, and the reduction to the single-species case."""
import math

import numpy as np
import pytest

import oracle
import scmf_inputs as si


def _two_species(n0=3000, N0=32, n1=5000, N1=8, chi=0.0, kappa=0.0, seed=21, n_single=None, grid=(8, 8, 8), box=(4.0, 4.0, 4.0)):
    pats = np.zeros((2, 32), dtype=np.uint8)
    pats[0, 16:] = 1                                   # species 0: AB diblocks of 32
    pats[1, :] = 2                                     # species 1: C homopolymers of 8 (first 8 entries of the row)
    cp = np.concatenate([np.zeros(n0, np.uint8), np.ones(n1, np.uint8)])
    c = [[0, chi, chi / 2], [chi, 0, chi / 3], [chi / 2, chi / 3, 0]]
    return si.species_system([(n0, N0), (n1, N1)], 32, 3, pats, cp, c, kappa, grid, box, seed=seed, n_single=n_single)


def test_layout_conservation_and_ideal_chain_closed_forms_per_species():
    s = _two_species()
    o = oracle.Oracle.from_system(s)
    assert o.B == 3000 * 32 + 5000 * 8
    o.load_state(s.x, s.y, s.z)
    d = o.density().reshape(3, -1)
    assert d.sum(1).tolist() == [3000 * 16, 3000 * 16, 5000 * 8]            # north_star check 2, per type
    types = s.bead_types()
    # density = histogram of the positions by (type, cell), computed in float64 numpy
    x, y, z = (v.astype(np.float64) for v in (s.x, s.y, s.z))
    cell = ((np.floor(x * 2).astype(int) % 8) * 8 + np.floor(y * 2).astype(int) % 8) * 8 + np.floor(z * 2).astype(int) % 8
    for t in range(3):
        assert np.array_equal(np.bincount(cell[types == t], minlength=512), d[t])
    acc = o.mc_steps(30)                                                     # chiN = kappaN = 0: ideal chains stay ideal
    assert 0 < acc < 30 * o.B
    px, py, pz = (v.astype(np.float64) for v in o.positions())
    off = 0
    for n_s, N_s in s.species:
        sl = slice(off, off + n_s * N_s)
        cx, cy, cz = (v[sl].reshape(n_s, N_s) for v in (px, py, pz))
        r2 = (cx[:, -1] - cx[:, 0]) ** 2 + (cy[:, -1] - cy[:, 0]) ** 2 + (cz[:, -1] - cz[:, 0]) ** 2
        want = (N_s - 1) * 1.0
        assert abs(r2.mean() - want) < 3.5 * want * math.sqrt(2.0 / (3.0 * n_s)), (N_s, r2.mean())   # north_star check 1, per species
        bond2 = np.diff(cx, axis=1) ** 2 + np.diff(cy, axis=1) ** 2 + np.diff(cz, axis=1) ** 2
        assert abs(bond2.mean() - 1.0) < 4 * math.sqrt(2.0 / 3.0 / bond2.size)
        off += n_s * N_s
    assert o.density().reshape(3, -1).sum(1).tolist() == [3000 * 16, 3000 * 16, 5000 * 8]


def test_equal_lengths_reduce_to_the_single_species_system_bit_for_bit():
    """Two species of the same length are the single-species system of all their chains: same chain ids, same
    draws, same trajectory."""
    n, N = 600, 16
    pats = [[0] * 8 + [1] * 8, [1] * 16]
    cp = (np.arange(n) % 3 == 0).astype(np.uint8)
    s1 = si.custom_system(n, N, 2, pats, cp, [[0, 18], [18, 0]], 45.0, (8, 8, 8), (4.0, 4.0, 4.0), seed=5)
    o1 = oracle.Oracle.from_system(s1)
    o2 = oracle.Oracle(n, N, 2, pats, cp, 1.0, [[0, 18], [18, 0]], 45.0, (8, 8, 8), (4.0, 4.0, 4.0), 0.5, 5, species=[(250, N), (350, N)])
    for o in (o1, o2):
        o.load_state(s1.x, s1.y, s1.z)
    assert o1.mc_steps(7) == o2.mc_steps(7)
    assert all(np.array_equal(a, b) for a, b in zip(o1.positions(), o2.positions()))
    assert np.array_equal(o1.omega().view(np.uint32), o2.omega().view(np.uint32))
    o1.generate_state(77)
    o2.generate_state(77)
    assert all(np.array_equal(a, b) for a, b in zip(o1.positions(), o2.positions()))
    phi = np.random.default_rng(1).uniform(0.1, 1.0, size=(2, 512)).astype(np.float32)
    o1.init_from_density(phi, 5, n_equil_steps=3, umbrella_k=0.5)
    o2.init_from_density(phi, 5, n_equil_steps=3, umbrella_k=0.5)
    assert all(np.array_equal(a, b) for a, b in zip(o1.positions(), o2.positions()))


def test_species_zero_moves_like_the_same_chains_alone_when_nothing_interacts():
    """chiN = kappaN = 0: omega = 0, chains do not see each other, and the random stream is keyed by the chain
    id -- so the chains of species 0 (ids 0..n0-1) follow exactly the trajectory they have in a system that
    holds only them."""
    s = _two_species(n0=400, n1=900)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(5)
    nb0 = 400 * 32
    alone = oracle.Oracle(400, 32, 3, s.type_patterns[:1], None, 1.0, s.chiN, 0.0, (8, 8, 8), (4.0, 4.0, 4.0), 0.5, 21)
    alone.load_state(s.x[:nb0], s.y[:nb0], s.z[:nb0])
    alone.mc_steps(5)
    for a, b in zip(o.positions(), alone.positions()):
        assert np.array_equal(a[:nb0], b)


def test_one_move_of_a_short_chain_recomputed_by_hand():
    """Bead 3 of chain n0 + 2 (species 1, N = 8) at step 4, half-sweep 1: trial position from the Philox words of
    counter (3, n0 + 2, 4, 1), bonded to beads 2 and 4 of the same chain at bead_off + 2*8 + {2, 4}; the last bead
    (i = 7) has one neighbour only."""
    s = _two_species(n0=50, n1=40, chi=12.0, kappa=20.0)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z, step0=4)
    c = 50 + 2
    j0 = 50 * 32 + 2 * 8
    for i, parity in ((3, 1), (7, 1), (0, 0)):
        j = j0 + i
        w = oracle.philox4x32_10([i, c, 4, parity], [21, 0])
        trial, u = o.trial(j, parity)
        want = [np.float32(v) + np.float32(0.5) * np.float32(oracle.tmap(int(w[d]))) for d, v in enumerate((s.x[j], s.y[j], s.z[j]))]
        assert [float(a) for a in trial] == [float(a) for a in want]
        # energy difference in double from the neighbours that exist
        r = np.array([s.x[j], s.y[j], s.z[j]], dtype=np.float64)
        t = trial.astype(np.float64)
        dq = 0.0
        for k in ([j - 1] if i > 0 else []) + ([j + 1] if i < 7 else []):
            nb = np.array([s.x[k], s.y[k], s.z[k]], dtype=np.float64)
            dq += ((t - nb) ** 2).sum() - ((r - nb) ** 2).sum()
        om = o.omega().reshape(3, -1)[2]
        dw = float(om[o.cell_index(*trial)]) - float(om[o.cell_index(*r.astype(np.float32))])
        assert o.delta_energy(j, *trial) == pytest.approx(1.5 * dq + dw, abs=2e-5)


def test_omega_uses_the_reference_length_and_all_beads():
    s = _two_species(n0=300, n1=500, chi=9.0, kappa=30.0, n_single=[0, 0, 700])
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    B = 300 * 32 + 500 * 8 + 700
    assert o.B == B
    n = o.density().reshape(3, -1).astype(np.float64)
    phi = n * 512.0 / B
    chi = np.asarray(s.chiN, dtype=np.float64)
    tot = phi.sum(0)
    want = np.stack([(30.0 * (tot - 1.0) + sum(chi[t, u] * phi[u] for u in range(3) if u != t)) / 32.0 for t in range(3)])   # N_ref = 32
    assert np.allclose(o.omega().reshape(3, -1), want, rtol=2e-5, atol=2e-5)
    assert o.constants()["invN"] == np.float32(1.0 / 32.0)


def test_order_independence_and_checkpoint_with_species():
    s = _two_species(n0=200, n1=300, chi=10.0, kappa=25.0, n_single=[50, 0, 0])
    a, b_ = oracle.Oracle.from_system(s), oracle.Oracle.from_system(s)
    a.load_state(s.x, s.y, s.z)
    b_.load_state(s.x, s.y, s.z)
    for parity in (0, 1):
        a.half_sweep(parity, order=0)
        b_.half_sweep(parity, order=1)
    assert all(np.array_equal(u, v) for u, v in zip(a.positions(), b_.positions()))
    a.finish_step()
    a.mc_steps(3)
    x, y, z = a.positions()
    c = oracle.Oracle.from_system(s)
    c.load_state(x, y, z, step0=a.step)
    a.mc_steps(2)
    c.mc_steps(2)
    assert all(np.array_equal(u, v) for u, v in zip(a.positions(), c.positions()))


def test_species_table_is_validated():
    pats = np.zeros((1, 8), dtype=np.uint8)
    for bad in ([(3, 8), (0, 4)], [(3, 9), (2, 4)], [(3, 8), (3, 4)]):        # empty species, longer than the pattern row, wrong total
        with pytest.raises((ValueError, AssertionError)):
            oracle.Oracle(5, 8, 1, pats, None, 1.0, [[0]], 0.0, (4, 4, 4), (2.0, 2.0, 2.0), 0.5, 1, species=bad)
