"""Polymer species of different chain lengths in one system (soma_params.n_species; SURVEY 8(f) row f2 "mixed
chain lengths"; R26) against the oracle: every kernel path, re-ordering, generated and placed states."""
import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system

pytestmark = pytest.mark.gpu


def _pats(rows, n_max):
    out = np.zeros((len(rows), n_max), dtype=np.uint8)
    for k, r in enumerate(rows):
        out[k, :len(r)] = r
    return out


def _mix(species, rows, chi, kappa, grid, box, seed, n_single=None, N_ref=None, b=1.0):
    """chains of species k take pattern k"""
    n_max = max(c for _, c in species)
    cp = np.concatenate([np.full(n, k, dtype=np.uint8) for k, (n, _) in enumerate(species)])
    T = len(chi)
    return si.species_system(species, N_ref or species[0][1], T, _pats(rows, n_max), cp, chi, kappa, grid, box, seed=seed, n_single=n_single, b=b)


CHI3 = [[0, 14, 6], [14, 0, 9], [6, 9, 0]]
CASES = {
    # both species on the lean fused kernel (N = 32 and N = 8), power-of-two grid
    "diblock32_homo8": lambda: _mix([(3000, 32), (7001, 8)], [[0] * 16 + [1] * 16, [2] * 8], CHI3, 40.0, (16, 16, 16), (8.0, 8.0, 8.0), 1),
    # a species the fused kernels cannot take (N = 5) next to one they can: mixed kernel paths in one step
    "diblock32_oligomer5": lambda: _mix([(2500, 32), (4000, 5)], [[0] * 16 + [1] * 16, [2, 2, 1, 1, 2]], CHI3, 35.0, (16, 16, 8), (8.0, 8.0, 4.0), 2),
    # three species, solvent molecules, reference length not any species' own, non-power-of-two grid (general fused kernel)
    "three_species_npot_solvent": lambda: _mix([(900, 16), (700, 64), (1500, 2)], [[0] * 8 + [1] * 8, [1] * 64, [2, 0]], CHI3, 30.0,
                                               (12, 10, 6), (6.0, 5.0, 3.0), 3, n_single=[0, 300, 4000], N_ref=32),
    # odd pattern row length (33): the fused kernels step aside (16-bit type loads), everything runs generic
    "odd_row_length": lambda: _mix([(500, 33), (800, 32)], [[0] * 17 + [1] * 16, [1] * 32], [[0, 11], [11, 0]], 25.0, (8, 8, 8), (4.0, 4.0, 4.0), 4),
    # single species given as a one-entry table
    "one_species_table": lambda: _mix([(2000, 16)], [[0] * 8 + [1] * 8], [[0, 15], [15, 0]], 45.0, (16, 8, 8), (8.0, 4.0, 4.0), 5),
}


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("case", sorted(CASES))
def test_species_parity_after_1_and_10_steps(case, path):
    s = CASES[case]()
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=path, options=dict(resort_interval=3)) as g:      # re-orderings inside the run, per species
        assert g.B == o.B
        g.load_state(s.x, s.y, s.z)
        assert_same_state(g, o, f"{case}: loaded")
        done = 0
        for upto in (1, 10):
            assert g.mc_steps(upto - done, want_accepted=True) == o.mc_steps(upto - done)
            done = upto
            assert_same_state(g, o, f"{case} path {path} after {upto} steps")
        assert g.counters()["resorts"] >= 3
        v, vo = g.validate(), o.validate()
        assert v["ok"] and v["density_per_type"][:o.T] == vo["density_per_type"][:o.T]
        assert v["max_bond_sq"] == np.float32(vo["max_bond_sq"]) and v["mean_bond_sq"] == pytest.approx(vo["mean_bond_sq"], rel=1e-12)


def test_species_use_the_kernels_their_length_allows():
    import paper_2606_09356_b200 as soma
    with gpu_system(CASES["diblock32_oligomer5"]()) as g:
        assert g.counters()["path"] == 2                  # N = 32 fused, N = 5 generic
        g.set_option("path", 1)
        assert g.counters()["path"] == 1
    with gpu_system(CASES["odd_row_length"]()) as g:
        assert g.counters()["path"] == 1
    s = _mix([(50, 5), (60, 3)], [[0] * 5, [1] * 3], [[0, 5], [5, 0]], 10.0, (4, 4, 4), (2.0, 2.0, 2.0), 6)
    with gpu_system(s) as g:
        with pytest.raises(soma.SomaError):
            g.set_option("path", 2)                       # no species the fused kernels could take


def test_generated_and_placed_states_with_species():
    s = CASES["three_species_npot_solvent"]()
    o = oracle.Oracle.from_system(s)
    with gpu_system(s) as g:
        o.generate_state(808, step0=1)
        g.generate_state(808, step0=1)
        same = all(np.array_equal(a, b) for a, b in zip(g.positions(), o.positions()))
        for a, b in zip(g.positions(), o.positions()):
            assert (a != b).mean() <= 1e-5
        if same:
            assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
            assert_same_state(g, o, "3 steps from the generated state")
        phi = np.random.default_rng(2).uniform(0.05, 1.0, size=(3, 12 * 10 * 6)).astype(np.float32)
        o.init_from_density(phi, 909, n_equil_steps=4, umbrella_k=0.8)
        g.init_from_density(phi, 909, n_equil_steps=4, umbrella_k=0.8)
        if all(np.array_equal(a, b) for a, b in zip(g.positions(), o.positions())):
            assert_same_state(g, o, "placed by density + umbrella steps")
        assert g.validate()["ok"]


def test_external_field_and_bond_force_biased_moves_with_species():
    s = CASES["diblock32_homo8"]()
    ext = np.random.default_rng(4).normal(0, 0.6, size=(3, 16 ** 3)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.set_smc(0.05)
    o.set_external_field(ext)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, smc_mobility=0.05) as g:
        g.set_external_field(ext)
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(4, want_accepted=True) == o.mc_steps(4)
        assert_same_state(g, o, "species + external field + bond-force-biased moves")


def test_species_parameters_are_validated():
    import paper_2606_09356_b200 as soma
    base = dict(n_chains=5, beads_per_chain=8, n_types=1, type_patterns=np.zeros((1, 8), np.uint8), chain_pattern=None, b=1.0,
                chiN=np.zeros((1, 1), np.float32), kappaN=0.0, grid=(4, 4, 4), box=(2.0, 2.0, 2.0), move_halfwidth=0.5, seed=1)
    for bad in ([(3, 8), (3, 4)], [(5, 8), (0, 4)], [(2, 8), (3, 0)], [(1, 8)] * 17):
        p, keep = soma.make_params(**base, species=bad)
        assert soma.soma_workspace_bytes(p) == 0, bad
    p, keep = soma.make_params(**base, species=[(2, 8), (3, 4)])
    assert soma.soma_workspace_bytes(p) > 0


@pytest.mark.parametrize("packed,otf", [(1, 1), (1, 0), (0, 0)])
def test_species_and_solvent_with_packed_counters_and_on_the_fly_omega(packed, otf):
    """Two types, three species (N = 32 and 8 on the lean kernel with omega on the fly, N = 5 on the generic
    kernels, which read the omega array) and single-bead solvent: all of them bin into the same packed counters,
    the omega array is filled every step because somebody needs it.  Then an external field switches the
    on-the-fly field off, and its removal on again."""
    s = _mix([(1500, 32), (2000, 8), (900, 5)], [[0] * 16 + [1] * 16, [1] * 8, [0, 0, 1, 1, 0]], [[0, 13], [13, 0]], 30.0,
             (16, 16, 8), (8.0, 8.0, 4.0), 7, n_single=[700, 1300])
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, options=dict(packed_counts=packed, omega_otf=otf, resort_interval=2)) as g:
        g.load_state(s.x, s.y, s.z)
        c = g.counters()
        assert c["packed_counts"] == bool(packed) and c["omega_otf"] == bool(otf)
        assert g.mc_steps(4, want_accepted=True) == o.mc_steps(4)
        assert_same_state(g, o, "species + solvent")
        ext = np.random.default_rng(3).normal(0, 0.4, size=(2, 16 * 16 * 8)).astype(np.float32)
        g.set_external_field(ext)
        o.set_external_field(ext)
        assert not g.counters()["omega_otf"]
        assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
        assert_same_state(g, o, "with an external field")
        g.set_external_field(None)
        o.set_external_field(None)
        assert g.counters()["omega_otf"] == bool(otf)
        assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
        assert_same_state(g, o, "field removed")
        assert g.validate()["ok"]
