"""Seeded random systems against the oracle: chain lengths, species tables, types, patterns, grids (power-of-two and
not), single-bead molecules, counter layouts, kernel paths and re-ordering intervals drawn at random; the whole state
must be the oracle's after every block of steps.  Catches what the hand-picked cases of the other files leave out."""
import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system

pytestmark = pytest.mark.gpu

STARTS = {}        # start kind -> cases run (second family)
RESYNCED = []      # cases whose device-side start differed from the oracle's in a last bit


def _random_system(rng):
    T = int(rng.integers(1, 4))
    pow2 = rng.random() < 0.6
    grid = tuple(int(g) for g in (rng.choice([4, 8, 16], 3) if pow2 else rng.choice([3, 5, 6, 10, 12], 3)))
    cell = 0.5 if rng.random() < 0.7 else float(rng.choice([0.25, 0.4, 1.0]))
    box = tuple(g * cell for g in grid)
    n_species = int(rng.integers(1, 4))
    lengths = [int(rng.choice([1, 2, 3, 4, 5, 8, 16, 32, 33, 64])) for _ in range(n_species)]
    counts = [int(rng.integers(1, 400)) for _ in range(n_species)]
    n_max = max(lengths)
    n_pat = int(rng.integers(1, 4))
    pats = rng.integers(0, T, size=(n_pat, n_max)).astype(np.uint8)
    n = sum(counts)
    cp = rng.integers(0, n_pat, size=n).astype(np.uint8) if n_pat > 1 else None
    chi = np.zeros((T, T))
    for a in range(T):
        for b_ in range(a + 1, T):
            chi[a, b_] = chi[b_, a] = float(rng.uniform(0, 25))
    kappa = float(rng.choice([0.0, 10.0, 50.0]))
    n_single = [int(rng.integers(0, 300)) for _ in range(T)] if rng.random() < 0.4 else None
    a = float(rng.choice([0.25, 0.5, 0.5, 0.3]))
    seed = int(rng.integers(1, 2 ** 40))
    if n_species == 1 and rng.random() < 0.5:
        return si.custom_system(counts[0], lengths[0], T, pats[:, :lengths[0]], cp, chi, kappa, grid, box, seed=seed, move_halfwidth=a, n_single=n_single)
    return si.species_system(list(zip(counts, lengths)), int(rng.choice(lengths)), T, pats, cp, chi, kappa, grid, box, seed=seed, move_halfwidth=a, n_single=n_single)


import os


@pytest.mark.parametrize("k", range(int(os.environ.get("SOMA_FUZZ_CASES", "100"))))
def test_random_system_matches_the_oracle(k):
    rng = np.random.default_rng(1000 + k)
    s = _random_system(rng)
    opts = dict(resort_interval=int(rng.choice([0, 1, 2, 5])), packed_counts=int(rng.choice([-1, 0, 1])), omega_otf=int(rng.choice([-1, 0, 1])),
                fused_lean=int(rng.choice([0, 1, 1])), omega_x4=int(rng.choice([0, 1])), fused_chunk=int(rng.choice([8, 24, 224])))
    path = int(rng.choice([0, 0, 1, 2]))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z, step0=int(rng.integers(0, 5)))
    import paper_2606_09356_b200 as soma
    with gpu_system(s, options=opts) as g:
        try:
            g.set_option("path", path)
        except soma.SomaError:
            path = 0                                   # no species the fused kernels could take
        g.load_state(s.x, s.y, s.z, step0=o.step)
        what = f"random system {k}: species {getattr(s, 'species', None)}, T={s.workload.n_types}, grid {s.workload.grid}, path {path}, {opts}"
        assert_same_state(g, o, what + " (loaded)")
        for steps in (1, 3, 2):
            assert g.mc_steps(steps, want_accepted=True) == o.mc_steps(steps), what
            assert_same_state(g, o, what)
        assert g.validate()["ok"]


@pytest.mark.parametrize("k", range(int(os.environ.get("SOMA_FUZZ_CASES", "100")) // 2))
def test_random_system_with_fields_moves_and_device_side_starts(k):
    """The same with what the rows of SURVEY 8(f) add: bond-force-biased moves, an external field switched on and
    off between blocks of steps, and states generated or placed by target concentrations on the device (those two
    agree with the oracle bit for bit except where double log / sin / cos differ in the last bit between libm and
    CUDA: the trajectory is compared only when the start is identical, which is the rule)."""
    rng = np.random.default_rng(5000 + k)
    s = _random_system(rng)
    w = s.workload
    smc = float(rng.choice([0.0, 0.0, 0.03, 0.1]))
    opts = dict(resort_interval=int(rng.choice([0, 1, 3])), packed_counts=int(rng.choice([-1, 0, 1])), omega_otf=int(rng.choice([-1, 0, 1])))
    start = str(rng.choice(["load", "generate", "density"]))
    o = oracle.Oracle.from_system(s)
    o.set_smc(smc)
    with gpu_system(s, options=opts, smc_mobility=smc) as g:
        what = f"random system {k}: species {getattr(s, 'species', None)}, T={w.n_types}, grid {w.grid}, smc {smc}, start {start}, {opts}"
        if start == "load":
            o.load_state(s.x, s.y, s.z)
            g.load_state(s.x, s.y, s.z)
        elif start == "generate":
            o.generate_state(77 + k, step0=2)
            g.generate_state(77 + k, step0=2)
        else:
            phi = rng.uniform(0.05, 1.5, size=(w.n_types, w.n_cells)).astype(np.float32)
            o.init_from_density(phi, 99 + k, n_equil_steps=2, umbrella_k=0.5)
            g.init_from_density(phi, 99 + k, n_equil_steps=2, umbrella_k=0.5)
        STARTS[start] = STARTS.get(start, 0) + 1
        if not all(np.array_equal(a, b) for a, b in zip(g.positions(), o.positions())):
            for a, b in zip(g.positions(), o.positions()):
                assert (a != b).mean() <= 1e-3 and np.all(np.abs(a.astype(np.float64) - b) <= 4 * np.spacing(np.abs(b)) + 1e-6), what
            # a last-bit difference of the double log / sin / cos: the documented case.  The device takes over the oracle's
            # start, so that the trajectory, the field switching and the move types of this seed are still compared
            RESYNCED.append(what)
            g.load_state(*o.positions(), step0=o.step)
        assert_same_state(g, o, what + " (start)")
        ext = rng.normal(0, 0.7, size=(w.n_types, w.n_cells)).astype(np.float32)
        for field in (None, ext, None):
            g.set_external_field(field)
            o.set_external_field(field)
            assert g.mc_steps(2, want_accepted=True) == o.mc_steps(2), what
            assert_same_state(g, o, what)


def test_how_many_device_side_starts_had_to_be_resynchronised():
    """Runs after the cases above (same file, later in it): says how many of the generated / density-placed starts
    differed from the oracle's in a last bit and were replaced by the oracle's start before the trajectory was compared.
    More than a few would mean the start generators disagree beyond the documented libm / CUDA cases."""
    n_device = STARTS.get("generate", 0) + STARTS.get("density", 0)
    print(f"fuzz: starts {STARTS}; {len(RESYNCED)} of {n_device} device-side starts resynchronised to the oracle's")
    for w in RESYNCED:
        print("  resynchronised:", w)
    assert len(RESYNCED) <= max(2, n_device // 10)
