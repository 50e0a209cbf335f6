"""GPU-vs-oracle parity of the whole SCMF Monte-Carlo step through the C ABI (BASELINE.json
`north_star` comparison rules).

Bar: density grids bit-exact, omega bit-exact, positions bit-identical (north_star's 1e-6 b is below
one fp32 ulp for |r| >= 16 b), accepted-move counts equal -- after 1 and after 10 MC steps from the
same seeded state, for both kernel paths.  With DESIGN.md reading R6b the accept decisions are
implementation-independent, so no flip is expected; the lock-step test keeps north_star's
allowance (|dE + ln u| < 1e-4, <= 1e-6 of the moves) as the outer bound and reports what it saw.
"""
import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system, lockstep

pytestmark = pytest.mark.gpu

FUSED, GENERIC = 2, 1


def _run_both(s, steps_list, path, **kw):
    """Advance GPU and oracle through cumulative step counts, comparing the full state at each."""
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=path, **kw) as g:
        g.load_state(s.x, s.y, s.z)
        assert_same_state(g, o, f"{s.workload.name} after load_state")
        done = 0
        for upto in steps_list:
            acc_g = g.mc_steps(upto - done, want_accepted=True)
            acc_o = o.mc_steps(upto - done)
            done = upto
            assert acc_g == acc_o, f"{s.workload.name} path {path}: accepted {acc_g} vs oracle {acc_o} after {upto} steps"
            assert_same_state(g, o, f"{s.workload.name} path {path} after {upto} steps")
            assert g.step == o.step == upto
            d = g.density()
            assert int(d.sum()) == s.workload.n_beads
        launches = g.counters()["launches"]
    assert launches > 0
    return launches


# ---- the five BASELINE.json configs, the small one at full size, the others scaled down so that the
# ---- oracle finishes in seconds but several tiles/warps and a ragged tail are covered ------------

def _scaled(i, n_chains, grid):
    return si.make_system(si.scaled(si.config(i), n_chains, grid))


CASES = {
    "cfg0_full": lambda: si.make_system(si.config(0)),
    "cfg1_scaled": lambda: _scaled(1, 4099, (16, 16, 16)),          # N=64, T=1, omega == 0; 4099 = ragged
    "cfg2_scaled": lambda: _scaled(2, 8193, (16, 16, 16)),          # N=32 diblock, 64 beads/cell
    "cfg3_scaled": lambda: _scaled(3, 4098, (32, 16, 16)),          # N=64 blend, 2 patterns, non-cubic
    "cfg4_scaled": lambda: _scaled(4, 16385, (32, 32, 16)),         # N=32 diblock, chiN=30
}


@pytest.mark.parametrize("path", [FUSED, GENERIC])
@pytest.mark.parametrize("case", sorted(CASES))
def test_parity_after_1_and_10_steps(case, path):
    _run_both(CASES[case](), [1, 10], path)


def test_cfg0_lockstep_protocol_no_flips():
    n_moves, n_flips, worst = lockstep(si.make_system(si.config(0)), 10)
    assert n_moves == 81920
    assert n_flips <= 1e-6 * n_moves          # = 0 for cfg 0
    print(f"lockstep cfg0: {n_moves} moves, {n_flips} flips, worst |margin| {worst:g}")


def test_scaled_cfg4_lockstep_protocol():
    n_moves, n_flips, worst = lockstep(_scaled(4, 16385, (32, 32, 16)), 5)
    assert n_flips <= max(0, int(1e-6 * n_moves))
    print(f"lockstep cfg4 scaled: {n_moves} moves, {n_flips} flips, worst |margin| {worst:g}")


# ---- degenerate and edge cases ---------------------------------------------------------------------

def _custom(n, N, T, pats, cp, chi, kappaN, grid, box, seed, **kw):
    return si.custom_system(n, N, T, pats, cp, chi, kappaN, grid, box, seed, **kw)


EDGE = {
    # N=1: no bonds, no odd beads;  N=2: one bond;  N=3, 5, 33: odd lengths -> generic path only
    "N1": lambda: _custom(777, 1, 2, [[0], [1]], np.arange(777) % 2, [[0, 9], [9, 0]], 30.0, (8, 8, 8), (4, 4, 4), 21),
    "N2": lambda: _custom(1001, 2, 2, [[0, 1]], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 22),
    "N3": lambda: _custom(513, 3, 2, [[0, 1, 0]], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 23),
    "N33": lambda: _custom(130, 33, 2, [[0] * 16 + [1] * 17], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 24),
    "N4": lambda: _custom(999, 4, 2, [[0, 0, 1, 1]], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 25),
    "N8": lambda: _custom(517, 8, 2, [[0, 0, 0, 1, 1, 1, 1, 0]], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 26),
    "N16": lambda: _custom(259, 16, 2, [[0] * 8 + [1] * 8], None, [[0, 15], [15, 0]], 40.0, (8, 8, 8), (4, 4, 4), 27),
    # three types with an asymmetric-valued chi matrix, three patterns, non-power-of-two non-cubic grid
    "T3_npot": lambda: _custom(600, 32, 3, [[0] * 10 + [1] * 12 + [2] * 10, [2] * 32, [1] * 16 + [0] * 16],
                               np.arange(600) % 3, [[0, 12, 5], [12, 0, 21], [5, 21, 0]], 35.0, (12, 10, 7), (6.0, 5.0, 3.5), 28),
    # T = 8 (the maximum), generic omega kernel
    "T8": lambda: _custom(300, 16, 8, [[0, 1, 2, 3, 4, 5, 6, 7] * 2], None,
                          (np.arange(64).reshape(8, 8) + np.arange(64).reshape(8, 8).T) * (1 - np.eye(8)) * 0.3, 25.0,
                          (6, 6, 6), (3, 3, 3), 29),
    # one chain, one cell, big moves, b != 1, a != 0.5, box far from cubic
    "one_chain": lambda: _custom(1, 32, 2, [[0] * 16 + [1] * 16], None, [[0, 20], [20, 0]], 50.0, (1, 1, 1), (3, 3, 3), 30),
    "b_and_a": lambda: _custom(700, 32, 2, [[0] * 16 + [1] * 16], None, [[0, 20], [20, 0]], 50.0, (20, 4, 9), (14.0, 2.8, 6.3), 31,
                               b=0.7, move_halfwidth=0.9),
    # zero move width: every trial equals the current position, dE = 0, all accepted, nothing changes
    "a0": lambda: _custom(100, 32, 2, [[0] * 16 + [1] * 16], None, [[0, 20], [20, 0]], 50.0, (8, 8, 8), (4, 4, 4), 32, move_halfwidth=0.0),
}


@pytest.mark.parametrize("case", sorted(EDGE))
def test_edge_cases_generic_path(case):
    _run_both(EDGE[case](), [1, 4], GENERIC)


@pytest.mark.parametrize("case", ["N2", "N4", "N8", "N16", "T3_npot", "T8", "one_chain", "b_and_a", "a0"])
def test_edge_cases_fused_path(case):
    _run_both(EDGE[case](), [1, 4], FUSED)


def test_fused_path_refuses_unsupported_chain_lengths():
    import paper_2606_09356_b200 as soma
    with gpu_system(EDGE["N33"]()) as g:
        with pytest.raises(soma.SomaError) as e:
            g.set_option("path", FUSED)
        assert e.value.code == soma.SOMA_EINVAL


def test_a0_accepts_everything_and_moves_nothing():
    s = EDGE["a0"]()
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(3, want_accepted=True) == 3 * s.workload.n_beads
        x, y, z = g.positions()
        assert np.array_equal(x, s.x) and np.array_equal(y, s.y) and np.array_equal(z, s.z)


def test_large_seed_step_and_chain_ids_reach_the_counter():
    """64-bit seed (both key words), step0 beyond 2^32 (counter word 3 bits 16..31)."""
    w = si.scaled(si.config(0), 300, (8, 8, 8))
    from dataclasses import replace
    s = si.make_system(replace(w, seed=0xFEDCBA9876543210))
    step0 = (5 << 32) + 0xFFFFFFFE           # crosses a 2^32 boundary during the run
    for path in (FUSED, GENERIC):
        o = oracle.Oracle.from_system(s)
        o.load_state(s.x, s.y, s.z, step0)
        with gpu_system(s, path=path) as g:
            g.load_state(s.x, s.y, s.z, step0)
            assert g.mc_steps(4, want_accepted=True) == o.mc_steps(4)
            assert_same_state(g, o, "large seed/step")
            assert g.step == step0 + 4
    # and the seed really matters
    s2 = si.make_system(replace(w, seed=0xFEDCBA9876543211))
    with gpu_system(s2) as g2:
        g2.load_state(s.x, s.y, s.z, step0)
        g2.mc_steps(1)
        assert not np.array_equal(g2.positions()[0], o.positions()[0])


# ---- further systems for the lean fused kernel (power-of-two grids, cell size 1/2): several warps per block
# with ragged tails, non-cubic grids, one to eight types, N = 2 ... 64, a single chain.

LEAN_CASES = {
    "cfg1_scaled_T1_N64": lambda: _scaled(1, 4099, (16, 16, 16)),
    "cfg2_scaled": lambda: _scaled(2, 8193, (32, 16, 32)),
    "cfg3_scaled_blend_N64": lambda: _scaled(3, 4098, (32, 16, 16)),
    "cfg4_scaled_noncubic": lambda: _scaled(4, 16385, (32, 32, 16)),
    "T3_three_patterns": lambda: _custom(900, 32, 3, [[0] * 10 + [1] * 12 + [2] * 10, [2] * 32, [1] * 16 + [0] * 16],
                                         np.arange(900) % 3, [[0, 12, 5], [12, 0, 21], [5, 21, 0]], 35.0, (16, 32, 16), (8.0, 16.0, 8.0), 41),
    "N2": lambda: _custom(3001, 2, 2, [[0, 1]], None, [[0, 15], [15, 0]], 40.0, (16, 16, 16), (8, 8, 8), 42),
    "N8": lambda: _custom(1517, 8, 2, [[0, 0, 0, 1, 1, 1, 1, 0]], None, [[0, 15], [15, 0]], 40.0, (16, 16, 16), (8, 8, 8), 43),
    "one_chain": lambda: _custom(1, 32, 2, [[0] * 16 + [1] * 16], None, [[0, 20], [20, 0]], 50.0, (16, 16, 16), (8, 8, 8), 44),
    "T8_sparse": lambda: _custom(300, 16, 8, [[0, 1, 2, 3, 4, 5, 6, 7] * 2], None,
                                 (np.arange(64).reshape(8, 8) + np.arange(64).reshape(8, 8).T) * (1 - np.eye(8)) * 0.3, 25.0,
                                 (8, 8, 8), (4, 4, 4), 46),
}


@pytest.mark.parametrize("threads", [256, 1024])
@pytest.mark.parametrize("case", sorted(LEAN_CASES))
def test_lean_kernel_parity_after_1_and_10_steps(case, threads):
    s = LEAN_CASES[case]()
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=FUSED, options=dict(lean_threads=threads, fused_chunk=24)) as g:    # small chunks: many blocks, ragged last one
        g.load_state(s.x, s.y, s.z)
        done = 0
        for upto in (1, 10):
            assert g.mc_steps(upto - done, want_accepted=True) == o.mc_steps(upto - done)
            done = upto
            assert_same_state(g, o, f"{case} lean kernel, {threads} threads, after {upto} steps")


@pytest.mark.parametrize("path", [FUSED, GENERIC])
@pytest.mark.parametrize("interval", [0, 1, 3])
def test_drift_and_resorts_do_not_change_the_trajectory(interval, path):
    """40 steps: without re-sorting the chains drift away from their neighbours in memory; with frequent
    re-sorting the slot order keeps changing.  The trajectory may not depend on either.  (Path 2 is the
    kernel bench.py times: its periodic re-ordering is compared with the oracle here.)"""
    s = _scaled(4, 6000, (16, 16, 16))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(40)
    with gpu_system(s, path=path, options=dict(resort_interval=interval)) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(40, want_accepted=True) == acc_o
        assert_same_state(g, o, f"path {path}, resort_interval={interval}")
        first = 1 if interval else 0                                 # never sorted when the interval is 0
        assert g.counters()["resorts"] == first + ((40 - 1) // interval if interval else 0)


@pytest.mark.parametrize("path", [FUSED, GENERIC])
@pytest.mark.parametrize("interval", [1, 3])
def test_parity_after_1_and_10_steps_with_resorts(interval, path):
    """The full-state comparison after 1 and 10 steps with the chain re-ordering inside the run."""
    s = _scaled(4, 16385, (32, 32, 16))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=path, options=dict(resort_interval=interval)) as g:
        g.load_state(s.x, s.y, s.z)
        done = 0
        for upto in (1, 10):
            assert g.mc_steps(upto - done, want_accepted=True) == o.mc_steps(upto - done)
            done = upto
            assert_same_state(g, o, f"path {path}, resort every {interval}, after {upto} steps")
        assert g.counters()["resorts"] >= 1 + 9 // interval


@pytest.mark.parametrize("lean", [0, 1])
def test_general_and_lean_fused_kernels_agree_with_the_oracle(lean):
    """fused_lean = 0 keeps the general fused kernel (any grid, any cell size) on a system where the lean
    one applies; both must give the oracle's state."""
    s = _scaled(2, 8193, (16, 16, 16))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=FUSED, options=dict(fused_lean=lean)) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(5, want_accepted=True) == o.mc_steps(5)
        assert_same_state(g, o, f"fused_lean={lean}")


def test_switching_paths_mid_run_keeps_the_trajectory():
    s = _scaled(2, 5000, (16, 16, 16))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(8)
    with gpu_system(s, path=FUSED) as g:
        g.load_state(s.x, s.y, s.z)
        for k, path in enumerate((FUSED, GENERIC, GENERIC, FUSED, FUSED, GENERIC, FUSED, FUSED)):
            g.set_option("path", path)
            g.set_option("fused_lean", k % 3 != 0)                   # the general fused kernel every third step
            g.mc_steps(1)
        assert_same_state(g, o, "path switched every step")


def test_path_option_is_validated():
    import paper_2606_09356_b200 as soma
    with gpu_system(EDGE["N33"]()) as g:                                     # odd N: no fused kernel
        with pytest.raises(soma.SomaError) as e:
            g.set_option("path", FUSED)
        assert e.value.code == soma.SOMA_EINVAL
        assert g.counters()["path"] == GENERIC
    with gpu_system(si.make_system(si.config(0))) as g:
        for bad in (3, -1):
            with pytest.raises(soma.SomaError) as e:
                g.set_option("path", bad)
            assert e.value.code == soma.SOMA_EINVAL


# ---- external field: omega = interaction part + ext, every kernel path -----

@pytest.mark.parametrize("path", [FUSED, GENERIC])
def test_external_field_parity(path):
    s = _scaled(4, 6000, (16, 16, 16))
    ext = np.random.default_rng(31).normal(0.0, 0.8, size=(2, 16 ** 3)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_external_field(ext)
    with gpu_system(s, path=path) as g:
        g.load_state(s.x, s.y, s.z)
        g.set_external_field(ext)
        assert np.array_equal(g.omega().view(np.uint32), o.omega().view(np.uint32))
        assert g.mc_steps(5, want_accepted=True) == o.mc_steps(5)
        assert_same_state(g, o, f"external field, path {path}, 5 steps")
        g.load_state(*g.positions(), step0=5)                     # the field survives a reload
        assert np.array_equal(g.omega().view(np.uint32), o.omega().view(np.uint32))
        g.set_external_field(None)
        o.set_external_field(None)
        assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
        assert_same_state(g, o, f"external field removed, path {path}")


def test_external_field_single_bead_molecules_on_device():
    """N = 1 (generic path): the oracle's Boltzmann pin, run on the GPU and compared bit for bit."""
    s = si.custom_system(20000, 1, 1, [[0]], None, [[0.0]], 0.0, (4, 4, 4), (2.0, 2.0, 2.0), seed=78)
    ext = np.random.default_rng(6).uniform(0.0, 2.0, size=(1, 64)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.set_external_field(ext)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        import torch
        g.set_external_field(torch.from_numpy(ext).cuda())        # device pointer in
        assert g.mc_steps(40, want_accepted=True) == o.mc_steps(40)
        assert_same_state(g, o, "N=1 in an external field")


# ---- single-bead molecules next to the chains (R23) ----------------

def _mixture(n_chains=3000, N=32, n_single=(7000, 0, 11000), grid=(16, 16, 16), seed=51):
    chi = np.array([[0, 18, 6], [18, 0, 9], [6, 9, 0.0]])
    pat = [[0] * (N // 2) + [1] * (N - N // 2)]
    return si.custom_system(n_chains, N, 3, pat, None, chi, 40.0, grid, tuple(g / 2 for g in grid), seed=seed, n_single=n_single)


@pytest.mark.parametrize("path", [FUSED, GENERIC])
def test_mixture_of_chains_and_single_bead_molecules(path):
    s = _mixture()
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, path=path) as g:
        g.load_state(s.x, s.y, s.z)
        assert_same_state(g, o, f"mixture loaded, path {path}")
        done = 0
        for upto in (1, 10):
            assert g.mc_steps(upto - done, want_accepted=True) == o.mc_steps(upto - done)
            done = upto
            assert_same_state(g, o, f"mixture, path {path}, {upto} steps")
        v = g.validate()
        assert v["ok"] and v["density_per_type"][:3] == o.validate()["density_per_type"]


def test_mixture_generic_chain_length_lockstep_and_generated_state():
    s = _mixture(n_chains=900, N=5, n_single=(0, 4000, 1), grid=(8, 8, 8), seed=52)       # odd N: generic kernels
    o = oracle.Oracle.from_system(s)
    o.generate_state(99)
    with gpu_system(s) as g:
        g.generate_state(99)
        assert all(np.array_equal(a, b_) for a, b_ in zip(g.positions(), o.positions()))
        assert g.mc_steps(6, want_accepted=True) == o.mc_steps(6)
        assert_same_state(g, o, "generated mixture, 6 steps")


# ---- bond-force-biased moves (R24) -----------------------------------

@pytest.mark.parametrize("path", [FUSED, GENERIC])
@pytest.mark.parametrize("case", ["cfg0_full", "cfg4_scaled", "cfg3_scaled_N64", "N5_T3_mixture"])
def test_bond_force_biased_moves_parity(case, path):
    A = 0.05
    if case == "cfg0_full":
        s = si.make_system(si.config(0))
    elif case == "cfg4_scaled":
        s = _scaled(4, 4097, (16, 16, 16))
    elif case == "cfg3_scaled_N64":
        s = _scaled(3, 2049, (16, 16, 16))
    else:
        s = _mixture(n_chains=900, N=5, n_single=(0, 2000, 300), grid=(8, 8, 8), seed=53)
    o = oracle.Oracle.from_system(s)
    o.set_smc(A)
    o.load_state(s.x, s.y, s.z)
    if case == "N5_T3_mixture" and path == FUSED:
        pytest.skip("odd N: generic kernels only")
    with gpu_system(s, path=path, smc_mobility=A) as g:
        assert g.counters()["path"] == path
        g.load_state(s.x, s.y, s.z)
        done = 0
        for upto in (1, 10):
            assert g.mc_steps(upto - done, want_accepted=True) == o.mc_steps(upto - done)
            done = upto
            assert_same_state(g, o, f"{case}, bond-force-biased moves, {upto} steps")


@pytest.mark.parametrize("x4", [0, 1])
def test_both_omega_kernels_give_the_oracle_field(x4):
    """omega_kernel (one cell per thread) and omega_kernel_x4 (four cells per thread, 128-bit accesses) on a
    system where both apply, with an external field: bit-identical omega after every step."""
    s = _custom(2500, 16, 3, [[0] * 5 + [1] * 6 + [2] * 5], None, [[0, 12, 5], [12, 0, 21], [5, 21, 0]], 35.0, (8, 12, 4), (4.0, 6.0, 2.0), 51)
    ext = np.random.default_rng(8).normal(0.0, 0.5, size=(3, 8 * 12 * 4)).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.set_external_field(ext)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, options=dict(omega_x4=x4)) as g:
        g.set_external_field(ext)
        g.load_state(s.x, s.y, s.z)
        for _ in range(3):
            assert g.mc_steps(1, want_accepted=True) == o.mc_steps(1)
            assert_same_state(g, o, f"omega_x4={x4}")


@pytest.mark.parametrize("packed,otf", [(0, 0), (1, 0), (1, 1)])
@pytest.mark.parametrize("case", ["cfg4_scaled_noncubic", "cfg1_scaled_T1_N64", "cfg3_scaled_blend_N64"])
def test_counter_layouts_and_on_the_fly_omega_give_the_same_trajectory(case, packed, otf):
    """32-bit counters, 16-bit counters two types to a word, and the lean kernel computing omega from the packed
    counters itself: the oracle's state after 1 and 10 steps in every combination, with re-orderings, a path
    switch in the middle (the generic kernels need the omega array: it is filled on demand) and a checkpoint."""
    s = LEAN_CASES[case]()
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s, options=dict(packed_counts=packed, omega_otf=otf, resort_interval=4)) as g:
        g.load_state(s.x, s.y, s.z)
        assert_same_state(g, o, "loaded")
        assert g.mc_steps(1, want_accepted=True) == o.mc_steps(1)
        assert_same_state(g, o, f"{case} packed={packed} otf={otf} after 1 step")
        g.mc_steps(3)
        g.set_option("path", GENERIC)
        g.mc_steps(2)
        g.set_option("path", 0)
        g.mc_steps(4)
        o.mc_steps(9)
        assert_same_state(g, o, f"{case} packed={packed} otf={otf} after 10 steps")
        x, y, z = g.positions()
        with gpu_system(s, options=dict(packed_counts=1 - packed)) as g2:       # resume with the other counter layout
            g2.load_state(x, y, z, g.step)
            assert g2.mc_steps(3, want_accepted=True) == o.mc_steps(3)
            assert_same_state(g2, o, "resumed")


def test_a_state_too_dense_for_16_bit_counters_falls_back_to_32_bit_ones():
    """45000 beads of each type in one cell: the load notices (guard level 2048) and keeps 32-bit counters; the
    trajectory is the oracle's."""
    n = 45000
    s = _custom(n, 2, 2, [[0, 1]], None, [[0, 3], [3, 0]], 2.0, (4, 4, 4), (2.0, 2.0, 2.0), 61)
    s.x[:] = 0.26 + 0.001 * (np.arange(2 * n) % 7)
    s.y[:] = 0.3
    s.z[:] = 1.1
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    assert int(o.density().max()) == n
    with gpu_system(s, options=dict(packed_counts=1)) as g:
        g.load_state(s.x, s.y, s.z)
        assert_same_state(g, o, "dense state loaded")
        assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
        assert_same_state(g, o, "dense state after 3 steps")


def test_a_16_bit_counter_reaching_its_guard_during_a_run_is_an_error_not_a_wrong_result():
    """2040 beads in one cell at load (below the guard level of 2048 for one-cell moves: packed counters are used),
    400 more next door and a field that pulls them in: as soon as the cell holds 2048 beads the next synchronising
    call fails with SOMA_EINVAL; with 32-bit counters the same run goes through and matches the oracle."""
    import paper_2606_09356_b200 as soma
    n0, n1 = 2040, 400
    s = _custom(n0 + n1, 1, 1, [[0]], None, [[0]], 0.0, (4, 4, 4), (2.0, 2.0, 2.0), 71)
    rng = np.random.default_rng(5)
    s.x[:n0] = 0.05 + 0.4 * rng.random(n0).astype(np.float32)       # cell (0, 1, 1)
    s.x[n0:] = 0.52 + 0.05 * rng.random(n1).astype(np.float32)      # cell (1, 1, 1), just across the face
    s.y[:] = 0.75
    s.z[:] = 0.75
    ext = np.zeros((1, 64), dtype=np.float32)
    ext[0, (0 * 4 + 1) * 4 + 1] = -25.0                             # the dense cell is a deep well: beads stay, neighbours come
    o = oracle.Oracle.from_system(s)
    o.set_external_field(ext)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(6)
    assert int(o.density().max()) >= 2048
    with gpu_system(s, options=dict(packed_counts=1)) as g:
        g.set_external_field(ext)
        g.load_state(s.x, s.y, s.z)
        assert g.counters()["packed_counts"]
        with pytest.raises(soma.SomaError) as e:
            for _ in range(6):
                g.mc_steps(1, want_accepted=True)
        assert e.value.code == soma.SOMA_EINVAL and "16-bit density counters" in str(e.value)
        with pytest.raises(soma.SomaError) as e2:
            g.mc_steps(1)                                           # the state is gone: load again
        assert e2.value.code == soma.SOMA_ESTATE
        g.set_option("packed_counts", 0)
        g.load_state(s.x, s.y, s.z)
        assert not g.counters()["packed_counts"]
        assert g.mc_steps(6, want_accepted=True) > 0
        assert_same_state(g, o, "the same run on 32-bit counters")


@pytest.mark.parametrize("reader", ["positions", "validate"])
def test_a_guard_hit_during_an_asynchronous_run_stops_the_checkpoint_calls(reader):
    """The same crowded cell, but run the way the wrapper runs by default: soma_mc_steps with accepted == NULL never
    synchronises, so the first call that does is the reader of the checkpoint -- soma_get_positions to host memory, or
    soma_validate_state.  It must fail with SOMA_EINVAL rather than hand out a state whose counters are past the guard."""
    import paper_2606_09356_b200 as soma
    n0, n1 = 2040, 400
    s = _custom(n0 + n1, 1, 1, [[0]], None, [[0]], 0.0, (4, 4, 4), (2.0, 2.0, 2.0), 71)
    rng = np.random.default_rng(5)
    s.x[:n0] = 0.05 + 0.4 * rng.random(n0).astype(np.float32)
    s.x[n0:] = 0.52 + 0.05 * rng.random(n1).astype(np.float32)
    s.y[:] = 0.75
    s.z[:] = 0.75
    ext = np.zeros((1, 64), dtype=np.float32)
    ext[0, (0 * 4 + 1) * 4 + 1] = -25.0
    with gpu_system(s, options=dict(packed_counts=1)) as g:
        g.set_external_field(ext)
        g.load_state(s.x, s.y, s.z)
        assert g.counters()["packed_counts"]
        g.mc_steps(6)                                               # asynchronous: returns without looking at the flag
        with pytest.raises(soma.SomaError) as e:
            g.positions() if reader == "positions" else g.validate()
        assert e.value.code == soma.SOMA_EINVAL and "16-bit density counters" in str(e.value)
        with pytest.raises(soma.SomaError) as e2:
            g.mc_steps(1)
        assert e2.value.code == soma.SOMA_ESTATE


@pytest.mark.parametrize("N,n", [(8, 517), (16, 259), (32, 131)])
def test_lanes_beyond_the_last_chain_do_not_depend_on_what_the_workspace_holds(N, n):
    """Chain counts that are not a multiple of 32/P leave lanes of the last warp of the lean kernel without a chain.  With
    several chain patterns such a lane used to read a pattern id past the end of the slot table; the lent workspace is filled
    with 0xFF here, so that id would be 255, the bead type 255 and the omega gather 255 grids past the array.  The lanes now
    look up the block's first slot.  32-bit counters, omega array (the default of grids below 2^20 cells); the run must also
    equal the oracle's."""
    half = N // 2
    pats = [[0] * half + [1] * half, [1] * half + [0] * half, [0] * N]
    s = _custom(n, N, 2, pats, np.arange(n) % 3, [[0, 12], [12, 0]], 35.0, (8, 8, 8), (4, 4, 4), 31 + N)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(3)
    with gpu_system(s, path=2, options=dict(packed_counts=0), workspace_fill=0xFF) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(3, want_accepted=True) == acc_o
        assert_same_state(g, o, f"N={N}, {n} chains of three patterns, workspace of 0xFF")
