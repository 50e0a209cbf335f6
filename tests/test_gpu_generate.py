"""Device-side initial state (soma_generate_state, R22) against the
oracle's generator, and the closed forms that pin the oracle's, on the device's own output."""
import math
import time

import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system, mean_sq_end_to_end

pytestmark = pytest.mark.gpu


def _ulp_check(a, b_, what):
    diff = a != b_
    frac = diff.mean()
    assert frac <= 1e-6, (what, frac)                                     # DESIGN.md R22: ~1e-8 expected
    if diff.any():
        assert np.all(np.abs(a[diff].astype(np.float64) - b_[diff]) <= np.spacing(np.abs(b_[diff]))), what
    return int(diff.sum())


@pytest.mark.parametrize("cfg,n,grid", [(4, 20000, (32, 32, 16)), (3, 6000, (32, 16, 16)), (1, 3000, (16, 16, 16))])
def test_generated_state_matches_the_oracle_and_evolves_identically(cfg, n, grid):
    s = si.make_system(si.scaled(si.config(cfg), n, grid))
    o = oracle.Oracle.from_system(s)
    o.generate_state(4242, step0=3)
    with gpu_system(s) as g:
        g.generate_state(4242, step0=3)
        assert g.step == 3
        n_diff = sum(_ulp_check(a, b_, "generated positions") for a, b_ in zip(g.positions(), o.positions()))
        if n_diff == 0:                                                   # identical start: identical trajectory
            assert_same_state(g, o, "generated state")
            assert g.mc_steps(4, want_accepted=True) == o.mc_steps(4)
            assert_same_state(g, o, "4 steps from the generated state")


def test_generate_full_size_cfg4_statistics_and_speed():
    """configs[4] (134 M beads) generated on the device: the closed forms of the configs' recipe hold,
    the state is binned, and it takes a small fraction of the host generator's time."""
    import paper_2606_09356_b200 as soma
    import torch
    w = si.config(4)
    pats = np.array([[0] * 16 + [1] * 16], dtype=np.uint8)
    chi = np.array([[0.0, w.chiN], [w.chiN, 0.0]], dtype=np.float32)
    with soma.Soma(w.n_chains, w.N, 2, pats, None, w.b, chi, w.kappaN, w.grid, w.box, w.move_halfwidth, w.seed) as g:
        g.generate_state(99)                                             # warm-up (first launch, sort)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g.generate_state(5)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        x, y, z = g.positions()
        dens = g.density()
        g.mc_steps(2)                                                    # and it runs
    n, N, b = w.n_chains, w.N, w.b
    assert int(dens.sum()) == w.n_beads
    r2, _ = mean_sq_end_to_end(x, y, z, n, N)
    want = (N - 1) * b * b
    assert abs(r2 - want) <= 3 * want * math.sqrt(2.0 / (3.0 * n)), (r2, want)
    for v, L in ((x, w.box[0]), (y, w.box[1]), (z, w.box[2])):
        v = v.reshape(n, N)
        first = v[:, 0].astype(np.float64) / L
        assert 0.0 <= first.min() and first.max() <= 1.0 and abs(first.mean() - 0.5) < 4 / math.sqrt(12 * n)
        d = np.diff(v[: 1 << 18].astype(np.float64), axis=1).reshape(-1)
        assert abs((d * d).mean() - b * b / 3) < 4 * math.sqrt(2.0 / d.size) * b * b / 3
    print(f"soma_generate_state, cfg4: {dt * 1e3:.1f} ms incl. binning, omega and the chain re-ordering")
    assert dt < 1.0


@pytest.mark.parametrize("cfg,n,grid", [(4, 20000, (32, 32, 16)), (3, 5001, (32, 16, 16))])
def test_validate_state_matches_the_oracle(cfg, n, grid):
    s = si.make_system(si.scaled(si.config(cfg), n, grid))
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        for steps in (0, 3):
            if steps:
                g.mc_steps(steps)
                o.mc_steps(steps)
            vg, vo = g.validate(), o.validate()
            assert vg["ok"] and vg["nonfinite"] == vo["nonfinite"] == 0
            assert vg["density_total"] == vo["density_total"] == s.workload.n_beads
            assert vg["density_per_type"][: s.workload.n_types] == vo["density_per_type"]
            assert vg["max_bond_sq"] == np.float32(vo["max_bond_sq"])                    # fp32 maximum: exact
            assert vg["mean_bond_sq"] == pytest.approx(vo["mean_bond_sq"], rel=1e-12)   # double sums in another order


def test_validate_single_bead_molecules_have_no_bonds():
    s = si.custom_system(5000, 1, 1, [[0]], None, [[0.0]], 0.0, (8, 8, 8), (4.0, 4.0, 4.0), seed=79)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        v = g.validate()
    assert v["ok"] and v["density_total"] == 5000 and v["max_bond_sq"] == 0.0 and v["mean_bond_sq"] == 0.0
