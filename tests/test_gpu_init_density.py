"""soma_init_from_density (second half; R25) against the oracle:
placement by target concentrations, umbrella-potential equilibration, error paths."""
import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system

pytestmark = pytest.mark.gpu


def _ulp_check(a, b_, what):
    diff = a != b_
    assert diff.mean() <= 1e-5, (what, diff.mean())                       # double libm vs CUDA log/sin/cos, R22/R25
    if diff.any():
        assert np.all(np.abs(a[diff].astype(np.float64) - b_[diff]) <= np.spacing(np.abs(b_[diff]))), what
    return int(diff.sum())


def _target(grid, T, seed):
    nx, ny, nz = grid
    ix = np.arange(nx)[:, None, None] + np.zeros((nx, ny, nz))
    iz = np.arange(nz)[None, None, :] + np.zeros((nx, ny, nz))
    a = 0.5 + 0.45 * np.cos(2 * np.pi * ix / nx) * np.cos(2 * np.pi * iz / nz)
    phi = np.stack([a, 1.0 - a] + [np.full((nx, ny, nz), 0.3)] * (T - 2))[:T]
    phi += np.random.default_rng(seed).uniform(0, 0.05, size=phi.shape)
    phi[0, 1] = 0.0                                                        # an empty slab for type 0
    return phi.reshape(T, -1).astype(np.float32)


CASES = {
    "cfg4_scaled": lambda: si.make_system(si.scaled(si.config(4), 20000, (32, 32, 16))),
    "cfg3_scaled_blend_N64": lambda: si.make_system(si.scaled(si.config(3), 6000, (32, 16, 16))),
    "N33_npot_T3": lambda: si.custom_system(700, 33, 3, [[0] * 11 + [1] * 11 + [2] * 11, [2] * 33], np.arange(700) % 2, [[0, 9, 4], [9, 0, 13], [4, 13, 0]],
                                            30.0, (6, 10, 12), (3.0, 5.0, 6.0), seed=3),
    "chains_and_solvent": lambda: si.custom_system(3000, 16, 3, [[0] * 8 + [1] * 8], None, [[0, 14, 3], [14, 0, 6], [3, 6, 0]], 40.0,
                                                   (16, 16, 16), (8.0, 8.0, 8.0), seed=4, n_single=[0, 500, 20000]),
    "single_beads_only_N1": lambda: si.custom_system(50000, 1, 2, [[0], [1]], np.arange(50000) % 2, [[0, 0], [0, 0]], 0.0, (8, 8, 8), (4.0, 4.0, 4.0), seed=5),
}


@pytest.mark.parametrize("case", sorted(CASES))
def test_placement_and_umbrella_equilibration_match_the_oracle(case):
    s = CASES[case]()
    w = s.workload
    phi = _target(w.grid, w.n_types, 7)
    o = oracle.Oracle.from_system(s)
    o.init_from_density(phi, gen_seed=31337, step0=2)
    with gpu_system(s) as g:
        g.init_from_density(phi, 31337, step0=2)
        assert g.step == 2
        n_diff = sum(_ulp_check(a, b_, f"{case}: placed positions") for a, b_ in zip(g.positions(), o.positions()))
        if n_diff == 0:
            assert_same_state(g, o, f"{case}: placed state")
            # the one-call form: placement + 6 steps under the umbrella, then plain steps
            acc_o = o.init_from_density(phi, 31337, step0=2, n_equil_steps=6, umbrella_k=1.5)
            g.init_from_density(phi, 31337, step0=2, n_equil_steps=6, umbrella_k=1.5)
            assert g.step == 8
            assert_same_state(g, o, f"{case}: after the umbrella equilibration")
            assert g.mc_steps(3, want_accepted=True) == o.mc_steps(3)
            assert_same_state(g, o, f"{case}: 3 plain steps later")
            assert acc_o > 0
        else:                                                              # densities still sum up, every chain is there
            assert int(g.density().sum()) == int(o.density().sum())
        v = g.validate()
        assert v["ok"] and v["density_total"] == o.B


def test_target_from_a_device_tensor_and_with_an_external_field():
    import torch
    s = CASES["cfg4_scaled"]()
    phi = _target(s.workload.grid, 2, 9)
    ext = np.random.default_rng(5).normal(0, 0.5, size=phi.shape).astype(np.float32)
    o = oracle.Oracle.from_system(s)
    o.set_external_field(ext)
    o.init_from_density(phi, 5, n_equil_steps=4, umbrella_k=0.7)
    with gpu_system(s) as g:
        g.set_external_field(ext)
        g.init_from_density(torch.from_numpy(phi).cuda(), 5, n_equil_steps=4, umbrella_k=0.7)
        if all(np.array_equal(a, b_) for a, b_ in zip(g.positions(), o.positions())):
            assert_same_state(g, o, "device target + external field + umbrella")   # omega: external field still on, umbrella off


def test_init_from_density_error_paths():
    import paper_2606_09356_b200 as soma
    s = si.custom_system(64, 4, 2, [[0, 0, 1, 1]], None, [[0, 5], [5, 0]], 10.0, (4, 4, 4), (2.0, 2.0, 2.0), seed=3)
    good = np.ones((2, 64), dtype=np.float32)
    with gpu_system(s) as g:
        for bad in (-0.1, np.nan, 65536.0):
            p = good.copy()
            p[1, 7] = bad
            with pytest.raises(soma.SomaError) as e:
                g.init_from_density(p, 1)
            assert e.value.code == soma.SOMA_EINVAL
        with pytest.raises(soma.SomaError) as e:
            g.init_from_density(np.zeros((2, 64), dtype=np.float32), 1)
        assert e.value.code == soma.SOMA_EINVAL and "zero total weight" in str(e.value)
        with pytest.raises(soma.SomaError) as e:
            g.mc_steps(1)                                                  # a refused call leaves no state behind
        assert e.value.code == soma.SOMA_ESTATE
        with pytest.raises(soma.SomaError):
            g.init_from_density(good, 1, step0=(1 << 48) - 2, n_equil_steps=5)
        g.init_from_density(good, 1)                                       # and a good call works afterwards
        assert int(g.density().sum()) == 256


def test_full_size_cfg4_from_a_lamellar_target():
    """configs[4] (134 M beads) placed from a target with polymer-rich and polymer-poor slabs on the device:
    totals, bond statistics, the slab profile of the density against the target (a symmetric diblock is placed
    by the total concentration; its beads are smeared over ~R_g around the target point), and the state runs."""
    w = si.config(4)
    s = si.System(w, np.array([[0] * 16 + [1] * 16], dtype=np.uint8), None, np.array([[0.0, w.chiN], [w.chiN, 0.0]], dtype=np.float32),
                  np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(0, np.float32))
    nx, ny, nz = w.grid
    ix = np.arange(nx, dtype=np.float32)[:, None, None]
    a = (0.5 + 0.4 * np.cos(2 * np.pi * ix / 32.0)) * np.ones((1, ny, nz), dtype=np.float32)     # slabs of period 32 cells = 16 b
    phi = np.stack([a, a]).reshape(2, -1).astype(np.float32)
    with gpu_system(s) as g:
        g.init_from_density(phi, 123)
        v = g.validate()
        assert v["ok"] and v["density_per_type"][:2] == [w.n_beads // 2, w.n_beads // 2]
        assert abs(v["mean_bond_sq"] - 1.0) < 0.001                       # the configs' Gaussian bonds, b = 1
        g.init_from_density(phi, 123, n_equil_steps=2, umbrella_k=1.0)
        assert g.validate()["ok"]
        dens = g.density().reshape(2, nx, ny * nz).sum(-1).sum(0).astype(np.float64)
        prof = dens / dens.mean() - 1.0
        want = 0.8 * np.cos(2 * np.pi * np.arange(nx) / 32.0)
        assert np.corrcoef(prof, want)[0, 1] > 0.99                       # polymer where the target has polymer
        amp = 2.0 * (prof * np.cos(2 * np.pi * np.arange(nx) / 32.0)).mean()
        assert 0.55 < amp < 0.8                                           # smeared by the chains' extent: exp(-(q R_g)^2 / 6)-ish
        assert g.step == 2
