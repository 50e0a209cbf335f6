"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (configs[4]: 134 M
beads, default kernel path): the whole state after one MC step against the oracle (one oracle step
takes ~20 s on one core), then properties that hold at any size after further steps."""
import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import gpu_system

pytestmark = pytest.mark.gpu


def test_cfg4_full_size_one_step_bit_exact_then_invariants():
    w = si.config(4)
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(1)
    ox, oy, oz = o.positions()
    dens_o, om_o = o.density(), o.omega()
    o.close()
    with gpu_system(s) as g:                              # path 0 = what bench.py runs
        g.load_state(s.x, s.y, s.z)
        acc_g = g.mc_steps(1, want_accepted=True)
        gx, gy, gz = g.positions()
        assert acc_g == acc_o
        for a, b_ in ((gx, ox), (gy, oy), (gz, oz)):
            assert np.array_equal(a, b_)                  # bit-identical: no decision flipped among 134 M moves
        del ox, oy, oz
        assert np.array_equal(g.density(), dens_o)
        assert np.array_equal(g.omega().view(np.uint32), om_o.view(np.uint32))
        # nine more steps (one chain re-ordering is not due yet; force one to cover it at this size)
        g.mc_steps(4)
        g.set_option("resort_now", 1)
        g.mc_steps(5)
        x, y, z = g.positions()
        dens = g.density()
    assert int(dens.sum()) == w.n_beads
    types = s.bead_types()
    for t in range(w.n_types):
        assert int(dens[t].sum()) == int((types == t).sum())
    # the densities are the histogram of the positions the library returns (cell rule of DESIGN.md section 2 step 1)
    cell = np.zeros(w.n_beads, dtype=np.int64)
    for v, n_ax, L_ax in ((x, w.grid[0], w.box[0]), (y, w.grid[1], w.box[1]), (z, w.grid[2], w.box[2])):
        inv_h = np.float32(n_ax) / np.float32(L_ax)
        gcoord = np.floor(v * inv_h).astype(np.int64) % n_ax
        cell = cell * n_ax + gcoord
    for t in range(w.n_types):
        hist = np.bincount(cell[types == t], minlength=w.n_cells)
        assert np.array_equal(hist, dens[t].reshape(-1).astype(np.int64))
    # beads move by less than the half-width per step and axis
    assert float(np.abs(x - s.x).max()) < 10 * w.move_halfwidth


@pytest.mark.parametrize("cfg,steps", [(1, 10), (2, 10), (3, 2)])
def test_full_size_configs_bit_exact(cfg, steps):
    """configs[1..3] at BASELINE.json's full sizes on the default kernel path (cfg1, cfg3: N = 64, one
    chain per warp; cfg3: two chain patterns), whole state against the oracle after `steps` MC steps."""
    w = si.config(cfg)
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(steps)
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(steps, want_accepted=True) == acc_o
        gx, gy, gz = g.positions()
        ox, oy, oz = o.positions()
        assert np.array_equal(gx, ox) and np.array_equal(gy, oy) and np.array_equal(gz, oz)
        assert np.array_equal(g.density(), o.density())
        assert np.array_equal(g.omega().view(np.uint32), o.omega().view(np.uint32))
    o.close()


def test_cfg2_full_size_bond_force_biased_moves_bit_exact():
    """configs[2] at full size (16.8 M beads) with the paper's bond-force-biased moves (R24) on
    the fused kernel: 33.6 M Gaussian-driven moves, every coordinate bit-identical to the oracle."""
    w = si.config(2)
    s = si.make_system(w)
    o = oracle.Oracle.from_system(s)
    o.set_smc(0.05)
    o.load_state(s.x, s.y, s.z)
    acc_o = o.mc_steps(2)
    with gpu_system(s, smc_mobility=0.05) as g:
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(2, want_accepted=True) == acc_o
        for a, b_ in zip(g.positions(), o.positions()):
            assert np.array_equal(a, b_)
        assert np.array_equal(g.density(), o.density())
    o.close()
