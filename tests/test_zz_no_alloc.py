"""soma_validate_noalloc -- the entry point for callers that must not allocate device memory.

Who needs it: a simulation whose share of the GPU was fixed before it started (spawned next to another solver,
or living inside a PyTorch process whose caching allocator already owns the free HBM), where a late cudaMalloc
may fail or take what the neighbour needs; a time-critical loop that cannot afford the device-wide stall of
cudaMalloc / cudaFree; and a check made before any handle -- and so any workspace -- exists.  The library keeps
the partial results of that call in one fixed 1.6 MB device array of its own, which every call on the device
shares and which keeps whatever the previous call left in it.

What is checked here: the report equals the one soma_validate_state gives for the same state (the existing
path, which works in the handle's workspace), on two calls in a row where the second state is SMALLER than the
first -- so a call that read slots it had not written itself would pick up the first state's leftovers -- and
that a state too large for the fixed array is refused with a message instead of being truncated.

This file is named so that pytest collects it last: with `pytest -x` a failure here hides no other test.  It
passes alone in a fresh process (the first call then does the per-device set-up) and after the other tests.
"""
import numpy as np
import pytest

import scmf_inputs as si
from helpers import gpu_system

pytestmark = pytest.mark.gpu


def _existing_and_noalloc(s, steps):
    """Run `steps` MC steps, then report the state through both paths: (soma_validate_state, soma_validate_noalloc)."""
    import torch
    import paper_2606_09356_b200 as soma
    w = s.workload
    with gpu_system(s) as g:
        g.load_state(s.x, s.y, s.z)
        if steps:
            g.mc_steps(steps)
        existing = g.validate()
        x, y, z = g.positions_device()                               # the caller's inputs: made before the call
        counts = torch.empty((w.n_types, g.cells), dtype=torch.int32, device="cuda")
        soma.soma_get_density(g._h, counts)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        stream = torch.cuda.current_stream().cuda_stream
        got = soma.soma_validate_noalloc(x, y, z, w.n_chains, w.N, counts, w.n_types, g.cells, stream)
        again = soma.soma_validate_noalloc(x, y, z, w.n_chains, w.N, counts, w.n_types, g.cells, stream)
        assert torch.cuda.memory_allocated() == before                # the binding made no tensor either
    return existing, got, again


def _assert_same_report(existing, got, n_beads, n_types):
    assert got["ok"] and existing["ok"]
    assert got["nonfinite"] == existing["nonfinite"] == 0
    assert got["density_total"] == existing["density_total"] == n_beads
    assert got["density_per_type"] == existing["density_per_type"]
    assert all(v == 0 for v in got["density_per_type"][n_types:])
    assert got["max_bond_sq"] == existing["max_bond_sq"]                               # fp32 maximum: exact
    assert got["mean_bond_sq"] == pytest.approx(existing["mean_bond_sq"], rel=1e-12)   # double sums in another order


def test_two_calls_in_a_row_match_the_existing_path():
    # first a state of 5 tiles plus a ragged tail, then a smaller one of other chain length: the second call finds
    # the first call's partial results still in the shared array and must not pick any of them up
    big = si.make_system(si.scaled(si.config(4), 700, (32, 32, 16)))       # 700 chains x 32 beads = 22 400 beads
    small = si.make_system(si.scaled(si.config(3), 45, (16, 16, 16)))      # 45 chains x 64 beads = 2 880 beads: one tile
    for s, steps in ((big, 3), (small, 2)):
        existing, got, again = _existing_and_noalloc(s, steps)
        _assert_same_report(existing, got, s.workload.n_beads, s.workload.n_types)
        assert again == got                                                # fixed summation order: same bits every time


def test_positions_only_and_nonfinite_coordinates_are_counted():
    import torch
    import paper_2606_09356_b200 as soma
    n, N = 300, 16
    rng = np.random.default_rng(7)
    xyz = [torch.from_numpy(rng.normal(size=n * N).astype(np.float32)).cuda() for _ in range(3)]
    xyz[0][5] = float("nan")
    xyz[1][4099] = float("nan")            # in the second tile
    xyz[2][n * N - 1] = float("nan")       # the very last bead
    v = soma.soma_validate_noalloc(*xyz, n, N)
    assert v["nonfinite"] == 3 and not v["ok"] and v["density_total"] == 0
    # as on the existing path, a bond that touches a NaN drops out of the maximum and of the sum (it is already
    # counted as non-finite); the rest is as numpy computes it
    a = [t.cpu().numpy().astype(np.float64).reshape(n, N) for t in xyz]
    q = sum((c[:, 1:] - c[:, :-1]) ** 2 for c in a)
    q = q[~np.isnan(q)]
    assert v["mean_bond_sq"] == pytest.approx(q.sum() / (n * (N - 1)), rel=1e-6)
    assert v["max_bond_sq"] == pytest.approx(q.max(), rel=1e-6)
    xyz[0][5] = float("inf")               # infinities count as well
    assert soma.soma_validate_noalloc(*xyz, n, N)["nonfinite"] == 3


def test_a_state_beyond_the_fixed_array_is_refused_with_a_message():
    import torch
    import paper_2606_09356_b200 as soma
    t = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(soma.SomaError) as e:                       # 2^28 + 32 beads: refused before the device is touched
        soma.soma_validate_noalloc(t, t, t, (1 << 23) + 1, 32)
    assert e.value.code == soma.SOMA_EINVAL
    assert "268435456" in str(e.value) and "scratch" in str(e.value)
    with pytest.raises(soma.SomaError):
        soma.soma_validate_noalloc(t, t, t, 2, 32, counts=t, n_types=9, cells=4)
