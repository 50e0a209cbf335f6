"""Host-side logic of bench.py that needs no GPU: the multi-rank aggregation ("replicas only":
barrier, max-over-ranks time, sum-over-ranks work) on the gloo backend with world_size 2, the
roofline bookkeeping, and the sampling of a workload for the timed oracle."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _rank_main(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    bench.barrier()
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
    out[rank] = (ms, units, bench.dist_env())
    dist.destroy_process_group()


def test_aggregate_over_two_gloo_ranks():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = mp.get_context("spawn").Manager().dict()
    mp.spawn(_rank_main, args=(2, port, out), nprocs=2, join=True)
    for rank in (0, 1):
        ms, units, env = out[rank]
        assert ms == 15.0                       # the slowest rank
        assert units == 3000.0                  # all ranks' moves
        assert env[0] == rank and env[2] == 2


def test_aggregate_is_identity_without_a_process_group():
    import bench
    assert bench.aggregate_over_ranks(3.5, 42.0) == (3.5, 42.0)


def test_algorithmic_bytes_match_design_section_7():
    import bench
    import scmf_inputs as si
    w = si.config(4)
    ab = bench.algorithmic_bytes(w)
    B, TC = w.n_beads, w.n_types * w.n_cells
    assert ab["step"] == 24 * B + 20 * TC == ab["move_bin_kernel"] + ab["omega_kernel"]
    assert abs(ab["step"] / B - 26.5) < 1e-9     # 26.5 B per attempted move on cfg4


def test_sample_workload_keeps_beads_per_cell():
    import bench
    import scmf_inputs as si
    w = si.config(4)
    ws = bench.sample_workload(w, 64)
    assert ws.n_chains == w.n_chains // 64 and ws.N == w.N
    assert ws.n_beads / ws.n_cells == pytest.approx(w.n_beads / w.n_cells)
