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


def test_gpus_flag_launches_the_ranks_itself():
    """`python bench.py --gpus 2` with no launcher around it starts 2 ranks (torch.distributed.run on
    127.0.0.1) and rank 0 prints one line with n_gpus = 2.  --dry --backend gloo: no GPU work."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry", "--backend", "gloo", "--steps", "4"],
                       capture_output=True, text=True, env=env, cwd=ROOT, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                       # rank 0 only
    line = json.loads(lines[0])
    import scmf_inputs as si
    assert line["n_gpus"] == 2 and line["dry"] is True
    assert line["ms_per_step"] == pytest.approx(15.0 / 4)        # the slower rank's time
    assert line["value"] == pytest.approx(2 * si.config(4).n_beads * 4 / 15e-3)
    assert line["config"]["parallelism"] == "replicas only"


def test_gpus_flag_must_agree_with_the_launcher():
    import subprocess
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT="29555")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--dry", "--backend", "gloo"],
                       capture_output=True, text=True, env=env, cwd=ROOT, timeout=120)
    assert r.returncode != 0 and "WORLD_SIZE=2" in r.stderr


def test_ncu_table_rows_are_keyed_by_the_kernel_sources(tmp_path):
    """bench.py quotes ncu counters only from a row captured on the kernel sources it runs."""
    import bench
    key = bench.kernel_source_hash()
    head = "path,config,source_hash,capture,dram_bytes_read,dram_bytes_write,lts_sectors,inst_executed,l1tex2xbar_req_pct,lsu_wavefronts_pct,issue_active_pct,limiter\n"
    t = tmp_path / "t.csv"
    t.write_text(head + f"2,4,{'0' * 12},old.txt,1,2,3,4,5,6,7,stale\n" + f"2,4,{key},new.txt,10,20,30,40,50,60,70,fresh\n")
    row = bench.ncu_counters(2, 4, str(t))
    assert row["capture"] == "new.txt" and row["limiter"] == "fresh"
    assert bench.ncu_counters(1, 4, str(t)) is None              # no capture of that path
    t.write_text(head + f"2,4,{'0' * 12},old.txt,1,2,3,4,5,6,7,stale\n")
    assert bench.ncu_counters(2, 4, str(t)) is None              # stale rows are never quoted
    assert bench.ncu_counters(2, 4, str(tmp_path / "missing.csv")) is None


def test_both_arms_time_the_oracle_on_the_same_sample():
    import bench
    import scmf_inputs as si
    w = si.config(4)
    ws_ours, f_ours = bench.oracle_sample(w, 4)                  # cpu_baseline of our arm
    ws_ref, f_ref = bench.oracle_sample(w, 20 + 5)               # --impl reference at the driver's K, W
    assert f_ours == f_ref == 8 and ws_ours.n_chains == ws_ref.n_chains == w.n_chains // 8
    _, f_long = bench.oracle_sample(w, 1000)                     # a long run is scaled down further
    assert f_long > 8
    ws0, f0 = bench.oracle_sample(si.config(0), 4)               # a small config is timed whole
    assert f0 == 1 and ws0.n_chains == si.config(0).n_chains
