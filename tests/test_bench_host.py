"""Host logic of bench.py's N > 1 paths (the max-over-ranks of the timing; the sum of the ranks' own segments in
the source-sharded mode; the --replicas rate), run as two gloo ranks on the CPU; and the --impl reference rule
that only rank 0 works.  The data path of the sharded mode (one all-reduce of the photon grid) is exercised
across two processes on a GPU in tests/test_gpu_multiproc.py."""
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(100.0 + 50.0 * rank, "cpu")        # rank 1 is the slow one
    out[rank] = (ms, bench.whole_job_rate(1000, ms, world), bench.sum_over_ranks(700 + 300 * rank, "cpu"))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_rate_is_all_units_over_slowest_rank():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29533, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, rate, seg_all = res[0]
    assert ms == 150.0 and abs(rate - 2 * 1000 / 0.150) < 1e-9
    assert seg_all == 1700.0                                      # sharded mode: the ranks' own segments add up


def test_single_process_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, "cpu") == 12.5
    assert bench.whole_job_rate(10, 1000.0, 1) == 10.0
    assert bench.sum_over_ranks(3.0, "cpu") == 3.0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_alu_roofs_come_from_the_committed_instruction_counts():
    """The march kernel's roofs are derived from profiles/march_instr.csv (last row), not from a constant in bench.py:
    148 SMs x 4 schedulers x clock x 32 lanes / cycles per warp-cell, 2 fp64-pipe cycles per fp64 warp instruction."""
    sys.path.insert(0, ROOT)
    import bench
    ipc, fpc, prof = bench.march_instruction_counts()
    assert 100 <= ipc <= 400 and 40 <= fpc < ipc and prof.endswith(".md")
    assert os.path.exists(os.path.join(ROOT, "profiles", prof))
    r = bench.alu_roofs(segments=1.0e12, march_ms=10_000.0, sm_mhz=1965.0, inst_per_cell=200.0, fp64_per_cell=80.0)
    slots = 148 * 4 * 1965e6 * 32
    assert abs(r["achieved"] - 1.0e11) < 1.0
    assert abs(r["fp64_peak"] - slots / 160.0) < 1.0 and abs(r["issue_peak"] - slots / 200.0) < 1.0
    assert abs(r["fp64_frac"] - 1.0e11 * 160.0 / slots) < 1e-12 and r["issue_frac"] > r["fp64_frac"]
