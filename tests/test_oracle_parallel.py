"""The multi-process form of the oracle (tests/parity.run_oracle_parallel: the source pass once, chunks of the
sorted catalogue traced by worker processes with the unchanged orc_trace loop, grids and counters added) gives
the serial oracle's step: Gamma is a sum over sources.  Also exercises orc_trace_add / orc_catalogue."""
import numpy as np
import pytest

from paper_2512_12466_b200 import synth
from parity import COUNTERS, run_oracle, run_oracle_parallel


@pytest.mark.parametrize("periodic", [0, 1])
def test_parallel_oracle_equals_serial(O, periodic):
    cfg = synth.make(4, n=40, n_src=300)
    go, ho, so, co = run_oracle(O, cfg, periodic=periodic)
    osum, cat = run_oracle_parallel(O, cfg, 3, periodic=periodic, chunk=7)
    try:
        assert all(np.array_equal(a, b) for a, b in zip(cat, co))
        st = osum.stats
        for name in COUNTERS:
            assert list(getattr(st, name)) == list(getattr(so, name)), name
        for name in ("segments", "zero_len_segments", "neighbour_deposits", "n_src_in", "n_src_dedup", "n_src_merged"):
            assert getattr(st, name) == getattr(so, name), name
        g, h = osum.gamma(), osum.heat()
        assert np.array_equal(g == 0, go == 0)
        assert np.all(np.abs(g - go) <= 1e-13 * go) and np.all(np.abs(h - ho) <= 1e-13 * ho)
        for name in ("photons_emitted", "photons_absorbed", "photons_escaped", "photons_residual"):
            assert abs(getattr(st, name) - getattr(so, name)) <= 1e-13 * so.photons_emitted
    finally:
        osum.close()


def test_a_dying_worker_leaves_no_process_and_no_shared_memory_behind(O, monkeypatch):
    """Process management only: when a worker ends without reporting (here: it exits at once, as after a SIGBUS on a
    full /dev/shm), step_parallel raises, joins or stops every worker and unlinks every segment it created."""
    import multiprocessing as mp
    import os

    def dies(*a):
        os._exit(7)

    monkeypatch.setattr(O, "_worker", dies)
    before = set(os.listdir("/dev/shm")) if os.path.isdir("/dev/shm") else None
    cfg = synth.make(4, n=24, n_src=20)
    with pytest.raises(RuntimeError, match="worker"):
        run_oracle_parallel(O, cfg, 3, chunk=2)
    assert not mp.active_children()
    if before is not None:
        assert set(os.listdir("/dev/shm")) <= before


def test_more_workers_than_shared_memory_can_hold_are_not_started(O, monkeypatch):
    import shutil
    from collections import namedtuple
    cfg = synth.make(4, n=24, n_src=20)
    per_proc = 2 * 24 ** 3 * 8
    U = namedtuple("U", "total used free")
    monkeypatch.setattr(shutil, "disk_usage", lambda path: U(10 * per_proc, 0, int(2.5 * per_proc / 0.9)))
    osum, _ = run_oracle_parallel(O, cfg, 6, chunk=2)
    try:
        assert osum.n_proc == 2 and len(osum._g) == 2                # asked for 6, room for 2
    finally:
        osum.close()
    monkeypatch.setattr(shutil, "disk_usage", lambda path: U(per_proc, 0, per_proc // 2))
    with pytest.raises(MemoryError, match="/dev/shm"):
        run_oracle_parallel(O, cfg, 2, chunk=2)
