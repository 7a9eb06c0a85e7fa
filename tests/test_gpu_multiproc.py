"""Source sharding across PROCESSES (Gamma is a sum over sources): two
processes, each with its own context on the one GPU at hand and a gloo group between them, run
Tracer.sharded_trace -- set_shard(rank, 2), trace_photons, ONE all-reduce of the photon grid, finalise -- the control
flow the NCCL path has on two GPUs (bench.py's default for N > 1).  Rank 0's result against the oracle's unsharded
step by the rule of tests/parity.py; both processes must build bit-identical catalogues (nothing is broadcast)."""
import os
import sys
import tempfile

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2512_12466_b200 import synth
from parity import compare, run_oracle

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, tmp, periodic):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2512_12466_b200 import nyxrt, synth as S
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    cfg = S.make(4, n=48, n_src=1500)
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=cfg["nH"].dtype,
                      max_sources=len(cfg["src_L"]), batch_rays=8192, periodic=periodic)
    try:
        tr.set_shard(rank, world)
        tr.set_fields(cfg["nH"].cuda(), cfg["xHI"].cuda())
        tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
        gam, heat, st, absorbed = tr.sharded_trace()
        cat = tr.catalog()
        torch.cuda.synchronize()
        # the ranks' own counters, added over the group like bench.py adds its segments
        cnt = torch.tensor([list(st.spawned), list(st.split), list(st.killed_tau), list(st.exited), list(st.killed_lmax)],
                           dtype=torch.int64)
        tot = torch.tensor([st.segments, st.zero_len_segments, st.neighbour_deposits], dtype=torch.int64)
        ph = torch.tensor([st.photons_emitted, st.photons_escaped, st.photons_residual, st.photons_lost], dtype=torch.float64)
        own_segments = int(st.segments)
        for t in (cnt, tot, ph):
            dist.all_reduce(t)
        np.savez(os.path.join(tmp, "rank%d.npz" % rank), gam=gam.cpu().numpy(), heat=heat.cpu().numpy(),
                 cat_cell=cat[0], cat_L=cat[1], cat_r=cat[2], cnt=cnt.numpy(), tot=tot.numpy(), ph=ph.numpy(),
                 absorbed=absorbed, own_segments=own_segments,
                 n_src=np.array([st.n_src_in, st.n_src_dedup, st.n_src_merged]))
    finally:
        tr.close()
        dist.barrier()
        dist.destroy_process_group()


class _Stats:
    pass


@pytest.mark.parametrize("periodic", [0, 1])
def test_two_processes_one_allreduce(O, periodic):
    import gc
    world = 2
    gc.collect()
    torch.cuda.empty_cache()          # the children need room for their own contexts next to this process's cache
    with tempfile.TemporaryDirectory() as tmp:
        mp.spawn(_worker, args=(world, 29541 + periodic, tmp, periodic), nprocs=world, join=True)
        r = [np.load(os.path.join(tmp, "rank%d.npz" % k)) for k in range(world)]
        r = [{k: v[k] for k in v.files} for v in r]
    # every process built the whole catalogue, identically (replicated, not broadcast)
    for k in ("cat_cell", "cat_L", "cat_r", "n_src"):
        assert np.array_equal(r[0][k], r[1][k]), k
    # both hold the same all-reduced result; each marched its own share of the rays
    assert np.array_equal(r[0]["gam"], r[1]["gam"]) and np.array_equal(r[0]["heat"], r[1]["heat"])
    assert 0 < r[0]["own_segments"] < r[0]["tot"][0] and r[0]["own_segments"] + r[1]["own_segments"] == r[0]["tot"][0]
    cfg = synth.make(4, n=48, n_src=1500)
    ro = run_oracle(O, cfg, periodic=periodic)
    st = _Stats()
    for i, name in enumerate(("spawned", "split", "killed_tau", "exited", "killed_lmax")):
        setattr(st, name, [int(v) for v in r[0]["cnt"][i]])
    st.segments, st.zero_len_segments, st.neighbour_deposits = (int(v) for v in r[0]["tot"])
    st.photons_emitted, st.photons_escaped, st.photons_residual, st.photons_lost = (float(v) for v in r[0]["ph"])
    st.photons_absorbed = float(r[0]["absorbed"])
    st.n_src_in, st.n_src_dedup, st.n_src_merged = (int(v) for v in r[0]["n_src"])
    worst = compare((r[0]["gam"], r[0]["heat"], st, (r[0]["cat_cell"], r[0]["cat_L"], r[0]["cat_r"])), ro, cfg)
    print("two processes, one all-reduce%s: worst relative Gamma error %.2e" % (" (periodic)" if periodic else "", worst))
