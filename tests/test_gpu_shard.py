"""Source sharding ("Gamma from each point source is accumulated"):
nyxrt_set_shard + nyxrt_trace_photons + (sum of the photon grids) + nyxrt_finalise.  Only one GPU is at hand,
so the `world` shards run one after the other on it and their photon grids are added with torch -- exactly
what the all-reduce of Tracer.sharded_trace does across processes; the sum must match the oracle's unsharded
step by the rule of tests/parity.py, and the shards' ray counters must add up to the oracle's exactly."""
import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import COUNTERS, compare, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def run_sharded(cfg, world, periodic=0, batch_rays=0):
    from paper_2512_12466_b200 import nyxrt
    nH, xHI = cfg["nH"].cuda().contiguous(), cfg["xHI"].cuda().contiguous()
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=nH.dtype, max_sources=len(L),
                      batch_rays=batch_rays, periodic=periodic)
    try:
        tr.set_fields(nH, xHI)
        tr.set_sources(pos, L)
        total = torch.zeros(cfg["shape"], dtype=torch.float64, device="cuda")
        stats = []
        for r in range(world):
            tr.set_shard(r, world)
            ph, st = tr.trace_photons()
            total += ph                                              # the all-reduce, on one device
            stats.append(st)
        gam, heat, absorbed = tr.finalise(total)
        cat = tr.catalog()
        torch.cuda.synchronize()
        return gam.cpu().numpy(), heat.cpu().numpy(), stats, cat, absorbed
    finally:
        tr.close()


class Sum:
    """The shards' statistics added up, shaped like nyxrt_stats for tests/parity.compare."""

    def __init__(self, stats, absorbed):
        for name in COUNTERS:
            setattr(self, name, [sum(getattr(s, name)[l] for s in stats) for l in range(16)])
        for name in ("segments", "zero_len_segments", "neighbour_deposits"):
            setattr(self, name, sum(getattr(s, name) for s in stats))
        for name in ("photons_emitted", "photons_escaped", "photons_residual", "photons_lost"):
            setattr(self, name, sum(getattr(s, name) for s in stats))
        self.photons_absorbed = absorbed
        for name in ("n_src_in", "n_src_dedup", "n_src_merged"):
            assert len({getattr(s, name) for s in stats}) == 1       # every shard builds the whole catalogue
            setattr(self, name, getattr(stats[0], name))


@pytest.mark.parametrize("world", [2, 3, 8])
def test_shards_add_up_to_the_oracle_step(O, world):
    cfg = synth.make(4, n=48, n_src=1500)
    gam, heat, stats, cat, absorbed = run_sharded(cfg, world, batch_rays=8192)
    ro = run_oracle(O, cfg)
    compare((gam, heat, Sum(stats, absorbed), cat), ro, cfg)
    assert all(s.segments > 0 for s in stats)
    n_cat = stats[0].n_src_merged
    assert sum(s.spawned[0] for s in stats) == 12 * n_cat
    for r, s in enumerate(stats):                                    # shard r holds entries r, r + world, ...
        assert s.spawned[0] == 12 * len(range(r, n_cat, world))


def test_more_shards_than_sources_and_periodic(O):
    cfg = synth.make(3, n=32, n_src=3)
    cfg["xHI"] = cfg["xHI"] * 0.02
    gam, heat, stats, cat, absorbed = run_sharded(cfg, 5, periodic=1)
    ro = run_oracle(O, cfg, periodic=1)
    compare((gam, heat, Sum(stats, absorbed), cat), ro, cfg)
    assert [s.segments > 0 for s in stats] == [True, True, True, False, False]


def test_world_one_equals_trace(O):
    cfg = synth.make(3, n=40, n_src=50)
    gam, heat, stats, cat, absorbed = run_sharded(cfg, 1)
    a = run_gpu(cfg)
    assert np.allclose(gam, a[0], rtol=1e-12, atol=0) and stats[0].segments == a[2].segments


def test_trace_refuses_when_a_shard_is_set():
    from paper_2512_12466_b200 import nyxrt
    tr = nyxrt.Tracer((8, 8, 8), 1e20, synth.default_params(), max_sources=1)
    f = torch.full((8, 8, 8), 1e-3, dtype=torch.float64, device="cuda")
    tr.set_fields(f, f)
    tr.set_sources(np.array([[4.5, 4.5, 4.5]]), np.array([1e48]))
    for rank, world in ((2, 2), (-1, 2), (0, 0)):
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.set_shard(rank, world)
        assert e.value.code == nyxrt.EINVAL
    tr.set_shard(1, 2)
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.trace()
    assert e.value.code == nyxrt.ESTATE
    tr.set_shard(0, 1)
    assert tr.trace()[2].segments > 0
    tr.close()
