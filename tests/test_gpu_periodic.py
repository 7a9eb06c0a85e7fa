"""GPU parity tests of the periodic box ("rays wrap around the box,
terminating when their travel distance exceeds sqrt(3) L_box", RAY_FLTR at 174, minimum-image merge at 321 and
380-383, wrapped shell samples at 351): the CUDA library with `grid.periodic = 1` against the oracle's
periodic mode (pinned in tests/test_oracle_periodic.py) on the same seeded inputs, by the rule of
tests/parity.py (counters exact, rates to 1e-9)."""
import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import compare, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def both(O, cfg, params=None, **kw):
    rg = run_gpu(cfg, params, periodic=1, **kw)
    ro = run_oracle(O, cfg, params, periodic=1)
    return compare(rg, ro, cfg, params), rg, ro


def s_max(shape):
    return float(np.sqrt(sum(int(v) ** 2 for v in shape)))


def test_thin_box_rays_wrap_to_the_travel_limit(O):
    """Optically thin box: every lineage wraps around several faces and ends at s >= sqrt(3) L_box."""
    cfg = synth.make(3, n=40, n_src=10)
    cfg["xHI"] = cfg["xHI"] * 1e-3
    worst, rg, ro = both(O, cfg, batch_rays=8192)
    st = rg[2]
    assert sum(st.exited) > 10000 and st.spawned[6] > 0
    # more segments than the open box can hold from the same sources
    open_gpu = run_gpu(cfg, batch_rays=8192)
    assert st.segments > 2 * open_gpu[2].segments


def test_mixed_medium_kills_and_wraps(O):
    cfg = synth.make(3, n=40, n_src=16)
    cfg["xHI"] = cfg["xHI"] * 0.02
    worst, rg, ro = both(O, cfg, batch_rays=4096)
    assert sum(rg[2].killed_tau) > 0 and sum(rg[2].exited) > 0


def test_merge_minimum_image(O):
    """Merging on: bubbles that overlap across a face link through the minimum image; centroid and snap use
    the images nearest to the first member."""
    cfg = synth.make(4, n=32, n_src=900)
    worst, rg, ro = both(O, cfg, batch_rays=16384)
    st = rg[2]
    assert st.n_src_merged < st.n_src_dedup
    # the open-box catalogue differs (some links exist only across the faces)
    open_gpu = run_gpu(cfg, batch_rays=16384)
    assert open_gpu[2].n_src_merged >= st.n_src_merged
    cfgb = synth.make(4, n=32, n_src=900, r_max=5.0)                       # bin width not dividing the box
    both(O, cfgb, params=dict(f_ov=0.8, f_req=0.9, n_min_samples=150))


def test_merge_only_across_faces(O):
    """Hand case: two sources in fully ionised gas at opposite faces, 4 cells apart through the wall and 28
    apart inside the box: they merge only in the periodic box."""
    n = 32
    cfg = dict(shape=(n, n, n), dx_cm=1e21, nH=torch.full((n, n, n), 1e-6, dtype=torch.float64),
               xHI=torch.full((n, n, n), 1e-3, dtype=torch.float64),
               src_pos=torch.tensor([[1.5, 10.5, 10.5], [29.5, 10.5, 10.5], [16.5, 30.5, 1.5], [16.5, 2.5, 30.5]],
                                    dtype=torch.float64),
               src_L=torch.tensor([1e50, 3e50, 2e50, 2e50], dtype=torch.float64),
               params=synth.default_params(merge=1, r_max=4.0))
    worst, rg, ro = both(O, cfg)
    assert rg[2].n_src_merged == 2
    cells = {tuple(c) for c in rg[3][0].tolist()}
    assert (29, 10, 10) in cells                                           # flux-weighted centroid snaps to the brighter
    assert run_gpu(cfg)[2].n_src_merged == 4


def test_f32_fields(O):
    cfg = synth.make(5, n=40, n_src=600)
    assert cfg["nH"].dtype == torch.float32
    both(O, cfg, batch_rays=20000)


@pytest.mark.parametrize("mode", [0, 1, 2, 4])
def test_geometry_modes(O, mode):
    cfg = synth.make(3, n=32, n_src=12)
    cfg["xHI"] = cfg["xHI"] * 0.01
    both(O, cfg, params=dict(geom_mode=mode))


@pytest.mark.parametrize("shape", [(20, 33, 47), (1, 9, 12), (7, 1, 1), (1, 1, 1)])
def test_non_cubic_and_degenerate_boxes(O, shape):
    """Non-cubic boxes, sources in corners, axes one cell wide (the ray re-enters the same cell; the cell is
    its own neighbour)."""
    g = torch.Generator().manual_seed(4)
    nz, ny, nx = shape
    pos = torch.tensor([[0.5, 0.5, 0.5], [nx - 0.1, ny - 0.1, nz - 0.1], [nx / 2.0, 0.0, nz / 2.0],
                        [0.01, ny - 0.01, 0.5]], dtype=torch.float64)
    cfg = dict(shape=shape, dx_cm=2e20,
               nH=10 ** (torch.rand(shape, generator=g, dtype=torch.float64) * 3 - 5),
               xHI=torch.rand(shape, generator=g, dtype=torch.float64) * 0.1,
               src_pos=pos, src_L=torch.tensor([1e50, 2e50, 3e49, 1e48], dtype=torch.float64),
               params=synth.default_params(n_th=3e-5, e_excess_erg=1e-11))
    if nz > 8:
        cfg["xHI"][5:9, 10:20, 30:40] = 0.0
    worst, rg, ro = both(O, cfg, batch_rays=1000)
    assert rg[2].segments > 0


def test_translation_invariance_on_the_device(O):
    """Rolling fields and sources rolls the result (to summation order): the device's wrap-around has no
    preferred origin."""
    cfg = synth.make(3, n=36, n_src=8)
    cfg["xHI"] = cfg["xHI"] * 0.01
    a = run_gpu(cfg, periodic=1)
    sh = (5, -7, 11)                                                       # (dz, dy, dx)
    cfg2 = dict(cfg)
    cfg2["nH"] = torch.roll(cfg["nH"], sh, (0, 1, 2))
    cfg2["xHI"] = torch.roll(cfg["xHI"], sh, (0, 1, 2))
    pos = cfg["src_pos"].clone()
    for ax, d in ((0, sh[2]), (1, sh[1]), (2, sh[0])):
        pos[:, ax] = torch.remainder(torch.floor(pos[:, ax]) + d, 36) + 0.5
    cfg2["src_pos"] = pos
    b = run_gpu(cfg2, periodic=1)
    assert list(a[2].spawned) == list(b[2].spawned) and a[2].segments == b[2].segments
    assert list(a[2].exited) == list(b[2].exited) and list(a[2].killed_tau) == list(b[2].killed_tau)
    ga = np.roll(a[0], sh, (0, 1, 2))
    assert np.allclose(b[0], ga, rtol=1e-9, atol=1e-30)
    assert np.array_equal(b[0] == 0, ga == 0)


def test_periodic_flag_is_validated():
    from paper_2512_12466_b200 import nyxrt
    bad = nyxrt.make_grid((16, 16, 16), 1e20, periodic=2)
    with pytest.raises(nyxrt.NyxrtError):
        nyxrt.nyxrt_create(bad, nyxrt.make_params(**synth.default_params()))
