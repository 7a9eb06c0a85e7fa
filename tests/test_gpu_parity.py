"""GPU parity tests: the CUDA library, called through the C ABI binding, against the CPU oracle on the
same seeded inputs (tests/parity.py states the comparison rule).  Sizes are chosen so the oracle takes
seconds while the work still spans several launches, several pool levels and ragged tails."""
import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import compare, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def both(O, cfg, params=None, **kw):
    rg = run_gpu(cfg, params, **kw)
    ro = run_oracle(O, cfg, params)
    return compare(rg, ro, cfg, params), rg, ro


def test_config1_stromgren(O):
    cfg = synth.make(1)
    worst, rg, ro = both(O, cfg)
    assert 3000 < rg[2].segments < 4500 and sum(rg[2].exited) == 0 and sum(rg[2].killed_tau) > 1000
    assert np.all(rg[1] == 0.0)                                              # 13.6 eV photons: e_excess = 0 exactly


@pytest.mark.parametrize("n", [48, 128])
def test_config2_shadow(O, n):
    cfg = synth.make(2, n=n)
    worst, rg, ro = both(O, cfg)
    g = rg[0]
    # the clump casts a shadow: cells on the axis well behind it get nothing
    s = n / 128.0
    src_x, cl_x = int(round(24 * s)), int(round(24 * s)) + int(round(40 * s))
    behind = g[n // 2, n // 2, cl_x + int(round(12 * s)):]
    ahead = g[n // 2, n // 2, src_x + 2:cl_x - int(round(10 * s))]
    assert np.all(behind == 0.0) and np.all(ahead > 0.0)


@pytest.mark.parametrize("batch", [0, 4096, 333])
def test_config3_many_sources_small(O, batch):
    cfg = synth.make(3, n=64, n_src=400)
    if batch == 333:
        batch = 352
    both(O, cfg, batch_rays=batch)


def test_config3_thin_long_rays(O):
    """rays crossing the whole (non-cubic would be nicer, see below) box: levels up to 7."""
    cfg = synth.make(3, n=96, n_src=12)
    cfg["xHI"] = cfg["xHI"] * 1e-3
    worst, rg, ro = both(O, cfg, batch_rays=8192)
    assert sum(rg[2].exited) > 1000 and rg[2].spawned[6] > 0


def test_config4_merge_small(O):
    cfg = synth.make(4, n=64, n_src=3000)
    worst, rg, ro = both(O, cfg, batch_rays=16384)
    st = rg[2]
    assert st.n_src_dedup < st.n_src_in and st.n_src_merged < st.n_src_dedup
    cfgb = synth.make(4, n=64, n_src=3000, r_max=3.0)
    both(O, cfgb, params=dict(f_ov=0.8, f_req=0.9, n_min_samples=150))


def test_config5_f32_small(O):
    cfg = synth.make(5, n=80, n_src=4000)
    assert cfg["nH"].dtype == torch.float32
    worst, rg, ro = both(O, cfg, batch_rays=20000)
    assert rg[2].n_src_merged < rg[2].n_src_dedup


def test_automerge_switch(O):
    cfg = synth.make(4, n=48, n_src=500)
    for thr, merged in ((0.018, True), (0.99, False)):
        worst, rg, ro = both(O, cfg, params=dict(merge=2, automerge_xmean=thr))
        assert (rg[2].n_src_merged < rg[2].n_src_dedup) == merged


@pytest.mark.parametrize("mode", [0, 1, 2, 4])
def test_geometry_modes(O, mode):
    cfg = synth.make(3, n=40, n_src=30)
    both(O, cfg, params=dict(geom_mode=mode))


@pytest.mark.parametrize("kw", [dict(n_min_ray=2.0), dict(n_min_ray=1.0), dict(level_max=3), dict(level_max=0),
                                dict(tau_max=2.0), dict(n_th=1e-6)])
def test_parameter_edges(O, kw):
    cfg = synth.make(3, n=40, n_src=25)
    cfg["xHI"] = cfg["xHI"] * 0.05
    worst, rg, ro = both(O, cfg, params=kw)
    if "level_max" in kw:
        assert sum(rg[2].killed_lmax) > 0


def test_non_cubic_grid_and_corner_sources(O):
    g = torch.Generator().manual_seed(4)
    nz, ny, nx = 20, 33, 47
    cfg = dict(shape=(nz, ny, nx), dx_cm=2e20,
               nH=10 ** (torch.rand((nz, ny, nx), generator=g, dtype=torch.float64) * 3 - 5),
               xHI=torch.rand((nz, ny, nx), generator=g, dtype=torch.float64) * 0.1,
               src_pos=torch.tensor([[0.5, 0.5, 0.5], [46.9, 32.9, 19.9], [23.0, 0.0, 10.0], [0.01, 32.99, 0.5],
                                     [23.2, 0.7, 10.1]], dtype=torch.float64),
               src_L=torch.tensor([1e50, 2e50, 3e49, 1e48, 5e49], dtype=torch.float64),
               params=synth.default_params(n_th=3e-5, e_excess_erg=1e-11))
    cfg["xHI"][5:9, 10:20, 30:40] = 0.0
    worst, rg, ro = both(O, cfg, batch_rays=1000)
    assert rg[2].n_src_dedup == 4


def test_no_sources_and_dark_sources(O):
    cfg = synth.make(1)
    cfg["src_pos"] = torch.zeros((0, 3), dtype=torch.float64)
    cfg["src_L"] = torch.zeros(0, dtype=torch.float64)
    worst, rg, ro = both(O, cfg)
    assert rg[2].segments == 0 and np.all(rg[0] == 0.0)
    cfg = synth.make(1)
    cfg["src_L"] = torch.zeros(1, dtype=torch.float64)
    worst, rg, ro = both(O, cfg)
    assert np.all(rg[0] == 0.0)


def test_fully_ionised_box(O):
    cfg = synth.make(1, n=24)
    cfg["xHI"] = torch.zeros_like(cfg["xHI"])
    worst, rg, ro = both(O, cfg)
    assert rg[2].photons_absorbed == 0.0 and abs(rg[2].photons_escaped - 5e48) < 1e36


def test_step_host_equals_device_path(O):
    cfg = synth.make(3, n=48, n_src=100)
    a = run_gpu(cfg)
    b = run_gpu(cfg, host=True)
    ro = run_oracle(O, cfg)
    compare(b, ro, cfg)
    assert list(a[2].spawned) == list(b[2].spawned) and a[2].segments == b[2].segments


def test_repeated_trace_is_stable(O):
    from paper_2512_12466_b200 import nyxrt
    cfg = synth.make(4, n=48, n_src=600)
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], max_sources=600, batch_rays=5000)
    tr.set_fields(cfg["nH"].cuda(), cfg["xHI"].cuda())
    tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
    g1, h1, s1 = tr.trace()
    c1 = tr.catalog()
    g2, h2, s2 = tr.trace()
    c2 = tr.catalog()
    assert list(s1.spawned) == list(s2.spawned) and s1.segments == s2.segments
    assert all(np.array_equal(x, y) for x, y in zip(c1, c2))
    assert torch.allclose(g1, g2, rtol=1e-12, atol=0)
    tr.close()


def test_directions_bit_exact(O):
    """DIR-SPEC: device and oracle directions are bit-identical (decisions depend on it)."""
    from paper_2512_12466_b200 import nyxrt
    tr = nyxrt.Tracer((8, 8, 8), 1e20, synth.default_params())
    for level in range(0, 7):
        d = tr.pix2dir(level, 0, 12 * 4 ** level)
        assert np.array_equal(d.view(np.uint64), O.pix2dir_all(level).view(np.uint64))
    rng = np.random.default_rng(0)
    for level in (9, 13):
        for p in rng.integers(0, 12 * 4 ** level - 64, 40):
            d = tr.pix2dir(level, int(p), 64)
            e = np.array([O.pix2dir(level, int(p) + k) for k in range(64)])
            assert np.array_equal(d.view(np.uint64), e.view(np.uint64))
    tr.close()


def test_error_paths():
    from paper_2512_12466_b200 import nyxrt
    p = synth.default_params()
    tr = nyxrt.Tracer((16, 16, 16), 1e20, p, max_sources=4)
    nH = torch.full((16, 16, 16), 1e-3, dtype=torch.float64, device="cuda")
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.trace()
    assert e.value.code == nyxrt.ESTATE
    tr.set_fields(nH, nH)
    for pos, L in (([[16.0, 1, 1]], [1.0]), ([[1.0, -0.1, 1]], [1.0]), ([[1.0, 1, 1]], [-1.0]),
                   ([[1.0, 1, 1]], [float("nan")]), ([[float("nan"), 1, 1]], [1.0])):
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.set_sources(np.array(pos), np.array(L))
        assert e.value.code == nyxrt.EINVAL
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.set_sources(np.ones((5, 3)), np.ones(5))
    assert e.value.code == nyxrt.ENOMEM
    tr.set_sources(np.array([[8.5, 8.5, 8.5]]), np.array([1e48]))
    g, h, st = tr.trace()
    assert st.segments > 0
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.step_host(nH.cpu(), nH.cpu(), np.ones((1, 3)), np.ones(1), torch.empty((16, 16, 16), dtype=torch.float64))
    assert e.value.code == nyxrt.ESTATE
    tr.close()
    bad = nyxrt.make_grid((16, 16, 16), 1e20)
    bad.periodic = 2
    with pytest.raises(nyxrt.NyxrtError):
        nyxrt.nyxrt_create(bad, nyxrt.make_params(**p))


@pytest.mark.parametrize("periodic", [0, 1])
def test_merge_large_groups(O, periodic):
    """Fully ionised gas: every bubble reaches R_max and the bubbles percolate, so almost all sources collapse
    into one group of thousands of members (collapse_big_kernel: one warp per large group, sums sequential in
    member order) next to a few small ones; the catalogue must equal the oracle's bit for bit."""
    cfg = synth.make(4, n=40, n_src=4000)
    cfg["xHI"] = torch.full_like(cfg["xHI"], 1e-3)
    rg = run_gpu(cfg, batch_rays=16384, periodic=periodic)
    ro = run_oracle(O, cfg, periodic=periodic)
    compare(rg, ro, cfg)
    st = rg[2]
    assert st.n_src_dedup > 1000 and st.n_src_merged < 40          # one giant group (and maybe a few loners)
    cfgb = synth.make(4, n=40, n_src=4000, r_max=2.0)             # many groups of tens to hundreds of members
    cfgb["xHI"] = torch.full_like(cfgb["xHI"], 1e-3)
    rgb = run_gpu(cfgb, batch_rays=16384, periodic=periodic)
    compare(rgb, run_oracle(O, cfgb, periodic=periodic), cfgb)
    assert 10 < rgb[2].n_src_merged < rgb[2].n_src_dedup


def test_graph_loop_and_profiling_loop_are_the_same_step(O):
    """Production runs the ray loop as one CUDA-graph launch (WHILE node over sched -> emit -> march); with
    NYXRT_FLAG_LAUNCH_TIMING the host enqueues the same kernels launch by launch with an event pair around every
    march launch (what bench.py's roofline needs).  Same counters, same rates, and both match the oracle; several
    traces on one context reuse the graph, a new spectrum table or shard rebuilds it."""
    from paper_2512_12466_b200 import nyxrt
    cfg = synth.make(4, n=64, n_src=3000)
    worst, rg, ro = both(O, cfg, batch_rays=16384)
    worst_t, rt, _ = both(O, cfg, params=dict(flags=nyxrt.FLAG_LAUNCH_TIMING), batch_rays=16384)
    sg, st = rg[2], rt[2]
    for name in ("spawned", "split", "killed_tau", "exited"):
        assert list(getattr(sg, name)) == list(getattr(st, name))
    assert sg.segments == st.segments and sg.iterations == st.iterations and sg.iterations > 10
    assert sg.ms_march == 0.0 and st.ms_march > 0.0 and sg.march_launches == st.march_launches
    assert np.all(np.abs(rg[0] - rt[0]) <= 1e-12 * rt[0])
    # one context, several traces: the graph is reused, then rebuilt for a shard, and reused again
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=cfg["nH"].dtype, max_sources=len(cfg["src_L"]),
                      batch_rays=16384)
    try:
        tr.set_fields(cfg["nH"].cuda(), cfg["xHI"].cuda())
        tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
        seg = [tr.trace()[2].segments for _ in range(3)]
        tr.set_shard(0, 2)
        s0 = tr.trace_photons()[1].segments
        tr.set_shard(1, 2)
        s1 = tr.trace_photons()[1].segments
        tr.set_shard(0, 1)
        seg.append(tr.trace()[2].segments)
    finally:
        tr.close()
    assert seg == [sg.segments] * 4 and s0 + s1 == sg.segments and 0 < s0 < sg.segments
