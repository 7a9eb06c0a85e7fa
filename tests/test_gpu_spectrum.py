"""GPU parity tests of the frequency-integrated flux (Sec. 2.2): the
CUDA library with a spectrum table set (march_kernel<..., LUT = true>) against the oracle with the SAME table
(an input, like the fields; each side has its own lookup), by the rule of tests/parity.py.  The library's own
black-body table generator is checked against the oracle's (pinned to scipy's quadrature in
tests/test_oracle_spectrum.py)."""
import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import compare

pytestmark = pytest.mark.gpu

E_LO, E_HI, M = -20, 12, 6


@pytest.fixture(scope="module")
def bb(O):
    return O.blackbody_table(1e5, E_LO, E_HI, M)


def run_both(O, cfg, table, params=None, periodic=0, batch_rays=0, geom=(E_LO, E_HI, M)):
    from paper_2512_12466_b200 import nyxrt
    p = dict(cfg["params"])
    p.update(params or {})
    nH, xHI = cfg["nH"], cfg["xHI"]
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, field_dtype=nH.dtype, max_sources=len(L), batch_rays=batch_rays,
                      periodic=periodic)
    try:
        tr.set_spectrum(*geom, table)
        tr.set_fields(nH.cuda().contiguous(), xHI.cuda().contiguous())
        tr.set_sources(pos, L)
        gam, heat, st = tr.trace()
        cat = tr.catalog()
        torch.cuda.synchronize()
        rg = (gam.cpu().numpy(), heat.cpu().numpy(), st, cat)
    finally:
        tr.close()
    g = O.make_grid(cfg["shape"], cfg["dx_cm"], field_dtype=nH.numpy().dtype, periodic=periodic)
    try:
        O.set_spectrum(*geom, table)
        ro = O.step(g, O.make_params(**p), nH.numpy(), xHI.numpy(), pos, L)
    finally:
        O.set_spectrum()
    return compare(rg, ro, cfg, params), rg, ro


def test_blackbody_many_sources(O, bb):
    cfg = synth.make(3, n=48, n_src=60)
    cfg["xHI"] = cfg["xHI"] * 0.05
    worst, rg, ro = run_both(O, cfg, bb, params=dict(tau_max=60.0), batch_rays=4096)
    st = rg[2]
    assert sum(st.killed_tau) > 0 and sum(st.exited) > 0 and st.segments > 10 ** 6
    # the hard tail leaves the box: far more escapes than the monochromatic trace of the same inputs
    from parity import run_gpu
    mono = run_gpu(cfg, params=dict(tau_max=60.0), batch_rays=4096)
    assert st.photons_escaped > 1.5 * mono[2].photons_escaped
    assert list(st.spawned) == list(mono[2].spawned)                      # tau does not depend on the spectrum


def test_blackbody_merge_f32_and_periodic(O, bb):
    cfg = synth.make(4, n=40, n_src=800)
    run_both(O, cfg, bb, batch_rays=8192)
    cfg = synth.make(5, n=40, n_src=500)
    assert cfg["nH"].dtype == torch.float32
    run_both(O, cfg, bb, batch_rays=8192)
    cfg = synth.make(3, n=32, n_src=8)
    cfg["xHI"] = cfg["xHI"] * 0.02
    run_both(O, cfg, bb, periodic=1)


def test_thick_cells_beyond_the_table(O):
    """A short table (2^-6 .. 2^3): thin cells fall below it (linear from 0), neutral cells above it (constant)."""
    t = np.array([O.spectrum_node_tau(-6, 3, k) for k in range(O.spectrum_nodes(-6, 3, 3))])
    q = 1.0 - 1.0 / (1.0 + t) ** 0.7                                      # any concave increasing curve
    cfg = synth.make(2, n=48)
    worst, rg, ro = run_both(O, cfg, q, geom=(-6, 3, 3))
    assert sum(rg[2].killed_tau) > 0


def test_table_of_the_exponential_is_the_monochromatic_kernel(O):
    from paper_2512_12466_b200 import nyxrt
    from parity import run_gpu
    cfg = synth.make(3, n=40, n_src=20)
    cfg["xHI"] = cfg["xHI"] * 0.1
    t = np.array([O.spectrum_node_tau(-30, 8, k) for k in range(O.spectrum_nodes(-30, 6, 8))])
    worst, rg, ro = run_both(O, cfg, -np.expm1(-t), geom=(-30, 6, 8))
    mono = run_gpu(cfg)
    lit = mono[0] > 0
    assert np.array_equal(rg[0] > 0, lit)
    assert np.median(np.abs(rg[0][lit] - mono[0][lit]) / mono[0][lit]) < 2e-4
    assert abs(rg[2].photons_absorbed - mono[2].photons_absorbed) < 1e-5 * mono[2].photons_absorbed


def test_library_blackbody_table_and_nodes(O):
    from paper_2512_12466_b200 import nyxrt
    assert nyxrt.nyxrt_spectrum_nodes(-4, 8, 2) == O.spectrum_nodes(-4, 8, 2) == 49
    for k in (0, 1, 7, 48):
        assert nyxrt.nyxrt_spectrum_node_tau(-4, 2, k) == O.spectrum_node_tau(-4, 2, k)
    for T in (3e4, 1e5):
        a = nyxrt.nyxrt_blackbody_table(T, -10, 10, 2)
        b = O.blackbody_table(T, -10, 10, 2)
        assert np.all(np.abs(a - b) <= 1e-8 * b), float(np.max(np.abs(a - b) / b))
        assert np.all(np.diff(a) >= 0) and a[-1] <= 1.0


def test_set_spectrum_validation_and_reset(O, bb):
    from paper_2512_12466_b200 import nyxrt
    cfg = synth.make(3, n=24, n_src=5)
    nH, xHI = cfg["nH"].cuda(), cfg["xHI"].cuda()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], max_sources=5)
    tr.set_fields(nH, xHI)
    tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
    g0 = tr.trace()[0].clone()
    for bad in (bb[:-1], bb[::-1].copy(), bb * 1.5):
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.set_spectrum(E_LO, E_HI, M, bad)
        assert e.value.code == nyxrt.EINVAL
    with pytest.raises(nyxrt.NyxrtError):
        tr.set_spectrum(3, 3, M, bb)
    tr.set_spectrum(E_LO, E_HI, M, bb)
    g1 = tr.trace()[0].clone()
    assert not torch.equal(g0, g1)
    tr.set_spectrum()                                                     # back to monochromatic
    assert torch.allclose(tr.trace()[0], g0, rtol=1e-12, atol=0)
    tr.close()
    p = dict(cfg["params"])
    p["geom_mode"] = 1
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, max_sources=5)
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.set_spectrum(E_LO, E_HI, M, bb)
    assert e.value.code == nyxrt.EINVAL
    tr.close()


def test_timestep_with_a_spectrum(O, bb):
    """The RT timestep on top of the frequency-integrated flux: the paper's full update."""
    from paper_2512_12466_b200 import nyxrt
    MYR = 3.1557e13
    cfg = synth.make(1)
    nH, y0 = cfg["nH"], cfg["xHI"].double()
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    p = dict(cfg["params"])
    p["tau_max"] = 200.0
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, max_sources=1)
    try:
        tr.set_spectrum(E_LO, E_HI, M, bb)
        tr.set_sources(pos, L)
        xe, xa, gam, heat, st, ts = tr.timestep(nyxrt.make_ode(1.0 * MYR), nH.cuda(), y0.cuda())
        xe, xa, gam = xe.cpu().numpy(), xa.cpu().numpy(), gam.cpu().numpy()
    finally:
        tr.close()
    g = O.make_grid(cfg["shape"], cfg["dx_cm"])
    try:
        O.set_spectrum(E_LO, E_HI, M, bb)
        oe, oa, ogam, oheat, ost, ots, cat = O.timestep(g, O.make_params(**p), O.make_ode(1.0 * MYR), nH.numpy(),
                                                        y0.numpy(), pos, L)
    finally:
        O.set_spectrum()
    assert ts.iterations == ots.iterations and ts.converged == ots.converged and ts.iterations >= 2
    assert st.segments == ost.segments and list(st.killed_tau) == list(ost.killed_tau)
    assert np.all(np.abs(gam - ogam) <= 1e-9 * np.abs(ogam) + 1e-30)
    assert np.all(np.abs(xe - oe) <= 1e-9 * np.abs(oe) + 1e-15)
    # a hard spectrum pre-ionises gas ahead of the front: the transition is wider than the monochromatic one
    assert float(np.sum((xe > 0.1) & (xe < 0.9))) > 0
