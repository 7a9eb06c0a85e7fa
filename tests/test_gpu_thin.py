"""GPU parity tests of the separate table for the optically thin case (PAPER.md:267 footnote 3; readings R40-R42;
SURVEY.md 8(f) item 2): the CUDA library with both tables set (march_kernel<..., LUT = 2>) against the oracle with
the SAME tables and threshold, by the rule of tests/parity.py; ionised boxes like config 4's, where almost every
segment is below the threshold, mixed media, fp32 fields, a periodic box, source shards, and the RT timestep on
top.  The library's own generator of T against the oracle's (pinned to quadrature in tests/test_oracle_thin.py)."""
import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import nyxrt, synth
from parity import compare

pytestmark = pytest.mark.gpu

E_LO, E_HI, M = -20, 12, 6


@pytest.fixture(scope="module")
def tabs(O):
    return O.blackbody_table(1e5, E_LO, E_HI, M), O.blackbody_thin_table(1e5, E_LO, E_HI, M)


def run_both(O, cfg, tabs, tau_thin, params=None, periodic=0, batch_rays=0):
    p = dict(cfg["params"])
    p.update(params or {})
    nH, xHI = cfg["nH"], cfg["xHI"]
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, field_dtype=nH.dtype, max_sources=len(L), batch_rays=batch_rays,
                      periodic=periodic)
    try:
        tr.set_spectrum(E_LO, E_HI, M, tabs[0])
        tr.set_spectrum_thin(tabs[1], tau_thin)
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
        O.set_spectrum(E_LO, E_HI, M, tabs[0])
        O.set_spectrum_thin(tabs[1], tau_thin)
        ro = O.step(g, O.make_params(**p), nH.numpy(), xHI.numpy(), pos, L)
    finally:
        O.set_spectrum()
    return compare(rg, ro, cfg, params), rg, ro


def test_generator_matches_the_oracles(O, tabs):
    t = nyxrt.nyxrt_blackbody_thin_table(1e5, E_LO, E_HI, M)
    assert t.shape == tabs[1].shape and np.all(np.abs(t - tabs[1]) <= 1e-7 * tabs[1] + 1e-300)


@pytest.mark.parametrize("periodic", [0, 1])
def test_ionised_box_with_merging(O, tabs, periodic):
    """config-4-like: x_HI = 1e-4 except neutral islands, merging on: almost every segment takes the thin form."""
    cfg = synth.make(4, n=48, n_src=400)
    worst, rg, ro = run_both(O, cfg, tabs, 2.0 ** -10, params=dict(tau_max=60.0), periodic=periodic, batch_rays=4096)
    assert rg[2].segments > 10 ** 5
    print("thin table, ionised box%s: %d segments, worst relative Gamma error %.2e"
          % (" (periodic)" if periodic else "", rg[2].segments, worst))


def test_mixed_medium_both_forms(O, tabs):
    """config-3-like (x_HI uniform in [0.01, 1], tau per cell around the threshold): both forms along every ray;
    and the result differs from the all-differenced one (the thin form is really in use)."""
    cfg = synth.make(3, n=40, n_src=60)
    worst, rg, ro = run_both(O, cfg, tabs, 0.05, params=dict(tau_max=60.0))
    _, rg0, _ = run_both(O, cfg, tabs, 0.0, params=dict(tau_max=60.0))
    lit = rg0[0] > 0
    rel = np.abs(rg[0][lit] - rg0[0][lit]) / rg0[0][lit]
    assert 1e-9 < rel.max() and np.median(rel) < 1e-2
    for name in ("spawned", "split", "killed_tau", "exited"):
        assert list(getattr(rg[2], name)) == list(getattr(rg0[2], name))       # tau_0 steers, not the form (R37)
    print("thin table, mixed medium: worst relative Gamma error %.2e; thin vs differenced form: median %.1e" % (worst, np.median(rel)))


def test_f32_fields_and_shards(O, tabs):
    cfg = synth.make(5, n=40, n_src=300)
    assert cfg["nH"].dtype == torch.float32
    worst, rg, ro = run_both(O, cfg, tabs, 2.0 ** -8, params=dict(tau_max=60.0))
    # the same step in three source shards: photon grids added, then finalised
    p = dict(cfg["params"])
    p["tau_max"] = 60.0
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, field_dtype=cfg["nH"].dtype, max_sources=len(cfg["src_L"]))
    try:
        tr.set_spectrum(E_LO, E_HI, M, tabs[0])
        tr.set_spectrum_thin(tabs[1], 2.0 ** -8)
        tr.set_fields(cfg["nH"].cuda(), cfg["xHI"].cuda())
        tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
        total, seg = None, 0
        for r in range(3):
            tr.set_shard(r, 3)
            ph, st = tr.trace_photons()
            total = ph.clone() if total is None else total + ph
            seg += st.segments
        gam, heat, absorbed = tr.finalise(total)
    finally:
        tr.close()
    assert seg == ro[2].segments
    go = torch.from_numpy(ro[0]).cuda()
    assert bool(((gam - go).abs() <= 1e-9 * go + 1e-30).all())


def test_set_spectrum_drops_the_thin_table_and_errors():
    cfg = synth.make(1)
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=cfg["nH"].dtype, max_sources=1)
    try:
        n = nyxrt.nyxrt_spectrum_nodes(-4, 4, 3)
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.set_spectrum_thin(np.ones(n), 1e-3)                              # no Q table yet
        assert e.value.code == nyxrt.ESTATE
        tr.set_spectrum(-4, 4, 3, np.linspace(0.1, 0.9, n))
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.set_spectrum_thin(np.ones(n - 1), 1e-3)
        assert e.value.code == nyxrt.EINVAL
        with pytest.raises(nyxrt.NyxrtError):
            tr.set_spectrum_thin(-np.ones(n), 1e-3)
        tr.set_spectrum_thin(np.ones(n), 1e-3)
        tr.set_spectrum_thin()                                                  # off again
        tr.set_spectrum()                                                       # monochromatic
    finally:
        tr.close()


def test_a_rejected_set_spectrum_leaves_both_tables_in_place(tabs):
    """A failed nyxrt_set_spectrum / nyxrt_set_spectrum_thin (bad length, non-monotone Q, negative T) must change
    nothing: the next trace still uses the Q table AND the thin table set before.  The thin table here is half the
    true one, so that a silently dropped table would move Gamma by tens of per cent, far beyond the run-to-run
    difference of the deposits' summation order."""
    cfg = synth.make(4, n=32, n_src=60)
    p = dict(cfg["params"], tau_max=60.0)
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, field_dtype=cfg["nH"].dtype, max_sources=60)
    try:
        tr.set_fields(cfg["nH"].cuda().contiguous(), cfg["xHI"].cuda().contiguous())
        tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
        tr.set_spectrum(E_LO, E_HI, M, tabs[0])
        g_one = tr.trace()[0].clone()                                           # Q table alone
        tr.set_spectrum_thin(0.5 * tabs[1], 2.0 ** -4)
        g_two = tr.trace()[0].clone()                                           # with the (halved) thin table
        assert float(((g_two - g_one).abs() > 0.1 * g_one).double().mean()) > 0.1
        bad_q = tabs[0].copy()
        bad_q[5] = bad_q[4] - 1e-3
        for call in (lambda: tr.set_spectrum(E_LO, E_HI, M, tabs[0][:-1]),      # wrong length
                     lambda: tr.set_spectrum(E_LO, E_HI + 1, M, tabs[0]),       # geometry does not match the length
                     lambda: tr.set_spectrum(E_LO, E_HI, M, bad_q),             # not monotone
                     lambda: tr.set_spectrum_thin(tabs[1][:-1], 2.0 ** -4),
                     lambda: tr.set_spectrum_thin(-tabs[1], 2.0 ** -4),
                     lambda: tr.set_spectrum_thin(tabs[1], -1.0)):
            with pytest.raises(nyxrt.NyxrtError) as e:
                call()
            assert e.value.code == nyxrt.EINVAL
            g = tr.trace()[0]
            assert bool(((g - g_two).abs() <= 1e-9 * g_two + 1e-30).all())
        tr.set_spectrum(E_LO, E_HI, M, tabs[0])                                 # a successful one does drop the thin table
        g = tr.trace()[0]
        assert bool(((g - g_one).abs() <= 1e-9 * g_one + 1e-30).all())
    finally:
        tr.close()


def test_timestep_with_both_tables(O, tabs):
    """The RT timestep on top of the two-table flux: the paper's full update, Stroemgren test A."""
    MYR = 3.1557e13
    cfg = synth.make(1)
    nH, y0 = cfg["nH"], cfg["xHI"].double()
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    p = dict(cfg["params"])
    p["tau_max"] = 200.0
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, max_sources=1)
    try:
        tr.set_spectrum(E_LO, E_HI, M, tabs[0])
        tr.set_spectrum_thin(tabs[1], 2.0 ** -6)
        tr.set_sources(pos, L)
        xe, xa, gam, heat, st, ts = tr.timestep(nyxrt.make_ode(1.0 * MYR), nH.cuda(), y0.cuda())
        xe, gam = xe.cpu().numpy(), gam.cpu().numpy()
    finally:
        tr.close()
    g = O.make_grid(cfg["shape"], cfg["dx_cm"])
    try:
        O.set_spectrum(E_LO, E_HI, M, tabs[0])
        O.set_spectrum_thin(tabs[1], 2.0 ** -6)
        oe, oa, ogam, oheat, ost, ots, cat = O.timestep(g, O.make_params(**p), O.make_ode(1.0 * MYR), nH.numpy(),
                                                        y0.numpy(), pos, L)
    finally:
        O.set_spectrum()
    assert ts.iterations == ots.iterations and ts.converged == ots.converged and ts.iterations >= 2
    assert st.segments == ost.segments and list(st.killed_tau) == list(ost.killed_tau)
    assert np.all(np.abs(gam - ogam) <= 1e-9 * np.abs(ogam) + 1e-30)
    assert np.all(np.abs(xe - oe) <= 1e-9 * np.abs(oe) + 1e-15)
