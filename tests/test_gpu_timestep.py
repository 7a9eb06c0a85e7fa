"""GPU parity tests of the RT timestep (monochromatic): the CUDA
library's nyxrt_timestep against the oracle's orc_timestep (pinned in tests/test_oracle_timestep.py) on the
same seeded inputs.  Bar: the number of RT<->ODE iterations, the convergence flag, the unconverged-cell
count and every ray counter of the last trace exactly equal; x_HI at the end of the step, its time average
and the last Gamma within 1e-9 relative (floors: 1e-15 on fractions, 1e-30 s^-1 on Gamma) -- the update is
a handful of fp64 operations on a Gamma that itself agrees to 1e-13."""
import math

import numpy as np
import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import COUNTERS, RTOL

pytestmark = pytest.mark.gpu

KPC, MYR = 3.0857e21, 3.1557e13
ODE_KEYS = ("alpha_cm3_s", "coll_cm3_s", "clumping", "tol_rel", "tol_abs", "unconv_frac", "max_iter", "inner_iter")


def run_both(O, cfg, dt, ode_kw=None, periodic=0, batch_rays=0):
    from paper_2512_12466_b200 import nyxrt
    ode_kw = ode_kw or {}
    nH = cfg["nH"]
    y0 = cfg["xHI"].double()
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=nH.dtype, max_sources=len(L),
                      batch_rays=batch_rays, periodic=periodic)
    try:
        tr.set_sources(pos, L)
        xe, xa, gam, heat, st, ts = tr.timestep(nyxrt.make_ode(dt, **ode_kw), nH.cuda().contiguous(), y0.cuda().contiguous())
        torch.cuda.synchronize()
        res_g = (xe.cpu().numpy(), xa.cpu().numpy(), gam.cpu().numpy(), heat.cpu().numpy(), st, ts)
    finally:
        tr.close()
    g = O.make_grid(cfg["shape"], cfg["dx_cm"], field_dtype=nH.numpy().dtype, periodic=periodic)
    oe, oa, ogam, oheat, ost, ots, cat = O.timestep(g, O.make_params(**cfg["params"]), O.make_ode(dt, **ode_kw),
                                                    nH.numpy(), y0.numpy(), pos, L)
    return res_g, (oe, oa, ogam, oheat, ost, ots)


def compare(res_g, res_o, f32=False):
    xe, xa, gam, heat, st, ts = res_g
    oe, oa, ogam, oheat, ost, ots = res_o
    assert ts.iterations == ots.iterations and ts.converged == ots.converged, (ts.iterations, ots.iterations)
    assert ts.unconverged_cells == ots.unconverged_cells and ts.segments_total == ots.segments_total
    for name in COUNTERS:
        assert list(getattr(st, name)) == list(getattr(ost, name)), name
    assert st.segments == ost.segments
    assert np.all(np.abs(gam - ogam) <= RTOL * np.abs(ogam) + 1e-30) and np.array_equal(gam == 0, ogam == 0)
    assert np.all(np.abs(heat - oheat) <= RTOL * np.abs(oheat) + 1e-45)
    assert np.all(np.abs(xe - oe) <= RTOL * np.abs(oe) + 1e-15)
    if f32:
        # <x_HI> is stored in f32: both sides round the same fp64 value unless it sits on a rounding boundary
        assert xa.dtype == np.float32 and np.all(np.abs(xa.astype(np.float64) - oa) <= 1.2e-7 * np.abs(oa) + 1e-30)
    else:
        assert np.all(np.abs(xa - oa) <= RTOL * np.abs(oa) + 1e-15)
    assert abs(ts.max_rel_change - ots.max_rel_change) <= 1e-6 * ots.max_rel_change + 1e-12


def test_stromgren_test_a(O):
    """Sec. 3.1 Test A on the device: three 1 Myr timesteps from a neutral box;
    parity with the oracle at every step and the I-front radius of Eq. 11 to 1 %."""
    from paper_2512_12466_b200 import nyxrt
    cfg = synth.make(1)
    n = cfg["shape"][0]
    dx, nH0, Nd, aB = cfg["dx_cm"], 1e-3, 5e48, 2.59e-13
    rs = (3 * Nd / (4 * math.pi * aB * nH0 ** 2)) ** (1 / 3)
    trec = 1.0 / (aB * nH0)
    y = cfg["xHI"].double()
    t = 0.0
    for k in range(3):
        c = dict(cfg)
        c["xHI"] = y
        rg, ro = run_both(O, c, 1.0 * MYR)
        compare(rg, ro)
        assert rg[5].iterations >= 2
        y = torch.from_numpy(rg[0])
        t += 1.0 * MYR
        vol = float((1.0 - y).sum()) * dx ** 3
        rn = (3 * vol / (4 * math.pi)) ** (1 / 3)
        ra = rs * (1 - math.exp(-t / trec)) ** (1 / 3)
        assert abs(rn / ra - 1.0) < 0.01, (k, rn / ra)


def test_many_sources_with_merging_and_collisions(O):
    cfg = synth.make(4, n=40, n_src=300)
    rg, ro = run_both(O, cfg, 200.0 * MYR, dict(coll_cm3_s=3e-14, clumping=2.5, max_iter=8), batch_rays=8192)
    compare(rg, ro)
    assert np.abs(rg[0] - cfg["xHI"].numpy()).max() > 0.05     # the step does something
    assert rg[4].n_src_merged == ro[4].n_src_merged and rg[5].iterations >= 2


def test_f32_fields(O):
    cfg = synth.make(5, n=40, n_src=200)
    rg, ro = run_both(O, cfg, 300.0 * MYR, dict(max_iter=6), batch_rays=8192)
    compare(rg, ro, f32=True)
    assert np.abs(rg[0] - cfg["xHI"].double().numpy()).max() > 0.05


def test_periodic_box(O):
    cfg = synth.make(3, n=32, n_src=6)
    cfg["xHI"] = cfg["xHI"] * 0.05
    rg, ro = run_both(O, cfg, 100.0 * MYR, dict(max_iter=5), periodic=1)
    compare(rg, ro)


def test_single_iteration_and_no_sources(O):
    cfg = synth.make(3, n=24, n_src=5)
    rg, ro = run_both(O, cfg, 100.0 * MYR, dict(max_iter=1))
    compare(rg, ro)
    assert rg[5].iterations == 1 and rg[5].converged == 0 and rg[5].unconverged_cells > 0
    cfg["src_pos"] = torch.zeros((0, 3), dtype=torch.float64)
    cfg["src_L"] = torch.zeros(0, dtype=torch.float64)
    rg, ro = run_both(O, cfg, 100.0 * MYR, dict(max_iter=3))
    compare(rg, ro)
    assert np.all(rg[2] == 0.0)                                  # no photons: recombination only
    assert np.all(rg[0] >= cfg["xHI"].numpy() - 1e-15)


def test_bad_arguments():
    from paper_2512_12466_b200 import nyxrt
    tr = nyxrt.Tracer((8, 8, 8), 1e20, synth.default_params(), max_sources=1)
    f = torch.full((8, 8, 8), 1e-3, dtype=torch.float64, device="cuda")
    with pytest.raises(nyxrt.NyxrtError) as e:
        tr.timestep(nyxrt.make_ode(1e12), f, f)
    assert e.value.code == nyxrt.ESTATE                          # no sources yet
    tr.set_sources(np.array([[4.5, 4.5, 4.5]]), np.array([1e48]))
    for kw in (dict(max_iter=0), dict(inner_iter=0), dict(alpha_cm3_s=-1.0), dict(tol_rel=float("nan"))):
        with pytest.raises(nyxrt.NyxrtError) as e:
            tr.timestep(nyxrt.make_ode(1e12, **kw), f, f)
        assert e.value.code == nyxrt.EINVAL
    with pytest.raises(nyxrt.NyxrtError):
        tr.timestep(nyxrt.make_ode(0.0), f, f)
    tr.close()


def test_correction_modes_stromgren_fig8c(O):
    """What the correction-mode switch is for (without the secondary correction the photons a
    ray cannot give to its own cell are lost, and "squaring f_c can increase photon loss"; Fig. 8c): Stroemgren Test A
    (Eq. 10-11) through nyxrt_timestep for every geom_mode, ten 1 Myr steps from a
    neutral box, the ionised volume's radius r_I(t) against Eq. 11 at every step.  GPU against the oracle by the
    parity rule at every step of every mode; then the shape: modes 0 (no correction), 2 (Eq. 5-6) and 3 (Eq. 7-8;
    the same as 2 here, the n_th rule is inactive in a uniform box) conserve photons and follow Eq. 11 to 2 %;
    mode 1 (Eq. 5 alone) loses about a tenth of the photons and lags; mode 4 (f_c squared, [59]) loses about twice
    as many and lags further.  The table in BASELINE.md section 4 is this test's output."""
    cfg = synth.make(1)
    dx, nH0, Nd, aB = cfg["dx_cm"], 1e-3, 5e48, 2.59e-13
    rs = (3 * Nd / (4 * math.pi * aB * nH0 ** 2)) ** (1 / 3)
    trec = 1.0 / (aB * nH0)
    ratio, lost = {}, {}
    for mode in (0, 1, 2, 3, 4):
        c = dict(cfg)
        c["params"] = dict(cfg["params"], geom_mode=mode)
        y, t, ratio[mode], lost[mode] = cfg["xHI"].double(), 0.0, [], []
        for k in range(10):
            c["xHI"] = y
            rg, ro = run_both(O, c, 1.0 * MYR)
            compare(rg, ro)
            assert abs(rg[4].photons_lost - ro[4].photons_lost) <= 1e-11 * ro[4].photons_emitted
            y = torch.from_numpy(rg[0])
            t += 1.0 * MYR
            rn = (3 * float((1.0 - y).sum()) * dx ** 3 / (4 * math.pi)) ** (1 / 3)
            ratio[mode].append(rn / (rs * (1 - math.exp(-t / trec)) ** (1 / 3)))
            lost[mode].append(rg[4].photons_lost / rg[4].photons_emitted)
        print("geom_mode %d: r_I / Eq. 11 at 1..10 Myr = %s; photons lost in the last trace %.4f"
              % (mode, " ".join("%.4f" % v for v in ratio[mode]), lost[mode][-1]))
    for mode in (0, 2, 3):
        assert all(abs(v - 1.0) < 0.02 for v in ratio[mode]) and max(lost[mode]) == 0.0, mode
    assert all(abs(a - b) <= 1e-9 for a, b in zip(ratio[2], ratio[3]))
    for k in range(10):
        assert ratio[4][k] < ratio[1][k] < ratio[2][k] - 0.03, k
        assert lost[4][k] > lost[1][k] > 0.02, k
    assert 0.93 < ratio[1][-1] < 0.97 and 0.88 < ratio[4][-1] < 0.93 and lost[4][-1] > 1.5 * lost[1][-1] > 0.05
