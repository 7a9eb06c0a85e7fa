"""Pins for the oracle's RT timestep (SURVEY.md 8(f) item 2 without the lookup table: time integration,
PAPER.md:97-103 Eq. 3, inside the iterative solve, "following [23]").  The per-cell update
is pinned to closed forms of Eq. 3 and to an independent numerical integration; the whole timestep to the
paper's own verification problem (Sec. 3.1: Eq. 10-11 with Table 1 Test A) and
to photon conservation in time (the property [23]'s time averaging exists for)."""
import math

import numpy as np
from scipy.integrate import solve_ivp

KPC, MYR = 3.0857e21, 3.1557e13


def test_photoionisation_only_closed_form(O):
    """alpha = C_H = 0: Eq. 3 is dy/dt = -Gamma y: y(dt) = y0 e^{-Gamma dt}, <y> = y0 (1 - e^{-Gamma dt})/(Gamma dt)."""
    for gam, dt, y0 in ((1e-12, 1e12, 1.0), (3e-14, 1e13, 0.4), (1e-10, 1e13, 1.0), (1e-20, 1e10, 0.7)):
        o = O.make_ode(dt, alpha_cm3_s=0.0, coll_cm3_s=0.0)
        ya, ye = O.ode_cell(o, gam, 1e-3, y0, y0)
        w = gam * dt
        assert abs(ye - y0 * math.exp(-w)) <= 1e-15 * y0
        assert abs(ya - y0 * (-math.expm1(-w)) / w) <= 4e-16 * y0


def test_nothing_acts_on_the_cell(O):
    """Gamma = 0 in a neutral cell (n_e = 0): nothing changes; dt -> 0: nothing changes."""
    o = O.make_ode(1e13)
    assert O.ode_cell(o, 0.0, 1e-3, 1.0, 1.0) == (1.0, 1.0)
    ya, ye = O.ode_cell(O.make_ode(1e-3), 1e-12, 1e-3, 0.25, 0.25)
    assert abs(ya - 0.25) < 1e-14 and abs(ye - 0.25) < 1e-14


def test_equilibrium_is_the_root_of_eq3(O):
    """dt >> t_i: x -> the root of (1 - x) Gamma = x^2 n_H alpha (Eq. 3 with C_H = 0, n_e = x n_H)."""
    gam, nH, aB = 2e-13, 1e-3, 2.59e-13
    o = O.make_ode(1e19, inner_iter=200)
    ya, ye = O.ode_cell(o, gam, nH, 1.0, 0.5)
    b = gam / (nH * aB)
    x_eq = (-b + math.sqrt(b * b + 4 * b)) / 2                       # x^2 + b x - b = 0
    assert abs((1 - ye) - x_eq) < 1e-9 and abs((1 - ya) - x_eq) < 1e-6
    # with collisional ionisation: (1 - x)(Gamma + x nH C) = x^2 nH alpha
    o = O.make_ode(1e19, inner_iter=400, coll_cm3_s=1e-13)
    ya, ye = O.ode_cell(o, gam, nH, 1.0, 0.5)
    x = 1 - ye
    assert abs((1 - x) * (gam + x * nH * 1e-13) - x * x * nH * aB) < 1e-5 * x * x * nH * aB      # <y> keeps (y0 - y_eq) t_i/dt of the transient


def test_against_numerical_integration_of_eq3(O):
    """Eq. 3 integrated numerically (n_e = x n_H varying in time) against the time-averaged
    semi-analytic update: equal up to the scheme's own error, which vanishes with dt (first order in the
    variation of n_e over the step); the clumping factor scales alpha (Eq. 10)."""
    nH, aB, CH, gam = 1e-3, 2.59e-13, 3e-14, 5e-16
    trec = 1.0 / (aB * nH)

    def rhs(t, x, C):
        ne = x[0] * nH
        return [(1 - x[0]) * (gam + ne * CH) - x[0] * ne * aB * C]

    errs = []
    for frac in (0.4, 0.1, 0.025):
        dt = frac * trec
        for C in (1.0, 3.0):
            sol = solve_ivp(rhs, (0, dt), [0.3], args=(C,), rtol=1e-11, atol=1e-14, dense_output=True)
            x_end = sol.y[0, -1]
            tt = np.linspace(0, dt, 4001)
            x_avg = np.trapezoid(sol.sol(tt)[0], tt) / dt
            o = O.make_ode(dt, coll_cm3_s=CH, clumping=C, inner_iter=50)
            ya, ye = O.ode_cell(o, gam, nH, 0.7, 0.7)
            errs.append((abs((1 - ye) - x_end), abs((1 - ya) - x_avg)))
    assert max(max(e) for e in errs) < 1e-2 and max(errs[-1]) < 1e-4
    for k in (0, 1):                                                 # both clumping factors, x_end and <x>
        for q in (0, 1):
            assert errs[4 + k][q] < errs[2 + k][q] / 3 < errs[k][q] / 9      # at least first order in dt


def test_time_average_is_the_mean_of_the_solution(O):
    """<y> = (1/dt) int y(t) dt of the update's own exponential solution (quadrature written out here)."""
    gam, nH, aB, dt, y0 = 4e-14, 2e-3, 2.59e-13, 2e13, 0.9
    o = O.make_ode(dt, inner_iter=60)
    ya, ye = O.ode_cell(o, gam, nH, y0, y0)
    ne = (1 - ya) * nH                                               # converged electron density
    rate = gam + ne * aB
    yeq = ne * aB / rate
    tt = np.linspace(0, dt, 200001)
    yt = yeq + (y0 - yeq) * np.exp(-rate * tt)
    assert abs(np.trapezoid(yt, tt) / dt - ya) < 1e-9 and abs(yt[-1] - ye) < 1e-9


def stromgren(O, n, dt, t_end, **ode):
    dx = 6.6 * KPC / n
    nH0, Nd, aB = 1e-3, 5e48, 2.59e-13
    rs = (3 * Nd / (4 * math.pi * aB * nH0 ** 2)) ** (1 / 3)
    trec = 1.0 / (aB * nH0)
    g = O.make_grid((n, n, n), dx)
    p = O.make_params()
    nH = np.full((n, n, n), nH0)
    y = np.ones((n, n, n))
    pos = np.array([[n / 2 + 0.5] * 3])
    t, out = 0.0, []
    while t < t_end - 1e-6 * dt:
        y0 = y
        y, ya, gam, _, st, ts, cat = O.timestep(g, p, O.make_ode(dt, **ode), nH, y0, pos, np.array([Nd]),
                                                 want_heat=False)
        t += dt
        vol = float(np.sum(1.0 - y)) * dx ** 3
        out.append(dict(t=t, rn=(3 * vol / (4 * math.pi)) ** (1 / 3), ra=rs * (1 - math.exp(-t / trec)) ** (1 / 3),
                        y0=y0, y=y, ya=ya, gam=gam, st=st, ts=ts, nH=nH, dx=dx))
    return out


def test_stromgren_front_with_large_timesteps(O):
    """Sec. 3.1, Test A of Table 1: r_I(t) = r_s [1 - e^{-t/t_rec}]^{1/3} with
    timesteps of 1 Myr (50 times the explicit step of tests/test_oracle_physics.py): the time-averaged
    scheme conserves photons, so the ionised volume follows Eq. 11 to better than 1 %."""
    out = stromgren(O, 32, 1.0 * MYR, 6.0 * MYR)
    for r in out:
        assert abs(r["rn"] / r["ra"] - 1.0) < 0.01, (r["t"] / MYR, r["rn"] / r["ra"])
        assert r["ts"].iterations >= 2
    assert sum(r["ts"].converged for r in out) >= len(out) - 1


def test_photon_conservation_in_time(O):
    """From Eq. 3 with constant coefficients: x_end - x_0 = dt [a_ion <y> - a_rec <x>] in every cell, so
    sum_c n_H V (x_end - x_0) = dt [absorbed photons/s of the last ray trace] - dt sum_c n_H V a_rec <x>
    when the solve has converged (the trace saw <y>).  Ties the ODE to the ray tracer's budget."""
    out = stromgren(O, 24, 0.5 * MYR, 1.0 * MYR, tol_rel=1e-6, tol_abs=1e-12, max_iter=80, unconv_frac=0.0)
    aB = 2.59e-13
    for r in out:
        V = r["dx"] ** 3
        dt = 0.5 * MYR
        lhs = float(np.sum(r["nH"] * V * (r["y0"] - r["y"])))       # new ionisations (x = 1 - y)
        x_avg = 1.0 - r["ya"]
        rec = float(np.sum(r["nH"] * V * (x_avg * r["nH"] * aB) * x_avg)) * dt
        absorbed = r["st"].photons_absorbed * dt
        assert r["ts"].converged == 1
        assert abs(lhs + rec - absorbed) < 2e-5 * absorbed, (lhs, rec, absorbed)
        # cell by cell with the last trace's Gamma (exact identity of the update, to rounding)
        cell = r["nH"] * ((r["gam"] * r["ya"]) - (x_avg * r["nH"] * aB) * x_avg) * dt
        assert np.allclose(r["nH"] * (r["y0"] - r["y"]), cell, rtol=1e-6, atol=1e-12 * 1e-3)


def test_first_trace_uses_the_field_at_the_start_and_f32_rounding(O):
    """R36 and the field dtype: with max_iter = 1 the timestep is one ray trace on x_HI(t0) followed by one
    update; with f32 fields <y> is rounded to f32 before it is traced."""
    n = 12
    rng = np.random.default_rng(3)
    nH = 10 ** rng.uniform(-3.5, -2.5, (n, n, n))
    y0 = rng.uniform(0.2, 1.0, (n, n, n))
    pos, L = np.array([[6.5, 6.5, 6.5]]), np.array([1e49])
    p = O.make_params()
    g = O.make_grid((n, n, n), 6e20)
    o = O.make_ode(3e12, max_iter=1)
    ye, ya, gam, heat, st, ts, cat = O.timestep(g, p, o, nH, y0, pos, L)
    gam1, heat1, st1, _ = O.step(g, p, nH, y0, pos, L)
    assert np.array_equal(gam, gam1) and ts.iterations == 1
    for c in ((6, 6, 6), (5, 7, 6), (0, 0, 0)):
        a, e = O.ode_cell(o, gam1[c], nH[c], y0[c], y0[c])
        assert ya[c] == a and ye[c] == e
    g32 = O.make_grid((n, n, n), 6e20, field_dtype=np.float32)
    ye2, ya2, *_ = O.timestep(g32, p, O.make_ode(3e12, max_iter=3), nH.astype(np.float32), y0, pos, L)
    assert ya2.dtype == np.float32 and ye2.dtype == np.float64
    ye3, ya3, *_ = O.timestep(g, p, O.make_ode(3e12, max_iter=3), nH, y0, pos, L)
    assert np.all(ye2 <= 1.0) and np.all(ye2 >= 0.0)
    assert np.allclose(ye2, ye3, rtol=1e-5, atol=1e-7) and not np.array_equal(ye2, ye3)
    assert np.array_equal(ya2, ya2.astype(np.float32))
