"""Pins for the oracle's separate table for the optically thin case (PAPER.md:267 footnote 3, "takes the limit as
n_H -> 0 to compute a separate LUT for the optically thin case", with the tau_0 table of; readings
R40-R42): T = dQ/dtau_0 against scipy's quadrature of the frequency integral; the thin form dtau T(tau + dtau/2)
against the quadrature of Eq. 1's numerator for one segment, next to the difference of two interpolants it
replaces; continuity at the switch; photon conservation with the counted-down ray; and the thin-limit rate
Gamma = sigma_0 T(tau) Ndot / (4 pi R^2)."""
import math

import numpy as np
import pytest
from scipy.integrate import quad

E_LO, E_HI, M = -20, 12, 8
T_EFF = 1e5
X0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * T_EFF)


@pytest.fixture()
def mono_after(O):
    yield
    O.set_spectrum()                                   # the tables are module state of the oracle: always reset


def planck(x):
    return x * x * math.exp(-x) / -math.expm1(-x)


NORM = quad(planck, X0, np.inf, epsabs=0, epsrel=1e-13)[0]


def t_ref(tau):
    """int phi (nu/nu_0)^-3 exp(-tau (nu/nu_0)^-3) dnu for the black body, by quadrature"""
    return quad(lambda x: planck(x) * (X0 / x) ** 3 * math.exp(-tau * (X0 / x) ** 3), X0, np.inf, epsabs=0,
                epsrel=1e-12)[0] / NORM


def dq_ref(tau, dtau):
    """Eq. 1's numerator for one segment: int phi exp(-tau_nu) (1 - exp(-dtau_nu)) dnu, no cancellation (expm1)"""
    return quad(lambda x: planck(x) * math.exp(-tau * (X0 / x) ** 3) * -math.expm1(-dtau * (X0 / x) ** 3), X0, np.inf,
                epsabs=0, epsrel=1e-12)[0] / NORM


@pytest.fixture(scope="module")
def tables(O):
    return O.blackbody_table(T_EFF, E_LO, E_HI, M), O.blackbody_thin_table(T_EFF, E_LO, E_HI, M)


def test_thin_table_is_dq_dtau_by_quadrature(O, tables, mono_after):
    q, t = tables
    assert len(t) == len(q) == O.spectrum_nodes(E_LO, E_HI, M)
    assert np.all(np.diff(t) <= 0) and t[0] > 0 and t[-1] >= 0              # T falls with tau_0 (hardening)
    O.set_spectrum(E_LO, E_HI, M, q)
    O.set_spectrum_thin(t, 1e-3)
    for k in (0, 1000, len(t) // 2, len(t) // 2 + 777, len(t) - 1500):
        tau = O.spectrum_node_tau(E_LO, M, k)
        assert O.spectrum_t(tau) == t[k]                                    # exact at the nodes
        assert abs(t[k] - t_ref(tau)) <= 1e-7 * t_ref(tau)
    for tau in (3e-7, 1e-3, 0.3, 1.0, 7.0, 40.0):                           # between nodes: linear interpolation
        assert abs(O.spectrum_t(tau) - t_ref(tau)) <= 1e-6 * t_ref(tau)
    assert O.spectrum_t(0.0) == t[0] and O.spectrum_t(2.0 ** (E_LO - 3)) == t[0]     # constant below the table
    assert O.spectrum_t(2.0 ** E_HI) == t[-1] and O.spectrum_t(1e9) == t[-1]         # and above it
    # T is the derivative of Q: centred differences of the Q NODES (no interpolation involved)
    for k in (5000, 6000, 7000):
        a, b = O.spectrum_node_tau(E_LO, M, k - 1), O.spectrum_node_tau(E_LO, M, k + 1)
        assert abs((q[k + 1] - q[k - 1]) / (b - a) - t[k]) <= 1e-4 * t[k]
    O.set_spectrum_thin()
    with pytest.raises(RuntimeError):
        O.set_spectrum_thin(t[:-1], 1e-3)                                   # wrong length
    O.set_spectrum()
    with pytest.raises(RuntimeError):
        O.set_spectrum_thin(t, 1e-3)                                        # no Q table set


def test_thin_form_keeps_the_digits_the_difference_loses(O, tables, mono_after):
    """One segment [tau, tau + dtau]: the thin form stays within 1e-6 of the quadrature for every dtau below 1e-3,
    the difference of two interpolants is off by up to the table's secant error (~ tau / 2^(M+1)) whatever dtau is,
    and below the table (where Q is linear from the origin) by rounding that grows as dtau falls."""
    q, t = tables
    O.set_spectrum(E_LO, E_HI, M, q)
    O.set_spectrum_thin(t, 1.0)
    worst_thin, worst_diff = 0.0, 0.0
    for tau in (1e-3, 0.03, 0.3, 1.0, 7.0):
        for dtau in (1e-3, 1e-4, 1e-5, 1e-6, 1e-7, 1e-8):
            ref = dq_ref(tau, dtau)
            thin = dtau * O.spectrum_t(tau + 0.5 * dtau)
            diff = O.spectrum_q(tau + dtau) - O.spectrum_q(tau)
            assert abs(thin - ref) <= 1e-6 * ref, (tau, dtau)
            worst_thin = max(worst_thin, abs(thin - ref) / ref)
            worst_diff = max(worst_diff, abs(diff - ref) / ref)
            assert abs(diff - ref) <= 2.0 ** -(M + 1) * max(tau, 1.0) * ref      # the secant of a bucket, no worse
    assert worst_diff > 1e-4 > 100 * worst_thin
    # rounding of the difference: the same segment length at a larger tau_0 has fewer digits left
    e_small = abs((O.spectrum_q(1e-3 + 1e-8) - O.spectrum_q(1e-3)) - dq_ref(1e-3, 1e-8)) / dq_ref(1e-3, 1e-8)
    e_large = abs((O.spectrum_q(1e-3 + 1e-3) - O.spectrum_q(1e-3)) - dq_ref(1e-3, 1e-3)) / dq_ref(1e-3, 1e-3)
    assert e_small > 50 * e_large


def test_forms_agree_at_the_switch(O, tables, mono_after):
    """At dtau = tau_thin the two forms differ by the secant error of the Q table only."""
    q, t = tables
    O.set_spectrum(E_LO, E_HI, M, q)
    O.set_spectrum_thin(t, 2.0 ** -12)
    for tau in (1e-4, 0.01, 0.5, 3.0, 15.0):
        d = 2.0 ** -12
        thin = d * O.spectrum_t(tau + 0.5 * d)
        diff = O.spectrum_q(tau + d) - O.spectrum_q(tau)
        assert abs(thin - diff) <= 2.0 ** -M * max(tau, 1.0) * thin


def _trace(O, n, nH, xHI, src, L, dx, **pk):
    g = O.make_grid((n, n, n), dx)
    p = O.make_params(**pk)
    a = np.full((n, n, n), float(nH)) if np.isscalar(nH) else nH
    x = np.full((n, n, n), float(xHI)) if np.isscalar(xHI) else xHI
    gam, heat, st = O.trace(g, p, a, x, np.array([src], np.int32), np.array([L]))
    return g, a, x, gam, heat, st


def test_budget_and_grid_sum_with_the_thin_table(O, tables, mono_after):
    """Photon conservation survives the mixture of the two forms because the ray's photons
    are counted down (R42): emitted = absorbed + escaped + residual to 1e-12, sum_c Gamma n_HI V = absorbed, and
    both forms are in use."""
    q, t = tables
    rng = np.random.default_rng(5)
    n = 24
    a = 10 ** rng.uniform(-6, -2, (n, n, n))                                # thin and thick cells side by side
    x = rng.uniform(0.0, 1.0, (n, n, n))
    x[rng.uniform(size=x.shape) < 0.1] = 0.0
    for tau_thin in (0.0, 2.0 ** -10, 1e9):
        O.set_spectrum(E_LO, E_HI, M, q)
        O.set_spectrum_thin(t, tau_thin)
        g, a, x, gam, heat, st = _trace(O, n, a, x, (11, 12, 13), 3e50, 3e20, n_th=1e-5, e_excess_erg=2e-11, tau_max=60.0)
        em, ab, es, re = st.photons_emitted, st.photons_absorbed, st.photons_escaped, st.photons_residual
        assert abs(ab + es + re - em) <= 1e-12 * em and ab > 0.2 * em and es > 0
        V = g.dx_cm ** 3
        assert abs(float(np.sum(gam * a * x)) * V - ab) <= 1e-12 * ab
        if tau_thin == 0.0:
            ref = (gam.copy(), ab)
        elif tau_thin < 1.0:
            # per cell within the Q table's secant error (~ tau_0 / 2^(M+1) of a segment) of the all-differenced
            # result, but not identical: the thin form is in use
            lit = ref[0] > 0
            rel = np.abs(gam[lit] - ref[0][lit]) / ref[0][lit]
            assert np.median(rel) < 1e-3 and np.quantile(rel, 0.99) < 0.05 and rel.max() > 1e-9
            assert abs(ab - ref[1]) < 2e-3 * ab
        # tau_thin = 1e9 forces the thin form on thick cells too (wrong physics there, on purpose): the budget
        # must still close, because it rests on the count-down, not on either form
        O.set_spectrum()


def test_thin_limit_rate(O, tables, mono_after):
    """The limit the footnote names: in a transparent uniform medium every segment takes the thin form and the rate
    per atom is Gamma(R) = sigma_0 T(tau_0(R)) Ndot / (4 pi R^2) (Eq. 1 with dtau -> 0), shell-averaged within a
    few per cent for R > 4 cells -- the normalisation of T, sigma-weighted by the spectrum, not sigma_0 alone."""
    q, t = tables
    O.set_spectrum(E_LO, E_HI, M, q)
    O.set_spectrum_thin(t, 1e-2)
    n, nH, dx, L, sig = 33, 1e-7, 1e20, 1e50, 6.3e-18
    g, a, x, gam, heat, st = _trace(O, n, nH, 1.0, (16, 16, 16), L, dx, tau_max=60.0)
    k = nH * sig * dx                                                       # tau_0 per cell: 6.3e-5, far below tau_thin
    zz, yy, xx = np.meshgrid(*(np.arange(n) - 16.0,) * 3, indexing="ij")
    r = np.sqrt(xx ** 2 + yy ** 2 + zz ** 2)
    assert t[0] < 0.5                                                       # sigma-weighted mean of (nu/nu_0)^-3 < 1
    for lo, hi in ((4, 6), (8, 10), (12, 14)):
        m = (r >= lo) & (r < hi)
        expect = np.mean(sig * O.spectrum_t(k * 0.5 * (lo + hi)) * L / (4 * math.pi * (r[m] * dx) ** 2))
        assert abs(gam[m].mean() - expect) < 0.05 * expect


def test_a_rejected_call_leaves_the_oracles_tables_in_place(O, tables, mono_after):
    """Host logic, no arithmetic: orc_set_spectrum / orc_set_spectrum_thin check their arguments before they touch
    the tables (the C ABI's rule, include/nyxrt.h), so a failed call changes neither lookup."""
    q, t = tables
    O.set_spectrum(E_LO, E_HI, M, q)
    O.set_spectrum_thin(t, 2.0 ** -8)
    q_at, t_at = O.spectrum_q(0.37), O.spectrum_t(0.37)
    for call in (lambda: O.set_spectrum(E_LO, E_HI, M, q[:-1]), lambda: O.set_spectrum(E_LO, E_HI + 1, M, q),
                 lambda: O.set_spectrum_thin(t[:-1], 2.0 ** -8), lambda: O.set_spectrum_thin(t, -1.0)):
        with pytest.raises(Exception):
            call()
        assert O.spectrum_q(0.37) == q_at and O.spectrum_t(0.37) == t_at
