"""Pins for the oracle's frequency-integrated flux (Sec. 2.2: Eq. 1 "precomputed as a function
of tau_0 ... a lookup table"): the table lookup against its own definition (nodes,
piecewise linearity, limits), the black-body table against scipy's quadrature of Eq. 1's frequency integral,
the traced result against the monochromatic oracle (a table of 1 - e^-tau must reproduce it), photon
conservation, and spectral hardening behind an absorber."""
import math

import numpy as np
import pytest
from scipy.integrate import quad

E_LO, E_HI, M = -20, 12, 5


@pytest.fixture()
def mono_after(O):
    yield
    O.set_spectrum()                                   # the table is module state of the oracle: always reset


def planck(x):
    """x^2 / (e^x - 1) without overflow"""
    return x * x * math.exp(-x) / -math.expm1(-x)


def nodes(O, e_lo, e_hi, m):
    n = O.spectrum_nodes(e_lo, e_hi, m)
    return np.array([O.spectrum_node_tau(e_lo, m, k) for k in range(n)])


def test_nodes_are_the_binary_buckets(O):
    t = nodes(O, -3, 2, 2)
    assert len(t) == 5 * 4 + 1 and t[0] == 0.125 and t[-1] == 4.0
    assert list(t[:5]) == [0.125, 0.125 * 1.25, 0.125 * 1.5, 0.125 * 1.75, 0.25]
    assert np.all(np.diff(t) > 0)


def test_lookup_is_the_piecewise_linear_interpolant(O, mono_after):
    rng = np.random.default_rng(0)
    t = nodes(O, -6, 4, 3)
    q = np.sort(rng.uniform(0, 1, len(t)))
    O.set_spectrum(-6, 4, 3, q)
    for k in range(len(t)):
        assert O.spectrum_q(t[k]) == q[k]                                   # exact at the nodes
    for k in rng.integers(0, len(t) - 1, 200):
        f = rng.uniform()
        tau = t[k] + f * (t[k + 1] - t[k])
        ref = q[k] + (tau - t[k]) / (t[k + 1] - t[k]) * (q[k + 1] - q[k])
        assert abs(O.spectrum_q(tau) - ref) < 1e-14
    assert O.spectrum_q(0.0) == 0.0 and O.spectrum_q(-1.0) == 0.0
    assert O.spectrum_q(t[0] / 4) == q[0] / 4                               # linear from the origin below the table
    assert O.spectrum_q(1e9) == q[-1] and O.spectrum_q(t[-1]) == q[-1]      # constant above it
    xs = np.concatenate([np.linspace(t[0] / 8, t[-1] * 1.1, 4001), [np.nextafter(v, 0) for v in t[1:]]])
    xs.sort()
    ys = np.array([O.spectrum_q(v) for v in xs])
    assert np.all(np.diff(ys) >= -1e-15)                                    # monotone, continuous at octave ends
    O.set_spectrum()
    with pytest.raises(RuntimeError):
        O.set_spectrum(-6, 4, 3, q[:-1])                                    # wrong length


def test_blackbody_table_against_quadrature(O):
    """Q(tau_0) = int phi (1 - exp(-tau_0 (nu/nu_0)^-3)) dnu for phi ~ nu^2/(e^{h nu/kT} - 1), nu >= nu_0."""
    for T in (5e4, 1e5):
        x0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * T)
        q = O.blackbody_table(T, -4, 8, 1)
        t = nodes(O, -4, 8, 1)
        norm = quad(planck, x0, np.inf, epsabs=0, epsrel=1e-12)[0]
        for k in (0, 3, 8, 11, 16, 24):
            val = quad(lambda x: planck(x) * -math.expm1(-t[k] * (x0 / x) ** 3), x0, np.inf, epsabs=0,
                       epsrel=1e-12, limit=200)[0] / norm
            assert abs(q[k] - val) < 1e-8 * val, (T, k, q[k], val)
        slope = np.diff(q) / np.diff(t)
        assert np.all(np.diff(q) > 0) and np.all(np.diff(slope) < 0) and 0 < q[0] and q[-1] < 1   # increasing, concave
        # thin limit: Q -> tau <(nu/nu_0)^-3>; harder spectrum (higher T) = smaller mean cross-section
        mean_s = quad(lambda x: planck(x) * (x0 / x) ** 3, x0, np.inf, epsrel=1e-12)[0] / norm
        q_thin = O.blackbody_table(T, -30, -29, 0)[0]
        assert abs(q_thin / 2.0 ** -30 - mean_s) < 1e-6 * mean_s
    assert O.blackbody_table(1e5, -4, 8, 1)[8] < O.blackbody_table(5e4, -4, 8, 1)[8]


def small_case(O, n=20, thick=1.0):
    rng = np.random.default_rng(5)
    nH = 10 ** rng.uniform(-3.3, -2.7, (n, n, n))
    xHI = rng.uniform(0.05, 1.0, (n, n, n)) * thick
    g = O.make_grid((n, n, n), 7e20)
    p = O.make_params(n_th=1e-3, e_excess_erg=1e-11)
    cell = np.array([[10, 9, 11], [3, 15, 4]], np.int32)
    return g, p, nH, xHI, cell, np.array([3e49, 1e49])


def test_table_of_the_exponential_reproduces_the_monochromatic_trace(O, mono_after):
    """Q = 1 - e^-tau tabulated: identical ray counters (tau does not depend on the table), the same photon
    budget, and Gamma equal up to the interpolation error, which falls 4x per extra table bit."""
    g, p, nH, xHI, cell, L = small_case(O)
    gam0, heat0, st0 = O.trace(g, p, nH, xHI, cell, L)
    errs = []
    for m in (4, 6, 8):
        t = nodes(O, -30, 6, m)
        O.set_spectrum(-30, 6, m, -np.expm1(-t))
        gam, heat, st = O.trace(g, p, nH, xHI, cell, L)
        for name in ("spawned", "split", "killed_tau", "exited", "killed_lmax"):
            assert list(getattr(st, name)) == list(getattr(st0, name))
        assert st.segments == st0.segments
        tot = st.photons_absorbed + st.photons_escaped + st.photons_residual
        assert abs(tot - st.photons_emitted) < 1e-12 * st.photons_emitted
        assert abs(st.photons_absorbed - st0.photons_absorbed) < 1e-3 * 4.0 ** (4 - m) * st0.photons_absorbed + 1e-9 * st0.photons_absorbed
        lit = gam0 > 0
        assert np.array_equal(gam > 0, lit)
        errs.append(float(np.median(np.abs(gam[lit] - gam0[lit]) / gam0[lit])))
    assert errs[2] < errs[1] / 8 < errs[0] / 64 and errs[2] < 2e-4, errs          # second order in the node spacing


def test_photons_telescope_along_a_lineage(O, mono_after):
    """Sum of the photons a lineage deposits = its share times Q(tau at its end): Eq. 1 integrated along the ray."""
    g, p, nH, xHI, cell, L = small_case(O, thick=0.05)
    O.set_spectrum(E_LO, E_HI, M, O.blackbody_table(1e5, E_LO, E_HI, M))
    gam, heat, st, log = O.trace(g, p, nH, xHI, cell[:1], L[:1], log_cap=2_000_000)
    tot = st.photons_absorbed + st.photons_escaped + st.photons_residual
    assert abs(tot - st.photons_emitted) < 1e-12 * st.photons_emitted
    assert st.photons_escaped > 0.05 * st.photons_emitted                  # hard photons leave the box
    # level-0 rays that never split (none here splits before leaving a 20^3 box? take any leaf lineage):
    # walk each (level, pix) path back to its level-0 ancestor and add dN / share over the path
    by = {}
    for r in log:
        by.setdefault((int(r["level"]), int(r["pix"])), []).append(r)
    leaves = [k for k in by if (k[0] + 1, 4 * k[1]) not in by and (k[0] + 1, 4 * k[1] + 1) not in by]
    checked = 0
    for (lev, pix) in leaves[:300]:
        frac, tau_end, l, q = 0.0, 0.0, lev, pix
        while l >= 0:
            share = L[0] / (12.0 * 4.0 ** l)
            for r in by.get((l, q), []):
                frac += r["dN"] / share
                tau_end = max(tau_end, 0.0)
            l, q = l - 1, q // 4
        tau_end = sum(r["dtau"] for ll, qq in [(lev - j, pix >> (2 * j)) for j in range(lev + 1)] for r in by.get((ll, qq), []))
        assert abs(frac - O.spectrum_q(tau_end)) < 1e-12 + 1e-9 * frac
        checked += 1
    assert checked > 50


def test_spectral_hardening_behind_an_absorber(O, mono_after):
    """Behind an optical depth of ~10 at threshold the monochromatic flux is down by e^-10; a 1e5 K black body
    still delivers its hard photons (1 - Q(10) ~ 0.3), and the rate per H I atom reflects it."""
    n = 24
    nH = np.full((n, n, n), 1e-3)
    xHI = np.full((n, n, n), 1e-6)
    xHI[:, :, 8:10] = 0.4                                  # a slab across the box, two cells thick
    g = O.make_grid((n, n, n), 2e21)
    p = O.make_params()
    cell = np.array([[2, 12, 12]], np.int32)
    L = np.array([1e50])
    tau_slab = 2 * 1e-3 * 0.4 * 6.3e-18 * 2e21
    assert 9 < tau_slab < 11
    gam0, _, st0 = O.trace(g, p, nH, xHI, cell, L, want_heat=False)
    O.set_spectrum(E_LO, E_HI, M, O.blackbody_table(1e5, E_LO, E_HI, M))
    gam1, _, st1 = O.trace(g, p, nH, xHI, cell, L, want_heat=False)
    behind0, behind1 = gam0[12, 12, 14], gam1[12, 12, 14]
    assert behind0 > 0 and behind1 > 50 * behind0
    front0, front1 = gam0[12, 12, 5], gam1[12, 12, 5]
    assert 0.15 < front1 / front0 < 0.35                   # thin limit: <(nu/nu_0)^-3> of the black body ~ 0.24
