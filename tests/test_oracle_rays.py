"""Pins for the oracle's ray loop (O3-O7): DDA geometry against the slab method and fine sampling,
tau against Eq. 2's closed form, the photon budget, Eq. 4 split radii, the tau_max kill, and the
Eq. 5-8 deposit shares recomputed by brute force from the segment log.  PAPER.md line numbers in each
docstring.  The checks use the oracle's optional per-segment log; every expected value is computed here
from geometry, never from the oracle's own formulas."""
import math

import numpy as np
import pytest

KPC = 3.0856775814913673e21


def uniform_case(O, n, nH, xHI, src, L=1e50, dx=1e20, log_cap=2_000_000, fields=None, **pk):
    g = O.make_grid((n, n, n), dx)
    p = O.make_params(**pk)
    if fields is None:
        a = np.full((n, n, n), float(nH))
        x = np.full((n, n, n), float(xHI))
    else:
        a, x = fields
    cell = np.array([src], np.int32)
    gam, heat, st, log = O.trace(g, p, a, x, cell, np.array([L]), log_cap=log_cap)
    return g, p, a, x, gam, heat, st, log


def slab(org, d, lo, hi):
    """Entry/exit parameters of the line org + t d through the box [lo,hi] (textbook slab method)."""
    t0, t1 = -math.inf, math.inf
    for a in range(3):
        if d[a] == 0.0:
            if not (lo[a] <= org[a] <= hi[a]):
                return math.inf, -math.inf
            continue
        ta, tb = (lo[a] - org[a]) / d[a], (hi[a] - org[a]) / d[a]
        if ta > tb:
            ta, tb = tb, ta
        t0, t1 = max(t0, ta), min(t1, tb)
    return t0, t1


def rays_of(log):
    """Group the log by ray (level, pix) preserving order."""
    out = {}
    for r in log:
        out.setdefault((int(r["level"]), int(r["pix"])), []).append(r)
    return out


def test_segments_are_exact_cell_chords(O):
    """PAPER.md:152 'advancing the ray one cell at a time using a fast voxel traversal technique [76]':
    every logged segment is the chord of the radial line src + s d through its cell, consecutive segments
    of a ray abut, and an exiting leaf ends at the slab-method exit distance from the box."""
    n, src = 9, (3, 4, 5)
    g, p, a, x, gam, heat, st, log = uniform_case(O, n, 1e-8, 1.0, src, dx=1e18)     # thin: nothing is killed
    org = np.array(src, float) + 0.5
    assert st.segments == len(log) > 3000
    byray = rays_of(log)
    n_leaf = 0
    for (lev, pix), segs in byray.items():
        d = O.pix2dir(lev, pix)
        prev_end = None
        for r in segs:
            lo = np.array(r["cell"], float)
            t0, t1 = slab(org, d, lo, lo + 1.0)
            s0, s1 = r["s0"], r["s0"] + r["ds"]
            assert t0 - 1e-12 <= s0 and s1 <= t1 + 1e-12, (lev, pix, r)
            assert abs(s1 - t1) < 1e-12                      # always leaves through the cell's exit face
            if prev_end is not None:
                assert s0 == prev_end                        # abutting (zero-length steps are not logged)
                assert abs(s0 - t0) < 1e-12
            prev_end = s1
        _, t_exit = slab(org, d, np.zeros(3), np.full(3, float(n)))
        last_end = segs[-1]["s0"] + segs[-1]["ds"]
        if abs(last_end - t_exit) < 1e-12:
            n_leaf += 1
        else:
            assert last_end < t_exit                         # stopped earlier: it must have split
            assert last_end ** 2 > 3.0 * 4 ** lev / (math.pi * p.n_min_ray)
    # rays without any segment: a child whose start point lies outside the box exits at once (Fig. 2(f),
    # a child may start in another subvolume than its parent), or splits again at once
    def no_segment_exits(lev, pix, s):
        if (lev, pix) in byray:
            return 0
        d = O.pix2dir(lev, pix)
        c = np.floor(org + s * d)
        if np.any(c < 0) or np.any(c >= n):
            return 1
        assert s * s > 3.0 * 4 ** lev / (math.pi * p.n_min_ray)
        return sum(no_segment_exits(lev + 1, 4 * pix + k, s) for k in range(4))
    extra = 0
    for (lev, pix), segs in byray.items():
        last_end = segs[-1]["s0"] + segs[-1]["ds"]
        _, t_exit = slab(org, O.pix2dir(lev, pix), np.zeros(3), np.full(3, float(n)))
        if last_end < t_exit - 1e-12:
            extra += sum(no_segment_exits(lev + 1, 4 * pix + k, last_end) for k in range(4))
    assert n_leaf + extra == sum(st.exited) and extra > 0


def test_cells_match_fine_sampling(O):
    """Brute force: walk each ray in steps of 1e-3 cells and list the cells it is in; the DDA must visit
    the same cells in the same order (cells clipped by less than two sampling steps may be missed by
    the sampler, never by the DDA)."""
    n, src = 7, (2, 3, 3)
    g, p, a, x, gam, heat, st, log = uniform_case(O, n, 1e-8, 1.0, src, dx=1e18)
    org = np.array(src, float) + 0.5
    h = 1e-3
    for (lev, pix), segs in list(rays_of(log).items())[::7]:
        d = O.pix2dir(lev, pix)
        s_a, s_b = segs[0]["s0"], segs[-1]["s0"] + segs[-1]["ds"]
        ss = np.arange(s_a + h / 2, s_b, h)
        cells = np.floor(org[None, :] + ss[:, None] * d[None, :]).astype(int)
        keep = np.ones(len(cells), bool)
        keep[1:] = np.any(cells[1:] != cells[:-1], axis=1)
        sampled = [tuple(c) for c in cells[keep]]
        logged = [tuple(int(v) for v in r["cell"]) for r in segs]
        big = [tuple(int(v) for v in r["cell"]) for r in segs if r["ds"] > 2 * h]
        assert set(sampled) <= set(logged)
        assert [c for c in sampled if c in set(big)] == big


def test_tau_closed_form_and_absorption(O):
    """Eq. 2 in a uniform medium: tau(s) = n_HI sigma dx s.  Eq. 1 with V_box
    (PAPER.md:205): photons absorbed in a segment = L_ray e^-tau (1 - e^-dtau), L_ray = L/(12 4^l)
    (PAPER.md:197)."""
    nH, xHI, dx, L = 2e-3, 0.5, 2e20, 7e49
    g, p, a, x, gam, heat, st, log = uniform_case(O, 15, nH, xHI, (7, 7, 7), L=L, dx=dx)
    k = nH * xHI * p.sigma_cm2 * dx
    assert len(log) > 1000
    for r in log:
        assert abs(r["dtau"] - k * r["ds"]) <= 1e-15 * k * r["ds"]
        Lray = L / (12 * 4 ** int(r["level"]))
        expect = Lray * math.exp(-k * r["s0"]) * -math.expm1(-k * r["ds"])
        assert abs(r["dN"] - expect) <= 1e-13 * expect * (1 + k * r["s0"])


def test_budget_and_grid_sum(O):
    """Photon conservation is the design goal of Eq. 1 and Eq. 6-8:
    emitted = absorbed + escaped + residual to 1e-12, and sum_c Gamma[c] n_HI[c] V = absorbed."""
    rng = np.random.default_rng(3)
    n = 24
    a = 10 ** rng.uniform(-5, -2, (n, n, n))
    x = rng.uniform(0.0, 1.0, (n, n, n))
    x[rng.uniform(size=x.shape) < 0.1] = 0.0                  # some fully ionised cells (a_c = 0)
    g, p, a, x, gam, heat, st, log = uniform_case(O, n, None, None, (11, 12, 13), L=3e50, dx=3e20, fields=(a, x),
                                                   n_th=1e-4, e_excess_erg=2e-11, log_cap=3_000_000)
    em, ab, es, re = st.photons_emitted, st.photons_absorbed, st.photons_escaped, st.photons_residual
    assert em == 3e50
    assert abs(ab + es + re - em) <= 1e-12 * em
    V = g.dx_cm ** 3
    tot = float(np.sum(gam * a * x) * V)
    assert abs(tot - ab) <= 1e-12 * ab
    # heating reading H1: heat = e_excess * photons absorbed per unit volume
    assert abs(float(heat.sum()) * V - 2e-11 * ab) <= 1e-12 * 2e-11 * ab
    # ... PER CELL: for a monochromatic source heat[c] = e_excess n_HI[c] Gamma[c], because
    # both grids receive the same photons (f_c dN in the cell, (1 - f_c) dN in the neighbour), Gamma divided by
    # the receiving cell's n_HI V (Eq. 6 / 8's factor a_abs / a'_abs) and the heating by V alone
    nHI = a * x
    lit = gam > 0
    assert lit.sum() > 1000
    assert np.all(np.abs(heat[lit] - 2e-11 * nHI[lit] * gam[lit]) <= 1e-12 * heat[lit])
    assert np.all(heat[~lit] == 0.0)
    assert np.all(gam[(a * x) == 0.0] == 0.0)
    # per level bookkeeping identities
    for l in range(15):
        assert st.spawned[l] == st.split[l] + st.killed_tau[l] + st.killed_lmax[l] + st.exited[l]
        assert st.spawned[l + 1] == 4 * st.split[l]
    assert st.spawned[0] == 12


def test_split_radii_eq4(O):
    """Eq. 4 with Omega_c = (dx/R)^2 and Omega(l) = 4 pi/(12 4^l): a ray of level l
    marches only while R <= r_split(l) = 2^l sqrt(3/(pi N_min)) dx, and level l >= 1 rays start beyond
    r_split(l-1).  In a thin medium around a centred source all 12 4^l pixels of a level exist while the
    splitting sphere fits in the box (Fig. 1)."""
    for nmin in (3.0, 2.0, 1.0):
        n = 33
        g, p, a, x, gam, heat, st, log = uniform_case(O, n, 1e-9, 1.0, (16, 16, 16), dx=1e18, n_min_ray=nmin)
        rs = [2 ** l * math.sqrt(3.0 / (math.pi * nmin)) for l in range(16)]
        if nmin == 3.0:
            assert abs(rs[0] - 0.5642) < 1e-4 and abs(rs[5] - 18.05) < 1e-2
        for r in log:
            l = int(r["level"])
            assert r["s0"] <= rs[l] * (1 + 1e-15)
            if l > 0:
                assert r["s0"] > rs[l - 1] * (1 - 1e-15)
        for l in range(1, 14):
            if rs[l - 1] + math.sqrt(3.0) < 16.0:
                assert st.spawned[l] == 12 * 4 ** l and st.split[l - 1] == 12 * 4 ** (l - 1)
        assert sum(st.killed_tau) == 0 and sum(st.exited) > 0


def test_kill_at_tau_max(O):
    """rays terminate once tau exceeds tau_max.  Thick uniform medium: every leaf dies
    at the first cell boundary whose tau >= tau_max (reading R14), none leaves the box."""
    nH, dx = 1e-3, 6.6 * KPC / 32
    g, p, a, x, gam, heat, st, log = uniform_case(O, 32, nH, 1.0, (16, 16, 16), L=5e48, dx=dx)
    k = nH * p.sigma_cm2 * dx
    assert sum(st.exited) == 0 and sum(st.killed_tau) > 0
    ends = {}
    for r in log:
        ends[(int(r["level"]), int(r["pix"]))] = (r["s0"], r["s0"] + r["ds"])
    n_kill = 0
    for (l, pix), (s0, s1) in ends.items():
        if k * s1 >= p.tau_max * (1 + 1e-13):
            n_kill += 1
            assert k * s0 < p.tau_max * (1 + 1e-13)
    assert n_kill == sum(st.killed_tau)
    assert st.photons_residual <= 1.01e-8 * st.photons_emitted         # BASELINE: killed at 1e-8


def test_deposit_shares_eq5_to_8(O):
    """Sec. 2.6.  Recompute D_edge (distance of the segment midpoint to the nearest
    face, brute force over the six faces) and L_pix = R sqrt(Omega(l)); then f_c must be 1/2 + D/L when
    D < L/2 and the neighbour qualifies (in the box, n_H' >= n_th, absorber > 0), else exactly 1, and the
    grid must hold exactly the shares f_c dN and (1-f_c) dN (Eq. 6/8 with a_abs/a'_abs)."""
    rng = np.random.default_rng(11)
    n = 6
    a = 10 ** rng.uniform(-4, -2, (n, n, n))
    x = rng.uniform(0.2, 1.0, (n, n, n))
    x[0, 1, 2] = 0.0
    n_th = 5e-4
    src = (2, 3, 2)
    e_ex = 3e-11
    g, p, a, x, gam, heat, st, log = uniform_case(O, n, None, None, src, L=1e49, dx=5e19, fields=(a, x), n_th=n_th,
                                                   e_excess_erg=e_ex)
    org = np.array(src, float) + 0.5
    V = g.dx_cm ** 3
    photons = np.zeros((n, n, n))
    n_nb = n_th_block = n_edge_block = n_tie = 0
    for r in log:
        if r["dN"] == 0.0:                                  # fully ionised cell: nothing to share out
            ci, cj, ck = (int(v) for v in r["cell"])
            assert a[ck, cj, ci] * x[ck, cj, ci] == 0.0
            continue
        l = int(r["level"])
        d = O.pix2dir(l, int(r["pix"]))
        sm = r["s0"] + 0.5 * r["ds"]
        pos = org + sm * d - np.array(r["cell"], float)
        dist = [pos[0], 1 - pos[0], pos[1], 1 - pos[1], pos[2], 1 - pos[2]]
        D = min(dist)
        Lp = sm * math.sqrt(4 * math.pi / (12 * 4 ** l))
        assert abs(r["d_edge"] - D) < 1e-12 and abs(r["l_pix"] - Lp) <= 1e-14 * Lp
        ci, cj, ck = (int(v) for v in r["cell"])
        fc_expect, nbc = 1.0, None
        ds_sorted = sorted(dist)
        tie = ds_sorted[1] - ds_sorted[0] < 1e-12          # midpoint equidistant from two faces (rays in a
        if tie:                                            # symmetry plane): either face is "nearest"
            n_tie += 1
            faces = [f for f in range(6) if dist[f] - D < 1e-12]
        else:
            faces = [int(np.argmin(dist))]
        if D < 0.5 * Lp - 1e-12:
            face = int(r["nb_face"]) if r["nb_face"] >= 0 else faces[0]
            assert face in faces
            if tie and r["nb_face"] < 0:
                fc_expect = r["fc"]                        # which tied face was tested is a DEC convention
                assert r["fc"] == 1.0
            else:
                nb = [ci, cj, ck]
                nb[face // 2] += 1 if face % 2 else -1
                if all(0 <= v < n for v in nb):
                    if a[nb[2], nb[1], nb[0]] >= n_th and a[nb[2], nb[1], nb[0]] * x[nb[2], nb[1], nb[0]] > 0:
                        fc_expect, nbc = 0.5 + D / Lp, nb
                    else:
                        n_th_block += 1
                else:
                    n_edge_block += 1
        elif D < 0.5 * Lp + 1e-12:
            fc_expect = r["fc"]
        assert abs(r["fc"] - fc_expect) < 1e-11, (r, fc_expect)
        assert 0.5 <= r["fc"] <= 1.0
        photons[ck, cj, ci] += r["fc"] * r["dN"]
        if nbc is not None:
            n_nb += 1
            assert r["nb_face"] >= 0
            photons[nbc[2], nbc[1], nbc[0]] += (1 - r["fc"]) * r["dN"]
        else:
            assert r["nb_face"] == -1
    assert n_nb > 100 and n_th_block > 10 and n_edge_block > 10 and n_tie < 0.1 * len(log)
    assert st.neighbour_deposits == n_nb                    # the counter of Eq. 6 / 8 deposits
    expect = np.divide(photons, a * x * V, out=np.zeros_like(photons), where=(a * x) > 0)
    assert np.allclose(gam, expect, rtol=1e-12, atol=0)
    # heating (reading H1): e_excess per photon absorbed, per unit volume -- f_c dN of it in the cell,
    # (1 - f_c) dN in the logged neighbour.  `photons` was rebuilt above from the log with exactly that split, so
    # a share put in the wrong cell (all of it in c, or f_c and 1 - f_c swapped) fails here.
    assert n_nb > 100 and np.count_nonzero(photons) > 50
    assert np.allclose(heat, e_ex * photons / V, rtol=1e-12, atol=0)
    assert np.array_equal(heat == 0.0, photons == 0.0)


@pytest.mark.parametrize("mode,conserves", [(0, True), (1, False), (2, True), (3, True), (4, False)])
def test_correction_modes(O, mode, conserves):
    """Fig. 8c legend: 'Uncorrected' (no factor), 'Linear' (Eq. 5 only), 'Corrected' (Eq. 5
    + Eq. 6), 'Squared' ([59]); mode 3 = Eq. 7-8.  Modes without the secondary correction
    lose photons, the others conserve them."""
    g, p, a, x, gam, heat, st, log = uniform_case(O, 16, 1e-3, 1.0, (8, 8, 8), L=5e48, dx=3e20, geom_mode=mode)
    em = st.photons_emitted
    tot = st.photons_absorbed + st.photons_escaped + st.photons_residual
    if conserves:
        assert st.photons_lost == 0.0 and abs(tot - em) <= 1e-12 * em
    else:
        assert st.photons_lost > 1e-3 * em and abs(tot + st.photons_lost - em) <= 1e-12 * em
    if mode == 0:
        assert np.all(log["fc"] == 1.0)
    if mode == 4:
        lin = uniform_case(O, 16, 1e-3, 1.0, (8, 8, 8), L=5e48, dx=3e20, geom_mode=1)[6]
        assert st.photons_lost > lin.photons_lost              # squaring f_c loses more
