"""Pins for the oracle's periodic mode ("rays ... wrap around,
terminating when their travel distance exceeds sqrt(3) L_box", RAY_FLTR at 174, minimum-image merge at 321
and 380-383).  The periodic code is pinned to the NON-periodic oracle (itself pinned by test_oracle_rays /
_merge) through translation invariance: a source whose rays never reach the boundary gives the same field
wherever the box is cut; and to geometry written out here (travel-distance limit, minimum image)."""
import math

import numpy as np

COUNTERS = ["spawned", "split", "killed_tau", "exited", "killed_lmax"]


def fields(n, seed, lo=0.05):
    rng = np.random.default_rng(seed)
    return 10 ** rng.uniform(-3.3, -2.7, (n, n, n)), rng.uniform(lo, 1.0, (n, n, n))


def test_translation_invariance_pins_wrapping(O):
    """Thick medium, source in the middle: no ray reaches a face, so the open-box result is also the periodic
    one.  Rolling fields and source so that the lit region straddles all three pairs of faces must give the
    rolled result bit for bit (one source: same deposits in the same order), with identical counters."""
    n, dx = 20, 7.0e20
    nH, xHI = fields(n, 1, lo=0.5)
    p = O.make_params(n_th=1e-3, e_excess_erg=1e-11)
    src = np.array([[10, 9, 11]], np.int32)
    L = np.array([3e49])
    g0 = O.make_grid((n, n, n), dx)
    gam0, heat0, st0 = O.trace(g0, p, nH, xHI, src, L)
    assert sum(st0.exited) == 0 and sum(st0.killed_tau) > 100 and st0.segments > 1000
    gp = O.make_grid((n, n, n), dx, periodic=1)
    gam_p, heat_p, st_p = O.trace(gp, p, nH, xHI, src, L)
    assert np.array_equal(gam_p, gam0) and np.array_equal(heat_p, heat0)
    shift = (9, -8, 10)                                   # (dz, dy, dx): source lands at cell (0, 1, 0)
    nH_r, xHI_r = np.roll(nH, shift, (0, 1, 2)), np.roll(xHI, shift, (0, 1, 2))
    src_r = np.array([[(10 + shift[2]) % n, (9 + shift[1]) % n, (11 + shift[0]) % n]], np.int32)
    gam_r, heat_r, st_r = O.trace(gp, p, nH_r, xHI_r, src_r, L)
    assert np.array_equal(gam_r, np.roll(gam0, shift, (0, 1, 2)))
    assert np.array_equal(heat_r, np.roll(heat0, shift, (0, 1, 2)))
    for name in COUNTERS:
        assert list(getattr(st_r, name)) == list(getattr(st0, name)), name
    assert st_r.segments == st0.segments and st_r.photons_absorbed == st0.photons_absorbed
    # the open box with the rolled inputs differs: the source sits in a corner and most rays leave at once
    gam_open, _, st_open = O.trace(g0, p, nH_r, xHI_r, src_r, L)
    assert sum(st_open.exited) > 0 and not np.array_equal(gam_open, gam_r)


def test_travel_distance_limit(O):
    """Empty periodic box: nothing is absorbed, no ray is killed, every lineage ends by the RAY_FLTR test
    p.s < sqrt(3) L_box: every segment starts below the limit, every leaf's last segment ends
    at or beyond it, and all photons are accounted as escaped.  While r_split(l-1) + sqrt(3) < sqrt(3) L_box
    every ray of level l-1 splits, so spawned[l] = 12 4^l (Eq. 4)."""
    n = 6
    g = O.make_grid((n, n, n), 1e18, periodic=1)
    p = O.make_params()
    nH = np.full((n, n, n), 1e-3)
    xHI = np.zeros((n, n, n))
    src = np.array([[1, 4, 2]], np.int32)
    gam, heat, st, log = O.trace(g, p, nH, xHI, src, np.array([1e50]), log_cap=3_000_000)
    s_max = math.sqrt(3.0) * n
    assert sum(st.killed_tau) == 0 and sum(st.killed_lmax) == 0 and not gam.any()
    assert abs(st.photons_escaped - 1e50) <= 1e-12 * 1e50 and st.photons_absorbed == 0.0
    assert np.all(log["s0"] < s_max)
    assert st.segments == len(log)
    ends = {}
    for r in log:
        ends[(int(r["level"]), int(r["pix"]))] = r["s0"] + r["ds"]
    top = max(l for l in range(16) if st.spawned[l])
    leaves = [v for (l, pix), v in ends.items() if st.split[l] == 0 or l == top]
    assert len(leaves) > 100 and min(leaves) >= s_max and max(leaves) < s_max + math.sqrt(3.0) + 1e-9
    for l in range(1, 16):
        r_split_prev = 2.0 ** (l - 1) * math.sqrt(3.0 / (math.pi * 3.0))
        if r_split_prev + math.sqrt(3.0) < s_max:
            assert st.spawned[l] == 12 * 4 ** l, l
    # cells of the wrapped path: every logged cell is inside the box, and far more distinct cells are
    # visited than an open box would allow from this corner-ish source
    assert log["cell"].min() >= 0 and log["cell"].max() < n
    assert len({tuple(c) for c in log["cell"]}) == n ** 3


def test_wrapped_cells_follow_the_line(O):
    """The cell of every segment is the wrapped cell of the segment's midpoint on the straight line
    src + s d (independent of the DDA bookkeeping)."""
    n = 5
    g = O.make_grid((n, n, n), 1e18, periodic=1)
    nH, xHI = np.full((n, n, n), 1e-6), np.full((n, n, n), 0.5)
    src = np.array([[4, 0, 2]], np.int32)
    _, _, st, log = O.trace(g, O.make_params(), nH, xHI, src, np.array([1e48]), log_cap=2_000_000)
    sel = log[log["ds"] > 1e-9][::7]
    assert len(sel) > 2000
    for r in sel:
        d = O.pix2dir(int(r["level"]), int(r["pix"]))
        mid = (src[0] + 0.5) + (r["s0"] + 0.5 * r["ds"]) * d
        assert tuple(np.floor(mid).astype(int) % n) == tuple(r["cell"]), r


def test_budget_and_uniform_symmetry(O):
    """Uniform periodic medium, moderately thin: emitted = absorbed + escaped + residual to 1e-12
    (BASELINE.json), sum_c Gamma n_HI V = absorbed, and the result does not depend on where the source is."""
    n, dx = 8, 5e19
    g = O.make_grid((n, n, n), dx, periodic=1)
    nH, xHI = np.full((n, n, n), 1e-3), np.full((n, n, n), 0.3)
    p = O.make_params()
    out = []
    for c in ((0, 0, 0), (7, 3, 5)):
        gam, _, st = O.trace(g, p, nH, xHI, np.array([c], np.int32), np.array([2e49]))
        tot = st.photons_absorbed + st.photons_escaped + st.photons_residual
        assert abs(tot - 2e49) <= 1e-12 * 2e49
        assert abs((gam * nH * xHI).sum() * dx ** 3 - st.photons_absorbed) <= 1e-12 * st.photons_absorbed
        out.append((np.roll(gam, tuple(-v for v in c[::-1]), (0, 1, 2)), st))
    assert np.array_equal(out[0][0], out[1][0])
    assert list(out[0][1].spawned) == list(out[1][1].spawned) and out[0][1].segments == out[1][1].segments


def test_merge_minimum_image(O):
    """PAPER.md:321 'coordinates ... computed under minimum-image (periodic) geometry', 380-383 'centroid
    (with periodic unwrapping) ... wrap back into domain ... snap'.  Hand cases + brute force in numpy."""
    n = 32
    gp, g0 = O.make_grid((n, n, n), 1.0, periodic=1), O.make_grid((n, n, n), 1.0)
    p = O.make_params(merge=1, f_ov=1.0, r_max=4.0)
    # two sources 4 cells apart through the x faces: linked only in the periodic box
    cell = np.array([[1, 5, 5], [29, 5, 5]], np.int32)
    L, r = np.array([1.0, 3.0]), np.array([2.0, 2.0])
    c0, L0, r0 = O.merge(g0, p, cell, L, r)
    assert len(L0) == 2
    cp, Lp, rp = O.merge(gp, p, cell, L, r)
    # unwrapped about the first member: x = 1 and 29 - 32 = -3; centroid (1*1 + 3*(-3))/4 = -2 -> wraps to
    # 30; nearest member by minimum image: x = 29 (distance 1) against x = 1 (distance 3)
    assert len(Lp) == 1 and Lp[0] == 4.0 and tuple(cp[0]) == (29, 5, 5) and rp[0] == 2.0
    # brute force on random sources
    rng = np.random.default_rng(5)
    m = 48
    cells = np.unique(rng.integers(0, n, (m, 3)).astype(np.int32), axis=0)
    order = np.lexsort((cells[:, 0], cells[:, 1], cells[:, 2]))
    cells = cells[order]
    m = len(cells)
    Ls, rs = rng.uniform(1, 2, m), rng.choice([0.0, 2.0, 4.0], m)
    oc, oL, orr = O.merge(gp, p, cells, Ls, rs)

    def mi(d):
        d = np.mod(d, n)
        return np.where(2 * d >= n, d - n, d)
    lab = np.arange(m)
    changed = True
    while changed:                                      # label propagation to a fixed point
        changed = False
        for a in range(m):
            for b in range(a + 1, m):
                if rs[a] > 0 and rs[b] > 0 and (mi(cells[a] - cells[b]) ** 2).sum() <= (rs[a] + rs[b]) ** 2 + 1e-9:
                    lo = min(lab[a], lab[b])
                    if lab[a] != lo or lab[b] != lo:
                        lab[a] = lab[b] = lo
                        changed = True
    exp = []
    for grp in sorted(set(lab)):
        mem = np.flatnonzero(lab == grp)
        if len(mem) == 1:
            exp.append((tuple(cells[mem[0]]), Ls[mem[0]], rs[mem[0]]))
            continue
        F = 0.0
        num = np.zeros(3)
        for b in mem:
            F = F + Ls[b]
            num = num + Ls[b] * (cells[mem[0]] + mi(cells[b] - cells[mem[0]])).astype(float)
        rc = np.mod(np.floor(num / F + 0.5).astype(int), n)
        d2 = [(mi(cells[b] - rc) ** 2).sum() for b in mem]
        exp.append((tuple(cells[mem[int(np.argmin(d2))]]), F, rs[mem].max()))
    exp.sort(key=lambda e: (e[0][2] * n + e[0][1]) * n + e[0][0])
    assert len(exp) == len(oL) < m
    for e, c, l, rr in zip(exp, oc, oL, orr):
        assert e[0] == tuple(c) and e[1] == l and e[2] == rr
    assert len(O.merge(g0, p, cells, Ls, rs)[1]) > len(oL)      # the open box links fewer pairs


def test_bubble_radius_wraps_samples(O):
    """Periodic shells are sampled through the faces (PAPER.md:351 'checked point samples'; every sample is
    checked): a fully ionised box gives exactly R_max at a corner, and the radius is translation invariant."""
    n = 24
    gp, g0 = O.make_grid((n, n, n), 1.0, periodic=1), O.make_grid((n, n, n), 1.0)
    p = O.make_params(r_max=8.0)
    x_all = np.zeros((n, n, n))
    assert O.bubble_radius(gp, p, x_all, np.array([[0, 0, 0]], np.int32))[0] == 8.0
    rng = np.random.default_rng(9)
    xHI = (rng.uniform(0, 1, (n, n, n)) < 0.12).astype(float)        # 12 % neutral cells
    xHI[10:14, 10:14, 10:14] = 0.0
    r_mid = O.bubble_radius(g0, p, xHI, np.array([[12, 12, 12]], np.int32))[0]
    shift = (11, 12, -12)
    r_rolled = O.bubble_radius(gp, p, np.roll(xHI, shift, (0, 1, 2)),
                               np.array([[(12 + shift[2]) % n, (12 + shift[1]) % n, (12 + shift[0]) % n]], np.int32))[0]
    assert r_rolled == O.bubble_radius(gp, p, xHI, np.array([[12, 12, 12]], np.int32))[0]
    assert r_mid <= 8.0 and r_rolled >= 0.0
