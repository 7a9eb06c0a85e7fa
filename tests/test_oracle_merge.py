"""Pins for the oracle's source pass (O1, M1-M8): dedup/sort, MAX_RADIUS and MERGE_SOURCES
(Alg. 3).  Expected values come from brute force written here (all pairs + DFS
labelling, direct shell counting) and from hand cases; the paper prints no values, so the shell sample
pattern and the defaults stay 'parity unpinned'."""
import math

import numpy as np


def grid(O, n):
    return O.make_grid((n, n, n), 1e20)


def test_dedup_and_sort(O):
    g = grid(O, 16)
    pos = np.array([[3.2, 4.9, 1.0], [15.99, 0.0, 0.5], [3.7, 4.1, 1.99], [0.1, 0.1, 0.1], [3.0, 4.0, 1.0]])
    L = np.array([1.0, 2.0, 4.0, 8.0, 16.0])
    cell, Lo = O.prepare_sources(g, pos, L)
    assert cell.tolist() == [[0, 0, 0], [15, 0, 0], [3, 4, 1]]          # ascending (k*ny + j)*nx + i
    assert Lo.tolist() == [8.0, 2.0, 21.0]                               # same-cell fluxes summed
    # sequential sum in input order (rounding is part of the contract: L later steers the centroid)
    vals = np.array([1e16, 1.0, -1e16, 1.0])
    cell, Lo = O.prepare_sources(g, np.tile([[5.5, 5.5, 5.5]], (4, 1)), np.abs(vals))
    s = 0.0
    for v in np.abs(vals):
        s = s + v
    assert Lo[0] == s
    # outside the box / negative flux are rejected
    for bad in ([[16.0, 1, 1]], [[-0.01, 1, 1]], [[1, 1, float("nan")]]):
        try:
            O.prepare_sources(g, np.array(bad, float), np.array([1.0]))
            assert False
        except RuntimeError:
            pass
    try:
        O.prepare_sources(g, np.array([[1.0, 1, 1]]), np.array([-1.0]))
        assert False
    except RuntimeError:
        pass
    c, l = O.prepare_sources(g, np.zeros((0, 3)), np.zeros(0))
    assert len(c) == 0


def brute_radius(O, p, xion, c, n):
    """MAX_RADIUS of Alg. 3 counted directly, shells of 12 4^samp_level directions."""
    if xion[c[2], c[1], c[0]] < p.x_th:
        return 0.0
    dirs = O.pix2dir_all(p.samp_level)
    r = p.delta_r
    while r <= p.r_max:
        pts = np.floor(np.array(c)[None, :] + 0.5 + r * dirs).astype(int)
        ok = np.all((pts >= 0) & (pts < n), axis=1)
        ntot = int(ok.sum())
        nion = int(sum(xion[k, j, i] >= p.x_th for i, j, k in pts[ok]))
        if ntot == 0:
            return r - p.delta_r
        if ntot < p.n_min_samples:
            if nion < ntot:
                return r - p.delta_r
        elif nion / ntot < p.f_req:
            return r - p.delta_r
        r += p.delta_r
    return p.r_max


def test_bubble_radius_hand_cases(O):
    n = 32
    g = grid(O, n)
    p = O.make_params(r_max=9.0, delta_r=2.0)
    xHI = np.full((n, n, n), 1e-4)
    c = np.array([[16, 16, 16], [2, 16, 16], [0, 0, 0]], np.int32)
    r = O.bubble_radius(g, p, xHI, c)
    assert r[0] == 9.0                           # all shells pass: exactly R_max even if not a multiple
    assert r[1] == 9.0                           # shells cut by the box: only in-box samples are 'checked'
    assert r[2] == 9.0
    xHI2 = xHI.copy()
    xHI2[16, 16, 16] = 1.0                       # source in a neutral cell: x0 < x_th -> 0
    assert O.bubble_radius(g, p, xHI2, c[:1])[0] == 0.0
    # ionised ball of radius 5.2 cells around the source, neutral outside: shells 2 and 4 pass, 6 fails -> 4
    ax = np.arange(n) - 16.0
    R = np.sqrt(ax[None, None, :] ** 2 + ax[None, :, None] ** 2 + ax[:, None, None] ** 2)
    xHI3 = np.where(R <= 5.2, 1e-4, 1.0)
    assert O.bubble_radius(g, p, xHI3, c[:1])[0] == 4.0
    # a ball of radius 1: first shell fails -> r - dr = 0
    assert O.bubble_radius(g, p, np.where(R <= 1.0, 1e-4, 1.0), c[:1])[0] == 0.0


def test_bubble_radius_brute_force(O):
    rng = np.random.default_rng(2)
    n = 24
    g = grid(O, n)
    from scipy.ndimage import gaussian_filter
    f = gaussian_filter(rng.normal(size=(n, n, n)), 2.0, mode="wrap")
    xHI = np.where(f > np.quantile(f, 0.7), 1.0, 1e-3)
    for kw in (dict(), dict(f_req=0.9, n_min_samples=100, r_max=11.0), dict(samp_level=1, delta_r=1.0, r_max=6.0)):
        p = O.make_params(**kw)
        cells = rng.integers(0, n, (60, 3)).astype(np.int32)
        r = O.bubble_radius(g, p, xHI, cells)
        for c, rr in zip(cells, r):
            assert rr == brute_radius(O, p, 1.0 - xHI, c, n)
        assert len(set(r.tolist())) > 2


def brute_merge(p, cells, L, r):
    """All pairs + DFS labelling + collapse, written independently of the oracle's union-find."""
    n = len(L)
    adj = [[] for _ in range(n)]
    for a in range(n):
        for b in range(a + 1, n):
            if r[a] > 0 and r[b] > 0:
                d2 = int(((cells[a].astype(np.int64) - cells[b]) ** 2).sum())
                if d2 <= (p.f_ov * (r[a] + r[b])) ** 2 + p.eps:
                    adj[a].append(b)
                    adj[b].append(a)
    label = [-1] * n
    groups = []
    for a in range(n):
        if label[a] >= 0:
            continue
        stack, mem = [a], []
        label[a] = len(groups)
        while stack:
            u = stack.pop()
            mem.append(u)
            for v in adj[u]:
                if label[v] < 0:
                    label[v] = len(groups)
                    stack.append(v)
        groups.append(sorted(mem))
    out = []
    for mem in groups:
        if len(mem) == 1:
            a = mem[0]
            out.append((tuple(cells[a]), L[a], r[a]))
            continue
        F = 0.0
        num = np.zeros(3)
        for b in mem:
            F = F + L[b]
            for ax in range(3):
                num[ax] = num[ax] + L[b] * float(cells[b][ax])
        rc = np.floor(num / F + 0.5).astype(np.int64)
        best = min(mem, key=lambda b: (int(((cells[b] - rc) ** 2).sum()), b))
        out.append((tuple(cells[best]), F, max(r[b] for b in mem)))
    return out


def test_merge_brute_force(O):
    rng = np.random.default_rng(9)
    n = 40
    g = grid(O, n)
    for trial in range(6):
        p = O.make_params(f_ov=[1.0, 0.7, 1.3][trial % 3])
        m = 64
        lin = np.sort(rng.choice(n ** 3, m, replace=False))
        cells = np.stack([lin % n, (lin // n) % n, lin // (n * n)], 1).astype(np.int32)
        L = 10 ** rng.uniform(48, 51, m)
        r = rng.choice([0.0, 2.0, 4.0, 6.0], m)
        oc, oL, orr = O.merge(g, p, cells, L, r)
        exp = brute_merge(p, cells, L, r)
        exp.sort(key=lambda e: (e[0][2] * n + e[0][1]) * n + e[0][0])
        assert 1 < len(oc) < m
        assert len(oc) == len(exp)
        for a in range(len(exp)):
            assert tuple(oc[a]) == exp[a][0] and oL[a] == exp[a][1] and orr[a] == exp[a][2]
        # invariants the paper states: flux sum, max radius, member cell, sorted order
        assert abs(oL.sum() - L.sum()) <= 1e-13 * L.sum()
        keys = (oc[:, 2].astype(np.int64) * n + oc[:, 1]) * n + oc[:, 0]
        assert np.all(np.diff(keys) > 0)
        assert set(map(tuple, oc)) <= set(map(tuple, cells))


def test_merge_hand_cases(O):
    g = grid(O, 64)
    p = O.make_params()
    L = np.array([1.0, 3.0])
    # two sources 10 apart: link iff d <= f_ov (ra + rb)
    c = np.array([[10, 10, 10], [20, 10, 10]], np.int32)
    assert len(O.merge(g, p, c, L, np.array([4.0, 6.0]))[0]) == 1
    assert len(O.merge(g, p, c, L, np.array([4.0, 5.9]))[0]) == 2
    assert len(O.merge(g, O.make_params(f_ov=1.1), c, L, np.array([4.0, 5.9]))[0]) == 1
    # r = 0 never links
    assert len(O.merge(g, p, c, L, np.array([0.0, 60.0]))[0]) == 2
    # merged: flux sum, max radius, centroid (10*1 + 20*3)/4 = 17.5 -> round 18 -> nearest member is x = 20
    oc, oL, orr = O.merge(g, p, c, L, np.array([4.0, 6.0]))
    assert oc.tolist() == [[20, 10, 10]] and oL[0] == 4.0 and orr[0] == 6.0
    # chain a-b-c merges transitively although a and c do not overlap (connected components)
    c3 = np.array([[10, 10, 10], [18, 10, 10], [26, 10, 10]], np.int32)
    oc, oL, orr = O.merge(g, p, c3, np.array([1.0, 1.0, 1.0]), np.array([4.0, 4.0, 4.0]))
    assert oc.tolist() == [[18, 10, 10]] and oL[0] == 3.0
    # equal-flux pair: centroid 14.0 -> tie between members at distance 4 -> first member (reading R10)
    oc, _, _ = O.merge(g, p, np.array([[10, 10, 10], [18, 10, 10]], np.int32), np.array([1.0, 1.0]), np.array([4.0, 4.0]))
    assert oc.tolist() == [[10, 10, 10]]


def test_step_merge_switch(O):
    """merge = 0/1/2 (PAPER.md:311 'automerge'; 0.018 in Fig. 7)."""
    n = 24
    g = grid(O, n)
    nH = np.full((n, n, n), 1e-5)
    xHI = np.full((n, n, n), 1e-3)
    xHI[:, :, :2] = 1.0
    pos = np.array([[10.5, 10.5, 10.5], [13.5, 10.5, 10.5], [10.2, 10.9, 10.1], [0.5, 5.5, 5.5]])
    L = np.array([1e49, 2e49, 4e49, 1e49])
    res = {}
    for m in (0, 1, 2):
        p = O.make_params(merge=m)
        gam, heat, st, cat = O.step(g, p, nH, xHI, pos, L)
        res[m] = (st, cat, gam)
        assert st.n_src_in == 4 and st.n_src_dedup == 3
        assert abs(st.photons_emitted - L.sum()) <= 1e-15 * L.sum()
    assert res[0][0].n_src_merged == 3 and res[1][0].n_src_merged == 2 and res[2][0].n_src_merged == 2
    assert res[1][1][0].tolist() == [[0, 5, 5], [10, 10, 10]]          # neutral-cell source stays alone
    assert res[1][1][1].tolist() == [1e49, 7e49]
    p = O.make_params(merge=2, automerge_xmean=0.95)                    # mean ionised fraction 0.916 < 0.95
    assert O.step(g, p, nH, xHI, pos, L)[2].n_src_merged == 3
    assert abs(O.mean_ionised(g, xHI) - (1 - (22 * 1e-3 + 2) / 24)) < 1e-12
