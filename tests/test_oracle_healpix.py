"""Pins for the oracle's HEALPix directions (O2 / DIR-SPEC) against what Gorski et al. 2005 fix
(PAPER.md:613 ref [63]; "twelve ray-casts ... coarsest level", "four HEALPix
subpixels").  None of these re-types the oracle's pix->vector formula: they use ring heights and
populations, symmetry, and the INVERSE map (vector -> nested pixel), which is a different algorithm."""
import math

import numpy as np
import pytest


def ang2pix_nest(level, v):
    """Inverse map (vector -> nested pixel) after the HEALPix library's `loc2pix` routine, the standard
    statement of Gorski et al.'s projection (equatorial: cylindrical equal-area; polar caps: Collignon): a
    restated public algorithm, used here only as a pin.  It shares nothing with the oracle's pix -> vector code."""
    ns = 1 << level
    x, y, z = v
    za = abs(z)
    tt = (math.atan2(y, x) % (2 * math.pi)) / (0.5 * math.pi)      # in [0,4)
    if tt >= 4.0:
        tt = 0.0
    if za <= 2.0 / 3.0:
        t1 = ns * (0.5 + tt)
        t2 = ns * z * 0.75
        jp = int(math.floor(t1 - t2))       # ascending edge line
        jm = int(math.floor(t1 + t2))       # descending edge line
        ifp, ifm = jp // ns, jm // ns
        if ifp == ifm:
            face = (ifp & 3) | 4
        elif ifp < ifm:
            face = ifp & 3
        else:
            face = (ifm & 3) + 8
        ix = jm & (ns - 1)
        iy = ns - (jp & (ns - 1)) - 1
    else:
        ntt = min(3, int(tt))
        tp = tt - ntt
        tmp = ns * math.sqrt(3.0 * (1.0 - za))
        jp = min(ns - 1, int(tp * tmp))
        jm = min(ns - 1, int((1.0 - tp) * tmp))
        if z >= 0:
            face, ix, iy = ntt, ns - jm - 1, ns - jp - 1
        else:
            face, ix, iy = ntt + 8, jp, jm
    pf = 0
    for b in range(level):
        pf |= ((ix >> b) & 1) << (2 * b)
        pf |= ((iy >> b) & 1) << (2 * b + 1)
    return face * ns * ns + pf


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5])
def test_roundtrip_through_inverse_map(O, level):
    d = O.pix2dir_all(level)
    for p in range(len(d)):
        assert ang2pix_nest(level, d[p]) == p


def test_roundtrip_sampled_deep_levels(O):
    rng = np.random.default_rng(5)
    for level in (8, 11, 13):
        for p in rng.integers(0, 12 * 4 ** level, 300):
            assert ang2pix_nest(level, O.pix2dir(level, int(p))) == int(p)


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_children_nest_inside_parent(O, level):
    """the four children of p are 4p..4p+3 (nested scheme) and lie inside p."""
    d = O.pix2dir_all(level + 1)
    for c in range(len(d)):
        assert ang2pix_nest(level, d[c]) == c // 4


def test_random_points_nest_consistently():
    rng = np.random.default_rng(1)
    v = rng.normal(size=(2000, 3))
    v /= np.linalg.norm(v, axis=1)[:, None]
    for w in v:
        p = [ang2pix_nest(l, w) for l in range(0, 9)]
        for l in range(8):
            assert p[l + 1] // 4 == p[l]


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5, 6])
def test_unit_norm_zero_sum_and_rings(O, level):
    ns = 1 << level
    d = O.pix2dir_all(level)
    npix = 12 * ns * ns
    assert d.shape == (npix, 3)
    assert np.max(np.abs(np.linalg.norm(d, axis=1) - 1.0)) < 4e-16
    assert np.max(np.abs(d.sum(0))) < 1e-13 * npix
    # ring heights and populations (Gorski et al. 2005 Eq. 4-9)
    zs = {}
    for z in d[:, 2]:
        zs[z] = zs.get(z, 0) + 1
    expect = {}
    for i in range(1, ns):                      # caps
        z = 1.0 - i * i / (3.0 * ns * ns)
        expect[z] = 4 * i
        expect[-z] = 4 * i
    for i in range(ns, 3 * ns + 1):             # belt
        expect[4.0 / 3.0 - 2.0 * i / (3.0 * ns)] = 4 * ns
    got = sorted(zs.items())
    exp = sorted(expect.items())
    assert len(got) == len(exp) == 4 * ns - 1
    for (zg, cg), (ze, ce) in zip(got, exp):
        assert abs(zg - ze) < 3e-16 and cg == ce
    # pixels of one ring are equally spaced in longitude
    for zg, cg in got[:: max(1, len(got) // 7)]:
        ph = np.sort(np.arctan2(d[d[:, 2] == zg, 1], d[d[:, 2] == zg, 0]) % (2 * np.pi))
        gaps = np.diff(np.concatenate([ph, [ph[0] + 2 * np.pi]]))
        assert np.max(np.abs(gaps - 2 * np.pi / cg)) < 1e-13


def test_level0_centres(O):
    d = O.pix2dir_all(0)
    for p in range(12):
        z = d[p, 2]
        phi = math.degrees(math.atan2(d[p, 1], d[p, 0])) % 360.0
        if p < 4:
            assert abs(z - 2 / 3) < 1e-16 and abs(phi - (45 + 90 * p)) < 1e-12
        elif p < 8:
            assert z == 0.0 and abs(phi - 90 * (p - 4)) < 1e-12
        else:
            assert abs(z + 2 / 3) < 1e-16 and abs(phi - (45 + 90 * (p - 8))) < 1e-12
    # equatorial base pixels are EXACTLY axis aligned (decisions rely on exact symmetry, DESIGN.md DEC)
    assert tuple(d[4]) == (1.0, 0.0, 0.0)
    assert abs(d[5, 0]) == 0.0 and d[5, 1] == 1.0
    assert d[6, 0] == -1.0 and abs(d[6, 1]) == 0.0
    assert abs(d[7, 0]) == 0.0 and d[7, 1] == -1.0


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5])
def test_exact_mirror_symmetry(O, level):
    """The pixelisation is symmetric under x->-x, y->-y, z->-z and x<->y; DIR-SPEC promises that mirrored
    pixels have bit-identical mirrored components (ties between faces are then exact ties)."""
    d = O.pix2dir_all(level)
    d = np.where(d == 0.0, 0.0, d)                      # -0.0 == 0.0
    s = set(map(tuple, d))
    for f in ([-1, 1, 1], [1, -1, 1], [1, 1, -1]):
        assert set(map(tuple, np.where(d == 0.0, 0.0, d * np.array(f, float)))) == s
    assert set(map(tuple, d[:, [1, 0, 2]])) == s


def test_polynomial_trig_matches_libm(O):
    """DIR-SPEC's polynomial sin/cos agree with libm to a few ulp, and phi sits on the equal-area ring
    lattice phi = (pi/4) m / nr of Gorski et al. (nr pixels per quadrant on the ring)."""
    for level in (3, 7, 12):
        ns = 1 << level
        rng = np.random.default_rng(level)
        for p in rng.integers(0, 12 * ns * ns, 400):
            d = O.pix2dir(level, int(p))
            z = d[2]
            st = math.hypot(d[0], d[1])
            assert abs(st * st + z * z - 1.0) < 1e-15
            za = abs(z)
            nr = ns if za <= 2 / 3 + 1e-15 else round(ns * math.sqrt(3 * (1 - za)))
            phi = math.atan2(d[1], d[0]) % (2 * math.pi)
            m = phi / (math.pi / (4 * nr))
            assert abs(m - round(m)) < 1e-6
            m = round(m)
            assert abs(d[0] / st - math.cos(math.pi * m / (4 * nr))) < 1e-15
            assert abs(d[1] / st - math.sin(math.pi * m / (4 * nr))) < 1e-15
