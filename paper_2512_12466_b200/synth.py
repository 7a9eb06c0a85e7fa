"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module holds NO ray-tracing arithmetic: it only draws fields and source lists.  The same arrays
are handed to the CPU oracle (tests, bench cpu_baseline) and to the CUDA library; neither side
generates its own.  They stand in for the paper's Nyx density / ionisation fields and halo catalogues
(40 h^-1 Mpc box, RT grids 256^3 / 512^3 / 1024^3), which are not available here.

Everything is torch on the given device (CPU by default; bench.py and the GPU tests pass "cuda" for the
1024^3 case so that the FFTs take seconds).  A config generated on one device type is deterministic for
that device type; the arrays are generated once per run and shared.
"""
import math

import torch

KPC_CM = 3.0856775814913673e21
MPC_CM = 3.0856775814913673e24
BOX_MPC = 40.0 / 0.67742            # 40 h^-1 Mpc, h = 0.67742  -> 59.05 Mpc comoving
SIGMA_HI = 6.3e-18                  # BASELINE.json config 1
TAU_MAX = math.log(1e8)             # BASELINE.json: "killed at 1e-8 of initial photons"


def _gen(seed, device):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _kgrid(n, device, dtype):
    k1 = torch.fft.fftfreq(n, d=1.0 / n, device=device, dtype=dtype)
    kr = torch.fft.rfftfreq(n, d=1.0 / n, device=device, dtype=dtype)
    return k1, kr


def gaussian_field(n, seed, slope, device="cpu", dtype=torch.float64):
    """Unit-variance Gaussian random field on n^3 with P(k) ~ k^slope (white noise -> rfftn -> filter)."""
    w = torch.randn((n, n, n), generator=_gen(seed, device), device=device, dtype=dtype)
    f = torch.fft.rfftn(w)
    del w
    k1, kr = _kgrid(n, device, dtype)
    k2 = (k1 * k1)[:, None, None] + (k1 * k1)[None, :, None] + (kr * kr)[None, None, :]
    amp = torch.where(k2 > 0, k2.clamp_min(1e-30) ** (slope / 4.0), torch.zeros_like(k2))
    del k2
    f *= amp
    del amp
    g = torch.fft.irfftn(f, s=(n, n, n))
    del f
    g -= g.mean()
    g /= g.std()
    return g


def smoothed_noise(n, seed, sigma_cells, device="cpu", dtype=torch.float64):
    """White noise smoothed with a Gaussian of width sigma_cells (periodic), zero mean, unit variance."""
    w = torch.randn((n, n, n), generator=_gen(seed, device), device=device, dtype=dtype)
    f = torch.fft.rfftn(w)
    del w
    k1, kr = _kgrid(n, device, dtype)
    c = -0.5 * (2.0 * math.pi * sigma_cells / n) ** 2
    f *= torch.exp(c * (k1 * k1))[:, None, None]
    f *= torch.exp(c * (k1 * k1))[None, :, None]
    f *= torch.exp(c * (kr * kr))[None, None, :]
    g = torch.fft.irfftn(f, s=(n, n, n))
    del f
    g -= g.mean()
    g /= g.std()
    return g


def quantile_hist(x, q, bins=1 << 16):
    """q-quantile of a (large) tensor by two histogram passes; deterministic, no sort."""
    lo, hi = float(x.min()), float(x.max())
    for _ in range(2):
        h = torch.histc(x.float() if x.dtype == torch.float64 and x.numel() > (1 << 28) else x, bins=bins,
                        min=lo, max=hi)
        c = torch.cumsum(h.double(), 0)
        below = float((x < lo).sum())
        target = q * x.numel() - below
        i = int(torch.searchsorted(c, torch.tensor([target], device=c.device, dtype=c.dtype)).item())
        i = min(max(i, 0), bins - 1)
        w = (hi - lo) / bins
        lo, hi = lo + i * w, lo + (i + 1) * w
    return 0.5 * (lo + hi)


def lognormal_density(n, seed, mean, sigma_ln, device, dtype):
    g = gaussian_field(n, seed, -2.5, device, dtype)
    g *= sigma_ln
    g -= 0.5 * sigma_ln * sigma_ln
    nH = torch.exp_(g)
    nH *= mean / float(nH.double().mean())
    return nH


def sample_sources(nH, n_src, seed_pos, seed_lum, mean_L, sigma_ln_L):
    """Cells drawn with probability ~ n_H^2 (inverse CDF in fp64; duplicates allowed, which exercises the
    dedup pass); luminosities lognormal with the given mean.  Positions are returned in cell units, inside
    the drawn cell (the library snaps them back).

    The inverse CDF is taken in two levels -- x-rows first, then the cell inside the drawn row -- with both
    running sums made sequentially on the host: a device-wide cumsum on CUDA is not reproducible from run
    to run (its partial sums are combined in a varying order), and the source list must be."""
    dev = nH.device
    n = nH.shape[0]
    w = nH.reshape(n * n, n).double()
    w = w * w
    rows = w.sum(1).cpu()                                  # per-row reduction: fixed order
    cdf_r = torch.cumsum(rows, 0)                          # host, sequential
    total = float(cdf_r[-1])
    u = torch.rand(n_src, generator=_gen(seed_pos, dev), device=dev, dtype=torch.float64).cpu() * total
    row = torch.searchsorted(cdf_r, u).clamp_(max=n * n - 1)
    before = torch.where(row > 0, cdf_r[(row - 1).clamp_(min=0)], torch.zeros_like(u))
    rem = u - before
    col = torch.empty(n_src, dtype=torch.int64)
    step = max(1, (1 << 27) // n)                          # <= 1 GiB of fp64 row copies at a time
    for a in range(0, n_src, step):
        r = row[a:a + step]
        cw = torch.cumsum(w[r.to(dev)].cpu(), 1)           # host, sequential along the row
        col[a:a + step] = torch.searchsorted(cw, rem[a:a + step, None]).squeeze(1).clamp_(max=n - 1)
    del w
    idx = (row * n + col).to(dev)
    k = idx // (n * n)
    j = (idx // n) % n
    i = idx % n
    off = 0.1 + 0.8 * torch.rand((n_src, 3), generator=_gen(seed_pos + 7919, dev), device=dev, dtype=torch.float64)
    pos = torch.stack([i, j, k], 1).double() + off
    gl = torch.randn(n_src, generator=_gen(seed_lum, dev), device=dev, dtype=torch.float64)
    L = mean_L * torch.exp(sigma_ln_L * gl - 0.5 * sigma_ln_L ** 2)
    return pos.cpu(), L.cpu()


def default_params(**kw):
    """Parameters of DESIGN.md's table; names follow the paper's symbols."""
    p = dict(sigma_cm2=SIGMA_HI, n_min_ray=3.0, tau_max=TAU_MAX, level_max=13, n_th=0.0, geom_mode=3,
             e_excess_erg=0.0, merge=0, automerge_xmean=0.018, delta_r=2.0, r_max=8.0, f_ov=1.0, x_th=0.9,
             f_req=0.75, eps=1e-9, n_min_samples=16, samp_level=2)
    p.update(kw)
    return p


def _pack(name, n, dx_cm, nH, xHI, pos, L, params, notes):
    return dict(name=name, n=n, shape=(n, n, n), dx_cm=float(dx_cm), nH=nH, xHI=xHI,
                src_pos=pos, src_L=L, params=params, notes=notes)


def config1(device="cpu", n=32):
    """Stroemgren test (BASELINE.json config 1; Table 1 Test A values)."""
    dx = 6.6 * KPC_CM / n
    nH = torch.full((n, n, n), 1e-3, dtype=torch.float64, device=device)
    xHI = torch.ones((n, n, n), dtype=torch.float64, device=device)
    c = n // 2
    pos = torch.tensor([[c + 0.5, c + 0.5, c + 0.5]], dtype=torch.float64)
    L = torch.tensor([5e48], dtype=torch.float64)
    return _pack("config1_stromgren_%d" % n, n, dx, nH, xHI, pos, L, default_params(e_excess_erg=0.0),
                 "uniform n_H=1e-3, x_HI=1, one source at cell (n/2,n/2,n/2)")


def config2(device="cpu", n=128):
    """Shadow test (BASELINE.json config 2).  Distances scale with n/128 so that small variants keep the
    geometry: clump radius 8, clump centre 40 cells from the source along +x."""
    s = n / 128.0
    dx = 6.6 * KPC_CM / n
    src = (int(round(24 * s)), n // 2, n // 2)
    clump = (src[0] + int(round(40 * s)), n // 2, n // 2)
    rad = 8.0 * s
    ax = torch.arange(n, dtype=torch.float64, device=device)
    d2 = ((ax - clump[0]) ** 2)[None, None, :] + ((ax - clump[1]) ** 2)[None, :, None] + ((ax - clump[2]) ** 2)[:, None, None]
    inside = d2 <= rad * rad
    nH = torch.where(inside, 200 * 2e-4, 2e-4).to(torch.float64)
    xHI = torch.where(inside, 1.0, 1e-3).to(torch.float64)
    pos = torch.tensor([[src[0] + 0.5, src[1] + 0.5, src[2] + 0.5]], dtype=torch.float64)
    L = torch.tensor([3e51], dtype=torch.float64)
    return _pack("config2_shadow_%d" % n, n, dx, nH.contiguous(), xHI.contiguous(), pos, L,
                 default_params(e_excess_erg=1.0e-11),
                 "clump centre %s radius %.1f, source cell %s" % (clump, rad, src))


def _cosmo(n, seed, device, dtype, z_eff):
    """Comoving lognormal n_H (mean 2e-7, sigma_ln 1.5, P(k)~k^-2.5) and the cell width that gives the
    proper optical depth per cell at redshift z_eff: tau = n_com (1+z)^3 sigma dx_com/(1+z), so the
    library is handed dx_cm = dx_com (1+z)^2 (z_eff = 0 is plain comoving)."""
    nH = lognormal_density(n, seed, 2e-7, 1.5, device, dtype)
    dx = BOX_MPC * MPC_CM / n * (1.0 + z_eff) ** 2
    return nH, dx


def config3(device="cpu", n=256, n_src=10_000, z_eff=0.0):
    """Many sources, merging disabled (BASELINE.json config 3)."""
    nH, dx = _cosmo(n, 1, device, torch.float64, z_eff)
    xHI = 0.01 + 0.99 * torch.rand((n, n, n), generator=_gen(1001, device), device=device, dtype=torch.float64)
    pos, L = sample_sources(nH, n_src, 1002, 1003, 1e50, 1.0)
    mean = float(nH.mean())
    return _pack("config3_many_%d" % n, n, dx, nH, xHI, pos, L,
                 default_params(merge=0, n_th=1e-2 * mean, e_excess_erg=1.0e-11),
                 "lognormal n_H seed 1, x_HI~U[0.01,1], %d sources ~ n_H^2, z_eff=%g" % (n_src, z_eff))


def config4(device="cpu", n=512, n_src=100_000, z_eff=7.0, smooth=8.0, r_max=8.0, x_ion=1e-4):
    """Late reionisation with merging (BASELINE.json config 4): x_HI = x_ion except 5 % neutral islands."""
    nH, dx = _cosmo(n, 2, device, torch.float64, z_eff)
    m = smoothed_noise(n, 2001, smooth * n / 512.0, device, torch.float64)
    thr = quantile_hist(m, 0.95)
    xHI = torch.where(m > thr, 1.0, x_ion).to(torch.float64)
    del m
    pos, L = sample_sources(nH, n_src, 2002, 2003, 1e50, 1.0)
    mean = float(nH.mean())
    return _pack("config4_late_%d" % n, n, dx, nH, xHI, pos, L,
                 default_params(merge=1, r_max=r_max, n_th=1e-2 * mean, e_excess_erg=1.0e-11),
                 "lognormal n_H seed 2, 5%% neutral islands (smooth %g), %d sources, z_eff=%g, r_max=%g"
                 % (smooth, n_src, z_eff, r_max))


def config5(device="cpu", n=1024, n_src=1_000_000, z_eff=7.0, smooth=16.0, r_max=8.0, x_ion=1e-4):
    """Production-scale coarse grid (BASELINE.json config 5): f32 fields, 50 % ionised by volume."""
    gen_dtype = torch.float32 if n >= 1024 else torch.float64
    nH, dx = _cosmo(n, 3, device, gen_dtype, z_eff)
    m = smoothed_noise(n, 3001, smooth * n / 1024.0, device, gen_dtype)
    thr = quantile_hist(m, 0.5)
    xHI = torch.where(m > thr, 1.0, x_ion).to(torch.float32)
    del m
    pos, L = sample_sources(nH, n_src, 3002, 3003, 1e50, 1.0)
    nH = nH.to(torch.float32)
    mean = float(nH.double().mean())
    return _pack("config5_prod_%d" % n, n, dx, nH, xHI, pos, L,
                 default_params(merge=1, r_max=r_max, n_th=1e-2 * mean, e_excess_erg=1.0e-11),
                 "lognormal n_H seed 3 (f32), 50%% ionised (smooth %g), %d sources, z_eff=%g, r_max=%g"
                 % (smooth, n_src, z_eff, r_max))


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make(config_id, device="cpu", **kw):
    return CONFIGS[int(config_id)](device=device, **kw)
