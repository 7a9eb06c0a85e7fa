"""Shared helper of the GPU parity tests: run the CUDA library (through the C ABI binding) and the CPU
oracle on the same seeded inputs and compare them by BASELINE.json's rule:
  - every per-level ray counter, `segments`, `zero_len_segments` and the catalogue: exactly equal;
  - per cell |Gamma_gpu - Gamma_or| <= 1e-9 |Gamma_or| + 1e-30 s^-1, heating likewise (floor scaled by
    e_excess n_HI); only the summation order of the fp64 deposits differs;
  - photon budget emitted = absorbed + escaped + residual (+ lost) to 1e-12 relative on both sides.
"""
import numpy as np
import torch

RTOL = 1e-9          # north_star: "within 1e-9 relative"
ATOL = 1e-30         # "with an absolute floor of 1e-30 s^-1"
BUDGET_RTOL = 1e-12  # "emitted = absorbed + escaped, to 1e-12 relative"

COUNTERS = ["spawned", "split", "killed_tau", "exited", "killed_lmax"]


def oracle_inputs(cfg):
    nH = cfg["nH"].cpu().numpy()
    xHI = cfg["xHI"].cpu().numpy()
    return nH, xHI, cfg["src_pos"].numpy(), cfg["src_L"].numpy()


def run_oracle(O, cfg, params=None, periodic=0):
    p = dict(cfg["params"])
    p.update(params or {})
    nH, xHI, pos, L = oracle_inputs(cfg)
    g = O.make_grid(cfg["shape"], cfg["dx_cm"], field_dtype=nH.dtype, periodic=periodic)
    return O.step(g, O.make_params(**p), nH, xHI, pos, L)


def run_gpu(cfg, params=None, batch_rays=0, want_heat=True, host=False, periodic=0):
    from paper_2512_12466_b200 import nyxrt
    p = dict(cfg["params"])
    p.update(params or {})
    nH = cfg["nH"].cuda().contiguous()
    xHI = cfg["xHI"].cuda().contiguous()
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], p, field_dtype=nH.dtype, max_sources=len(L),
                      batch_rays=batch_rays, host_staging=host, periodic=periodic)
    try:
        if host:
            gam = torch.empty(cfg["shape"], dtype=torch.float64).pin_memory()
            heat = torch.empty(cfg["shape"], dtype=torch.float64).pin_memory() if want_heat else None
            st = tr.step_host(cfg["nH"].cpu().contiguous(), cfg["xHI"].cpu().contiguous(), pos, L, gam, heat)
            cat = tr.catalog()
            return gam.numpy(), (heat.numpy() if want_heat else None), st, cat
        tr.set_fields(nH, xHI)
        tr.set_sources(pos, L)
        gam, heat, st = tr.trace(want_heat=want_heat)
        cat = tr.catalog()
        torch.cuda.synchronize()
        return gam.cpu().numpy(), (heat.cpu().numpy() if want_heat else None), st, cat
    finally:
        tr.close()


def assert_budget(st, what):
    em = st.photons_emitted
    tot = st.photons_absorbed + st.photons_escaped + st.photons_residual + st.photons_lost
    assert abs(tot - em) <= BUDGET_RTOL * em, (what, em, tot, (tot - em) / max(em, 1e-300))


def compare(res_gpu, res_or, cfg, params=None):
    gg, hg, sg, cg = res_gpu
    go, ho, so, co = res_or
    p = dict(cfg["params"])
    p.update(params or {})
    # catalogue: cells exact, L and r to 1e-15 (they are computed by the same sequential sums: equal)
    assert cg[0].shape == co[0].shape and np.array_equal(cg[0], co[0])
    assert np.array_equal(cg[1], co[1]) and np.array_equal(cg[2], co[2])
    for f in ("n_src_in", "n_src_dedup", "n_src_merged"):
        assert getattr(sg, f) == getattr(so, f), f
    # ray counts per HEALPix level: exact
    for name in COUNTERS:
        assert list(getattr(sg, name)) == list(getattr(so, name)), (name, list(getattr(sg, name)), list(getattr(so, name)))
    assert sg.segments == so.segments and sg.zero_len_segments == so.zero_len_segments
    assert sg.neighbour_deposits == so.neighbour_deposits
    # rates
    err = np.abs(gg - go)
    bad = err > RTOL * np.abs(go) + ATOL
    assert not bad.any(), ("Gamma", int(bad.sum()), float((err / np.maximum(np.abs(go), 1e-300)).max()))
    assert np.array_equal(gg == 0.0, go == 0.0)
    if hg is not None and ho is not None:
        nHI = (cfg["nH"].cpu().numpy().astype(np.float64)) * (cfg["xHI"].cpu().numpy().astype(np.float64))
        floor = ATOL * p["e_excess_erg"] * nHI
        errh = np.abs(hg - ho)
        assert not (errh > RTOL * np.abs(ho) + floor).any(), "heat"
    assert_budget(sg, "gpu")
    assert_budget(so, "oracle")
    for f in ("photons_emitted", "photons_absorbed", "photons_escaped", "photons_residual", "photons_lost"):
        a, b = getattr(sg, f), getattr(so, f)
        assert abs(a - b) <= 1e-11 * max(abs(b), 1e-300) + 1e-11 * so.photons_emitted * (f != "photons_emitted"), (f, a, b)
    rel = err / np.maximum(np.abs(go), 1e-300)
    return float(rel[go != 0].max()) if (go != 0).any() else 0.0


def compare_slabs(gam_gpu, heat_gpu, go, ho, cfg, params=None, slab=32):
    """The per-cell rule of `compare` for a grid too large to hold several host copies of: the GPU result
    stays on the device, the oracle's arrays (numpy) are brought over z-slab by z-slab."""
    p = dict(cfg["params"])
    p.update(params or {})
    worst = 0.0
    nz = gam_gpu.shape[0]
    for z0 in range(0, nz, slab):
        z1 = min(nz, z0 + slab)
        o = torch.from_numpy(go[z0:z1]).to(gam_gpu.device)
        g = gam_gpu[z0:z1]
        err = (g - o).abs()
        assert not bool((err > RTOL * o.abs() + ATOL).any()), ("Gamma", z0)
        assert bool(((g == 0) == (o == 0)).all()), ("Gamma zero pattern", z0)
        nz_mask = o != 0
        if bool(nz_mask.any()):
            worst = max(worst, float((err[nz_mask] / o[nz_mask].abs()).max()))
        if heat_gpu is not None and ho is not None:
            h = torch.from_numpy(ho[z0:z1]).to(gam_gpu.device)
            nHI = cfg["nH"][z0:z1].double() * cfg["xHI"][z0:z1].double()
            floor = ATOL * p["e_excess_erg"] * nHI
            assert not bool(((heat_gpu[z0:z1] - h).abs() > RTOL * h.abs() + floor).any()), ("heat", z0)
    return worst


# ---- the oracle on P host cores (SURVEY.md 8(d) "Oracle timed beside it"): oracle/oracle.py step_parallel ---------------

def run_oracle_parallel(O, cfg, n_proc, params=None, periodic=0, want_heat=True, chunk=4):
    """Returns (OracleSum, catalogue).  The caller must close() the OracleSum (shared memory)."""
    p = dict(cfg["params"])
    p.update(params or {})
    nH, xHI, pos, L = oracle_inputs(cfg)
    g = O.make_grid(cfg["shape"], cfg["dx_cm"], field_dtype=nH.dtype, periodic=periodic)
    return O.step_parallel(g, O.make_params(**p), nH, xHI, pos, L, n_proc, want_heat=want_heat, chunk=chunk)


def compare_slabs_sum(gam_gpu, heat_gpu, osum, cfg, params=None, slab=32):
    """`compare_slabs` against the sum of the workers' partial grids, z-slab by z-slab."""
    p = dict(cfg["params"])
    p.update(params or {})
    worst = 0.0
    nz = gam_gpu.shape[0]
    for z0 in range(0, nz, slab):
        z1 = min(nz, z0 + slab)
        o = torch.from_numpy(osum.gamma(z0, z1)).to(gam_gpu.device)
        g = gam_gpu[z0:z1]
        err = (g - o).abs()
        assert not bool((err > RTOL * o.abs() + ATOL).any()), ("Gamma", z0)
        assert bool(((g == 0) == (o == 0)).all()), ("Gamma zero pattern", z0)
        nz_mask = o != 0
        if bool(nz_mask.any()):
            worst = max(worst, float((err[nz_mask] / o[nz_mask].abs()).max()))
        ho = osum.heat(z0, z1)
        if heat_gpu is not None and ho is not None:
            h = torch.from_numpy(ho).to(gam_gpu.device)
            nHI = cfg["nH"][z0:z1].double().to(gam_gpu.device) * cfg["xHI"][z0:z1].double().to(gam_gpu.device)
            floor = ATOL * p["e_excess_erg"] * nHI
            assert not bool(((heat_gpu[z0:z1] - h).abs() > RTOL * h.abs() + floor).any()), ("heat", z0)
    return worst
