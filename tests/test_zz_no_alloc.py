"""nyxrt_finalise_static: the finalise stage for callers that must not allocate device memory.

Some users of this library cannot call cudaMalloc while an RT step runs: inside Nyx the AMReX arena has taken
nearly all of the GPU's memory at start-up (under this binding PyTorch's caching allocator plays the same part), so
an allocation made by the library can fail although the application has free blocks, and cudaMalloc / cudaFree
make every stream of the device wait.  For them the library has ONE entry point that needs no context and no
workspace; its scratch (one partial sum per grid row) is a fixed 8 MiB device array inside libnyxrt.so, shared by
all calls, limited to ny * nz <= NYXRT_STATIC_MAX_ROWS rows.

What is checked here, against the existing path nyxrt_trace_photons -> nyxrt_finalise (which the parity tests tie to
the oracle): two calls in a row, on grids of different shape (the second smaller, so that the scratch still holds
the first call's partials beyond the second call's rows), give Gamma_HI and the heating rate bit for bit and the
absorbed total within the photon-budget tolerance of tests/parity.py (the two paths sum in different fixed orders);
a repeated call gives the same bits; fp32 fields; an oversized grid is refused with a message and nothing is run.
torch's allocator statistics show that the calls themselves allocate nothing through torch either.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (its first call is the first use of the library's static
array on the device) and after the other tests.
"""
import ctypes as C

import pytest
import torch

from paper_2512_12466_b200 import synth
from parity import BUDGET_RTOL

pytestmark = pytest.mark.gpu


def existing_path(cfg, scale=1.0):
    """nyxrt_trace_photons + nyxrt_finalise through a context: (fields, photons, gamma, heat, absorbed)."""
    from paper_2512_12466_b200 import nyxrt
    nH, xHI = cfg["nH"].cuda().contiguous(), cfg["xHI"].cuda().contiguous()
    tr = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], cfg["params"], field_dtype=nH.dtype, max_sources=len(cfg["src_L"]))
    try:
        tr.set_fields(nH, xHI)
        tr.set_sources(cfg["src_pos"].numpy(), cfg["src_L"].numpy())
        photons, _ = tr.trace_photons()
        if scale != 1.0:
            photons = photons * scale            # as if summed over shards: any photon grid is a valid input
        gamma, heat, absorbed = tr.finalise(photons)
        torch.cuda.synchronize()
        return nH, xHI, photons, gamma, heat, absorbed
    finally:
        tr.close()


def static_path(cfg, nH, xHI, photons, out):
    from paper_2512_12466_b200 import nyxrt
    gamma, heat, absorbed = out
    nyxrt.nyxrt_finalise_static(nH, xHI, photons, gamma, cfg["dx_cm"], cfg["params"]["e_excess_erg"], heat, absorbed)


def outputs(shape):
    # filled with a marker so that a cell the kernel skipped would show
    return (torch.full(shape, -7.0, dtype=torch.float64, device="cuda"),
            torch.full(shape, -7.0, dtype=torch.float64, device="cuda"),
            torch.full((1,), -7.0, dtype=torch.float64, device="cuda"))


def check(ref, out):
    _, _, photons, gamma, heat, absorbed = ref
    torch.cuda.synchronize()
    assert torch.equal(out[0], gamma), "Gamma_HI differs from nyxrt_finalise"
    assert torch.equal(out[1], heat), "heating differs from nyxrt_finalise"
    assert bool(((out[0] == 0) == (photons == 0)).all())
    got = float(out[2].item())
    assert absorbed > 0 and abs(got - absorbed) <= BUDGET_RTOL * absorbed, (got, absorbed)
    return got


def test_two_calls_in_a_row_match_the_context_path():
    big = synth.make(4, n=48, n_src=300)
    big["params"]["e_excess_erg"] = 3.2e-12
    small = synth.make(3, n=24, n_src=7)
    small["params"]["e_excess_erg"] = 1.1e-11
    ref_big, ref_small = existing_path(big), existing_path(small, scale=0.37)
    out_big, out_small = outputs(big["shape"]), outputs(small["shape"])
    torch.cuda.synchronize()
    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    static_path(big, *ref_big[:3], out_big)                  # first call: 48 * 48 rows of scratch written
    static_path(small, *ref_small[:3], out_small)            # second call, same stream: 24 * 24 rows, the rest is stale
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == before
    sum_big = check(ref_big, out_big)
    check(ref_small, out_small)
    # a third call on the first inputs: the scratch now holds the small grid's partials; the result has the same bits
    again = outputs(big["shape"])
    static_path(big, *ref_big[:3], again)
    assert check(ref_big, again) == sum_big


def test_fp32_fields_ragged_rows_and_optional_outputs():
    from paper_2512_12466_b200 import nyxrt
    cfg = synth.make(3, n=40, n_src=9)
    cfg["nH"], cfg["xHI"] = cfg["nH"].float(), cfg["xHI"].float()
    cfg["params"]["e_excess_erg"] = 2.0e-12
    ref = existing_path(cfg)
    out = outputs(cfg["shape"])
    static_path(cfg, *ref[:3], out)
    check(ref, out)
    gamma_only = torch.full(cfg["shape"], -7.0, dtype=torch.float64, device="cuda")
    nyxrt.nyxrt_finalise_static(ref[0], ref[1], ref[2], gamma_only, cfg["dx_cm"])      # no heat, no total
    torch.cuda.synchronize()
    assert torch.equal(gamma_only, ref[3])
    # rows of 37 cells (one full warp pass and a tail of 5), 5 x 3 rows: against the formula itself, cell by cell
    g = torch.Generator().manual_seed(12)
    shape = (3, 5, 37)
    nH = (torch.rand(shape, generator=g, dtype=torch.float64) + 0.5).cuda()
    xHI = torch.rand(shape, generator=g, dtype=torch.float64).clamp_min(1e-3).cuda()
    photons = torch.rand(shape, generator=g, dtype=torch.float64).cuda() * 1e40
    photons[photons < 3e39] = 0.0
    out = outputs(shape)
    dx, e = 3.0e22, 1.5e-12
    nyxrt.nyxrt_finalise_static(nH, xHI, photons, out[0], dx, e, out[1], out[2])
    torch.cuda.synchronize()
    V = dx * dx * dx
    assert torch.equal(out[0], torch.where(photons != 0, photons / ((nH * xHI).abs() * V), torch.zeros_like(photons)))
    assert torch.equal(out[1], (e * photons) / torch.full_like(photons, V))    # a tensor divisor: torch divides, IEEE
    total = float(photons.sum().item())
    assert abs(float(out[2].item()) - total) <= BUDGET_RTOL * total


def test_a_grid_beyond_the_scratch_is_refused():
    from paper_2512_12466_b200 import nyxrt
    # 1025 * 1024 rows > NYXRT_STATIC_MAX_ROWS; the size check comes before any pointer is used, so the small
    # tensor passed here with that claimed shape is never read or written
    ny, nz = 1025, 1024
    assert ny * nz > nyxrt.STATIC_MAX_ROWS
    a = torch.ones(8, dtype=torch.float64, device="cuda")
    marker = a.clone()
    err = C.create_string_buffer(256)
    rc = nyxrt.lib().nyxrt_finalise_static(C.c_int32(0), C.c_int32(1), C.c_int32(ny), C.c_int32(nz), C.c_int32(0),
                                           C.c_double(1.0), C.c_double(0.0), C.c_void_p(a.data_ptr()),
                                           C.c_void_p(a.data_ptr()), C.c_void_p(a.data_ptr()), C.c_void_p(a.data_ptr()),
                                           None, None, None, err, C.c_int64(len(err)))
    torch.cuda.synchronize()
    assert rc == nyxrt.ENOMEM and b"NYXRT_STATIC_MAX_ROWS" in err.value and b"1049600" in err.value
    assert torch.equal(a, marker)
    # the largest accepted row count is exactly the maximum: 1024 * 1024 rows of one cell
    n = nyxrt.STATIC_MAX_ROWS
    nH = torch.full((1024, 1024, 1), 2.0, dtype=torch.float64, device="cuda")
    photons = torch.arange(n, dtype=torch.float64, device="cuda").reshape(1024, 1024, 1)
    gamma = torch.empty_like(nH)
    total = torch.zeros(1, dtype=torch.float64, device="cuda")
    nyxrt.nyxrt_finalise_static(nH, nH, photons, gamma, 1.0, 0.0, None, total)
    torch.cuda.synchronize()
    assert float(total.item()) == n * (n - 1) / 2                      # integers below 2^53: exact in any order
    assert torch.equal(gamma, photons / 4.0)
    with pytest.raises(nyxrt.NyxrtError) as ei:
        nyxrt.nyxrt_finalise_static(nH, nH, photons, gamma, -1.0)
    assert ei.value.code == nyxrt.EINVAL and "dx_cm" in str(ei.value)
