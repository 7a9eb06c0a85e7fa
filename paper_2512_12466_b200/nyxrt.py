"""ctypes binding of include/nyxrt.h.  Same names as the C ABI; argument marshalling only.

torch is used for what the task assigns to it: device memory (workspace, fields, outputs) and streams.
"""
import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

MAXLEV = 16
OK, EINVAL, ESTATE, ENOMEM, ECUDA, EOVERFLOW = 0, -1, -2, -3, -4, -5
FLAG_LAUNCH_TIMING = 1
STATIC_MAX_ROWS = 1 << 20      # NYXRT_STATIC_MAX_ROWS: largest ny * nz nyxrt_finalise_static accepts
_ERRNAME = {EINVAL: "NYXRT_EINVAL", ESTATE: "NYXRT_ESTATE", ENOMEM: "NYXRT_ENOMEM", ECUDA: "NYXRT_ECUDA",
            EOVERFLOW: "NYXRT_EOVERFLOW"}


class NyxrtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s (%d): %s" % (_ERRNAME.get(code, "?"), code, msg))
        self.code = code


class nyxrt_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("field_dtype", C.c_int32),
                ("dx_cm", C.c_double), ("box_lo", C.c_double * 3), ("pos_unit_cm", C.c_double),
                ("periodic", C.c_int32), ("device", C.c_int32)]


class nyxrt_params(C.Structure):
    _fields_ = [("sigma_cm2", C.c_double), ("n_min_ray", C.c_double), ("tau_max", C.c_double),
                ("n_th", C.c_double), ("e_excess_erg", C.c_double), ("automerge_xmean", C.c_double),
                ("delta_r", C.c_double), ("r_max", C.c_double), ("f_ov", C.c_double), ("x_th", C.c_double),
                ("f_req", C.c_double), ("eps", C.c_double),
                ("level_max", C.c_int32), ("geom_mode", C.c_int32), ("merge", C.c_int32),
                ("n_min_samples", C.c_int32), ("samp_level", C.c_int32), ("flags", C.c_int32)]


class nyxrt_stats(C.Structure):
    _fields_ = [("spawned", C.c_uint64 * MAXLEV), ("split", C.c_uint64 * MAXLEV),
                ("killed_tau", C.c_uint64 * MAXLEV), ("exited", C.c_uint64 * MAXLEV),
                ("killed_lmax", C.c_uint64 * MAXLEV),
                ("segments", C.c_uint64), ("zero_len_segments", C.c_uint64), ("neighbour_deposits", C.c_uint64),
                ("n_src_in", C.c_uint64), ("n_src_dedup", C.c_uint64), ("n_src_merged", C.c_uint64),
                ("iterations", C.c_uint64), ("peak_pool_rays", C.c_uint64),
                ("photons_emitted", C.c_double), ("photons_absorbed", C.c_double),
                ("photons_escaped", C.c_double), ("photons_residual", C.c_double), ("photons_lost", C.c_double),
                ("march_launches", C.c_uint64), ("kernel_launches", C.c_uint64),
                ("ms_sources", C.c_float), ("ms_loop", C.c_float), ("ms_finalise", C.c_float),
                ("ms_total", C.c_float), ("ms_march", C.c_float), ("pad_", C.c_float)]

    def as_dict(self):
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


class nyxrt_ode(C.Structure):
    _fields_ = [("dt_s", C.c_double), ("alpha_cm3_s", C.c_double), ("coll_cm3_s", C.c_double),
                ("clumping", C.c_double), ("tol_rel", C.c_double), ("tol_abs", C.c_double),
                ("unconv_frac", C.c_double), ("max_iter", C.c_int32), ("inner_iter", C.c_int32)]


class nyxrt_tstats(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("converged", C.c_int32), ("unconverged_cells", C.c_uint64),
                ("segments_total", C.c_uint64), ("kernel_launches", C.c_uint64), ("max_rel_change", C.c_double),
                ("ms_total", C.c_float), ("ms_rt", C.c_float), ("ms_ode", C.c_float), ("pad_", C.c_float)]


EXPORTS = ["nyxrt_create", "nyxrt_workspace_bytes", "nyxrt_set_workspace", "nyxrt_set_fields", "nyxrt_set_sources",
           "nyxrt_trace", "nyxrt_get_catalog", "nyxrt_step_host", "nyxrt_pix2dir", "nyxrt_last_error",
           "nyxrt_destroy", "nyxrt_version", "nyxrt_sizeof_grid", "nyxrt_sizeof_params", "nyxrt_sizeof_stats",
           "nyxrt_timestep", "nyxrt_sizeof_ode", "nyxrt_sizeof_tstats", "nyxrt_set_shard", "nyxrt_trace_photons",
           "nyxrt_finalise", "nyxrt_spectrum_nodes", "nyxrt_spectrum_node_tau", "nyxrt_set_spectrum",
           "nyxrt_blackbody_table", "nyxrt_set_spectrum_thin", "nyxrt_blackbody_thin_table", "nyxrt_finalise_static"]

_lib = None


def lib():
    """Loads libnyxrt.so; raises (never falls back) when it is missing."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path):
            raise ImportError("libnyxrt.so is not built: run `python -m paper_2512_12466_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(path)
        for name in EXPORTS:
            getattr(L, name)
        L.nyxrt_last_error.restype = C.c_char_p
        L.nyxrt_last_error.argtypes = [C.c_void_p]
        L.nyxrt_destroy.restype = None
        L.nyxrt_destroy.argtypes = [C.c_void_p]
        assert L.nyxrt_sizeof_grid() == C.sizeof(nyxrt_grid)
        assert L.nyxrt_sizeof_params() == C.sizeof(nyxrt_params)
        assert L.nyxrt_sizeof_stats() == C.sizeof(nyxrt_stats)
        assert L.nyxrt_sizeof_ode() == C.sizeof(nyxrt_ode)
        assert L.nyxrt_sizeof_tstats() == C.sizeof(nyxrt_tstats)
        _lib = L
    return _lib


def _check(ctx, rc):
    if rc != OK:
        msg = lib().nyxrt_last_error(ctx).decode() if ctx else "no context"
        raise NyxrtError(rc, msg)


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


# ---- the C ABI, one Python function per entry point ---------------------------------------------------

def nyxrt_create(grid, params):
    ctx = C.c_void_p()
    rc = lib().nyxrt_create(C.byref(grid), C.byref(params), C.byref(ctx))
    if rc != OK:
        raise NyxrtError(rc, "nyxrt_create failed (no CUDA device, or bad grid/params)")
    return ctx


def nyxrt_workspace_bytes(ctx, max_sources, batch_rays=0, host_staging=False):
    n = C.c_uint64(0)
    _check(ctx, lib().nyxrt_workspace_bytes(ctx, C.c_int64(max_sources), C.c_int64(batch_rays),
                                            C.c_int32(1 if host_staging else 0), C.byref(n)))
    return n.value


def nyxrt_set_workspace(ctx, workspace, max_sources, batch_rays=0, host_staging=False):
    assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()
    _check(ctx, lib().nyxrt_set_workspace(ctx, C.c_void_p(workspace.data_ptr()), C.c_uint64(workspace.numel()),
                                          C.c_int64(max_sources), C.c_int64(batch_rays),
                                          C.c_int32(1 if host_staging else 0)))


def nyxrt_set_fields(ctx, nH, xHI, stream=None):
    assert nH.is_cuda and xHI.is_cuda and nH.is_contiguous() and xHI.is_contiguous() and nH.dtype == xHI.dtype
    _check(ctx, lib().nyxrt_set_fields(ctx, C.c_void_p(nH.data_ptr()), C.c_void_p(xHI.data_ptr()), _stream_ptr(stream)))


def nyxrt_set_sources(ctx, pos, L, stream=None):
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64).reshape(-1)
    assert len(pos) == len(L)
    _check(ctx, lib().nyxrt_set_sources(ctx, C.c_int64(len(L)), pos.ctypes.data_as(C.c_void_p),
                                        L.ctypes.data_as(C.c_void_p), _stream_ptr(stream)))


def nyxrt_trace(ctx, gamma, heat=None, stream=None):
    assert gamma.is_cuda and gamma.dtype == torch.float64 and gamma.is_contiguous()
    assert heat is None or (heat.is_cuda and heat.dtype == torch.float64 and heat.is_contiguous())
    st = nyxrt_stats()
    _check(ctx, lib().nyxrt_trace(ctx, C.c_void_p(gamma.data_ptr()),
                                  C.c_void_p(heat.data_ptr()) if heat is not None else None,
                                  C.byref(st), _stream_ptr(stream)))
    return st


def nyxrt_spectrum_nodes(e_lo, e_hi, m):
    n = C.c_int64(0)
    rc = lib().nyxrt_spectrum_nodes(C.c_int32(e_lo), C.c_int32(e_hi), C.c_int32(m), C.byref(n))
    if rc != OK:
        raise NyxrtError(rc, "bad table geometry")
    return n.value


def nyxrt_spectrum_node_tau(e_lo, m, k):
    t = C.c_double(0.0)
    rc = lib().nyxrt_spectrum_node_tau(C.c_int32(e_lo), C.c_int32(m), C.c_int64(k), C.byref(t))
    if rc != OK:
        raise NyxrtError(rc, "bad node")
    return t.value


def nyxrt_set_spectrum(ctx, e_lo=0, e_hi=0, m=0, q=None):
    """q: host array of Q at the nodes (None: back to monochromatic)."""
    if q is None:
        _check(ctx, lib().nyxrt_set_spectrum(ctx, 0, 0, 0, None, C.c_int64(0)))
        return
    q = np.ascontiguousarray(q, dtype=np.float64)
    _check(ctx, lib().nyxrt_set_spectrum(ctx, C.c_int32(e_lo), C.c_int32(e_hi), C.c_int32(m),
                                         q.ctypes.data_as(C.c_void_p), C.c_int64(len(q))))


def nyxrt_blackbody_table(t_eff_K, e_lo, e_hi, m):
    n = nyxrt_spectrum_nodes(e_lo, e_hi, m)
    q = np.zeros(n)
    rc = lib().nyxrt_blackbody_table(C.c_double(t_eff_K), C.c_int32(e_lo), C.c_int32(e_hi), C.c_int32(m),
                                     q.ctypes.data_as(C.c_void_p), C.c_int64(n))
    if rc != OK:
        raise NyxrtError(rc, "blackbody_table: bad argument")
    return q


def nyxrt_set_spectrum_thin(ctx, t=None, tau_thin=0.0):
    """t: host array of T = dQ/dtau_0 at the nodes of the Q table (None: thin table off)."""
    if t is None:
        _check(ctx, lib().nyxrt_set_spectrum_thin(ctx, None, C.c_int64(0), C.c_double(0.0)))
        return
    t = np.ascontiguousarray(t, dtype=np.float64)
    _check(ctx, lib().nyxrt_set_spectrum_thin(ctx, t.ctypes.data_as(C.c_void_p), C.c_int64(len(t)), C.c_double(tau_thin)))


def nyxrt_blackbody_thin_table(t_eff_K, e_lo, e_hi, m):
    n = nyxrt_spectrum_nodes(e_lo, e_hi, m)
    t = np.zeros(n)
    rc = lib().nyxrt_blackbody_thin_table(C.c_double(t_eff_K), C.c_int32(e_lo), C.c_int32(e_hi), C.c_int32(m),
                                          t.ctypes.data_as(C.c_void_p), C.c_int64(n))
    if rc != OK:
        raise NyxrtError(rc, "blackbody_thin_table: bad argument")
    return t


def nyxrt_set_shard(ctx, rank, world):
    _check(ctx, lib().nyxrt_set_shard(ctx, C.c_int32(rank), C.c_int32(world)))


def nyxrt_trace_photons(ctx, photons, stream=None):
    assert photons.is_cuda and photons.dtype == torch.float64 and photons.is_contiguous()
    st = nyxrt_stats()
    _check(ctx, lib().nyxrt_trace_photons(ctx, C.c_void_p(photons.data_ptr()), C.byref(st), _stream_ptr(stream)))
    return st


def nyxrt_finalise(ctx, photons, gamma, heat=None, stream=None):
    """Returns the sum of `photons` (absorbed photons per second)."""
    for t in (photons, gamma) + ((heat,) if heat is not None else ()):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    absorbed = C.c_double(0.0)
    _check(ctx, lib().nyxrt_finalise(ctx, C.c_void_p(photons.data_ptr()), C.c_void_p(gamma.data_ptr()),
                                     C.c_void_p(heat.data_ptr()) if heat is not None else None, C.byref(absorbed),
                                     _stream_ptr(stream)))
    return absorbed.value


def nyxrt_finalise_static(nH, xHI, photons, gamma, dx_cm, e_excess_erg=0.0, heat=None, absorbed=None, stream=None):
    """nyxrt_finalise without a context or workspace, for code that must not allocate device memory (the host
    application's arena or torch's caching allocator owns the GPU, and cudaMalloc stalls every stream): the scratch
    is a fixed 8 MiB array inside the library, so grids are limited to ny * nz <= STATIC_MAX_ROWS rows and calls that
    overlap on one GPU race on it.  All tensors are the caller's CUDA tensors of shape [nz][ny][nx]; `absorbed` is a
    1-element fp64 CUDA tensor that receives the sum of `photons` (or None).  Enqueues on `stream`, does not
    synchronise.  This wrapper only marshals: it creates no tensor."""
    for t in (photons, gamma) + tuple(x for x in (heat, absorbed) if x is not None):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    assert nH.is_cuda and xHI.is_cuda and nH.is_contiguous() and xHI.is_contiguous() and nH.dtype == xHI.dtype
    assert nH.dtype in (torch.float32, torch.float64) and nH.dim() == 3
    assert nH.shape == xHI.shape == photons.shape == gamma.shape and (heat is None or heat.shape == nH.shape)
    nz, ny, nx = nH.shape
    err = C.create_string_buffer(256)
    rc = lib().nyxrt_finalise_static(
        C.c_int32(nH.device.index or 0), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
        C.c_int32(1 if nH.dtype == torch.float32 else 0), C.c_double(dx_cm), C.c_double(e_excess_erg),
        C.c_void_p(nH.data_ptr()), C.c_void_p(xHI.data_ptr()), C.c_void_p(photons.data_ptr()),
        C.c_void_p(gamma.data_ptr()), C.c_void_p(heat.data_ptr()) if heat is not None else None,
        C.c_void_p(absorbed.data_ptr()) if absorbed is not None else None, _stream_ptr(stream), err, C.c_int64(len(err)))
    if rc != OK:
        raise NyxrtError(rc, err.value.decode())


def nyxrt_timestep(ctx, ode, nH, xHI_begin, xHI_end, xHI_avg, gamma, heat=None, stream=None):
    """One RT timestep; all arrays are CUDA tensors (xHI_begin / xHI_end / gamma / heat fp64, nH / xHI_avg of the
    field dtype).  Returns (stats of the last ray trace, timestep stats)."""
    for t in (nH, xHI_begin, xHI_end, xHI_avg, gamma) + ((heat,) if heat is not None else ()):
        assert t.is_cuda and t.is_contiguous()
    assert xHI_begin.dtype == xHI_end.dtype == gamma.dtype == torch.float64 and nH.dtype == xHI_avg.dtype
    st, ts = nyxrt_stats(), nyxrt_tstats()
    _check(ctx, lib().nyxrt_timestep(ctx, C.byref(ode), C.c_void_p(nH.data_ptr()), C.c_void_p(xHI_begin.data_ptr()),
                                     C.c_void_p(xHI_end.data_ptr()), C.c_void_p(xHI_avg.data_ptr()),
                                     C.c_void_p(gamma.data_ptr()),
                                     C.c_void_p(heat.data_ptr()) if heat is not None else None,
                                     C.byref(st), C.byref(ts), _stream_ptr(stream)))
    return st, ts


def nyxrt_get_catalog(ctx):
    n = C.c_int64(0)
    _check(ctx, lib().nyxrt_get_catalog(ctx, C.c_int64(0), None, None, None, C.byref(n)))
    m = n.value
    cell = np.zeros((m, 3), np.int32)
    L = np.zeros(m)
    r = np.zeros(m)
    if m:
        _check(ctx, lib().nyxrt_get_catalog(ctx, C.c_int64(m), cell.ctypes.data_as(C.c_void_p),
                                            L.ctypes.data_as(C.c_void_p), r.ctypes.data_as(C.c_void_p), C.byref(n)))
    return cell, L, r


def nyxrt_step_host(ctx, nH, xHI, pos, L, gamma, heat=None):
    """Host buffers in, host buffers out (torch CPU tensors or numpy arrays; pinned memory is fastest)."""
    def hp(a):
        return C.c_void_p(a.data_ptr()) if isinstance(a, torch.Tensor) else a.ctypes.data_as(C.c_void_p)
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64).reshape(-1)
    st = nyxrt_stats()
    _check(ctx, lib().nyxrt_step_host(ctx, hp(nH), hp(xHI), C.c_int64(len(L)), pos.ctypes.data_as(C.c_void_p),
                                      L.ctypes.data_as(C.c_void_p), hp(gamma), hp(heat) if heat is not None else None,
                                      C.byref(st)))
    return st


def nyxrt_pix2dir(ctx, level, pix_begin, n):
    out = np.zeros((n, 3))
    _check(ctx, lib().nyxrt_pix2dir(ctx, C.c_int32(level), C.c_int64(pix_begin), C.c_int64(n),
                                    out.ctypes.data_as(C.c_void_p)))
    return out


def nyxrt_destroy(ctx):
    lib().nyxrt_destroy(ctx)


# ---- small convenience wrapper used by tests / bench (still marshalling only) --------------------------

def make_grid(shape_zyx, dx_cm, field_dtype=torch.float64, box_lo=(0.0, 0.0, 0.0), pos_unit_cm=None, device=0,
              periodic=0):
    g = nyxrt_grid()
    g.nz, g.ny, g.nx = [int(v) for v in shape_zyx]
    g.field_dtype = 1 if field_dtype == torch.float32 else 0
    g.dx_cm = float(dx_cm)
    g.box_lo[:] = [float(v) for v in box_lo]
    g.pos_unit_cm = float(dx_cm if pos_unit_cm is None else pos_unit_cm)
    g.periodic = int(periodic)
    g.device = int(device)
    return g


def make_ode(dt_s, **kw):
    """Defaults: DESIGN.md "Parameters" (alpha_B(1e4 K) = 2.59e-13 cm^3/s)."""
    d = dict(alpha_cm3_s=2.59e-13, coll_cm3_s=0.0, clumping=1.0, tol_rel=1e-2, tol_abs=1e-5, unconv_frac=1e-4,
             max_iter=30, inner_iter=8)
    d.update(kw)
    o = nyxrt_ode()
    o.dt_s = float(dt_s)
    for k, v in d.items():
        setattr(o, k, v)
    return o


def make_params(**kw):
    p = nyxrt_params()
    for k, v in kw.items():
        setattr(p, k, v)
    return p


class Tracer:
    """Owns a context and its torch-allocated workspace."""

    def __init__(self, shape_zyx, dx_cm, params, field_dtype=torch.float64, max_sources=1, batch_rays=0,
                 host_staging=False, device=0, periodic=0):
        if not torch.cuda.is_available():
            raise RuntimeError("nyxrt needs a CUDA device; there is no CPU fallback")
        self.grid = make_grid(shape_zyx, dx_cm, field_dtype, device=device, periodic=periodic)
        self.params = make_params(**params)
        self.shape = tuple(int(v) for v in shape_zyx)
        self.device = torch.device("cuda", device)
        self.ctx = nyxrt_create(self.grid, self.params)
        self.max_sources = max(int(max_sources), 1)
        nbytes = nyxrt_workspace_bytes(self.ctx, self.max_sources, batch_rays, host_staging)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        nyxrt_set_workspace(self.ctx, self.workspace, self.max_sources, batch_rays, host_staging)

    def set_fields(self, nH, xHI, stream=None):
        self._fields = (nH, xHI)            # keep the borrowed tensors alive
        nyxrt_set_fields(self.ctx, nH, xHI, stream)

    def set_sources(self, pos, L, stream=None):
        nyxrt_set_sources(self.ctx, pos, L, stream)

    def trace(self, gamma=None, heat=None, want_heat=True, stream=None):
        if gamma is None:
            gamma = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        if heat is None and want_heat:
            heat = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        st = nyxrt_trace(self.ctx, gamma, heat, stream)
        return gamma, heat, st

    def timestep(self, ode, nH, xHI_begin, want_heat=True, stream=None):
        """Returns (xHI_end, xHI_avg, gamma, heat, stats, tstats); the sources must have been set."""
        xe = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        xa = torch.empty(self.shape, dtype=nH.dtype, device=self.device)
        gamma = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        heat = torch.empty(self.shape, dtype=torch.float64, device=self.device) if want_heat else None
        self._fields = (nH, xa)
        st, ts = nyxrt_timestep(self.ctx, ode, nH, xHI_begin, xe, xa, gamma, heat, stream)
        return xe, xa, gamma, heat, st, ts

    def set_spectrum(self, e_lo=0, e_hi=0, m=0, q=None):
        nyxrt_set_spectrum(self.ctx, e_lo, e_hi, m, q)

    def set_spectrum_thin(self, t=None, tau_thin=0.0):
        nyxrt_set_spectrum_thin(self.ctx, t, tau_thin)

    def set_shard(self, rank, world):
        nyxrt_set_shard(self.ctx, rank, world)

    def trace_photons(self, photons=None, stream=None):
        if photons is None:
            photons = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        return photons, nyxrt_trace_photons(self.ctx, photons, stream)

    def finalise(self, photons, want_heat=True, stream=None):
        gamma = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        heat = torch.empty(self.shape, dtype=torch.float64, device=self.device) if want_heat else None
        absorbed = nyxrt_finalise(self.ctx, photons, gamma, heat, stream)
        return gamma, heat, absorbed

    def sharded_trace(self, group=None, want_heat=True, stream=None):
        """One RT step sharded by source over the ranks of a torch.distributed group (NCCL): this rank's shard
        must have been set with set_shard(rank, world).  One all-reduce of the per-cell photon counts."""
        import torch.distributed as dist
        photons, st = self.trace_photons(stream=stream)
        if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
            dist.all_reduce(photons, op=dist.ReduceOp.SUM, group=group)
        gamma, heat, absorbed = self.finalise(photons, want_heat, stream)
        return gamma, heat, st, absorbed

    def catalog(self):
        return nyxrt_get_catalog(self.ctx)

    def step_host(self, nH, xHI, pos, L, gamma, heat=None):
        return nyxrt_step_host(self.ctx, nH, xHI, pos, L, gamma, heat)

    def pix2dir(self, level, pix_begin, n):
        return nyxrt_pix2dir(self.ctx, level, pix_begin, n)

    def close(self):
        if self.ctx is not None:
            nyxrt_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
