"""ctypes front end of the CPU oracle (oracle/nyxrt_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports the product package, and the product package never imports it.
Everything here is argument marshalling; the arithmetic is in nyxrt_oracle.c, which cites the paper.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nyxrt_oracle.c")
_LIB = os.path.join(_HERE, "libnyxrt_oracle.so")
MAXLEV = 16


def build(force=False):
    """gcc -O2 -ffp-contract=off (no fast-math): decisions must not be contracted (DESIGN.md DEC)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-Wall",
                               "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("field_dtype", C.c_int32),
                ("dx_cm", C.c_double), ("box_lo", C.c_double * 3), ("pos_unit_cm", C.c_double),
                ("periodic", C.c_int32), ("pad_", C.c_int32)]


class Params(C.Structure):
    _fields_ = [("sigma_cm2", C.c_double), ("n_min_ray", C.c_double), ("tau_max", C.c_double),
                ("n_th", C.c_double), ("e_excess_erg", C.c_double), ("automerge_xmean", C.c_double),
                ("delta_r", C.c_double), ("r_max", C.c_double), ("f_ov", C.c_double), ("x_th", C.c_double),
                ("f_req", C.c_double), ("eps", C.c_double),
                ("level_max", C.c_int32), ("geom_mode", C.c_int32), ("merge", C.c_int32),
                ("n_min_samples", C.c_int32), ("samp_level", C.c_int32), ("pad_", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("spawned", C.c_uint64 * MAXLEV), ("split", C.c_uint64 * MAXLEV),
                ("killed_tau", C.c_uint64 * MAXLEV), ("exited", C.c_uint64 * MAXLEV),
                ("killed_lmax", C.c_uint64 * MAXLEV),
                ("segments", C.c_uint64), ("zero_len_segments", C.c_uint64), ("neighbour_deposits", C.c_uint64),
                ("n_src_in", C.c_uint64), ("n_src_dedup", C.c_uint64), ("n_src_merged", C.c_uint64),
                ("photons_emitted", C.c_double), ("photons_absorbed", C.c_double),
                ("photons_escaped", C.c_double), ("photons_residual", C.c_double),
                ("photons_lost", C.c_double)]

    def as_dict(self):
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


SEG_DTYPE = np.dtype([("src", "<i4"), ("level", "<i4"), ("pix", "<i8"), ("cell", "<i4", (3,)),
                      ("nb_face", "<i4"), ("s0", "<f8"), ("ds", "<f8"), ("dtau", "<f8"), ("dN", "<f8"),
                      ("fc", "<f8"), ("d_edge", "<f8"), ("l_pix", "<f8")], align=True)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_mean_ionised.restype = C.c_double
        assert _lib.orc_sizeof_stats() == C.sizeof(Stats)
        assert _lib.orc_sizeof_seg() == SEG_DTYPE.itemsize, (_lib.orc_sizeof_seg(), SEG_DTYPE.itemsize)
    return _lib


def make_grid(shape_zyx, dx_cm, field_dtype=np.float64, box_lo=(0.0, 0.0, 0.0), pos_unit_cm=None, periodic=0):
    g = Grid()
    g.periodic = int(periodic)
    g.nz, g.ny, g.nx = [int(v) for v in shape_zyx]
    g.field_dtype = 1 if np.dtype(field_dtype) == np.float32 else 0
    g.dx_cm = float(dx_cm)
    g.box_lo[:] = [float(v) for v in box_lo]
    g.pos_unit_cm = float(dx_cm if pos_unit_cm is None else pos_unit_cm)   # default: positions in cells
    return g


def make_params(**kw):
    """Field names follow the paper's symbols; defaults are DESIGN.md's table of parameters."""
    d = dict(sigma_cm2=6.3e-18, n_min_ray=3.0, tau_max=float(np.log(1e8)), n_th=0.0, e_excess_erg=0.0,
             automerge_xmean=0.018, delta_r=2.0, r_max=8.0, f_ov=1.0, x_th=0.9, f_req=0.75, eps=1e-9,
             level_max=13, geom_mode=3, merge=0, n_min_samples=16, samp_level=2)
    d.update(kw)
    p = Params()
    for k, v in d.items():
        setattr(p, k, v)
    return p


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("oracle %s failed with code %d" % (what, rc))


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def pix2dir(level, pix):
    out = np.zeros(3)
    _chk(lib().orc_pix2dir(C.c_int(level), C.c_int64(int(pix)), _ptr(out)), "pix2dir")
    return out


def pix2dir_all(level):
    n = 12 * 4 ** level
    out = np.zeros((n, 3))
    f = lib().orc_pix2dir
    for p in range(n):
        f(C.c_int(level), C.c_int64(p), C.c_void_p(out.ctypes.data + 24 * p))
    return out


def prepare_sources(g, pos, L):
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64)
    n = len(L)
    cell = np.zeros((max(n, 1), 3), np.int32)
    Lo = np.zeros(max(n, 1))
    nout = C.c_int64(0)
    _chk(lib().orc_prepare_sources(C.byref(g), C.c_int64(n), _ptr(pos), _ptr(L), _ptr(cell), _ptr(Lo),
                                   C.byref(nout)), "prepare_sources")
    return cell[:nout.value].copy(), Lo[:nout.value].copy()


def _field(g, a):
    want = np.float32 if g.field_dtype else np.float64
    a = np.ascontiguousarray(a)
    assert a.dtype == want, (a.dtype, want)
    assert a.shape == (g.nz, g.ny, g.nx), (a.shape, (g.nz, g.ny, g.nx))
    return a


def bubble_radius(g, p, xHI, cell):
    xHI = _field(g, xHI)
    cell = np.ascontiguousarray(cell, np.int32).reshape(-1, 3)
    r = np.zeros(len(cell))
    _chk(lib().orc_bubble_radius(C.byref(g), C.byref(p), _ptr(xHI), C.c_int64(len(cell)), _ptr(cell), _ptr(r)),
         "bubble_radius")
    return r


def merge(g, p, cell, L, r):
    cell = np.ascontiguousarray(cell, np.int32).reshape(-1, 3)
    L = np.ascontiguousarray(L, np.float64)
    r = np.ascontiguousarray(r, np.float64)
    n = len(L)
    oc = np.zeros((max(n, 1), 3), np.int32)
    oL = np.zeros(max(n, 1))
    orr = np.zeros(max(n, 1))
    nout = C.c_int64(0)
    _chk(lib().orc_merge(C.byref(g), C.byref(p), C.c_int64(n), _ptr(cell), _ptr(L), _ptr(r), _ptr(oc), _ptr(oL),
                         _ptr(orr), C.byref(nout)), "merge")
    m = nout.value
    return oc[:m].copy(), oL[:m].copy(), orr[:m].copy()


def trace(g, p, nH, xHI, cell, L, want_heat=True, log_cap=0):
    """Returns (gamma, heat, stats[, seglog])."""
    nH = _field(g, nH)
    xHI = _field(g, xHI)
    cell = np.ascontiguousarray(cell, np.int32).reshape(-1, 3)
    L = np.ascontiguousarray(L, np.float64)
    gamma = np.zeros((g.nz, g.ny, g.nx))
    heat = np.zeros((g.nz, g.ny, g.nx)) if want_heat else None
    st = Stats()
    log = np.zeros(log_cap, SEG_DTYPE) if log_cap else None
    nlog = C.c_int64(0)
    _chk(lib().orc_trace(C.byref(g), C.byref(p), _ptr(nH), _ptr(xHI), C.c_int64(len(L)), _ptr(cell), _ptr(L),
                         _ptr(gamma), _ptr(heat) if want_heat else None, C.byref(st),
                         _ptr(log) if log_cap else None, C.c_int64(log_cap), C.byref(nlog)), "trace")
    if log_cap:
        if nlog.value > log_cap:
            raise RuntimeError("segment log overflow: %d > %d" % (nlog.value, log_cap))
        return gamma, heat, st, log[:nlog.value]
    return gamma, heat, st


def step(g, p, nH, xHI, pos, L, want_heat=True):
    """The whole RT step.  Returns (gamma, heat, stats, (cat_cell, cat_L, cat_r))."""
    nH = _field(g, nH)
    xHI = _field(g, xHI)
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64)
    n = len(L)
    gamma = np.zeros((g.nz, g.ny, g.nx))
    heat = np.zeros((g.nz, g.ny, g.nx)) if want_heat else None
    st = Stats()
    cc = np.zeros((max(n, 1), 3), np.int32)
    cL = np.zeros(max(n, 1))
    cr = np.zeros(max(n, 1))
    ncat = C.c_int64(0)
    _chk(lib().orc_step(C.byref(g), C.byref(p), _ptr(nH), _ptr(xHI), C.c_int64(n), _ptr(pos), _ptr(L),
                        _ptr(gamma), _ptr(heat) if want_heat else None, C.byref(st), _ptr(cc), _ptr(cL), _ptr(cr),
                        C.byref(ncat)), "step")
    m = ncat.value
    return gamma, heat, st, (cc[:m].copy(), cL[:m].copy(), cr[:m].copy())


def catalogue(g, p, xHI, pos, L):
    """The source pass alone (dedup + sort, bubble radii + merge when merging is on).
    Returns (stats with the n_src_* fields, (cat_cell, cat_L, cat_r))."""
    xHI = _field(g, xHI)
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64)
    n = len(L)
    st = Stats()
    cc = np.zeros((max(n, 1), 3), np.int32)
    cL = np.zeros(max(n, 1))
    cr = np.zeros(max(n, 1))
    ncat = C.c_int64(0)
    _chk(lib().orc_catalogue(C.byref(g), C.byref(p), _ptr(xHI), C.c_int64(n), _ptr(pos), _ptr(L), C.byref(st),
                             _ptr(cc), _ptr(cL), _ptr(cr), C.byref(ncat)), "catalogue")
    m = ncat.value
    return st, (cc[:m].copy(), cL[:m].copy(), cr[:m].copy())


def trace_add(g, p, nH, xHI, cell, L, gamma, heat, st):
    """orc_trace of a slice of the catalogue, ADDED to gamma / heat (numpy fp64 grids; heat may be None) and to
    the counters of st.  nH / xHI must already have the grid's dtype and shape (no copy is made)."""
    cell = np.ascontiguousarray(cell, np.int32).reshape(-1, 3)
    L = np.ascontiguousarray(L, np.float64)
    _chk(lib().orc_trace_add(C.byref(g), C.byref(p), _ptr(nH), _ptr(xHI), C.c_int64(len(L)), _ptr(cell), _ptr(L),
                             _ptr(gamma), _ptr(heat) if heat is not None else None, C.byref(st)), "trace_add")


def mean_ionised(g, xHI):
    return lib().orc_mean_ionised(C.byref(g), _ptr(_field(g, xHI)))


# ---- RT timestep: time integration + iterative solve (following [23]) ---------------

class Ode(C.Structure):
    _fields_ = [("dt_s", C.c_double), ("alpha_cm3_s", C.c_double), ("coll_cm3_s", C.c_double),
                ("clumping", C.c_double), ("tol_rel", C.c_double), ("tol_abs", C.c_double),
                ("unconv_frac", C.c_double),
                ("max_iter", C.c_int32), ("inner_iter", C.c_int32)]


class TStats(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("converged", C.c_int32), ("unconverged_cells", C.c_uint64),
                ("segments_total", C.c_uint64), ("max_rel_change", C.c_double)]


def make_ode(dt_s, **kw):
    """Defaults: DESIGN.md "Parameters" (alpha_B(1e4 K) = 2.59e-13)."""
    d = dict(alpha_cm3_s=2.59e-13, coll_cm3_s=0.0, clumping=1.0, tol_rel=1e-2, tol_abs=1e-5, unconv_frac=1e-4,
             max_iter=30, inner_iter=8)
    d.update(kw)
    o = Ode()
    o.dt_s = float(dt_s)
    for k, v in d.items():
        setattr(o, k, v)
    assert lib().orc_sizeof_ode() == C.sizeof(Ode) and lib().orc_sizeof_tstats() == C.sizeof(TStats)
    return o


def ode_cell(o, gamma, nH, y0, yavg):
    """One cell of T2.  Returns (y_avg, y_end)."""
    ya, ye = C.c_double(yavg), C.c_double(0.0)
    f = lib().orc_ode_cell
    f.restype = None
    f(C.byref(o), C.c_double(gamma), C.c_double(nH), C.c_double(y0), C.byref(ya), C.byref(ye))
    return ya.value, ye.value


def timestep(g, p, o, nH, xHI_begin, pos, L, want_heat=True):
    """One RT timestep.  Returns (xHI_end f64, xHI_avg field dtype, gamma, heat, stats, tstats, catalogue)."""
    nH = _field(g, nH)
    xb = np.ascontiguousarray(xHI_begin, dtype=np.float64)
    assert xb.shape == (g.nz, g.ny, g.nx)
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    L = np.ascontiguousarray(L, dtype=np.float64)
    n = len(L)
    shape = (g.nz, g.ny, g.nx)
    xe = np.zeros(shape)
    xa = np.zeros(shape, np.float32 if g.field_dtype else np.float64)
    gamma = np.zeros(shape)
    heat = np.zeros(shape) if want_heat else None
    st, ts = Stats(), TStats()
    cc = np.zeros((max(n, 1), 3), np.int32)
    cL = np.zeros(max(n, 1))
    cr = np.zeros(max(n, 1))
    ncat = C.c_int64(0)
    _chk(lib().orc_timestep(C.byref(g), C.byref(p), C.byref(o), _ptr(nH), _ptr(xb), C.c_int64(n), _ptr(pos), _ptr(L),
                            _ptr(xe), _ptr(xa), _ptr(gamma), _ptr(heat) if want_heat else None, C.byref(st),
                            C.byref(ts), _ptr(cc), _ptr(cL), _ptr(cr), C.byref(ncat)), "timestep")
    m = ncat.value
    return xe, xa, gamma, heat, st, ts, (cc[:m].copy(), cL[:m].copy(), cr[:m].copy())


# ---- frequency-integrated flux: the tau_0 lookup table of PAPER.md:95 -------------------------------------

def spectrum_nodes(e_lo, e_hi, m):
    f = lib().orc_spectrum_nodes
    f.restype = C.c_int64
    return f(C.c_int(e_lo), C.c_int(e_hi), C.c_int(m))


def spectrum_node_tau(e_lo, m, k):
    f = lib().orc_spectrum_node_tau
    f.restype = C.c_double
    return f(C.c_int(e_lo), C.c_int(m), C.c_int64(k))


def set_spectrum(e_lo=0, e_hi=0, m=0, q=None):
    """q = None: monochromatic (the default).  The table is copied; it is module state of the oracle."""
    if q is None:
        _chk(lib().orc_set_spectrum(0, 0, 0, None, C.c_int64(0)), "set_spectrum")
        return
    q = np.ascontiguousarray(q, dtype=np.float64)
    _chk(lib().orc_set_spectrum(C.c_int(e_lo), C.c_int(e_hi), C.c_int(m), _ptr(q), C.c_int64(len(q))), "set_spectrum")


def set_spectrum_thin(t=None, tau_thin=0.0):
    """The separate table for thin segments (PAPER.md:267 footnote 3), on the nodes of the table set with
    set_spectrum; t = None: off."""
    if t is None:
        _chk(lib().orc_set_spectrum_thin(None, C.c_int64(0), C.c_double(0.0)), "set_spectrum_thin")
        return
    t = np.ascontiguousarray(t, dtype=np.float64)
    _chk(lib().orc_set_spectrum_thin(_ptr(t), C.c_int64(len(t)), C.c_double(tau_thin)), "set_spectrum_thin")


def spectrum_t(tau):
    f = lib().orc_spectrum_t
    f.restype = C.c_double
    return f(C.c_double(tau))


def blackbody_thin_table(t_eff_K, e_lo, e_hi, m):
    n = spectrum_nodes(e_lo, e_hi, m)
    t = np.zeros(n)
    _chk(lib().orc_blackbody_thin_table(C.c_double(t_eff_K), C.c_int(e_lo), C.c_int(e_hi), C.c_int(m), _ptr(t),
                                        C.c_int64(n)), "blackbody_thin_table")
    return t


def spectrum_q(tau):
    f = lib().orc_spectrum_q
    f.restype = C.c_double
    return f(C.c_double(tau))


def blackbody_table(t_eff_K, e_lo, e_hi, m):
    n = spectrum_nodes(e_lo, e_hi, m)
    q = np.zeros(n)
    _chk(lib().orc_blackbody_table(C.c_double(t_eff_K), C.c_int(e_lo), C.c_int(e_hi), C.c_int(m), _ptr(q), C.c_int64(n)),
         "blackbody_table")
    return q


# ---- the step on P host cores (SURVEY.md 8(d) "Oracle timed beside it") ---------------------------------------------
# Gamma is a sum over sources: the parent runs the source pass once (dedup, radii, merge, sort), P
# single-threaded worker processes then trace disjoint chunks of the sorted catalogue with the unchanged
# orc_trace loop (orc_trace_add), each adding into its own grids (shared memory, zero-filled by the OS), and the
# parent adds the counters; the grids are added by the caller, slab by slab.  Process management only.

def _worker(g, p, nH, xHI, cat, chunks, counter, shm_names, shape, want_heat, conn):
    import time
    from multiprocessing import shared_memory
    shms = [shared_memory.SharedMemory(name=n) for n in shm_names]
    gam = np.ndarray(shape, np.float64, buffer=shms[0].buf)
    heat = np.ndarray(shape, np.float64, buffer=shms[1].buf) if want_heat else None
    st = Stats()
    t0 = time.perf_counter()
    while True:
        with counter.get_lock():
            k = counter.value
            counter.value += 1
        if k >= len(chunks):
            break
        a, b = chunks[k]
        trace_add(g, p, nH, xHI, cat[0][a:b], cat[1][a:b], gam, heat, st)
    conn.send((bytes(st), time.perf_counter() - t0))
    conn.close()
    del gam, heat
    for s in shms:
        s.close()


class OracleSum:
    """Partial results of the worker processes: the summed counters (a Stats) and the partial grids;
    gamma(z0, z1) / heat(z0, z1) add the partial grids of a z-slab."""

    def __init__(self, stats, gam_parts, heat_parts, shms, cpu_seconds, n_proc):
        self.stats, self._g, self._h, self._shms = stats, gam_parts, heat_parts, shms
        self.cpu_seconds, self.n_proc = cpu_seconds, n_proc

    def gamma(self, z0=0, z1=None):
        return np.sum([g[z0:z1] for g in self._g], axis=0)

    def heat(self, z0=0, z1=None):
        return np.sum([h[z0:z1] for h in self._h], axis=0) if self._h else None

    def close(self):
        self._g = self._h = None
        for s in self._shms:
            s.close()
            s.unlink()
        self._shms = []


def step_parallel(g, p, nH, xHI, pos, L, n_proc, want_heat=True, chunk=4):
    """The whole RT step with the ray loop on n_proc processes.  Returns (OracleSum, catalogue); the caller must
    close() the OracleSum."""
    import multiprocessing as mp
    from multiprocessing import shared_memory
    nH = _field(g, nH)
    xHI = _field(g, xHI)
    st0, cat = catalogue(g, p, xHI, pos, L)
    n_cat = len(cat[1])
    chunks = [(a, min(n_cat, a + chunk)) for a in range(0, n_cat, chunk)]
    shape = (g.nz, g.ny, g.nx)
    nbytes = int(np.prod(shape)) * 8
    # The workers' partial grids live in /dev/shm: never ask for more of it than is free (a worker that touches
    # a page the tmpfs cannot back dies of SIGBUS), and say so instead of failing half-way.
    import shutil
    per_proc = nbytes * (2 if want_heat else 1)
    try:
        shm_free = shutil.disk_usage("/dev/shm").free
    except OSError:
        shm_free = None
    if shm_free is not None:
        fit = int(0.9 * shm_free // per_proc)
        if fit < 1:
            raise MemoryError("step_parallel: /dev/shm has %.1f GB free, one worker's grids need %.1f GB"
                              % (shm_free / 1e9, per_proc / 1e9))
        n_proc = min(n_proc, fit)
    # fork: the children inherit the fields and the catalogue without a copy and never touch CUDA or threads of the
    # parent (they only run the single-threaded C oracle), which is what makes forking a process that has
    # initialised CUDA safe here.
    ctx = mp.get_context("fork")
    counter = ctx.Value(C.c_int64, 0)
    shms, procs, conns, gam_parts, heat_parts = [], [], [], [], []
    total = Stats()
    cpu = 0.0
    try:
        for _ in range(n_proc):
            pair = []
            for _k in range(2 if want_heat else 1):
                pair.append(shared_memory.SharedMemory(create=True, size=nbytes))
                shms.append(pair[-1])
            gam_parts.append(np.ndarray(shape, np.float64, buffer=pair[0].buf))
            if want_heat:
                heat_parts.append(np.ndarray(shape, np.float64, buffer=pair[1].buf))
            rx, tx = ctx.Pipe(duplex=False)
            pr = ctx.Process(target=_worker, args=(g, p, nH, xHI, cat, chunks, counter, [s.name for s in pair], shape,
                                                   want_heat, tx))
            pr.start()
            tx.close()
            procs.append(pr)
            conns.append(rx)
        for pr, rx in zip(procs, conns):
            try:
                raw, secs = rx.recv()
            except EOFError:
                pr.join()
                raise RuntimeError("oracle worker died (exit code %s) before it reported" % pr.exitcode)
            pr.join()
            if pr.exitcode != 0:
                raise RuntimeError("oracle worker failed (exit code %s)" % pr.exitcode)
            st = Stats.from_buffer_copy(raw)
            cpu += secs
            for name, _ in Stats._fields_:
                v = getattr(st, name)
                if hasattr(v, "__len__"):
                    t = getattr(total, name)
                    for l in range(len(v)):
                        t[l] += v[l]
                else:
                    setattr(total, name, getattr(total, name) + v)
    except BaseException:
        # no orphans and no leaked segments: stop every worker, then give the shared memory back
        for pr in procs:
            if pr.is_alive():
                pr.terminate()
        for pr in procs:
            pr.join()
        gam_parts.clear()
        heat_parts.clear()
        for s_ in shms:
            try:
                s_.close()
                s_.unlink()
            except (OSError, BufferError):
                pass
        raise
    total.n_src_in, total.n_src_dedup, total.n_src_merged = st0.n_src_in, st0.n_src_dedup, st0.n_src_merged
    return OracleSum(total, gam_parts, heat_parts, shms, cpu, n_proc), cat
