"""No-GPU checks of the boundary: the C-ABI library loads, exports every symbol include/nyxrt.h declares,
its struct sizes match the binding, and it fails loudly (no fallback) without a CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nyxrt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nyxrt_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__
    __graft_entry__.build()
    from paper_2512_12466_b200 import nyxrt
    L = nyxrt.lib()
    names = declared_symbols()
    assert len(names) >= 15 and set(nyxrt.EXPORTS) == set(names)
    for n in names:
        assert getattr(L, n) is not None
    assert L.nyxrt_version() >= 100
    assert L.nyxrt_sizeof_grid() == ctypes.sizeof(nyxrt.nyxrt_grid)
    assert L.nyxrt_sizeof_params() == ctypes.sizeof(nyxrt.nyxrt_params)
    assert L.nyxrt_sizeof_stats() == ctypes.sizeof(nyxrt.nyxrt_stats)


def test_argument_validation_without_gpu():
    from paper_2512_12466_b200 import nyxrt, synth
    L = nyxrt.lib()
    ctx = ctypes.c_void_p()
    assert L.nyxrt_create(None, None, ctypes.byref(ctx)) == nyxrt.EINVAL
    g = nyxrt.make_grid((8, 8, 8), 1e20)
    p = nyxrt.make_params(**synth.default_params())
    g.nx = 0
    assert L.nyxrt_create(ctypes.byref(g), ctypes.byref(p), ctypes.byref(ctx)) == nyxrt.EINVAL
    g.nx = 8
    p.level_max = 14
    assert L.nyxrt_create(ctypes.byref(g), ctypes.byref(p), ctypes.byref(ctx)) == nyxrt.EINVAL
    assert L.nyxrt_last_error(None) is not None
    L.nyxrt_destroy(None)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2512_12466_b200 import nyxrt, synth
    with pytest.raises(RuntimeError):
        nyxrt.Tracer((8, 8, 8), 1e20, synth.default_params())
    g = nyxrt.make_grid((8, 8, 8), 1e20)
    with pytest.raises(nyxrt.NyxrtError) as e:
        nyxrt.nyxrt_create(g, nyxrt.make_params(**synth.default_params()))
    assert e.value.code == nyxrt.ECUDA


def test_product_never_imports_oracle():
    """The product path must not route through the oracle: no import, include, path or symbol of it."""
    pat = re.compile(r"(import|from)\s+oracle|oracle[./\\]|nyxrt_oracle|orc_[a-z]")
    pkg = os.path.join(ROOT, "paper_2512_12466_b200")
    n = 0
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                n += 1
                assert not pat.search(open(os.path.join(dp, f)).read()), f
    assert n >= 8
    assert not pat.search(open(os.path.join(ROOT, "include", "nyxrt.h")).read())
