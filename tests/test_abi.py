"""CPU-side checks of the C-ABI: the library loads, exports every symbol include/catapult.h declares,
and rejects bad arguments before any launch (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_07617_b200 import build, binding
    build.build()
    return binding.load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "catapult.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(catapult_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 15
    from paper_2604_07617_b200 import binding
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.catapult_version()
    # the product library exports nothing beyond its header: measurement / test hooks live in the probe library
    import subprocess
    syms = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r"\b(catapult_[a-z0-9_]+)\b", syms))
    assert exported == declared, exported ^ declared


def test_probe_library_exports_its_header():
    from paper_2604_07617_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "catapult_probe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(catapult_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.PROBE_EXPORTS)
    P = binding.load_probe()
    for name in declared:
        assert hasattr(P, name), name


def test_struct_layouts_match_header(lib):
    from paper_2604_07617_b200 import binding
    assert C.sizeof(binding.FieldDesc) == 4 * (6 + 16) + 8 * 6 + 8 * 5 + 8 * 3
    assert C.sizeof(binding.TraceParams) == 8 * 8 + 8 + 4 * 4 + 8 * 4 + 4 * 2   # + loss_time_mode, reserved_


def test_argument_validation_without_gpu(lib):
    from paper_2604_07617_b200 import binding
    from paper_2604_07617_b200 import workloads as W
    h = C.c_void_p()
    assert lib.catapult_field_build(None, None, None, C.byref(h)) == binding.EINVAL
    assert b"desc" in lib.catapult_last_error()
    fd = W.config(0, n=1, with_nodes=False)
    base = dict(coord=0, ncell=[2, 2, 2], lo=[0, 0, 0], hi=[1, 6.28, 1.57], nfp=4, nquant=4, G0=44.0, I0=0.0,
                iota0=0.4, iota1=0.1, psi0=8.0)
    bad = [dict(base, ncell=[0, 2, 2]), dict(base, nquant=7), dict(base, hi=[1, 6.28, 0.0]), dict(base, coord=5),
           dict(base, G0=0.0), dict(base, nfp=0)]
    dummy = C.c_void_p(16)
    for b in bad:
        d = binding.make_desc(b)
        assert lib.catapult_field_build(C.byref(d), dummy, None, C.byref(h)) == binding.EINVAL, b
    d = binding.make_desc(dict(base, I0=1.0))
    assert lib.catapult_field_build(C.byref(d), dummy, None, C.byref(h)) == binding.EUNSUPPORTED
    # more cells than a 32-bit flat index can carry; column tags: the canonical order or nothing
    d = binding.make_desc(dict(base, ncell=[2048, 2048, 2048]))
    assert lib.catapult_field_build(C.byref(d), dummy, None, C.byref(h)) == binding.EINVAL
    d = binding.make_desc(dict(base, quant=[1, 3, 2, 4]))
    assert lib.catapult_field_build(C.byref(d), dummy, None, C.byref(h)) == binding.EUNSUPPORTED
    d = binding.make_desc(dict(base, quant=[1, 2, 3, 4]))
    assert lib.catapult_field_build(C.byref(d), None, None, C.byref(h)) == binding.EINVAL      # tags fine, nodes NULL
    d = binding.make_desc(base)
    assert lib.catapult_field_build(C.byref(d), None, None, C.byref(h)) == binding.EINVAL
    p = binding.make_params(fd["params"])
    assert lib.catapult_trace(None, C.byref(p), 4, dummy, dummy, dummy, dummy, None, None, None, None) == binding.EINVAL
    assert lib.catapult_estimate(7, 4, dummy, None, None, dummy, None, None) == binding.EINVAL
    assert lib.catapult_estimate(0, -1, dummy, None, None, dummy, None, None) == binding.EINVAL
    assert lib.catapult_estimate(0, 4, None, None, None, dummy, None, None) == binding.EINVAL
    assert lib.catapult_field_eval(None, 1, dummy, dummy, None) == binding.EINVAL
    assert lib.catapult_field_destroy(None) == binding.OK


def test_binding_fails_loudly_when_library_missing(monkeypatch, tmp_path):
    from paper_2604_07617_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        binding.load()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2604_07617_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "catapult_oracle" not in src and "import oracle" not in src and "from oracle" not in src, fn
