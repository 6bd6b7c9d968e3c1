"""The C-ABI library loads on a CPU-only box and exports every symbol include/gwmf.h declares
(no compute calls without a GPU); host-only entry points behave."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_0906_4175_b200 import build, gwmf
    build.build()
    return gwmf.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "gwmf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gwmf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    from paper_0906_4175_b200 import gwmf
    names = _declared()
    assert "gwmf_make_bank" in names and "gwmf_load_segment" in names and "gwmf_filter" in names \
        and "gwmf_triggers" in names                              # the four calls BASELINE.json names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/gwmf.h but not exported by libgwmf.so"
    assert sorted(gwmf.EXPORTS) == names                          # the binding carries the same names


def test_struct_layouts_match_header():
    from paper_0906_4175_b200 import gwmf
    assert ctypes.sizeof(gwmf.Params) == 64       # int64, 2 doubles, int32(+pad), double, 5 int32 (+pad)
    assert ctypes.sizeof(gwmf.MassPair) == 16
    assert gwmf.TRIGGER_DTYPE.itemsize == 16


def test_workspace_bytes_host_only(lib):
    from paper_0906_4175_b200 import gwmf
    assert gwmf.workspace_bytes(1000, 4, 8, 1) == 0
    assert gwmf.workspace_bytes(1 << 13, 4, 4096, 1) == 0         # below the supported range
    assert gwmf.workspace_bytes(1 << 23, 4, 4096, 1) == 0
    assert gwmf.workspace_bytes(1 << 14, 33, 4096, 1) == 0
    b = gwmf.workspace_bytes(1 << 20, 16, 4096, 1024)
    # band intermediate: 256 n-point transforms * n * 8 B = 2 GiB, and as much again for the pre-passed bands (vbuf);
    # per-band power spectra of the decimated path (2 * 128 templates * p * 4 sub-grid rows * 32768 * 8 B = 4 GiB);
    # double-buffered correlated spectra (2 * 128 * 4 MiB = 1 GiB); tables / slots / staging
    assert (9 << 30) < b < (9 << 30) + (512 << 20)
    assert gwmf.workspace_bytes(1 << 20, 16, 4096, 1024, batch=2) < (700 << 20)
    # chi^2 on demand runs no band-power stage: its 4 GiB of per-band spectra (and U+, and the job lists) are not carved
    assert gwmf.workspace_bytes(1 << 20, 16, 4096, 1024, chisq_on_demand=True) < b - (4 << 30)
    assert lib.gwmf_strerror(-2).decode().startswith("empty template")
    assert lib.gwmf_strerror(0).decode() == "ok"


def test_null_arguments_are_rejected_without_a_gpu(lib):
    assert lib.gwmf_filter(None, 0, 1) == -1
    assert lib.gwmf_make_bank(None, None, 1) == -1
    assert lib.gwmf_load_segment(None, None, None) == -1
    n = ctypes.c_int64(0)
    assert lib.gwmf_triggers(None, None, 0, ctypes.byref(n)) == -1
    h = ctypes.c_void_p()
    from paper_0906_4175_b200 import gwmf
    prm = gwmf.Params(1 << 14, 4096.0, 40.0, 4, 6.0, 4096, 8, 0, 0, 0)
    assert lib.gwmf_create(ctypes.byref(prm), None, 0, None, ctypes.byref(h)) == -1     # no workspace


def test_product_has_no_cpu_fallback():
    import torch
    from paper_0906_4175_b200 import gwmf
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        gwmf.Filter(1 << 14, 4, 4096, 8)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_0906_4175_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in text and "from oracle" not in text and "gwmf_oracle" not in text, fn
    otext = open(os.path.join(ROOT, "oracle", "gwmf_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "#include \"gwmf" not in otext and "include/gwmf.h" not in otext
    assert "import paper_0906_4175_b200" not in otext and "from paper_0906_4175_b200" not in otext
