"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/wdm.h declares, and
validates arguments (no compute calls, no GPU needed)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def wdm():
    from paper_2606_25026_b200 import build
    build.build()
    import paper_2606_25026_b200 as w
    w.lib()
    return w


def test_exports_every_declared_symbol(wdm):
    header = open(os.path.join(ROOT, "include", "wdm.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(wdm_[a-z_0-9]+)\s*\(", header))
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(wdm.lib(), name), f"{name} declared in include/wdm.h but not exported"
    assert declared == set(wdm.EXPORTS)
    for name in wdm.EXPORTS:
        assert callable(getattr(wdm, name))          # binding has the same names


def test_argument_validation_without_gpu(wdm):
    for n in (0, 4, 100, 2048, -8):
        with pytest.raises(wdm.WdmError) as e:
            wdm.wdm_create(n, 1.0, 1.0, 1.0, wdm.WDM_C64)
        assert e.value.code == wdm.WDM_EUNSUPPORTED
    for args in ((64, 0.0, 1.0, 1.0, 0), (64, 1.0, -1.0, 1.0, 0), (64, 1.0, 1.0, -0.1, 0), (64, 1.0, 1.0, 1.0, 7)):
        with pytest.raises(wdm.WdmError) as e:
            wdm.wdm_create(*args)
        assert e.value.code == wdm.WDM_EINVAL
    assert "N must be a power of two" in wdm.wdm_last_error(None) or wdm.wdm_last_error(None)
    # null context
    assert wdm.lib().wdm_step(None, 1, 0.1) == wdm.WDM_EINVAL
    assert wdm.lib().wdm_destroy(None) == wdm.WDM_OK


def test_workspace_bytes(wdm):
    b = wdm.wdm_workspace_bytes(512, wdm.WDM_C64, 0)
    n = 512 ** 3
    # psi (8 B) + Phi (4 B) + half spectrum (4 B (1 + 2/N)) per cell, plus small tables
    assert n * 16 < b < n * 16.2
    assert wdm.wdm_workspace_bytes(512, wdm.WDM_C128, 0) > 2 * n * 16
    bp = wdm.wdm_workspace_bytes(256, wdm.WDM_C64, 1 << 20)
    assert bp - wdm.wdm_workspace_bytes(256, wdm.WDM_C64, 0) > 256 ** 3 * 4 + (1 << 20) * 24
    with pytest.raises(wdm.WdmError):
        wdm.wdm_workspace_bytes(100, 0, 0)


def test_missing_library_fails_loudly(wdm, monkeypatch):
    import paper_2606_25026_b200 as w
    monkeypatch.setattr(w, "_lib", None)
    monkeypatch.setattr(w, "LIB_PATH", "/nonexistent/libwdm.so")
    with pytest.raises(ImportError):
        w.lib()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_25026_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep)[-1:]:
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "wdmo" not in text, f
    text = open(os.path.join(ROOT, "oracle", "wdmo.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "import paper_2606_25026_b200" not in text and "libwdm.so" not in text and "csrc/wdm" not in text.replace("paper_2606_25026_b200/csrc/", "")
