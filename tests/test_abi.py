"""CPU-only: the C-ABI library builds, loads and exports every symbol include/wstack.h declares; no compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "wstack.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ws_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported():
    import paper_2301_06061_b200 as ws
    names = _declared()
    assert len(names) >= 20
    lib = ctypes.CDLL(ws.library_path()) if os.path.exists(ws.library_path()) else ws.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in wstack.h but not exported"
    assert sorted(ws.EXPORTED_SYMBOLS) == names


def test_host_only_calls():
    import paper_2301_06061_b200 as ws
    L = ws.lib()
    assert L.ws_version() == ws.WS_VERSION
    hdr = open(os.path.join(ROOT, "include", "wstack.h")).read()
    assert int(re.search(r"#define WS_VERSION (\d+)", hdr).group(1)) == ws.WS_VERSION
    assert L.ws_strerror(-3) == b"workspace too small"
    assert L.ws_grid_bytes(None) == 0 and L.ws_launch_count(None) == 0


def test_no_fallback_without_gpu():
    """On a box without a GPU the product path must fail loudly, not fall back to anything."""
    import torch
    import paper_2301_06061_b200 as ws
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(ws.WStackError):
        ws.Plan(256, 4, 7, 1e-3, -1.0, 1.0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2301_06061_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle performs", "").replace("oracle performs", "") or f == "ws_bin.cu", f
    txt = open(os.path.join(pkg, "csrc", "ws_bin.cu")).read()
    assert "#include \"ws_internal.h\"" in txt and "wstack_oracle" not in txt
