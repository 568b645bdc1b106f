"""Host-side checks of the boundary that need no GPU: the library loads, exports every symbol include/tpctrack.h
declares, the binding's struct layouts match the header, defaults agree with the oracle's independent copy, and
creation fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def tr():
    from paper_1712_09416_b200 import _build
    _build.build_tracker()
    from paper_1712_09416_b200 import tracker
    return tracker


def declared_functions():
    src = (ROOT / "include" / "tpctrack.h").read_text()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(tr):
    names = declared_functions()
    assert len(names) >= 12 and "tpc_track_event" in names and "tpc_tracker_create" in names
    for n in names:
        assert hasattr(tr.lib, n), n
    assert set(tr.EXPORTS) == set(names)


def test_struct_layouts_match_header(tr):
    assert C.sizeof(tr.tpc_params) == 27 * 4
    assert C.sizeof(tr.tpc_event_in) == 8 + 8 * 5 + 8          # int32 + pad, 5 pointers, int32 + pad
    assert C.sizeof(tr.tpc_event_out) == 8 + 8 * 31
    assert C.sizeof(tr.tpc_counters) == 13 * 8
    assert C.sizeof(tr.tpc_geometry) == 8 + 8 + 16 + 8


def test_defaults_equal_the_oracles_independent_copy(tr, oracle_mod):
    a, b = tr.tpc_default_params().as_dict(), oracle_mod.default_params().as_dict()
    assert a == b


def test_status_strings(tr):
    assert tr.tpc_status_string(0) == "ok"
    for s in (-1, -2, -3, -4):
        assert tr.tpc_status_string(s) not in ("ok", "unknown status")


def test_no_cpu_fallback_and_argument_errors(tr):
    import torch
    rx = np.linspace(85, 245, 159).astype(np.float32)
    if not torch.cuda.is_available():
        with pytest.raises(tr.TpcError) as ei:
            tr.Tracker(36, rx, 0.176, 0.06, 0.06, 0.5)
        assert "no CUDA device" in str(ei.value)
    # geometry errors are caught before any device work
    for bad in (rx[::-1].copy(), rx[:2]):
        with pytest.raises(tr.TpcError):
            tr.Tracker(36, bad, 0.176, 0.06, 0.06, 0.5)
    with pytest.raises(tr.TpcError):
        tr.Tracker(36, rx, 0.176, 0.0, 0.06, 0.5)
    p = tr.tpc_default_params(); p.link_step = 3
    with pytest.raises(tr.TpcError):
        tr.Tracker(36, rx, 0.176, 0.06, 0.06, 0.5, params=p)


def test_product_never_imports_the_oracle():
    for f in list((ROOT / "paper_1712_09416_b200").rglob("*.py")) + list((ROOT / "paper_1712_09416_b200").rglob("*.cu*")):
        txt = f.read_text()
        assert "import oracle" not in txt and "from oracle" not in txt and "tpc_oracle" not in txt, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".cpp", ".h"):
            txt = f.read_text()
            assert "#include \"../paper_1712_09416_b200" not in txt and "csrc/" not in txt, f   # no product source
            assert "#include \"tpctrack.h\"" not in txt and "libtpctrack" not in txt, f


def test_baseline_md_quotes_table_1_of_the_paper_unchanged():
    """tests/golden/table1_tracking_time.txt = Table 1 of the paper: context numbers only."""
    root = Path(__file__).resolve().parent.parent
    text = (root / "BASELINE.md").read_text()
    rows = [l.split() for l in (root / "tests" / "golden" / "table1_tracking_time.txt").read_text().splitlines()
            if l and not l.startswith("#")]
    assert len(rows) == 5
    for dev, ms in rows:
        assert any(dev in line and ms + " ms" in line.replace("*", "") for line in text.splitlines()), (dev, ms)
