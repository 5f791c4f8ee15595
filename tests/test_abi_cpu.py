"""The C-ABI library loads and exports every symbol include/dedisp.h declares
(no GPU; no compute calls)."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def dd():
    from paper_1112_0065_b200 import build
    build.build()
    import paper_1112_0065_b200 as dd
    return dd


def _declared():
    text = (ROOT / "include" / "dedisp.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dedisp_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported_and_bound(dd):
    names = _declared()
    assert "dedisp_plan_create" in names and "dedisp_execute_batch" in names and len(names) >= 15
    L = dd.lib()
    for n in names:
        assert hasattr(L, n), n           # exported by the .so
        assert n in dd.ABI, n             # typed in the binding
        assert callable(getattr(dd, n)), n  # wrapper with the same name
    assert sorted(dd.ABI) == names


def test_host_side_validation(dd):
    # plan_create is host-only: geometry validation works without a device
    for bad in [(0, 64e-6, 1500.0, -1.0), (4, 0.0, 1500.0, -1.0), (4, 64e-6, -5.0, -1.0),
                (4, 64e-6, 1500.0, 1.0), (4, 64e-6, 1500.0, 0.0), (4, 64e-6, 3.0, -1.0),
                (4, float("nan"), 1500.0, -1.0)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_plan_create(*bad)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    p = dd.dedisp_plan_create(4, 1e-3, 1500.0, -100.0)
    assert dd.dedisp_get_nchans(p) == 4 and dd.dedisp_get_ndm(p) == 0
    assert dd.dedisp_get_max_delay(p) == -1
    assert dd.dedisp_get_in_row_stride_bytes(p, 100, 2) == 0
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_set_dm_list(p, [1.0, -2.0])
    assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_execute(p, 16, 1 << 20, 2, 1 << 21, dd.DEDISP_OUT_U32)
    assert e.value.status == dd.DEDISP_ERR_NO_DM_LIST
    with pytest.raises(dd.DedispError):
        dd.dedisp_set_kernel(p, 9)
    dd.dedisp_destroy(p)
    assert dd.lib().dedisp_get_error_string(7) == b"CUDA error"
    assert dd.lib().dedisp_destroy(None) == 0


def test_no_cpu_fallback_in_product():
    # the product package never imports the oracle, and the oracle never imports the product
    pkg = ROOT / "paper_1112_0065_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.h")) \
            + list(pkg.rglob("*.cuh")):
        s = f.read_text()
        assert "import oracle" not in s and "from oracle" not in s and "dedisp_oracle" not in s, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c", ".h"):
            s = f.read_text()
            assert "import paper_1112_0065_b200" not in s and "from paper_1112_0065_b200" not in s \
                and "dedisp.h" not in s and "libdedisp_b200" not in s, f


def test_host_only_size_functions(dd):
    """The workspace / stride / block-count queries are host arithmetic (no device): documented values for the HTRU
    gulp, 0 on bad arguments, never shrinking with the problem."""
    w7 = [1, 2, 4, 8, 16, 32, 64]
    assert dd.dedisp_static_scratch_bytes() == 32 << 20
    fe = dd.dedisp_find_events_workspace_bytes(8400, 65536)
    assert 70e6 < fe < 80e6                                              # "73 MB" for 7 widths x 1200 rows
    assert dd.dedisp_find_events_workspace_bytes(0, 65536) == 0 and dd.dedisp_find_events_workspace_bytes(8400, 0) == 0
    assert dd.dedisp_find_events_workspace_bytes(8400, 131072) >= fe <= dd.dedisp_find_events_workspace_bytes(16800, 65536)
    mf = dd.dedisp_matched_filter_rms_workspace_bytes(1200, 65536, 7)
    assert mf > 0 and mf % 8 == 0
    assert dd.dedisp_matched_filter_rms_workspace_bytes(0, 65536, 7) == 0
    assert dd.dedisp_matched_filter_rms_workspace_bytes(1200, 65536, 0) == 0
    assert dd.dedisp_matched_filter_rms_workspace_bytes(2400, 65536, 7) >= mf
    # block maxima: blocks of 2048 outputs, offset by the largest width, enough blocks to cover nsamps + offset
    assert dd.dedisp_matched_filter_hint_blocks(65536, w7) == (33, 2048, 64)
    assert dd.dedisp_matched_filter_hint_blocks(100, [1]) == (1, 2048, 1)
    assert dd.dedisp_matched_filter_hint_blocks(2048, [1, 64])[0] == 2
    se = dd.dedisp_search_events_workspace_bytes(1200, 65536, w7, 16384)
    assert se >= 16384 * 2048 * 4 + fe and se % 256 == 0                 # the compact z + the f2 workspace inside it
    assert dd.dedisp_search_events_workspace_bytes(1200, 65536, w7, 0) == 0
    assert dd.dedisp_search_events_workspace_bytes(0, 65536, w7, 16) == 0
    assert dd.dedisp_search_events_workspace_bytes(1200, 65536, w7, 32768) > se
    # strides need the delay table (max_delay): 0 before set_dm_list, which needs a device
    p = dd.dedisp_plan_create(1024, 64e-6, 1581.8046875, -0.390625)
    assert dd.dedisp_get_in_row_stride_bytes(p, 100, 2) == 0
    dd.dedisp_destroy(p)
