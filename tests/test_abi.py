"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/hsg.h declares; argument validation that needs no GPU."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _declared_symbols():
    text = (ROOT / "include" / "hsg.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hsg_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported_by_the_library():
    import paper_1204_6192_b200 as hsg
    L = hsg.lib()
    declared = _declared_symbols()
    assert len(declared) >= 18
    assert sorted(hsg.SYMBOLS) == declared
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in hsg.hsg_version()


def test_query_bytes_and_descriptor_validation_without_a_gpu():
    import paper_1204_6192_b200 as hsg
    temps = np.array([0.1, 0.2, 0.3], dtype=np.float32)
    state, scratch = hsg.hsg_query_bytes(8, 2, 2, temps)
    assert state >= 4 * 3 * 512 * 12 + 4 * 6 * 512 * 2 and state % 256 == 0
    assert scratch > 0 and scratch % 256 == 0
    s4, _ = hsg.hsg_query_bytes(32, 64, 2, np.linspace(0.06, 0.25, 32))
    assert s4 >= 4096 * 32768 * 12            # the c4 state is 1.6 GB of spins
    for bad in [(7, 1, 1, temps), (8, 0, 1, temps), (8, 1, 0, temps), (8, 1, 1, temps[::-1].copy()),
                (8, 1, 1, np.array([0.0, 0.1], np.float32)), (0, 1, 1, temps)]:
        with pytest.raises(hsg.HsgError):
            hsg.hsg_query_bytes(*bad)
    # hsg_desc.flags: the fast-math heat-bath variant is the only defined bit; unknown bits are refused
    assert hsg.hsg_query_bytes(8, 2, 2, temps, flags=hsg.HSG_FLAG_FAST_MATH) == (state, scratch)
    for flags in (2, 4, 0x80000000, 3):
        with pytest.raises(hsg.HsgError):
            hsg.hsg_query_bytes(8, 2, 2, temps, flags=flags)
    text = (ROOT / "include" / "hsg.h").read_text()
    assert re.search(r"HSG_FLAG_FAST_MATH\s*=\s*1\b", text) and hsg.HSG_FLAG_FAST_MATH == 1


def test_null_handles_are_rejected():
    import paper_1204_6192_b200 as hsg
    L = hsg.lib()
    assert L.hsg_sweep(None, 1, 1) == hsg.HSG_EINVAL
    assert L.hsg_destroy(None) == hsg.HSG_EINVAL
    assert L.hsg_pt_swap(None, None) == hsg.HSG_EINVAL
    assert L.hsg_measure(None, None, None, None, None) == hsg.HSG_EINVAL
    assert L.hsg_launch_count(None) == 0
    out = C.c_void_p(123)
    assert L.hsg_create(None, None, 0, None, 0, None, C.byref(out)) == hsg.HSG_EINVAL and not out.value


def test_product_path_does_not_touch_the_oracle():
    """The package must not import, link or read anything under oracle/ (and vice versa)."""
    for p in (ROOT / "paper_1204_6192_b200").rglob("*"):
        if p.suffix in {".py", ".cu", ".cuh", ".h"}:
            assert "oracle" not in p.read_text().lower(), p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in {".py", ".cpp"}:
            t = p.read_text()
            assert "import paper_1204_6192_b200" not in t and "from paper_1204_6192_b200" not in t
            assert "#include \"../paper" not in t and "csrc" not in t
