"""CPU-side checks of the boundary: libhigs.so builds with nvcc (cross-compile, no GPU needed),
loads, and exports every function include/higs.h declares; the ctypes structs match the header's
layout.  No compute call is made here."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "higs.h").read_text()


def _declared_functions():
    body = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    return sorted(set(re.findall(r"\b(higs_[a-z_0-9]+)\s*\(", body)))


def test_header_declares_the_expected_entry_points():
    names = _declared_functions()
    for must in ("higs_create", "higs_destroy", "higs_render", "higs_render_host", "higs_get_stats", "higs_get_lists",
                 "higs_strerror"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2606_00352_b200 as hg
    lib = hg.load()
    for name in _declared_functions():
        assert hasattr(lib, name), f"libhigs.so does not export {name}"
    assert sorted(hg.EXPORTS) == _declared_functions()
    assert lib.higs_abi_version() == int(re.search(r"#define HIGS_ABI_VERSION (\d+)", HEADER).group(1))
    assert lib.higs_strerror(0) == b"ok"
    assert b"capacity" in lib.higs_strerror(-3)


def test_struct_layouts_match_the_header():
    import paper_2606_00352_b200 as hg
    assert C.sizeof(hg.higs_camera) == 80
    assert C.sizeof(hg.higs_stats) == 6 * 8 + 6 * 4 + 2 * 8 + 8 * 4
    assert C.sizeof(hg.higs_lists) == 2 * 8 + 8 + 6 * 8            # int32 n_mt padded to 8
    assert C.sizeof(hg.higs_records) == 8 + 2 * 8
    for macro, val in (("HIGS_TILE", hg.HIGS_TILE), ("HIGS_MT_W", hg.HIGS_MT_W), ("HIGS_MT_H", hg.HIGS_MT_H),
                       ("HIGS_MT_TILES", hg.HIGS_MT_TILES), ("HIGS_BATCH_CAP", hg.HIGS_BATCH_CAP)):
        assert int(re.search(rf"#define {macro}\s+(\d+)", HEADER).group(1)) == val
    for macro, val in (("HIGS_FLAG_STAGE_TIMERS", 1), ("HIGS_FLAG_COUNT_EVALS", 2), ("HIGS_FLAG_NO_XBATCH_CUT", 4)):
        assert int(re.search(rf"#define {macro}\s+(\d+)u", HEADER).group(1)) == val


def test_product_fails_loudly_without_a_gpu():
    import torch
    import paper_2606_00352_b200 as hg
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        hg.higs_create(0, 10, 64, 64)


def test_product_does_not_import_the_oracle():
    for p in (ROOT / "paper_2606_00352_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            txt = p.read_text()
            assert "import oracle" not in txt and "from oracle" not in txt and "higs_oracle" not in txt, p
