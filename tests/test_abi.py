"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU and exports
every symbol include/rosefusion_b200.h declares.  No compute call is made here."""
import ctypes
import os
import re

import paper_2105_05600_b200 as rf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "rosefusion_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rf_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert "rf_pfo_track" in names and "rf_volume_create" in names and len(names) >= 15
    lib = rf.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(rf.EXPORTS) == names
    lib.rf_version.restype = ctypes.c_int
    assert lib.rf_version() >= 100


def test_struct_sizes_match_the_header():
    from paper_2105_05600_b200 import api
    assert ctypes.sizeof(api.VolumeOpts) == 40
    assert ctypes.sizeof(api.TrackState) == 4 * (12 + 12 + 6 + 4)
    assert ctypes.sizeof(api.TrackTrace) == 6 * 4 + 8 * (4 + 6 + 12 + 6)
    assert ctypes.sizeof(api.TrackResult) == 32
    assert ctypes.sizeof(api.Frame) == 40
    assert ctypes.sizeof(api.PstSet) == 48


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2105_05600_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(base, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
