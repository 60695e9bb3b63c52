"""CPU-side checks of the C-ABI boundary (no GPU needed): libbemcub.so builds for sm_100a, loads,
exports every symbol include/bemcub.h declares, refuses to work without a CUDA device (no CPU
fallback), and its host-side rule tables agree with the oracle's independent transcription."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "bemcub.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bemcub_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound():
    from paper_1606_03743_b200 import bemcub
    names = _declared_symbols()
    assert len(names) >= 17
    lib = ctypes.CDLL(bemcub.library_path())
    for name in names:
        assert hasattr(lib, name), f"{name} declared in bemcub.h but not exported"
        assert hasattr(bemcub, name), f"{name} has no Python binding of the same name"
    assert sorted(bemcub.EXPORTED) == names


def test_library_is_sm100a_only():
    import subprocess
    from paper_1606_03743_b200 import bemcub
    out = subprocess.run(["cuobjdump", "-lelf", bemcub.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    from paper_1606_03743_b200 import bemcub
    with pytest.raises(bemcub.BemcubError) as ei:
        bemcub.bemcub_create(0, 0)
    assert ei.value.code == bemcub.ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1606_03743_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "oracle/" not in txt.replace("oracle/ ", ""), f


@pytest.mark.parametrize("etype", [0, 1])
@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_rule_tables_match_oracle_transcription(etype, level):
    """Two independent transcriptions of Appendix A/B: same point sets and
    weights (order may differ, it only affects rounding)."""
    from paper_1606_03743_b200 import bemcub
    n, d = bemcub.bemcub_rule_info(etype, level)
    on, od = oracle.rule_info(etype, level)
    assert (n, d) == (on, od)
    c, w = bemcub.bemcub_rule_points(etype, level)
    oc, ow = oracle.rule_nodes(etype, level)
    assert abs(w.sum() - 1.0) < 4e-16
    a = np.round(np.column_stack([c, w]), 13)
    b = np.round(np.column_stack([oc, ow]), 13)
    a = a[np.lexsort(a.T[::-1])]
    b = b[np.lexsort(b.T[::-1])]
    np.testing.assert_allclose(a, b, atol=2e-13)


def test_rule_info_errors():
    from paper_1606_03743_b200 import bemcub
    for et, lv in ((2, 0), (0, 5), (0, -1)):
        with pytest.raises(bemcub.BemcubError) as ei:
            bemcub.bemcub_rule_info(et, lv)
        assert ei.value.code == bemcub.ERR_BAD_RULE
    p = bemcub.bemcub_default_policy(False)
    assert [p.dr[0][i] for i in range(5)] == [3, 8, 20, 80, 1500]
    assert p.allow_upgrade == 1 and p.use_levels_mask == 63


def test_limit_errors_say_what_the_limit_is():
    """A refused size names its limit (bemcub.h documents both next to the calls they belong to)."""
    from paper_1606_03743_b200 import bemcub
    assert "2^25" in bemcub.bemcub_strerror(bemcub.ERR_TOO_MANY_ELEMENTS)
    assert "64 field points" in bemcub.bemcub_strerror(bemcub.ERR_FIXED_SCRATCH)
    hdr = open(os.path.join(ROOT, "include", "bemcub.h")).read()
    assert "BEMCUB_ERR_TOO_MANY_ELEMENTS" in hdr and "2^25" in hdr
    codes = dict(re.findall(r"(BEMCUB_ERR_[A-Z_]+) = (-\d+)", hdr))
    for name, val in codes.items():
        assert bemcub.bemcub_strerror(int(val)) != "unknown error code", name
