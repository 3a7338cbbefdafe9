"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/axg.h declares, and refuses to work (loudly) without a CUDA device."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "axg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(axg_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1405_3331_b200 import axg
    L = axg.lib()
    names = _declared()
    assert len(names) >= 18 and "axg_step" in names and "axg_read_state" in names
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(axg.EXPORTS)


def test_field_and_phase_constants_match_header():
    from paper_1405_3331_b200 import axg
    src = open(os.path.join(ROOT, "include", "axg.h")).read()
    for name, val in axg.FIELDS.items():
        m = re.search(r"\bAXG_%s = (\d+)" % name, src)
        assert m and int(m.group(1)) == val, name
    for name, val in (("DIFFUSE", 1), ("BIN", 2), ("SENSE", 4), ("ADVANCE", 8), ("COMMIT", 16), ("ALL", 31)):
        assert re.search(r"\bAXG_PHASE_%s = %d\b" % (name, val), src)
        assert getattr(axg, "PHASE_" + name) == val


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1405_3331_b200 import axg
    with pytest.raises(axg.AxgError) as e:
        axg.Axg((8, 8, 8), 0.5, 1, 2.0, 0.25, 0.1, 1, torch_memory=False)
    assert e.value.code == -4 and "no CPU fallback" in str(e.value)


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1405_3331_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "axo_" not in txt, f
