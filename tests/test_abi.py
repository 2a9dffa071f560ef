"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/gwi.h
declares; host-side argument validation that needs no GPU; no CPU fallback."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "gwi.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gwi_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2201_11133_b200 as gwi
    L = gwi.lib()
    decl = _declared_symbols()
    assert "gwi_load_model" in decl and "gwi_infer" in decl and "gwi_ensemble_triggers" in decl
    for s in decl:
        assert hasattr(L, s), s
    assert sorted(gwi.EXPORTED_SYMBOLS) == decl
    assert gwi.version() >= 100


def test_no_torch_types_in_header():
    src = open(os.path.join(ROOT, "include", "gwi.h")).read()
    assert "torch" not in src and "at::" not in src and 'extern "C"' in src


def test_host_side_errors_without_gpu(tmp_path):
    import paper_2201_11133_b200 as gwi
    import gwsynth as gs
    with pytest.raises(gwi.GwiError) as e:
        gwi.load_model(str(tmp_path / "missing.gwim"))
    assert e.value.status == 2
    p = tmp_path / "bad.gwim"
    p.write_bytes(b"GWIM" + b"\x02" + b"\0" * 60)
    with pytest.raises(gwi.GwiError) as e:
        gwi.load_model(str(p))
    assert e.value.status == 3
    good = tmp_path / "good.gwim"
    gs.make_model_file(str(good), gs.CFG1_ARCH, 0)
    raw = good.read_bytes()
    (tmp_path / "trunc.gwim").write_bytes(raw[:-8])
    with pytest.raises(gwi.GwiError) as e:
        gwi.load_model(str(tmp_path / "trunc.gwim"))
    assert e.value.status == 2
    (tmp_path / "trail.gwim").write_bytes(raw + b"\0")
    with pytest.raises(gwi.GwiError) as e:
        gwi.load_model(str(tmp_path / "trail.gwim"))
    assert e.value.status == 3
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(gwi.GwiError) as e:          # the product path fails loudly without a GPU
            gwi.load_model(str(good))
        assert e.value.status == 5 and "no CPU fallback" in str(e.value)
    L = gwi.lib()
    assert L.gwi_infer_workspace_bytes(None, 1, 1) == 0
    assert L.gwi_carry_bytes() >= 32 and L.gwi_triggers_workspace_bytes(0) == 0
    assert L.gwi_triggers_workspace_bytes(1 << 20) > (1 << 20) // 8


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2201_11133_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                s = open(os.path.join(dp, f)).read()
                assert "oracle" not in s.replace("the oracle", "").replace("fp64 oracle", "").replace("The oracle", "") \
                    or "import" not in s.split("oracle")[0][-30:], f
                assert "from oracle" not in s and "import oracle" not in s and "gwo_" not in s, f
