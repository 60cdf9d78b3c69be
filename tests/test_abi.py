"""The C-ABI library loads and exports every symbol include/dr.h declares (no compute calls: no GPU needed)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dr_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_2605_08916_b200 import build
    lib = ctypes.CDLL(build.build())
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_names():
    from paper_2605_08916_b200 import build
    build.build()
    from paper_2605_08916_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    # struct sizes match the C layout
    assert ctypes.sizeof(binding.dr_material) == 36
    assert ctypes.sizeof(binding.dr_config) == 64
    assert ctypes.sizeof(binding.dr_stats) == 88
    assert ctypes.sizeof(binding.dr_scene_info) == 32


def test_product_path_does_not_touch_the_oracle():
    """The oracle is test infrastructure: nothing in the package or the inputs module imports it."""
    for folder in ("paper_2605_08916_b200", "dr_inputs"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, folder)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                    text = open(os.path.join(dirpath, f)).read()
                    for needle in ("import oracle", "from oracle", "liboracle", "orc_", "oracle/", "oracle."):
                        assert needle not in text, (dirpath, f, needle)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2605_08916_b200" not in text and "libdr" not in text and "dr.h" not in text, f
