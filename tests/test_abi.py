"""-m "not gpu": the C-ABI library builds, loads, and exports every symbol include/ikv.h declares.
No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ikv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ikv_[a-z_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2606_09916_b200 import build
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    syms = declared_symbols()
    assert len(syms) >= 16 and "ikv_memory_update" in syms and "ikv_score" in syms
    assert "ikv_select_evict" in syms and "ikv_decode_attn" in syms
    for name in syms:
        assert hasattr(lib, name), f"{name} declared in include/ikv.h but not exported by libikv.so"


def test_binding_names_match_header():
    from paper_2606_09916_b200 import ikv
    assert sorted(ikv.EXPORTS) == declared_symbols()
    assert "sm_100a" in ikv.version()
    for name in declared_symbols():
        meth = name[len("ikv_"):]
        if meth in ("create", "destroy", "last_error", "version"):
            continue
        assert hasattr(ikv.Context, meth), f"binding lacks Context.{meth}"


def test_struct_layouts_match_header_sizes():
    """ctypes mirrors of ikv_config / ikv_request have the C sizes (LP64)."""
    from paper_2606_09916_b200 import ikv
    assert ctypes.sizeof(ikv.Config) == 64
    assert ctypes.sizeof(ikv.Request) == 72
    assert ctypes.sizeof(ikv.ResidualWeights) == 88


def test_product_does_not_touch_the_oracle():
    """The product path may not import, link or execute anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2606_09916_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "ikv_oracle" not in src and "from oracle" not in src and "import oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_09916_b200" not in src and "from paper_2606_09916_b200" not in src, f
            assert "libikv.so" not in src and "csrc/" not in src.replace("paper_2606_09916_b200/csrc)", ""), f
