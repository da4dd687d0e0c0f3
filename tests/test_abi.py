"""The C-ABI library builds, loads and exports every symbol include/*.h declares (no GPU)."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        text = open(h).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)          # strip comments
        for m in re.finditer(r"\b(cs_[A-Za-z0-9_]+)\s*\(", text):
            names.add(m.group(1))
    return sorted(names)


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for want in ("cs_computeBox", "cs_computeKeys", "cs_sortKeys", "cs_buildLeaves", "cs_linkOctree",
                 "cs_nodeCounts", "cs_buildOctree", "cs_buildOctreeHost", "cs_create", "cs_destroy"):
        assert want in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2307_06345_b200 import build
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/ but not exported"


def test_binding_signatures_cover_the_header():
    from paper_2307_06345_b200 import binding
    lib = binding.lib()
    for name in _declared_symbols():
        fn = getattr(lib, name)
        assert fn.argtypes is not None, f"binding has no signature for {name}"
    assert binding.version().startswith("cornerstone-b200")
    assert binding.workspaceBytes(1 << 20, 1 << 16) > (1 << 20) * 12


def test_no_cpu_fallback_without_device():
    import torch
    from paper_2307_06345_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        binding.Context(1024, 64)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2307_06345_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text, f
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "binding" not in orc.replace("never imports\nthe product's CUDA binding", "")
