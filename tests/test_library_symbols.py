"""The C-ABI library loads and exports every symbol include/lsd.h declares (no compute calls without a GPU)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_declared_symbol_is_exported():
    import paper_2606_02455_b200 as P
    from paper_2606_02455_b200 import build
    build.build()
    lib = P.load_library()
    header = open(os.path.join(ROOT, "include", "lsd.h")).read()
    declared = set(re.findall(r"^(?:lsd_status|void|const char\*|int64_t|int32_t)\s+(lsd_[a-z_]+)\s*\(", header, re.M))
    assert declared, "no declarations found"
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/lsd.h but not exported"
    assert set(P.EXPORTED_SYMBOLS) <= declared
    assert "sm_100a" in P.lsd_version()


def test_no_cpu_fallback_without_device():
    import torch
    import lsd_inputs as L
    import paper_2606_02455_b200 as P
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(P.LsdError) as ei:
        P.context_from_workload(L.make_workload("cfg1"))
    assert ei.value.status == -2


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_02455_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "lsd_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_02455_b200", src, re.M), f
            assert "liblsd_b200" not in src and "lsd.h" not in src, f
