"""CPU-side boundary checks: the C-ABI library loads and exports every symbol include/mdsm.h declares."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "mdsm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mdsm_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for n in ("mdsm_plan_create", "mdsm_rfi_clip", "mdsm_dedisperse", "mdsm_detect"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1307_5700_b200 import build
    path = build.build()
    lib = ctypes.CDLL(path)
    for n in _declared():
        assert hasattr(lib, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (mdsm_[a-z_0-9]+)\b", out))
    assert set(_declared()) <= exported


def test_binding_has_the_same_names():
    import paper_1307_5700_b200 as m
    for n in _declared():
        assert hasattr(m, n), n


def test_no_oracle_or_cpu_fallback_in_product_path():
    pkg = os.path.join(ROOT, "paper_1307_5700_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                s = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "mdsm_oracle" not in s, f
    s = "".join(open(os.path.join(ROOT, "oracle", f)).read() for f in ("__init__.py", "mdsm_oracle.c", "mdsm_oracle_next.c"))
    assert "import paper_1307_5700_b200" not in s and "from paper_1307_5700_b200" not in s and "mdsm.h" not in s


def test_plan_create_fails_loudly_without_a_gpu_or_with_bad_args():
    import torch
    import paper_1307_5700_b200 as m
    with pytest.raises(m.MdsmError):
        m.mdsm_plan_create(0, 64, 418.0, -0.3125, 51.2e-6, 4096, 0.0, 0.1, 32)       # nbeams < 1
    with pytest.raises(m.MdsmError):
        m.mdsm_plan_create(1, 64, 418.0, +0.3125, 51.2e-6, 4096, 0.0, 0.1, 32)       # foff >= 0
    with pytest.raises(m.MdsmError):
        m.mdsm_plan_create(1, 64, 418.0, -0.3125, 51.2e-6, 100, 0.0, 0.1, 32)        # nsamps <= max_delay
    if not torch.cuda.is_available():
        with pytest.raises(m.MdsmError):
            m.mdsm_plan_create(1, 64, 418.0, -0.3125, 51.2e-6, 4096, 0.0, 0.1, 32)   # no device: no fallback
