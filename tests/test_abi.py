"""The C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol include/wolff.h declares."""
import ctypes
import os
import re

import pytest

from paper_1110_0899_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "wolff.h")).read()
    return sorted(set(re.findall(r"WOLFF_API[^;(]*?\b(wolff_\w+)\s*\(", text)))


def test_header_declares_the_calls_north_star_names():
    syms = declared_symbols()
    for required in ("wolff_create", "wolff_run", "wolff_observables", "wolff_get_spins", "wolff_destroy"):
        assert required in syms
    assert sorted(binding._SIGNATURES) == syms      # the Python binding has the same names, no more, no fewer


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert binding.load() is not None


def test_built_for_sm_100a_only():
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_argument_validation_needs_no_gpu():
    lib = binding.load()
    for args in [(1, 8, 1.0, 1.0, 0), (2, 1, 1.0, 1.0, 0), (2, 8, -1.0, 1.0, 0), (2, 8, 1.0, 0.0, 0), (3, 4096, 1.0, 1.0, 0)]:
        assert not lib.wolff_create(*args)
        assert binding.last_error()
    assert lib.wolff_run(None, 1, None) == binding.WOLFF_EINVAL
    assert lib.wolff_destroy(None) == binding.WOLFF_OK


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1110_0899_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "wolff_oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert "paper_1110_0899_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_1110_0899_b200``", "").replace("paper_1110_0899_b200/csrc/", ""), f


def test_header_documents_every_option_key_the_library_accepts():
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    api = open(os.path.join(root, "paper_1110_0899_b200", "csrc", "api.cu")).read()
    header = open(os.path.join(root, "include", "wolff.h")).read()
    keys = set(re.findall(r'!strcmp\(key, "([a-z_]+)"\)', api))
    assert len(keys) >= 15
    missing = sorted(k for k in keys if '"%s"' % k not in header)
    assert not missing, "option keys accepted by wolff_set_option but not documented in include/wolff.h: %s" % missing
