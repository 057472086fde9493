"""CPU-only checks of the boundary: the C-ABI library builds, loads without a GPU and exports
every symbol include/tdlike.h declares; the binding names them all; no compute call is made."""
import os
import re
import subprocess

import pytest

from paper_2603_06010_b200 import binding as tdb
from paper_2603_06010_b200 import build as tdbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tdlike.h")
PROBE_HEADER = os.path.join(ROOT, "include", "tdprobe.h")


def _declared(header=HEADER):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(td_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_loads_without_gpu():
    path = tdbuild.build()
    assert os.path.exists(path)
    lib = tdb.load()
    assert lib.td_strerror(0) == b"ok"
    assert b"positive definite" in lib.td_strerror(tdb.TD_ENOTSPD)


def test_every_declared_symbol_is_exported_and_bound():
    names = _declared()
    assert {"td_create", "td_destroy", "td_loglike_batch", "td_inner_batch", "td_set_path", "td_get_info",
            "td_strerror"} <= set(names)
    nm = subprocess.run(["nm", "-D", "--defined-only", tdb.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r"\bT (td_[a-z0-9_]+)\b", nm))
    assert set(names) <= exported, set(names) - exported
    assert set(names) == set(tdb.SYMBOLS), set(names) ^ set(tdb.SYMBOLS)


def test_probe_library_is_separate_from_the_product_library():
    """include/tdprobe.h is served by the bench-only libtdprobe.so; the product library exports no probe."""
    names = _declared(PROBE_HEADER)
    assert names == ["td_probe_throughput"]
    nm = subprocess.run(["nm", "-D", "--defined-only", tdb.PROBE_LIB_PATH], capture_output=True, text=True, check=True).stdout
    assert set(names) <= set(re.findall(r"\bT (td_[a-z0-9_]+)\b", nm))
    nm = subprocess.run(["nm", "-D", "--defined-only", tdb.LIB_PATH], capture_output=True, text=True, check=True).stdout
    assert "probe" not in nm


def test_library_is_sm100a_with_no_other_arch():
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", tdb.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_binding_argument_validation_needs_no_gpu():
    import numpy as np
    with pytest.raises(ValueError):
        tdb.TDLikelihood(np.ones(5), [2, 2])          # lengths do not sum to the ACF size


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_06010_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    assert "paper_2603_06010_b200" not in open(os.path.join(ROOT, "oracle", "td_oracle.py")).read().replace(
        "paper_2603_06010_b200/csrc", "")
