"""CPU checks of the boundary: libccake.so builds for sm_100a, loads, and exports every symbol include/ccake.h
declares; the binding restates the header's ids; the library refuses to run without a CUDA device (no fallback)."""
import ctypes as C
import os
import re

import pytest

from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import build as cuda_build
from paper_2511_22852_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ccake.h")


def _header_text():
    with open(HEADER) as fh:
        return fh.read()


def test_library_builds_and_exports_every_declared_symbol():
    cuda_build.build()
    L = B.lib()
    declared = set(re.findall(r"\b(ccake_[a-z0-9_]+)\s*\(", re.sub(r"/\*.*?\*/", "", _header_text(), flags=re.S)))
    assert declared, "no declarations found in include/ccake.h"
    for name in declared:
        assert hasattr(L, name), f"libccake.so does not export {name}"
    assert declared == set(B.EXPORTS), (declared ^ set(B.EXPORTS))


def test_binding_restates_header_ids():
    txt = re.sub(r"/\*.*?\*/", "", _header_text(), flags=re.S)
    ids = {}
    for body in re.findall(r"enum\s*\{(.*?)\}", txt, flags=re.S):
        nxt = 0
        for item in body.split(","):
            item = item.strip()
            if not item:
                continue
            m = re.match(r"(\w+)\s*(?:=\s*(-?\w+))?$", item)
            assert m, item
            if m.group(2) is not None:
                nxt = ids[m.group(2)] if m.group(2) in ids else int(m.group(2), 0)
            ids[m.group(1)] = nxt
            nxt += 1
    for name, val in ids.items():
        short = name.replace("CCAKE_", "")
        if short.startswith("COL_") or short in ("NCOLS_MAX",):
            continue
        if hasattr(B, short):
            assert getattr(B, short) == val, (name, val, getattr(B, short))
    assert ids["CCAKE_NSTATE"] == B.NSTATE == 28 and ids["CCAKE_RATE"] == B.RATE
    assert [ids[f"CCAKE_COL_{c}"] for c in ("T", "MUB", "MUS", "MUQ", "P", "CS2", "E", "WS", "WB", "WSQ", "WQ")] == list(range(11))


def test_params_struct_layout_matches_header():
    """sizeof(ccake_params): 8 int32 + pointer + 13 doubles + 9 + 3 + 8 doubles."""
    assert C.sizeof(B.Params) == 8 * 4 + 8 + 8 * (13 + 9 + 3 + 8)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(B.CcakeError) as e:
        B.Ccake(**W.base_params())
    assert e.value.rc == B.ECUDA


def test_null_arguments_are_rejected_without_a_device():
    L = B.lib()
    assert L.ccake_create(None, None) == B.EINVAL
    assert L.ccake_step(None, 1) == B.EINVAL
    assert L.ccake_destroy(None) == B.OK
    assert L.ccake_last_error(None) == b"null context"
