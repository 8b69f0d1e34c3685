"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/prefixflow.h declares; host-only entry points behave.  No compute call is made."""
import ctypes
import os
import re

from paper_2606_01143_b200 import binding as pf
from paper_2606_01143_b200 import build as pf_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "prefixflow.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pf_[a-zA-Z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    pf_build.build_library()
    L = ctypes.CDLL(pf_build.SO_PATH)
    names = declared_symbols()
    assert len(names) >= 14
    for n in names:
        assert hasattr(L, n), f"{n} declared in prefixflow.h but not exported"
    assert set(names) == set(pf.SYMBOLS)


def test_version_and_workspace_bytes_are_host_only():
    assert pf.pf_version() >= 100
    d = pf.make_desc(28, 4, 128)
    small = pf.pf_workspace_bytes(d, 1024, 256)
    big = pf.pf_workspace_bytes(d, 5120, 1024)
    assert 0 < small < big
    assert pf.pf_workspace_bytes(d, -1, 0) == 0


def test_static_scratch_limits_are_host_only():
    """pf_causal_bwd_static's limit is computable without a GPU: 32 MiB / bytes per token, a multiple of 64."""
    assert pf.pf_static_scratch_bytes() == 32 << 20
    d = pf.make_desc(28, 4, 128)
    cap = pf.pf_causal_bwd_static_max_tokens(d)
    per_tok = 8 * 28 + 4 * 28 * 128 + 8 * 4 * 128
    assert cap % 64 == 0 and cap == ((32 << 20) - 6 * 256) // per_tok // 64 * 64 == 1792
    assert pf.pf_causal_bwd_static_max_tokens(pf.make_desc(2, 2, 64)) > cap
    assert pf.pf_workspace_bytes(d, cap, 0) > 32 << 20 >= cap * per_tok   # the caller-side formula keeps 16 x 64 spare rows


def test_struct_layout_matches_header():
    assert ctypes.sizeof(pf.pf_desc) == 16
    assert ctypes.sizeof(pf.pf_tensor) == 24
