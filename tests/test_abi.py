"""The C-ABI library loads and exports every symbol include/fcp.h declares; host-only entry
points report errors through status codes (no GPU needed)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_08476_b200.build import build
    return ctypes.CDLL(build())


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fcp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fcp_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), n
    import paper_2606_08476_b200 as m
    assert sorted(m.EXPORTS) == names


def test_status_codes(fcp):
    with pytest.raises(fcp.FcpError) as e:
        fcp.Plan([3, 4], 2)                       # C % N != 0
    assert e.value.status == -1
    with pytest.raises(fcp.FcpError):
        fcp.Plan([0, 4], 2)
    with pytest.raises(fcp.FcpError):
        fcp.Plan([4, 4], 2, imbalance_ppm=999_999)
    with pytest.raises(fcp.FcpError) as e:
        fcp.Plan([4, 4], 2, strategy=7)
    assert e.value.status == -2
    with pytest.raises(fcp.FcpError) as e:
        fcp.Sched.create([0, 4], [0], [0], [0, 4], 4, 2, 96)      # head_dim
    assert e.value.status == -2
    with pytest.raises(fcp.FcpError) as e:
        fcp.Sched.create([0, 4], [0], [0], [0, 4], 3, 2, 64)      # Hq % Hkv
    assert e.value.status == -2
    assert fcp.version().startswith("sm_100a")


def test_buffer_too_small_protocol(lib, fcp):
    p = fcp.Plan([512, 256, 128, 128], 2)
    n = ctypes.c_int32()
    st = lib.fcp_plan_shards(ctypes.c_void_p(p._h.value), -1, None, 0, ctypes.byref(n))
    assert st == -3 and n.value == 8
    assert len(p.shards()) == 8 and len(p.shards(0)) == 5 and len(p.shards(1)) == 3
