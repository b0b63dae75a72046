"""The C-ABI library loads and exports every symbol include/shd.h declares (no compute calls: CPU box)."""
import ctypes
import re
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def declared():
    names = set()
    for header in ("shd.h", "shd_bench.h"):          # the hot-path boundary and the measurement tooling
        text = (ROOT / "include" / header).read_text()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(shd_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_exported():
    from paper_2304_09139_b200 import build
    lib = ctypes.CDLL(str(build.build()))
    names = declared()
    assert "shd_create" in names and "shd_energy_grad" in names and "shd_smax" in names and "shd_minimize" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in shd.h but not exported"


def test_binding_lists_every_symbol():
    from paper_2304_09139_b200 import shd
    assert sorted(shd.EXPORTS) == declared()


def test_no_device_fails_loudly():
    """There is no CPU fallback: without a CUDA device shd_create reports SHD_ECUDA."""
    import torch
    if torch.cuda.is_available():
        return
    from paper_2304_09139_b200 import shd
    try:
        shd.Shd(2, 16, 4.0, m_star=4)
    except shd.ShdError as e:
        assert e.code == shd.SHD_ECUDA
    else:
        raise AssertionError("shd_create succeeded without a device")


def test_bad_arguments():
    from paper_2304_09139_b200 import shd
    h = ctypes.c_void_p()
    assert shd.lib.shd_create_shell(5, 16, 4.0, 4, None, ctypes.byref(h)) == shd.SHD_EINVAL   # d = 5 (D:R14)
    assert shd.lib.shd_create_shell(0, 16, 4.0, 4, None, ctypes.byref(h)) == shd.SHD_EINVAL
    assert shd.lib.shd_create_shell(2, 0, 4.0, 4, None, ctypes.byref(h)) == shd.SHD_EINVAL
    assert shd.lib.shd_create_shell(2, 16, -1.0, 4, None, ctypes.byref(h)) == shd.SHD_EINVAL
    assert shd.lib.shd_create(2, 16, 4.0, float("nan"), None, ctypes.byref(h)) == shd.SHD_EINVAL


def test_bench_reads_ncu_traffic_from_profiles():
    """bench.py's roofline.traffic is parsed from the newest committed ncu summary that states it (nothing hard-coded)."""
    import sys
    sys.path.insert(0, str(ROOT))
    import bench
    b, src = bench.ncu_traffic("k_grad8", "cfg4")
    assert src and src.startswith("profiles/r") and 1e8 < b < 1e11
    b2, src2 = bench.ncu_traffic("k_rho8", "cfg4")
    assert src2 == src and 1e8 < b2 < 1e11
    assert bench.ncu_traffic("k_grad8", "no_such_workload") == (None, None)
    assert bench.ncu_traffic("k_no_such_kernel", "cfg4") == (None, None)
