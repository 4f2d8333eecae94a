"""CPU-only checks of the boundary: the C-ABI library builds, loads without a GPU and exports every symbol that
include/gw.h declares; host-side argument validation works without touching a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gwlib():
    from paper_2206_07660_b200 import build as gwbuild
    gwbuild.build()
    import paper_2206_07660_b200 as gw
    return gw


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "gw.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(gw_[a-z0-9_]+)\s*\(", txt)))


def test_exports_every_declared_symbol(gwlib):
    syms = declared_symbols()
    assert {"gw_polarization", "gw_screened_interaction", "gw_selfenergy", "gw_exchange"} <= set(syms)
    L = ctypes.CDLL(gwlib.lib_path())
    for s in syms:
        assert hasattr(L, s), s


def test_no_torch_or_python_in_abi():
    txt = open(os.path.join(ROOT, "include", "gw.h")).read()
    assert "torch" not in re.sub(r"/\*.*?\*/", "", txt, flags=re.S).lower()
    assert "at::" not in txt and "pybind" not in txt.lower()


def test_strerror_and_version(gwlib):
    assert gwlib.gw_version() >= 100
    assert gwlib.gw_strerror(0) == "ok"
    assert "sm_100" in gwlib.gw_strerror(-3)
    assert "nw > ntau" in gwlib.gw_strerror(-4) and "positive definite" in gwlib.gw_strerror(-5)


def test_validation_without_device(gwlib):
    # host-only argument checks: bad sizes / null pointers are rejected before any CUDA call
    from paper_2206_07660_b200.binding import _CProblem
    L = gwlib.lib()
    c = _CProblem(2, 2, 2, 26, 100, 104, 104, 2, 0, 8, 700.0, None, None, None, None, 0)
    assert L.gw_polarization(ctypes.byref(c), None, None, None) == -1          # GW_EINVAL: null V
    c.V = 4096
    c.nao = 0
    assert L.gw_polarization(ctypes.byref(c), ctypes.c_void_p(4096), ctypes.c_void_p(4096), None) == -1
    c.nao = 26; c.q_begin = 5; c.q_end = 3
    assert L.gw_polarization(ctypes.byref(c), ctypes.c_void_p(4096), ctypes.c_void_p(4096), None) == -1
    c.q_begin = 0; c.q_end = 8; c.nao = 80
    assert L.gw_polarization(ctypes.byref(c), ctypes.c_void_p(4096), ctypes.c_void_p(4096), None) == -4   # GW_ESHAPE
    c.nao = 26
    # every documented GW_ESHAPE condition (gw.h), refused before any launch; the workspace query answers 0 for them
    for field, bad, good in (("ntau", 201, 104), ("nw", 105, 104), ("naux", 897, 100), ("nao", 65, 26)):
        setattr(c, field, bad)
        assert L.gw_polarization(ctypes.byref(c), ctypes.c_void_p(4096), ctypes.c_void_p(4096), None) == -4, field
        assert L.gw_workspace_bytes(ctypes.byref(c)) == 0, field
        setattr(c, field, good)
    c.ntau = 200; c.nw = 150; c.naux = 896; c.nao = 64          # the documented maxima are accepted by the planner
    assert L.gw_workspace_bytes(ctypes.byref(c)) > 0
    c.ntau = 104; c.nw = 104; c.naux = 100; c.nao = 26
    assert L.gw_polarization(ctypes.byref(c), ctypes.c_void_p(4097), ctypes.c_void_p(4096), None) == -1  # misaligned
    assert L.gw_workspace_bytes(ctypes.byref(c)) > 0
    assert L.gw_launch_count(ctypes.byref(c)) == 8


def test_missing_library_fails_loudly(monkeypatch, gwlib):
    import paper_2206_07660_b200.binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "_SO", "/nonexistent/libgw_b200.so")
    with pytest.raises(b.GWError):
        b.lib()


def test_product_path_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2206_07660_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "import oracle" not in txt and "gwref" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2206_07660_b200" not in txt.replace("paper_2206_07660_b200/csrc", ""), f


def test_every_documented_shape_is_plannable(gwlib):
    """gw.h documents nao <= 64, naux <= 896, nw <= ntau <= 200: the planners of all four stages must place every such problem
    (gw_workspace_bytes answers 0 as soon as one stage cannot)."""
    from paper_2206_07660_b200.binding import _CProblem
    L = gwlib.lib()
    bad = []
    for nao in range(1, 65):
        for naux in (1, 37, 200, 448, 449, 640, 896):
            for ntau, nw in ((8, 8), (200, 200), (200, 13)):
                c = _CProblem(2, 1, 3, nao, naux, ntau, nw, 2, 0, 6, 10.0, 4096, 4096, 4096, None, 0)
                if L.gw_workspace_bytes(ctypes.byref(c)) == 0:
                    bad.append((nao, naux, ntau, nw))
    assert not bad, bad[:10]


def test_traffic_recording_from_ncu_csv(tmp_path, monkeypatch):
    """bench.py --traffic-from-ncu: per-launch DRAM bytes of the two dominant kernels from an ncu --csv log, keyed by the kernel-source hash,
    optionally scaled to another config with the same mesh and basis (host logic only)."""
    import importlib.util
    import json
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    csv_path = tmp_path / "k.csv"
    hdr = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"\n'
    row = lambda i, k, m, u, v: f'"{i}","1","python","h","{k}","1","7","(512, 1, 1)","(148, 1, 1)","0","10.0","s","{m}","{u}","{v}"\n'
    csv_path.write_text(hdr + row(0, "void s1::p0_kernel<7, 1>(x)", "dram__bytes_read.sum", "Gbyte", "10") + row(0, "void s1::p0_kernel<7, 1>(x)", "dram__bytes_write.sum", "Gbyte", "2")
                        + row(1, "void s3w::sigma_ws_kernel<7>(x)", "dram__bytes_read.sum", "byte", "5000000000") + row(1, "void s3w::sigma_ws_kernel<7>(x)", "dram__bytes_write.sum", "byte", "1000000000"))
    monkeypatch.setattr(bench, "TRAFFIC_JSON", str(tmp_path / "traffic.json"))
    assert bench.traffic_from_ncu(str(csv_path), "cfgQ", "4") == 0
    rec = json.load(open(tmp_path / "traffic.json"))
    assert rec["cfgQ"]["stage1_bytes"] == 12e9 and rec["cfgQ"]["stage3_bytes"] == 6e9
    assert rec["cfg4"]["stage1_bytes"] == 12e9 * 15 and "scaled_from" in rec["cfg4"]
    assert bench.traffic_lookup("cfgQ", 0) == 12e9 and bench.traffic_lookup("cfg2", 0) is None
