"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/tcp.h declares; calls fail loudly without a GPU (no CPU fallback); the product
package never imports the oracle; the bench's roofline model is consistent with DESIGN.md."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_header_symbols():
    from paper_2209_08450_b200 import build as b
    so = b.build()
    assert os.path.exists(so)
    import paper_2209_08450_b200 as tcp
    L = tcp.lib()
    header = open(os.path.join(ROOT, "include", "tcp.h")).read()
    declared = set(re.findall(r"\b(tcp_[a-z0-9_]+)\s*\(", header)) - {"tcp_set_option(ctx"}
    declared = {d for d in declared if not d.startswith("tcp_ctx") and d != "tcp_stream_t"}
    assert declared == set(tcp.EXPORTS), declared ^ set(tcp.EXPORTS)
    for s in declared:
        assert hasattr(L, s), s
    # sm_100a SASS is embedded
    out = subprocess.run(["cuobjdump", "--list-elf", so], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2209_08450_b200 as tcp
    with pytest.raises(tcp.TcpError, match="no usable CUDA device"):
        tcp.tcp_create(128, 180, 8, 64.0, "f32", "shepp")
    with pytest.raises(tcp.TcpError):
        tcp.Recon(128, 180, 8, 64.0)


def test_product_never_imports_oracle_and_oracle_never_imports_product():
    pkg = os.path.join(ROOT, "paper_2209_08450_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "oracle" not in src.lower().replace("no cpu fallback", ""), os.path.join(dp, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2209_08450_b200" not in src and "libtcp" not in src
            assert "_work" not in src


def test_stage_model_matches_survey_bytes_per_voxel():
    sys.path.insert(0, ROOT)
    import bench
    import synthgen as sg
    w = sg.make_workload.__wrapped__("C4") if hasattr(sg.make_workload, "__wrapped__") else None
    # avoid building the 500-ellipsoid phantom: a stub with the sizes is enough
    class W:  # noqa: D401
        n, nproj = 2048, 2048
    model = bench.stage_model(W, 16, 4, True, True)
    per_voxel = sum(v["bytes"] for v in model.values()) / (16 * 2048 * 2048)
    # 2 rho + 2 rho B_r + 2 rho B_c + 6 B_c + B_o = 40 B/voxel at rho = 1, fp16
    assert per_voxel == pytest.approx(40.0, rel=1e-12)
    flops = sum(v["flops"] for v in model.values()) / (16 * 2048 * 2048)
    assert 600 < flops < 660      # ~620 flop/voxel at m = 4


def test_slice_range_host_logic():
    """tcp_slice_range: contiguous, in rank order, sizes differ by at most one, empty ranges when world > nz_total."""
    import paper_2209_08450_b200 as tcp
    for nz, world in [(2048, 1), (2048, 8), (2049, 8), (10, 3), (3, 8), (0, 2)]:
        rs = [tcp.tcp_slice_range(nz, r, world) for r in range(world)]
        assert rs[0][0] == 0 and rs[-1][1] == nz
        assert all(rs[i][1] == rs[i + 1][0] for i in range(world - 1))
        sizes = [b - a for a, b in rs]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    for bad in [(10, 2, 2), (10, -1, 2), (10, 0, 0), (-1, 0, 1)]:
        with pytest.raises(tcp.TcpError):
            tcp.tcp_slice_range(*bad)


def test_check_angles_host_logic():
    import numpy as np
    import paper_2209_08450_b200 as tcp
    tcp.tcp_check_angles(np.linspace(0, np.pi, 180, endpoint=False).astype(np.float32))
    tcp.tcp_check_angles(np.array([0.3], np.float32))
    tcp.tcp_check_angles(np.linspace(-1.0, 2.0, 50).astype(np.float32))           # any start, span < pi
    for bad in (np.linspace(0, 2 * np.pi, 360, endpoint=False), np.array([0.0, 0.2, 0.2, 0.4]), np.array([0.5, 0.4]),
                np.array([0.0, np.nan, 1.0]), np.array([0.0, np.inf]), np.array([0.0, np.pi])):
        with pytest.raises(tcp.TcpError):
            tcp.tcp_check_angles(bad.astype(np.float32))
