"""tcp_ring_remove_static: the allocation-free ring removal (scratch in a file-scope device array) against the
existing path (tcp_set_param(TCP_PARAM_RING_ALPHA) inside tcp_recon, scratch from cudaMalloc), on two calls in a row.
Collected last on purpose (the run is `pytest -x`); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import synthgen as sg

pytestmark = pytest.mark.gpu

# the tolerances test_gpu_parity.py puts on the sinogram workspace after pre-processing
SINO_TOL = {"f32": 3e-6, "f16": 2e-3}


def _ringy_inputs(w, rows, cols):
    """Seeded C2-like counts with miscalibrated detector columns (gain errors common to all projections: rings)."""
    raw, _ = sg.make_counts(w, rows)
    flat, dark, _, _ = sg.make_flat_dark(w, rows)
    raw = raw.astype(np.float64)
    for col, gain in cols:
        raw[:, :, col] = (raw[:, :, col] - dark[None, :, col]) * gain + dark[None, :, col]
    raw = np.clip(np.rint(raw), 0, 65535).astype(np.uint16)
    return (torch.from_numpy(raw.view(np.int16)).cuda().view(torch.uint16), torch.from_numpy(flat).cuda(),
            torch.from_numpy(dark).cuda(), torch.from_numpy(w.theta).cuda())


def _existing_path(tcp, w, nz, dtype, dev, alpha):
    """(p, p with rings removed) of the context path: S1+S2 into the sinogram workspace, then the ring step of tcp_recon."""
    r = tcp.Recon(w.n, w.nproj, nz, w.center, dtype, w.filter, 3)
    p = r.normalize(dev[0], dev[1], dev[2]).clone()
    r.set_ring(alpha)
    r.recon(*dev)
    after = r.workspace("sinogram").clone()
    r.close()
    return p, after


@pytest.mark.parametrize("dtype", ["f32", "f16"])
def test_ring_remove_static_matches_context_path_twice(dtype):
    import paper_2209_08450_b200 as tcp
    w = sg.make_workload("C2", scale=4)
    # call 1: 5 slices out of place; call 2: 3 other slices, another alpha, IN PLACE, right behind it on the same stream
    # (different shapes: the second call finds the first one's values at other offsets of the shared scratch array)
    cases = [(list(range(30, 35)), [(40, 1.02), (77, 0.97)], 2e-3, False),
             (list(range(50, 53)), [(10, 0.98), (64, 1.03), (101, 1.01)], 5e-4, True)]
    tcp.tcp_ring_static_setup()
    prepared = []
    for rows, cols, alpha, inplace in cases:
        dev = _ringy_inputs(w, rows, cols)
        p, want = _existing_path(tcp, w, len(rows), dtype, dev, alpha)
        assert float((want.float() - p.float()).abs().max()) > 5e-3          # the step matters on this input
        prepared.append((p, want, alpha, inplace, torch.empty_like(p)))
    # warm the kernels (module loading may allocate), then the two calls in a row with free device memory watched
    tcp.tcp_ring_remove_static(prepared[0][0], prepared[0][4], prepared[0][2])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    outs = []
    for p, want, alpha, inplace, buf in prepared:
        if inplace:
            buf.copy_(p)
            tcp.tcp_ring_remove_static(buf, buf, alpha)
        else:
            buf.fill_(float("nan"))
            tcp.tcp_ring_remove_static(p, buf, alpha)
        outs.append(buf)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                              # nothing was allocated
    for (p, want, alpha, inplace, _), got in zip(prepared, outs):
        assert got.dtype == want.dtype and got.shape == want.shape
        err = float((got.double() - want.double()).abs().max())
        assert err <= SINO_TOL[dtype] * max(1.0, float(want.float().abs().max())), (dtype, inplace, err)


def test_ring_remove_static_rejects_what_it_cannot_hold():
    import paper_2209_08450_b200 as tcp
    x = torch.zeros((33, 4, 2048), dtype=torch.float32, device="cuda")        # nz * n = 67584 > 65536
    with pytest.raises(tcp.TcpError, match="TCP_RING_STATIC_MAX"):
        tcp.tcp_ring_remove_static(x, x, 1e-3)
    ok = torch.zeros((32, 4, 2048), dtype=torch.float32, device="cuda")       # exactly the limit
    tcp.tcp_ring_remove_static(ok, ok, 1e-3)
    torch.cuda.synchronize()
    assert float(ok.abs().max()) == 0.0
    for bad in (0.0, -1.0, float("nan")):
        with pytest.raises(tcp.TcpError):
            tcp.tcp_ring_remove_static(ok, ok, bad)
    with pytest.raises(tcp.TcpError):
        tcp.tcp_ring_remove_static(ok, ok.half(), 1e-3)                       # mixed types
    with pytest.raises(tcp.TcpError):
        tcp.tcp_ring_remove_static(ok.cpu(), ok.cpu(), 1e-3)                  # host tensors
