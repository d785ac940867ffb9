"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Gates (BASELINE.json north_star): fp32 vs oracle gridding <= 1e-5
rel-L2 per slice; fp16 <= 5e-3 rel-L2 and <= 1e-2 max-abs on the normalised volume."""
import numpy as np
import pytest
import torch

import oracle as orc
import synthgen as sg

pytestmark = pytest.mark.gpu

FP32_GATE = 1e-5
FP32_GATE_MAX = 5e-5     # of max |oracle|: fp32 rounding of ~40 sequential stages, see DESIGN.md section 3
FP16_GATE_L2 = 5e-3
FP16_GATE_MAX = 1e-2


def rl2(a, b):
    a = np.asarray(a).astype(np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64)
    b = np.asarray(b).astype(a.dtype)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def check(got, ref, dtype="f32", vol=None, tag=None):
    """One slice against the oracle at north_star's gates.  fp32: rel-L2 <= 1e-5 (north_star) AND, element by element,
    max-abs <= FP32_GATE_MAX of max |oracle| over the volume `vol` (a norm alone lets a single wrong
    pixel through at n >= 512).  fp16 storage: rel-L2 <= 5e-3 and max-abs <= 1e-2 of max |oracle|."""
    scale = float(np.abs(ref if vol is None else vol).max())
    e2, emax = rl2(got, ref), float(np.abs(np.asarray(got, np.float64) - ref).max()) / scale
    if dtype == "f32":
        assert e2 < FP32_GATE and emax < FP32_GATE_MAX, (tag, e2, emax)
    else:
        assert e2 < FP16_GATE_L2 and emax < FP16_GATE_MAX, (tag, e2, emax)


def _tcp():
    import paper_2209_08450_b200 as tcp
    return tcp


def _inputs(w, rows):
    raw, _ = sg.make_counts(w, rows)
    flat, dark, _, _ = sg.make_flat_dark(w, rows)
    return raw, flat, dark, w.theta


def _to_dev(raw, flat, dark, theta):
    return (torch.from_numpy(raw.view(np.int16)).cuda().view(torch.uint16), torch.from_numpy(flat).cuda(),
            torch.from_numpy(dark).cuda(), torch.from_numpy(theta).cuda())


def _gpu_recon(w, rows, dtype, m=3, filt=None, impl=None, keep=False):
    tcp = _tcp()
    raw, flat, dark, theta = _inputs(w, rows)
    r = tcp.Recon(w.n, w.nproj, len(rows), w.center, dtype, filt or w.filter, m)
    if impl is not None:        # default: "tile" for f32, "mma" (tensor cores) for fp16 storage
        r.set_grid_impl(impl)
    out = r.recon(*_to_dev(raw, flat, dark, theta))
    torch.cuda.synchronize()
    res = out.float().cpu().numpy()
    if keep:
        return res, r, (raw, flat, dark, theta)
    r.close()
    return res, None, (raw, flat, dark, theta)


# ------------------------------------------------------------------ the tensor-core transform on its own
@pytest.mark.parametrize("inverse", [False, True])
def test_mma_fft_lines_against_the_dft(inverse):
    """tcp_fft_lines: the length-4096 transform whose radix-16 butterflies run as mma.sync products (mmafft.cuh), on its
    own, against the DFT definition in fp64 (numpy.fft of the same fp16 inputs; the oracle's orc.fft on the first lines).
    Index and sign conventions: a delta at i0 gives e^{-/+ 2 pi i k i0 / N} exactly; a constant gives N delta_k.  Random
    lines: operands are rounded to fp16 once per pass, so rel-L2 stays at a few 2^-11."""
    tcp = _tcp()
    N, B = 4096, 24
    rng = np.random.default_rng(5)
    x = (rng.standard_normal((B, N)) + 1j * rng.standard_normal((B, N)))
    x[0] = 0; x[0, 1] = 1.0                       # delta at 1
    x[1] = 0; x[1, 2049] = 1j                     # delta in the upper half
    x[2] = 1.0 - 0.5j                             # constant
    x[3, N // 2:] = 0                             # zero-padded, as the row kernel's inputs
    x[4] *= 100.0                                 # large
    x[5] *= 1e-2                                  # small
    xh = np.stack([x.real, x.imag], -1).astype(np.float16)
    xq = xh[..., 0].astype(np.float64) + 1j * xh[..., 1].astype(np.float64)
    r = tcp.Recon(2048, 8, 2, 1024.0, "f16", "ramp")
    got = r.fft_lines(torch.from_numpy(xh).cuda(), inverse=inverse).cpu().numpy().astype(np.complex128)
    r.close()
    ref = np.fft.ifft(xq, axis=1) * N if inverse else np.fft.fft(xq, axis=1)
    for b in range(2):
        o = orc.fft(xq[b], sign=+1 if inverse else -1)
        assert rl2(o, ref[b]) < 1e-12
    for b in range(B):
        assert rl2(got[b], ref[b]) < 1.5e-3, (b, rl2(got[b], ref[b]))
    assert np.abs(got[0] - ref[0]).max() < 2e-3 and np.abs(got[2] - ref[2]).max() < 2e-3 * N


# ------------------------------------------------------------------ C1, stage by stage
@pytest.mark.parametrize("m", [3, 4, 16 + 2, 16 + 3])
def test_c1_fp32_stages_and_volume(m):
    """m: kernel code (3, 4: Gaussian half-width; 16 + 2, 16 + 3: Kaiser-Bessel window, reading Q21)."""
    w = sg.make_workload("C1")
    rows = list(range(w.nz_total))
    out, r, (raw, flat, dark, theta) = _gpu_recon(w, rows, "f32", m=m, keep=True)
    n, M = w.n, 2 * w.n
    # S1+S2
    p = orc.neglog(raw, flat, dark)
    sino = r.workspace("sinogram").cpu().numpy()
    assert np.abs(sino - p).max() < 2e-6 * max(1.0, np.abs(p).max())
    # S3+S4 (pairs packed: slice 2p real, 2p+1 imaginary)
    spec = r.workspace("spectrum").cpu().numpy()
    for pair in (0, 3):
        GA = orc.spectrum(orc.filter_rows(p[2 * pair], w.filter), w.center)
        GB = orc.spectrum(orc.filter_rows(p[2 * pair + 1], w.filter), w.center)
        assert rl2(spec[pair], GA + 1j * GB) < 2e-6
    # S5
    grid = r.workspace("grid").cpu().numpy()
    GA = orc.spectrum(orc.filter_rows(p[0], w.filter), w.center)
    GB = orc.spectrum(orc.filter_rows(p[1], w.filter), w.center)
    Fo = orc.grid(GA + 1j * GB, theta, n, m)
    assert rl2(grid[0], Fo) < 3e-6
    # S1..S7
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, m, "grid")
    for z in rows:
        check(out[z], ref[z], "f32")
    r.close()


@pytest.mark.parametrize("dtype", ["f32", "f16", "f16_out32"])
@pytest.mark.parametrize("cfg,scale,nz", [("C1", 1, 8), ("C2", 4, 5), ("C3", 4, 18)])
def test_kaiser_bessel_kernel(dtype, cfg, scale, nz):
    """The half-width-2 Kaiser-Bessel kernel (tcp_create_ex code 16 + 2: 16 taps per sample instead of 36) through both
    production griddings (CUDA-core tile kernel for fp32, tensor cores for fp16 storage) against the oracle with the same
    kernel code, at the gates of north_star; odd and multi-group chunks, an off-centre axis (C3)."""
    w = sg.make_workload(cfg, scale=scale)
    rows = list(range(min(nz, w.nz_total)))
    out, _, (raw, flat, dark, theta) = _gpu_recon(w, rows, dtype, m=16 + 2)
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 16 + 2, "grid")
    for z in range(len(rows)):
        check(out[z], ref[z], "f32" if dtype == "f32" else dtype, vol=ref, tag=z)
    tcp = _tcp()
    r = tcp.Recon(w.n, w.nproj, 2, w.center, dtype, w.filter, 16 + 2)
    for impl in ("gather", "scatter"):
        with pytest.raises(tcp.TcpError):
            r.set_grid_impl(impl)
    r.close()
    for bad in (16 + 4, 16 + 1, 32 + 2, 2):
        with pytest.raises(tcp.TcpError):
            tcp.tcp_create_ex(w.n, w.nproj, 2, w.center, dtype, w.filter, bad)


def test_c1_gridding_implementations_agree():
    """tile (default), per-cell gather and fp32-atomic scatter compute the same sum."""
    w = sg.make_workload("C1")
    rows = list(range(w.nz_total))
    t, _, _ = _gpu_recon(w, rows, "f32", impl="tile")
    a, _, _ = _gpu_recon(w, rows, "f32", impl="gather")
    b, _, _ = _gpu_recon(w, rows, "f32", impl="scatter")
    assert rl2(a, b) < 3e-6
    assert rl2(t, a) < 3e-6
    th, _, _ = _gpu_recon(w, rows, "f16", impl="tile")
    ah, _, _ = _gpu_recon(w, rows, "f16", impl="gather")
    mh, _, _ = _gpu_recon(w, rows, "f16", impl="mma")
    assert rl2(th, ah) < 2e-3
    # tile (FHFMA) and mma (tcgen05) accumulate in fp32; mma rounds wx, wy and wx*wy to fp16 (three roundings, tile one)
    assert rl2(mh, th) < 1e-3


@pytest.mark.parametrize("dtype,nz", [("f32", 18), ("f16", 18), ("f16", 5), ("f16", 32), ("f16", 36)])
def test_several_pair_groups_and_ragged_chunk(dtype, nz):
    """nz = 18 -> 9 slice pairs = two pair groups of 8 (tile) / one of 16 (mma), ragged; nz = 5 -> odd;
    nz = 32 -> one full group of 16 pairs; nz = 36 -> 18 pairs = two mma groups."""
    w = sg.make_workload("C2", scale=4)
    rows = list(range(40, 40 + nz))
    out, _, (raw, flat, dark, theta) = _gpu_recon(w, rows, dtype)
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid")
    for z in range(nz):
        check(out[z], ref[z], dtype, vol=ref, tag=z)


def test_limited_and_uneven_angles():
    """theta increasing but neither equispaced nor spanning [0, pi): the projection windows of the
    tiles and the split of the near-DC tiles must not depend on an even spread.  (The counts are
    those of the equispaced scan: parity against the oracle does not need a meaningful image.)"""
    tcp = _tcp()
    w = sg.make_workload("C1")
    rng = np.random.default_rng(5)
    th = np.sort(rng.uniform(0.3, 2.6, w.nproj)).astype(np.float32)
    raw, flat, dark, _ = _inputs(w, [2, 3])
    r = tcp.Recon(w.n, w.nproj, 2, w.center, "f32", w.filter, 3)
    out = r.recon(*_to_dev(raw, flat, dark, th))
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    r.close()
    ref = orc.recon(raw, flat, dark, th, w.center, w.filter, 3, "grid")
    for z in range(2):
        check(out[z], ref[z], "f32")


def test_c1_fp16_grid_stage_strip_layout():
    """fp16 storage: the tcgen05 gridding writes the grid strip-major (tcp_grid_strip); read back in
    row-major order it must equal the oracle's gridding of the oracle's spectrum to fp16 accuracy."""
    w = sg.make_workload("C1")
    rows = list(range(w.nz_total))
    out, r, (raw, flat, dark, theta) = _gpu_recon(w, rows, "f16", keep=True)
    assert r.grid_strip > 0
    p = orc.neglog(raw, flat, dark)
    for pair in (0, 2):
        GA = orc.spectrum(orc.filter_rows(p[2 * pair], w.filter), w.center)
        GB = orc.spectrum(orc.filter_rows(p[2 * pair + 1], w.filter), w.center)
        Fo = orc.grid(GA + 1j * GB, theta, w.n, 3)
        got = r.workspace("grid").cpu().numpy()[pair] / r.scale
        assert rl2(got, Fo) < 2e-3
    r.set_grid_impl("tile")
    assert r.grid_strip == 0
    r.close()


@pytest.mark.parametrize("dtype", ["f16", "f16_out32"])
def test_c1_fp16(dtype):
    w = sg.make_workload("C1")
    rows = list(range(w.nz_total))
    out, _, (raw, flat, dark, theta) = _gpu_recon(w, rows, dtype)
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid")
    scale = np.abs(ref).max()
    for z in rows:
        assert rl2(out[z], ref[z]) < FP16_GATE_L2
    assert np.abs(out - ref).max() / scale < FP16_GATE_MAX


# ------------------------------------------------------------------ other sizes / filters / centres
@pytest.mark.parametrize("cfg,scale,dtype", [
    ("C2", 8, "f32"), ("C2", 4, "f32"), ("C2", 2, "f32"), ("C2", 2, "f16"),
    ("C3", 8, "f32"), ("C3", 4, "f16"), ("C4", 16, "f16"), ("C4", 8, "f32"), ("C5", 16, "f16_out32"),
    ("C2", 1, "f32"), ("C2", 1, "f16"), ("C3", 1, "f16"),
])
def test_downscaled_configs(cfg, scale, dtype):
    w = sg.make_workload(cfg, scale=scale)
    # pairs of ADJACENT slices, as in a real chunk: the two slices of a pair share one complex
    # transform, so rounding error is relative to the larger of the two
    h = w.nz_total // 2
    rows = [0, 1, h, h + 1, w.nz_total - 2, w.nz_total - 1]
    out, _, (raw, flat, dark, theta) = _gpu_recon(w, rows, dtype)
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid")
    if dtype == "f32":
        for z in range(len(rows)):
            check(out[z], ref[z], "f32")
    else:
        for z in range(len(rows)):
            assert rl2(out[z], ref[z]) < FP16_GATE_L2, (cfg, scale, z, rl2(out[z], ref[z]))
        assert np.abs(out - ref).max() / np.abs(ref).max() < FP16_GATE_MAX


@pytest.mark.parametrize("filt", ["ramp", "shepp", "parzen", "cosine", "hann", "hamming"])
def test_filters_and_offcentre(filt):
    w = sg.make_workload("C1")
    w.center = 61.75
    rows = [3, 4]
    out, _, (raw, flat, dark, theta) = _gpu_recon(w, rows, "f32", filt=filt)
    ref = orc.recon(raw, flat, dark, theta, w.center, filt, 3, "grid")
    for z in range(2):
        check(out[z], ref[z], "f32")


@pytest.mark.parametrize("dtype", ["f32", "f16"])
def test_centre_try_mode(dtype):
    """tcp_recon_try: one slice, several candidate centres in one call.  Entry i must equal the
    oracle's reconstruction of that slice with centre centers[i] (odd count: the last pair carries one
    centre; non-integer centres included), and an out-of-range centre or count is refused."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    raw, flat, dark, theta = _inputs(w, [4])
    centers = [61.0, 64.0, 66.5, 63.25, 70.0]
    r = tcp.Recon(w.n, w.nproj, 8, w.center, dtype, w.filter, 3)
    d = _to_dev(raw, flat, dark, theta)
    out = r.recon_try(d[0], d[1], d[2], d[3], centers)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    assert out.shape == (len(centers), w.n, w.n)
    for i, c in enumerate(centers):
        ref = orc.recon(raw, flat, dark, theta, c, w.filter, 3, "grid")[0]
        if dtype == "f32":
            check(out[i], ref, "f32")
        else:
            assert rl2(out[i], ref) < FP16_GATE_L2, (c, rl2(out[i], ref))
            assert np.abs(out[i] - ref).max() / np.abs(ref).max() < FP16_GATE_MAX
    # the context still reconstructs chunks afterwards (the try tables are per call)
    raw8, flat8, dark8, _ = _inputs(w, list(range(8)))
    full = r.recon(*_to_dev(raw8, flat8, dark8, theta)).float().cpu().numpy()
    ref8 = orc.recon(raw8[:, 4:5], flat8[4:5], dark8[4:5], theta, w.center, w.filter, 3, "grid")[0]
    check(full[4], ref8, dtype)
    with pytest.raises(tcp.TcpError):
        r.recon_try(d[0], d[1], d[2], d[3], [float(w.n)])
    with pytest.raises(tcp.TcpError):
        r.recon_try(d[0], d[1], d[2], d[3], [64.0] * 9)
    r.close()


@pytest.mark.parametrize("dtype,cfg,scale,nz", [("f32", "C1", 1, 8), ("f16", "C1", 1, 5), ("f32", "C2", 2, 3), ("f16", "C3", 4, 10)])
def test_line_summation_operator(dtype, cfg, scale, nz):
    """TCP_ALG_LINE (the paper's LineRec): filtered sinogram backprojected by direct
    line summation with linear interpolation, against the oracle's B_lin (pinned by P5, P6, P8) on the same
    counts: C1 as is, C2 / C3 down-scaled (off-centre C3, ragged slice groups)."""
    tcp = _tcp()
    w = sg.make_workload(cfg, scale=scale) if scale > 1 else sg.make_workload(cfg)
    rows = list(range(w.nz_total // 2 - nz // 2, w.nz_total // 2 - nz // 2 + nz))
    raw, flat, dark, theta = _inputs(w, rows)
    r = tcp.Recon(w.n, w.nproj, nz, w.center, dtype, w.filter, 3)
    r.set_algorithm("line")
    out = r.recon(*_to_dev(raw, flat, dark, theta))
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "lin")
    scale_v = np.abs(ref).max()
    for z in range(nz):
        if dtype == "f32":
            check(out[z], ref[z], "f32")
        else:
            assert rl2(out[z], ref[z]) < FP16_GATE_L2, (z, rl2(out[z], ref[z]))
            assert np.abs(out[z] - ref[z]).max() / scale_v < FP16_GATE_MAX
    # back to FourierRec on the same context
    r.set_algorithm("fourier")
    out2 = r.recon(*_to_dev(raw, flat, dark, theta)).float().cpu().numpy()
    ref2 = orc.recon(raw[:, :1], flat[:1], dark[:1], theta, w.center, w.filter, 3, "grid")[0]
    check(out2[0], ref2, dtype)
    r.close()


@pytest.mark.parametrize("dtype,alg", [("f32", "fourier"), ("f16", "fourier"), ("f32", "line")])
def test_edge_padding(dtype, alg):
    """TCP_OPT_PAD = edge against the oracle with pad="edge", on rows whose edge values are far
    from zero (C1 counts with the centre pushed off so the phantom touches the detector edge), for both
    backprojection operators; and back to zero padding on the same context."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    w.center = 40.0
    raw, flat, dark, theta = _inputs(w, [2, 3, 4])
    r = tcp.Recon(w.n, w.nproj, 3, w.center, dtype, w.filter, 3)
    r.set_pad("edge")
    r.set_algorithm(alg)
    dev = _to_dev(raw, flat, dark, theta)
    out = r.recon(*dev).float().cpu().numpy()
    method = "grid" if alg == "fourier" else "lin"
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, method, pad="edge")
    refz = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, method)
    assert rl2(ref[1], refz[1]) > 1e-2                       # the option matters on this input
    for z in range(3):
        check(out[z], ref[z], dtype, vol=ref, tag=z)
    r.set_pad("zero")
    outz = r.recon(*dev).float().cpu().numpy()
    for z in range(3):
        check(outz[z], refz[z], dtype, vol=refz, tag=z)
    r.close()


@pytest.mark.parametrize("dtype", ["f32", "f16"])
def test_recon_under_cuda_graph_capture(dtype):
    """tcp_recon only enqueues kernels on the caller's stream (no allocation, no host sync), so a chunk can be
    captured into a CUDA graph and replayed: the small configs are launch-bound (8 launches of a few
    microseconds each).  The replay on new data must equal the eager call bit for bit."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    raw, flat, dark, theta = _inputs(w, list(range(8)))
    d = list(_to_dev(raw, flat, dark, theta))
    r = tcp.Recon(w.n, w.nproj, 8, w.center, dtype, w.filter, 3)
    eager = r.recon(*d).clone()
    static_raw = torch.zeros_like(d[0].view(torch.int16))
    out = torch.empty_like(eager)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        r.recon(static_raw.view(torch.uint16), d[1], d[2], d[3], out=out, stream=side)      # warm-up outside capture
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        r.recon(static_raw.view(torch.uint16), d[1], d[2], d[3], out=out, stream=torch.cuda.current_stream())
    static_raw.copy_(d[0].view(torch.int16))
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager)
    ref = orc.recon(raw[:, :1], flat[:1], dark[:1], theta, w.center, w.filter, 3, "grid")[0]
    check(out[0].float().cpu().numpy(), ref, dtype)
    r.close()


@pytest.mark.parametrize("dtype,pad", [("f32", "zero"), ("f32", "edge"), ("f16", "zero")])
def test_fused_filter_option(dtype, pad):
    """TCP_OPT_FILTER_FUSED (the uncropped reading of S3 + S4, one transform per row) against the oracle with
    fused=True; it is a different image from the default chain, which the same context still produces after
    the option is switched off."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    w.center = 58.5
    raw, flat, dark, theta = _inputs(w, [1, 2, 3, 4, 5])
    r = tcp.Recon(w.n, w.nproj, 5, w.center, dtype, w.filter, 3)
    r.set_filter_fused(True)
    r.set_pad(pad)
    dev = _to_dev(raw, flat, dark, theta)
    out = r.recon(*dev).float().cpu().numpy()
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid", pad=pad, fused=True)
    lit = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid", pad=pad)
    gate = FP32_GATE if dtype == "f32" else FP16_GATE_L2
    assert rl2(ref[2], lit[2]) > 10 * gate or dtype == "f16"
    for z in range(5):
        check(out[z], ref[z], dtype, vol=ref, tag=z)
    r.set_filter_fused(False)
    out2 = r.recon(*dev).float().cpu().numpy()
    for z in range(5):
        check(out2[z], lit[z], dtype, vol=lit, tag=z)
    r.close()


@pytest.mark.parametrize("m", [3, 16 + 2])
def test_gridding_weight_cache(m):
    """TCP_OPT_WEIGHT_CACHE: the cached replay equals the direct kernel bit for bit (m = 3: the 52-byte records; Kaiser-Bessel
    half-width 2: the compact 28-byte records, k_grid_mma.cu compact_record / expand_record); the cache follows a change of
    the angles between calls (rebuilt on the device) and of nothing else."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    raw, flat, dark, theta = _inputs(w, list(range(8)))
    d = _to_dev(raw, flat, dark, theta)
    r = tcp.Recon(w.n, w.nproj, 8, w.center, "f16", w.filter, m)
    r.set_weight_cache(False)
    direct = r.recon(*d).clone()
    r.set_weight_cache(True)
    first = r.recon(*d).clone()          # builds the cache
    second = r.recon(*d).clone()         # replays it
    assert torch.equal(first, direct) and torch.equal(second, direct)
    # other angles: uneven, limited range
    th2 = np.sort((w.theta * 0.8 + 0.05 + 0.002 * np.sin(np.arange(w.nproj))).astype(np.float32))
    d2 = (d[0], d[1], d[2], torch.from_numpy(th2).cuda())
    a = r.recon(*d2).clone()
    r.set_weight_cache(False)
    b = r.recon(*d2).clone()
    assert torch.equal(a, b)
    ref = orc.recon(raw[:, 3:4], flat[3:4], dark[3:4], th2, w.center, w.filter, m, "grid")[0]
    assert rl2(a[3].float().cpu().numpy(), ref) < FP16_GATE_L2
    # back to the first angles
    r.set_weight_cache(True)
    assert torch.equal(r.recon(*d), direct)
    r.close()


def test_mean_frames_and_errors():
    tcp = _tcp()
    rng = np.random.default_rng(0)
    fr = rng.integers(0, 65536, (10, 5, 64), dtype=np.uint16)
    d = torch.from_numpy(fr.view(np.int16)).cuda().view(torch.uint16)
    mean = torch.empty((5, 64), dtype=torch.float32, device="cuda")
    tcp.tcp_mean_frames_u16(d, mean)
    torch.cuda.synchronize()
    ref = (fr.astype(np.float64).sum(0) / 10.0)
    assert np.abs(mean.cpu().numpy() - ref).max() <= np.abs(ref).max() * 2 ** -23
    for bad in [(100, 10, 2, 50.0), (128, 0, 2, 50.0), (128, 10, 0, 50.0), (128, 10, 2, 200.0), (8192, 10, 2, 50.0)]:
        with pytest.raises(tcp.TcpError):
            tcp.tcp_create(bad[0], bad[1], bad[2], bad[3], "f32", "ramp")
    with pytest.raises(tcp.TcpError):
        tcp.tcp_create_ex(128, 10, 2, 50.0, "f32", "ramp", 7)


def test_pipeline_host_matches_direct():
    """a7: chunked, stream-overlapped host->host pipeline equals chunk-by-chunk tcp_recon."""
    tcp = _tcp()
    w = sg.make_workload("C2", scale=4)           # 128^2 x 128 slices
    nzt = 22                                       # 5 chunks of 4 + a partial chunk of 2
    rows = list(range(nzt))
    raw, flat, dark, theta = _inputs(w, rows)
    r = tcp.Recon(w.n, w.nproj, 4, w.center, "f32", w.filter)
    raw_h = torch.from_numpy(raw.view(np.int16)).view(torch.uint16).pin_memory()
    out_h, ms = r.recon_volume_host(raw_h, torch.from_numpy(flat).pin_memory(), torch.from_numpy(dark).pin_memory(),
                                    torch.from_numpy(theta).pin_memory(), nbuf=3)
    assert ms > 0
    out_h = out_h.numpy()
    for z0 in range(0, 20, 4):
        sl = slice(z0, z0 + 4)
        d = r.recon(*_to_dev(np.ascontiguousarray(raw[:, sl]), flat[sl], dark[sl], theta))
        torch.cuda.synchronize()
        assert np.array_equal(out_h[sl], d.cpu().numpy())
    ref = orc.recon(np.ascontiguousarray(raw[:, 20:22]), flat[20:22], dark[20:22], theta, w.center, w.filter, orc.KB + 2, "grid")   # default kernel
    for z in range(2):
        check(out_h[20 + z], ref[z], "f32")
    r.close()
    # the partial last chunk runs as a chunk of its own size: equal to a 2-slice context, bit for bit
    r2 = tcp.Recon(w.n, w.nproj, 2, w.center, "f32", w.filter)
    d = r2.recon(*_to_dev(np.ascontiguousarray(raw[:, 20:22]), flat[20:22], dark[20:22], theta))
    torch.cuda.synchronize()
    assert np.array_equal(out_h[20:22], d.cpu().numpy())
    r2.close()


# ------------------------------------------------------------------ stored oracle values (tests/golden)
@pytest.mark.parametrize("m", [3, 4])
def test_c1_against_stored_oracle_values(m):
    """The CUDA path against values the oracle wrote to tests/golden/c1_oracle_samples.txt (make_golden.py calls only
    oracle/): fp32 path, sampled pixels of three C1 slices, within 1e-5 of the volume's scale."""
    import os
    stored = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c1_oracle_samples.txt")) as f:
        for ln in f:
            if ln.startswith("#") or not ln.strip():
                continue
            method, mm, z, iy, ix, v = ln.split()
            if method == "grid" and int(mm) == m:
                stored[(int(z), int(iy), int(ix))] = float(v)
    assert len(stored) == 24
    w = sg.make_workload("C1")
    out, _, _ = _gpu_recon(w, list(range(w.nz_total)), "f32", m=m)
    scale = max(abs(v) for v in stored.values())
    for (z, iy, ix), v in stored.items():
        assert abs(out[z, iy, ix] - v) < 1e-5 * scale, (z, iy, ix, out[z, iy, ix], v)


# ------------------------------------------------------------------ S1+S2 fused into the row kernel's loader
@pytest.mark.parametrize("dtype,nz,pad", [("f16", 8, "zero"), ("f16", 5, "edge"), ("f16_out32", 18, "zero")])
def test_fused_normalize_is_bit_identical(dtype, nz, pad):
    """TCP_OPT_FUSE_NORMALIZE (default on with fp16 storage): S1+S2 inside rows_kernel's loader give the same bits as
    the separate normalise kernel + sinogram round trip (also on an odd chunk, with edge padding, with the angle
    weights), one launch fewer; tcp_normalize still fills the sinogram workspace."""
    tcp = _tcp()
    w = sg.make_workload("C2", scale=4)
    rows = list(range(30, 30 + nz))
    raw, flat, dark, theta = _inputs(w, rows)
    dev = _to_dev(raw, flat, dark, theta)
    r = tcp.Recon(w.n, w.nproj, nz, w.center, dtype, w.filter, 3)
    r.set_pad(pad)
    n_fused = r.launches_per_recon
    a = r.recon(*dev).clone()
    r.set_angle_weights(True)
    aw = r.recon(*dev).clone()
    r.set_fuse_normalize(False)
    assert r.launches_per_recon == n_fused + 1
    bw = r.recon(*dev).clone()
    r.set_angle_weights(False)
    b = r.recon(*dev).clone()
    torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(aw, bw)
    sino = r.normalize(dev[0], dev[1], dev[2]).float().cpu().numpy()
    p = orc.neglog(raw, flat, dark)
    assert np.abs(sino - p).max() < 2e-3 * max(1.0, np.abs(p).max())
    r.close()
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid", pad=pad)
    out = a.float().cpu().numpy()
    for z in range(nz):
        assert rl2(out[z], ref[z]) < FP16_GATE_L2


# ------------------------------------------------------------------ unequally spaced angles
@pytest.mark.parametrize("dtype,alg", [("f32", "fourier"), ("f16", "fourier"), ("f32", "line")])
def test_angle_weights_for_unequally_spaced_angles(dtype, alg):
    """TCP_OPT_ANGLE_WEIGHTS: angles in two interleaved spacings; the GPU's trapezoid weights (trig_kernel, fp64 from
    the float32 angles) against the oracle's (pin P11); also through tcp_recon_try; with equispaced angles the
    option changes nothing beyond rounding; switching it off restores the default bit for bit."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    raw, flat, dark, _ = _inputs(w, [2, 3, 4])
    nproj = w.nproj
    na = 2 * nproj // 3
    theta = np.concatenate([np.arange(na) * (np.pi / 2 / na), np.pi / 2 + np.arange(nproj - na) * (np.pi / 2 / (nproj - na))]).astype(np.float32)
    r = tcp.Recon(w.n, nproj, 3, w.center, dtype, w.filter, 3)
    dev = _to_dev(raw, flat, dark, theta)
    base = r.recon(*dev).float().cpu().numpy()
    r.set_algorithm(alg)
    r.set_angle_weights(True)
    out = r.recon(*dev).float().cpu().numpy()
    method = "grid" if alg == "fourier" else "lin"
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, method, angle_weighted=True)
    plain = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, method)
    assert rl2(plain[0], ref[0]) > 0.05                      # the weights matter for these angles
    for z in range(3):
        if dtype == "f32":
            check(out[z], ref[z], "f32")
        else:
            assert rl2(out[z], ref[z]) < FP16_GATE_L2
            assert np.abs(out[z] - ref[z]).max() / np.abs(ref).max() < FP16_GATE_MAX
    if alg == "fourier":
        t = r.recon_try(dev[0][:, 1:2].contiguous(), dev[1][1:2], dev[2][1:2], dev[3], [w.center, w.center + 1.5]).float().cpu().numpy()
        check(t[0], ref[1], dtype)
        r.set_angle_weights(False)
        again = r.recon(*dev).float().cpu().numpy()
        assert np.array_equal(again, base)
    r.close()
    # equispaced: weights are 1 to float32 rounding of the angles
    r = tcp.Recon(w.n, nproj, 3, w.center, "f32", w.filter, 3)
    d2 = _to_dev(raw, flat, dark, w.theta)
    a = r.recon(*d2).cpu().numpy()
    r.set_angle_weights(True)
    b = r.recon(*d2).cpu().numpy()
    r.close()
    assert rl2(b, a) < 2e-5


# ------------------------------------------------------------------ degenerate cases of the method
@pytest.mark.parametrize("dtype", ["f32", "f16"])
@pytest.mark.parametrize("case", ["one_projection", "axis_angles", "centre_at_edges", "guards"])
def test_degenerate_cases(dtype, case):
    """The smallest problem the ABI accepts and the method's special points: a single projection at theta = 0
    (every sample on a grid point: 2m-1 taps, reading Q7), angles on the axes and diagonals, the rotation centre on
    the first / last detector pixel, a single slice (paired with zeros), and (fp32) the guards of S1:
    raw = 0, raw = 65535, raw < dark, flat = dark."""
    tcp = _tcp()
    n, nz = 64, 1
    rng = np.random.default_rng(77)
    if case == "one_projection":
        theta, centers = np.array([0.0], np.float32), [32.0]
    elif case == "axis_angles":
        theta, centers = (np.arange(4) * np.float32(np.pi / 4)).astype(np.float32), [31.5]
    elif case == "centre_at_edges":
        theta, centers = sg.make_theta(12), [0.0, float(n - 1)]
    else:
        # fp16 storage holds |f| < 1.9 per pixel: with 90 projections a p = 13.8 sample
        # backprojects to ~0.15 per pixel, inside that range, and the clamps of S1 are compared at the fp16 gates
        theta, centers = sg.make_theta(9 if dtype == "f32" else 90), [30.25]
    nproj = theta.size
    flat = rng.uniform(20000, 30000, (nz, n)).astype(np.float32)
    dark = rng.uniform(90, 110, (nz, n)).astype(np.float32)
    raw = np.rint((flat - dark)[None] * np.exp(-rng.uniform(0.0, 1.5, (nproj, nz, n))) + dark[None]).astype(np.uint16)
    if case == "guards":
        raw[0, 0, 3], raw[1, 0, 4], raw[2, 0, 5] = 0, 65535, 50
        flat[0, 9] = dark[0, 9]
    for c in centers:
        r = tcp.Recon(n, nproj, nz, c, dtype, "ramp", 3)
        out = r.recon(*_to_dev(raw, flat, dark, theta)).float().cpu().numpy()
        r.close()
        ref = orc.recon(raw, flat, dark, theta, c, "ramp", 3, "grid")
        assert np.isfinite(out).all()
        if dtype == "f32":
            check(out[0], ref[0], "f32")
        else:
            assert rl2(out[0], ref[0]) < FP16_GATE_L2, (case, c, rl2(out[0], ref[0]))
            assert np.abs(out[0] - ref[0]).max() / np.abs(ref).max() < FP16_GATE_MAX


@pytest.mark.parametrize("dtype", ["f16", "f16_out32"])
def test_fp16_storage_saturates_instead_of_overflowing(dtype):
    """A dead detector pixel (raw = 0 in every projection, p = 13.8: a ring through the whole slice) and a hot one on
    few projections drive |f| Phi^2 S past 65504, the largest half.  Every half store of the path saturates
    (cvt.rn.satfinite: sinogram, spectrum, grid, pass-1, output), so the result stays finite -- no inf in the grid,
    hence no NaN slice pair after S6 -- and the slice that shares the complex transform with the damaged one is
    reconstructed as if it were alone, away from where the damaged slice saturates."""
    tcp = _tcp()
    n, nz, nproj = 64, 2, 9
    rng = np.random.default_rng(78)
    theta = sg.make_theta(nproj)
    flat = rng.uniform(20000, 30000, (nz, n)).astype(np.float32)
    dark = rng.uniform(90, 110, (nz, n)).astype(np.float32)
    raw = np.rint((flat - dark)[None] * np.exp(-rng.uniform(0.0, 1.5, (nproj, nz, n))) + dark[None]).astype(np.uint16)
    raw[:, 0, 20] = 0                       # dead pixel of slice 0
    raw[0:2, 0, 40] = 65535                 # hot pixel on two projections
    r = tcp.Recon(n, nproj, nz, 31.5, dtype, "ramp", 3)
    out = r.recon(*_to_dev(raw, flat, dark, theta)).float().cpu().numpy()
    r.close()
    assert np.isfinite(out).all()
    ref = orc.recon(raw, flat, dark, theta, 31.5, "ramp", 3, "grid")
    assert np.abs(ref[0]).max() > 1.0       # the damaged slice does leave the range fp16 storage is scaled for
    check(out[1], ref[1], dtype, tag="partner slice")


def test_empty_inputs_are_refused():
    tcp = _tcp()
    r = tcp.Recon(64, 4, 2, 32.0, "f32", "ramp")
    e = torch.empty((4, 0, 64), dtype=torch.uint16)
    f = torch.empty((0, 64), dtype=torch.float32)
    with pytest.raises(tcp.TcpError):
        r.recon_volume_host(e, f, f, torch.zeros(4), torch.empty((0, 64, 64)))
    with pytest.raises(tcp.TcpError):
        tcp.tcp_create(64, 0, 2, 32.0, "f32", "ramp")
    with pytest.raises(tcp.TcpError):
        tcp.tcp_create(64, 4, 0, 32.0, "f32", "ramp")
    r.close()


# ------------------------------------------------------------------ detector width not a power of two (8(f-2))
def _cut(w, rows, lo, hi):
    """Columns lo..hi of a workload's detector: a narrower (possibly odd, possibly truncating) detector."""
    raw, flat, dark, theta = _inputs(w, rows)
    return (np.ascontiguousarray(raw[:, :, lo:hi]), np.ascontiguousarray(flat[:, lo:hi]),
            np.ascontiguousarray(dark[:, lo:hi]), theta, w.center - lo)


@pytest.mark.parametrize("dtype", ["f32", "f16", "f16_out32"])
@pytest.mark.parametrize("cfg,scale,lo,hi", [("C1", 1, 14, 114), ("C1", 1, 14, 113), ("C2", 2, 60, 190), ("C2", 4, 38, 100)])
def test_detector_width_not_a_power_of_two(dtype, cfg, scale, lo, hi):
    """tcp_create_det: widths 100, 99 (odd), 130 (just above a power of two, object truncated)
    and 62 (below the smallest transform) against the oracle's recon_padded, whose padding, centre shift and
    cut-out pin P10 fixes; 5 slices = an odd chunk."""
    tcp = _tcp()
    w = sg.make_workload(cfg, scale=scale)
    rows = list(range(w.nz_total // 2 - 2, w.nz_total // 2 + 3))
    raw, flat, dark, theta, c = _cut(w, rows, lo, hi)
    ndet = hi - lo
    r = tcp.Recon(ndet, w.nproj, len(rows), c, dtype, w.filter, 3)
    assert r.npad == orc.padded_size(ndet)[0] and r.npad != ndet
    out = r.recon(*_to_dev(raw, flat, dark, theta))
    torch.cuda.synchronize()
    assert out.shape == (len(rows), ndet, ndet)
    out = out.float().cpu().numpy()
    ref = orc.recon_padded(raw, flat, dark, theta, c, w.filter, 3, "grid")
    scale_v = np.abs(ref).max()
    for z in range(len(rows)):
        if dtype == "f32":
            check(out[z], ref[z], "f32")
        else:
            assert rl2(out[z], ref[z]) < FP16_GATE_L2, (z, rl2(out[z], ref[z]))
            assert np.abs(out[z] - ref[z]).max() / scale_v < FP16_GATE_MAX
    # the padded sinogram workspace: air outside the detector, S1+S2 inside
    sino = r.workspace("sinogram").float().cpu().numpy()
    pad_l = orc.padded_size(ndet)[1]
    assert sino.shape == (len(rows), w.nproj, r.npad)
    assert not sino[:, :, :pad_l].any() and not sino[:, :, pad_l + ndet:].any()
    p = orc.neglog(raw, flat, dark)
    assert np.abs(sino[:, :, pad_l:pad_l + ndet] - p).max() < (2e-6 if dtype == "f32" else 2e-3) * max(1.0, np.abs(p).max())
    r.close()


def test_detector_width_variants_pipeline_try_line_and_errors():
    """The other entry points on a padded context: LineRec, the rotation-centre try mode, the host pipeline with
    a partial last chunk; tcp_create_det on a power of two is tcp_create_ex bit for bit; argument errors."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    rows = list(range(8))
    raw, flat, dark, theta, c = _cut(w, rows, 14, 113)            # ndet = 99
    ndet = 99
    r = tcp.Recon(ndet, w.nproj, 4, c, "f32", w.filter, 3)
    # host pipeline: 2 chunks of 4 ... of a 7-slice stack (partial last chunk)
    raw_h = torch.from_numpy(np.ascontiguousarray(raw[:, :7]).view(np.int16)).view(torch.uint16).pin_memory()
    out_h, ms = r.recon_volume_host(raw_h, torch.from_numpy(flat[:7].copy()).pin_memory(),
                                    torch.from_numpy(dark[:7].copy()).pin_memory(), torch.from_numpy(theta).pin_memory(), nbuf=2)
    ref = orc.recon_padded(raw[:, :7], flat[:7], dark[:7], theta, c, w.filter, 3, "grid")
    assert out_h.shape == (7, ndet, ndet)
    for z in range(7):
        check(out_h[z].numpy(), ref[z], "f32")
    # try mode
    centers = [c - 2.0, c, c + 1.5]
    d = _to_dev(np.ascontiguousarray(raw[:, 3:4]), flat[3:4], dark[3:4], theta)
    t = r.recon_try(d[0], d[1], d[2], d[3], centers).cpu().numpy()
    assert t.shape == (3, ndet, ndet)
    for i, ci in enumerate(centers):
        ri = orc.recon_padded(raw[:, 3:4], flat[3:4], dark[3:4], theta, ci, w.filter, 3, "grid")[0]
        check(t[i], ri, "f32")
    with pytest.raises(tcp.TcpError):
        r.recon_try(d[0], d[1], d[2], d[3], [float(ndet)])        # centre range is the caller's detector
    with pytest.raises(tcp.TcpError):                              # the padded row's edges are air, not the detector's
        r.set_pad("edge")
    # LineRec
    r.set_algorithm("line")
    o = r.recon(*_to_dev(np.ascontiguousarray(raw[:, :4]), flat[:4], dark[:4], theta)).cpu().numpy()
    rl = orc.recon_padded(raw[:, :4], flat[:4], dark[:4], theta, c, w.filter, 3, "lin")
    for z in range(4):
        check(o[z], rl[z], "f32")
    r.close()
    # a power of two: tcp_create_det == tcp_create_ex
    raw8, flat8, dark8, _ = _inputs(w, rows)
    dev = _to_dev(raw8, flat8, dark8, theta)
    outs = []
    for create in (tcp.tcp_create_det, tcp.tcp_create_ex):
        h = create(w.n, w.nproj, 8, w.center, "f16", w.filter, 3)
        assert tcp.tcp_padded_n(h) == w.n
        o = torch.empty((8, w.n, w.n), dtype=torch.float16, device="cuda")
        tcp.tcp_recon(h, *dev, o)
        torch.cuda.synchronize()
        outs.append(o.cpu())
        tcp.tcp_destroy(h)
    assert torch.equal(outs[0], outs[1])
    for bad in [(7, 10, 2, 3.0), (4097, 10, 2, 50.0), (100, 10, 2, 99.5), (100, 10, 2, -1.0), (100, 0, 2, 50.0)]:
        with pytest.raises(tcp.TcpError):
            tcp.tcp_create_det(bad[0], bad[1], bad[2], bad[3], "f32", "ramp", 0)


def test_pipeline_slice_ranges_equal_the_whole_volume():
    """tcp_recon_volume_host_rows ("--start-row/--end-row"; the multi-GPU recipe of PAPER.md:145-149):
    three "ranks" (one after the other on this GPU, each with its own context; nothing waits on anything) reconstruct
    their tcp_slice_range of shared full-stack host arrays; the union equals the one-call volume bit for bit, rows
    outside a rank's range are left untouched, bad ranges are refused."""
    tcp = _tcp()
    w = sg.make_workload("C2", scale=4)
    nzt = 23
    raw, flat, dark, theta = _inputs(w, list(range(nzt)))
    raw_h = torch.from_numpy(raw.view(np.int16)).view(torch.uint16).pin_memory()
    flat_h, dark_h, th_h = torch.from_numpy(flat).pin_memory(), torch.from_numpy(dark).pin_memory(), torch.from_numpy(theta).pin_memory()
    r = tcp.Recon(w.n, w.nproj, 4, w.center, "f16", w.filter)
    whole, _ = r.recon_volume_host(raw_h, flat_h, dark_h, th_h, nbuf=3)
    whole = whole.clone()
    r.close()
    out = torch.full((nzt, w.n, w.n), -7.0, dtype=torch.float16).pin_memory()
    world = 3
    for rank in range(world):
        z0, z1 = tcp.tcp_slice_range(nzt, rank, world)
        rr = tcp.Recon(w.n, w.nproj, 4, w.center, "f16", w.filter)
        before = out.clone()
        rr.recon_volume_host(raw_h, flat_h, dark_h, th_h, out_host=out, nbuf=2, rows=(z0, z1))
        assert torch.equal(out[:z0], before[:z0]) and torch.equal(out[z1:], before[z1:])
        rr.close()
    assert torch.equal(out, whole)
    r = tcp.Recon(w.n, w.nproj, 4, w.center, "f16", w.filter)
    for bad in [(5, 5), (-1, 3), (20, 24), (7, 3)]:
        with pytest.raises(tcp.TcpError):
            r.recon_volume_host(raw_h, flat_h, dark_h, th_h, out_host=out, rows=bad)
    with pytest.raises(tcp.TcpError):               # angles over a full turn: refused on the host, before any copy
        r.recon_volume_host(raw_h, flat_h, dark_h, (th_h * 2.0).pin_memory(), out_host=out)
    r.close()


# ------------------------------------------------------------------ BASELINE full sizes, bench launch configuration
@pytest.mark.parametrize("cfg,nz,tcfft,where", [("C4", 32, None, "mid"), ("C4", 32, None, "first"), ("C4", 32, None, "last"),
                                                ("C4", 32, 0, "mid"), ("C4", 32, 1, "mid"), ("C4", 32, 6, "mid"), ("C4kb", 32, None, "mid"),
                                                ("C5", 32, None, "mid"), ("C5", 32, None, "first"), ("C5", 32, None, "last")])
def test_full_size_chunk_sampled_against_oracle(cfg, nz, tcfft, where):
    """C4 (2048^2, 2048 projections, fp16, one 32-slice chunk exactly as bench.py launches it: tcgen05
    gridding with 16 pairs per accumulator group) and C5 (4096^2, 4000 projections, M = 8192, off-centre,
    fp16 -> fp32 output).  Inputs are manufactured on the GPU (synthgen.make_counts_torch, frame averaging
    through tcp_mean_frames_u16) and the SAME arrays go to the oracle, which reconstructs a sample of the
    chunk's slices one by one.  tcfft: TCP_OPT_TCFFT, which transforms run their butterflies on the tensor cores
    (None = the default, every transform at M = 4096; 0 = the fp32 CUDA-core transforms; 1 = the row kernel only;
    6 = the inverse 2D transform only): same gates for every combination."""
    tcp = _tcp()
    kcode = 16 + 2 if cfg.endswith("kb") else 3          # "C4kb": C4 with the half-width-2 Kaiser-Bessel kernel
    cfg = cfg[:2]
    w = sg.make_workload(cfg)
    z0 = {"mid": w.nz_total // 2 - nz // 2, "first": 0, "last": w.nz_total - nz}[where]
    rows = list(range(z0, z0 + nz))
    raw_d, ff, df = sg.make_counts_torch(w, rows, device="cuda")
    flat_d = torch.empty((nz, w.n), dtype=torch.float32, device="cuda")
    dark_d = torch.empty_like(flat_d)
    tcp.tcp_mean_frames_u16(ff.contiguous(), flat_d)
    tcp.tcp_mean_frames_u16(df.contiguous(), dark_d)
    theta = w.theta
    r = tcp.Recon(w.n, w.nproj, nz, w.center, w.dtype, w.filter, kcode)
    if tcfft is not None:
        r.set_tcfft(tcfft)
    out = r.recon(raw_d.contiguous(), flat_d, dark_d, torch.from_numpy(theta).cuda())
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    r.close()
    sample = sorted({0, 1, nz // 2, nz - 1}) if where == "mid" else [0, nz - 1]     # first / last chunk: the stack's end slices (phantom edge, air rows)
    raw_h = raw_d.view(torch.int16)[:, sample].contiguous().cpu().numpy().view(np.uint16)
    ref = orc.recon(raw_h, flat_d[sample].cpu().numpy(), dark_d[sample].cpu().numpy(), theta, w.center, w.filter, kcode, "grid")
    scale = np.abs(ref).max()
    for i, z in enumerate(sample):
        print("full size %s tcfft=%s %s slice %d: rel-L2 %.3e max-abs %.3e" % (cfg, tcfft, where, z, rl2(out[z], ref[i]), np.abs(out[z] - ref[i]).max() / scale))
        assert rl2(out[z], ref[i]) < FP16_GATE_L2, (cfg, z, rl2(out[z], ref[i]))
        assert np.abs(out[z] - ref[i]).max() / scale < FP16_GATE_MAX


# ------------------------------------------------------------------ pre-processing between S2 and S3
@pytest.mark.parametrize("dtype", ["f32", "f16"])
@pytest.mark.parametrize("which", ["zinger", "ring", "both"])
def test_preprocessing_zingers_and_rings(dtype, which):
    """TCP_PARAM_ZINGER_DIF / TCP_PARAM_RING_ALPHA against the oracle's recon_pre (readings Q22, Q23; pins
    P13, P14).  Input: C2 at quarter size with bright detector hits (counts x 3 on isolated samples: p lower by ln 3, far
    from the 0.3 threshold on either side, so the fp32 and fp64 decisions agree) and two miscalibrated detector columns
    (+2 %, -3 % gain in every projection: rings).  Gates of north_star; the options must matter on this input; 5 slices
    (an odd chunk); try mode and LineRec run the same steps; padded-detector contexts and bad values are refused."""
    tcp = _tcp()
    w = sg.make_workload("C2", scale=4)
    rows = list(range(30, 35))
    raw, flat, dark, theta = _inputs(w, rows)
    rng = np.random.default_rng(31)
    raw = raw.astype(np.float64)
    for _ in range(40):
        j, z, i = rng.integers(w.nproj), rng.integers(len(rows)), rng.integers(w.n)
        raw[j, z, i] = (raw[j, z, i] - dark[z, i]) * 3.0 + dark[z, i]
    raw[:, :, 40] = (raw[:, :, 40] - dark[None, :, 40]) * 1.02 + dark[None, :, 40]
    raw[:, :, 77] = (raw[:, :, 77] - dark[None, :, 77]) * 0.97 + dark[None, :, 77]
    raw = np.clip(np.rint(raw), 0, 65535).astype(np.uint16)
    zd = 0.3 if which in ("zinger", "both") else 0.0
    ra = 2e-3 if which in ("ring", "both") else 0.0
    r = tcp.Recon(w.n, w.nproj, len(rows), w.center, dtype, w.filter, 3)
    dev = _to_dev(raw, flat, dark, theta)
    plain = r.recon(*dev).float().cpu().numpy()
    r.set_zinger(zd)
    r.set_ring(ra)
    out = r.recon(*dev).float().cpu().numpy()
    ref = orc.recon_pre(raw, flat, dark, theta, w.center, w.filter, 3, "grid", zinger_dif=zd, ring_alpha=ra)
    ref0 = orc.recon(raw, flat, dark, theta, w.center, w.filter, 3, "grid")
    assert rl2(ref[2], ref0[2]) > 2e-2                      # the steps matter on this input
    assert rl2(plain[2], ref0[2]) < (FP32_GATE if dtype == "f32" else FP16_GATE_L2)
    for z in range(len(rows)):
        check(out[z], ref[z], dtype, vol=ref, tag=(which, z))
    # the sinogram workspace after the steps
    p = orc.neglog(raw, flat, dark)
    if zd:
        p = orc.remove_zingers(p, zd)
    if ra:
        p = orc.remove_rings(p, ra)
    sino = r.workspace("sinogram").float().cpu().numpy()
    assert np.abs(sino - p).max() < (3e-6 if dtype == "f32" else 2e-3) * max(1.0, np.abs(p).max())
    # try mode and LineRec take the same steps
    t = r.recon_try(dev[0][:, 2:3].contiguous(), dev[1][2:3], dev[2][2:3], dev[3], [w.center]).float().cpu().numpy()
    check(t[0], ref[2], dtype, vol=ref, tag="try")
    r.set_algorithm("line")
    ol = r.recon(*dev).float().cpu().numpy()
    rl_ = orc.recon_pre(raw, flat, dark, theta, w.center, w.filter, 3, "lin", zinger_dif=zd, ring_alpha=ra)
    check(ol[1], rl_[1], dtype, vol=rl_, tag="line")
    for bad in (-1.0, float("nan")):
        with pytest.raises(tcp.TcpError):
            r.set_zinger(bad)
    r.close()
    rp = tcp.Recon(100, w.nproj, 2, 50.0, dtype, w.filter, 3)
    with pytest.raises(tcp.TcpError):
        rp.set_ring(1e-3)
    rp.close()


def test_binding_checks_host_tensors_and_device_angles():
    """The binding validates what the library cannot (advisor findings): host tensors of the pipeline call must be CPU,
    contiguous, of the right dtype and shape (a CUDA theta would be dereferenced on the host); device angles of
    Recon.recon are checked once per tensor on a host copy (unsorted or >= pi spans are refused, not silently mis-gridded)."""
    tcp = _tcp()
    w = sg.make_workload("C1")
    raw, flat, dark, theta = _inputs(w, list(range(4)))
    r = tcp.Recon(w.n, w.nproj, 4, w.center, "f32", w.filter)
    raw_h = torch.from_numpy(raw.view(np.int16)).view(torch.uint16).pin_memory()
    flat_h, dark_h, th_h = torch.from_numpy(flat).pin_memory(), torch.from_numpy(dark).pin_memory(), torch.from_numpy(theta).pin_memory()
    out, _ = r.recon_volume_host(raw_h, flat_h, dark_h, th_h, nbuf=2)
    assert np.isfinite(out.numpy()).all()
    for bad in [dict(theta=th_h.cuda()), dict(theta=th_h.double()), dict(flat=flat_h[:, ::2]), dict(dark=dark_h[:3]),
                dict(flat=flat_h.cuda())]:
        a = dict(raw=raw_h, flat=flat_h, dark=dark_h, theta=th_h)
        a.update(bad)
        with pytest.raises(tcp.TcpError):
            r.recon_volume_host(a["raw"], a["flat"], a["dark"], a["theta"], nbuf=2)
    dev = _to_dev(raw, flat, dark, theta)
    r.recon(*dev)
    with pytest.raises(tcp.TcpError):
        r.recon(dev[0], dev[1], dev[2], (dev[3] * 2.0).contiguous())          # a full turn
    with pytest.raises(tcp.TcpError):
        r.recon(dev[0], dev[1], dev[2], dev[3].flip(0).contiguous())          # decreasing
    # tcp.h: on a power-of-two context the device arrays must be 16-byte aligned (rows move as 16-byte vectors / bulk copies)
    shifted = torch.empty(dev[1].numel() + 1, dtype=torch.float32, device="cuda")[1:].view_as(dev[1])
    shifted.copy_(dev[1])
    with pytest.raises(tcp.TcpError, match="16-byte"):
        r.recon(dev[0], shifted, dev[2], dev[3])
    r.close()


def test_grid_corners_stay_zero_across_option_changes():
    """The tile and tensor-core griddings have no work item for the corner tiles no sample can reach; the grid is zeroed once
    per context and again after an option that changes its layout or writer.  Switching the gridding implementation back
    and forth on one context (strip-major <-> row-major grid) must therefore reproduce the first result bit for bit, and the
    corner cells of the grid workspace must read zero."""
    tcp = _tcp()
    w = sg.make_workload("C2", scale=2)               # n = 256: the corner tiles exist (M = 512, 16 x 16 tiles)
    rows = list(range(40, 46))
    raw, flat, dark, theta = _inputs(w, rows)
    dev = _to_dev(raw, flat, dark, theta)
    r = tcp.Recon(w.n, w.nproj, len(rows), w.center, "f16", w.filter)
    first = r.recon(*dev).clone()
    g = r.workspace("grid")                             # [npair][M l2][M l1], FFT order
    M = 2 * w.n
    assert float(g[:, M // 2 - 8:M // 2 + 8, M // 2 - 8:M // 2 + 8].abs().max()) == 0.0      # |l1|, |l2| ~ n: the far corner
    assert float(g.abs().max()) > 0.0
    r.set_grid_impl("tile")
    tile = r.recon(*dev).clone()
    r.set_grid_impl("mma")
    again = r.recon(*dev).clone()
    assert torch.equal(again, first)
    ref = orc.recon(raw, flat, dark, theta, w.center, w.filter, orc.KB + 2, "grid")
    for z in range(len(rows)):
        check(tile[z].float().cpu().numpy(), ref[z], "f16", vol=ref, tag=("tile", z))
        check(first[z].float().cpu().numpy(), ref[z], "f16", vol=ref, tag=("mma", z))
    r.close()
