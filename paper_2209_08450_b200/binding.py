"""ctypes binding of include/tcp.h.  Same names as the C ABI; marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtcp.so")

DTYPES = {"f32": 0, "f16": 1, "f16_out32": 2}
FILTERS = {"ramp": 0, "shepp": 1, "parzen": 2, "cosine": 3, "hann": 4, "hamming": 5}
WS = {"sinogram": 0, "spectrum": 1, "grid": 2, "pass1": 3, "trig": 4}
GRID_IMPLS = {"gather": 0, "scatter": 1, "tile": 2, "mma": 3}

# every symbol include/tcp.h declares (tests check the library exports them all)
EXPORTS = [
    "tcp_create", "tcp_create_ex", "tcp_recon", "tcp_destroy", "tcp_last_error",
    "tcp_mean_frames_u16", "tcp_normalize", "tcp_workspace", "tcp_read_workspace", "tcp_scale", "tcp_grid_strip",
    "tcp_workspace_bytes", "tcp_launches_per_recon", "tcp_set_option", "tcp_profile_collect",
    "tcp_recon_volume_host", "tcp_recon_try", "tcp_create_det", "tcp_padded_n",
    "tcp_recon_volume_host_rows", "tcp_slice_range", "tcp_check_angles", "tcp_pass1_layout", "tcp_grid_swizzled", "tcp_fft_lines", "tcp_measure_rates", "tcp_set_param",
    "tcp_ring_static_setup", "tcp_ring_remove_static",
]


class TcpError(RuntimeError):
    pass


def lib_path() -> str:
    return _SO


_lib = None


def lib():
    """Load libtcp.so (built in-tree by paper_2209_08450_b200.build).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise TcpError("libtcp.so is not built: run `python -m paper_2209_08450_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(_SO)
    vp, ci, cf = C.c_void_p, C.c_int, C.c_float
    L.tcp_create.restype = vp
    L.tcp_create.argtypes = [ci, ci, ci, cf, ci, ci]
    L.tcp_create_ex.restype = vp
    L.tcp_create_ex.argtypes = [ci, ci, ci, cf, ci, ci, ci]
    L.tcp_create_det.restype = vp
    L.tcp_create_det.argtypes = [ci, ci, ci, cf, ci, ci, ci]
    L.tcp_padded_n.restype = ci
    L.tcp_padded_n.argtypes = [vp]
    L.tcp_recon.restype = ci
    L.tcp_recon.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.tcp_destroy.restype = None
    L.tcp_destroy.argtypes = [vp]
    L.tcp_last_error.restype = C.c_char_p
    L.tcp_mean_frames_u16.restype = ci
    L.tcp_mean_frames_u16.argtypes = [vp, ci, ci, ci, vp, vp]
    L.tcp_normalize.restype = ci
    L.tcp_normalize.argtypes = [vp, vp, vp, vp, vp]
    L.tcp_workspace.restype = ci
    L.tcp_workspace.argtypes = [vp, ci, C.POINTER(vp), C.POINTER(C.c_size_t)]
    L.tcp_read_workspace.restype = ci
    L.tcp_read_workspace.argtypes = [vp, ci, vp, C.c_size_t, vp]
    L.tcp_scale.restype = C.c_double
    L.tcp_scale.argtypes = [vp]
    L.tcp_grid_strip.restype = C.c_int
    L.tcp_grid_strip.argtypes = [vp]
    L.tcp_workspace_bytes.restype = C.c_size_t
    L.tcp_workspace_bytes.argtypes = [vp]
    L.tcp_launches_per_recon.restype = ci
    L.tcp_launches_per_recon.argtypes = [vp]
    L.tcp_set_option.restype = ci
    L.tcp_set_option.argtypes = [vp, ci, ci]
    L.tcp_profile_collect.restype = ci
    L.tcp_profile_collect.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(ci)]
    L.tcp_recon_volume_host.restype = ci
    L.tcp_recon_volume_host.argtypes = [vp, vp, vp, vp, vp, vp, ci, ci, C.POINTER(cf)]
    L.tcp_recon_volume_host_rows.restype = ci
    L.tcp_recon_volume_host_rows.argtypes = [vp, vp, vp, vp, vp, vp, ci, ci, ci, ci, C.POINTER(cf)]
    L.tcp_check_angles.restype = ci
    L.tcp_check_angles.argtypes = [vp, ci]
    L.tcp_slice_range.restype = ci
    L.tcp_slice_range.argtypes = [ci, ci, ci, C.POINTER(ci), C.POINTER(ci)]
    L.tcp_pass1_layout.restype = ci
    L.tcp_pass1_layout.argtypes = [vp]
    L.tcp_grid_swizzled.restype = ci
    L.tcp_grid_swizzled.argtypes = [vp]
    L.tcp_fft_lines.restype = ci
    L.tcp_fft_lines.argtypes = [vp, vp, vp, ci, ci, vp]
    L.tcp_set_param.restype = ci
    L.tcp_set_param.argtypes = [vp, ci, C.c_double]
    L.tcp_ring_static_setup.restype = ci
    L.tcp_ring_static_setup.argtypes = []
    L.tcp_ring_remove_static.restype = ci
    L.tcp_ring_remove_static.argtypes = [vp, vp, ci, ci, ci, ci, C.c_double, vp]
    L.tcp_measure_rates.restype = ci
    L.tcp_measure_rates.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.tcp_recon_try.restype = ci
    L.tcp_recon_try.argtypes = [vp, vp, vp, vp, vp, C.POINTER(cf), ci, vp, vp]
    _lib = L
    return L


def _swz(nl: int, size: int):
    """Position of element k of a line in the layouts the tensor-core transforms read (mmafft.cuh swz<NL>; marshalling of
    test read-backs only): the inverse permutation is the same function (an XOR with bits it does not change)."""
    import numpy as np
    k = np.arange(size, dtype=np.int64)
    if nl == 2:
        f = lambda x: np.where(x & 1, 12, 0) ^ np.where(x & 2, 5, 0)
        return k ^ f((k >> 8) & 3) ^ f((k >> 4) & 3)
    f = lambda x: ((x & 3) << 1) | (x & 1)
    return k ^ f((k >> 8) & 3) ^ f((k >> 4) & 3)


def tcp_last_error() -> str:
    return lib().tcp_last_error().decode()


def _check(rc: int):
    if rc != 0:
        raise TcpError("tcp error %d: %s" % (rc, tcp_last_error()))


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t: torch.Tensor, dtype, shape=None) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TcpError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise TcpError("expected shape %s, got %s" % (tuple(shape), tuple(t.shape)))
    return t.data_ptr()


def tcp_create(n, nproj, nz_chunk, center, dtype, filter):
    h = lib().tcp_create(n, nproj, nz_chunk, float(center), DTYPES.get(dtype, dtype), FILTERS.get(filter, filter))
    if not h:
        raise TcpError("tcp_create failed: " + tcp_last_error())
    return h


def tcp_measure_rates():
    """(fp32 FFMA TFLOP/s, fp16 mma.sync TFLOP/s) measured on the current device (tcp_measure_rates)."""
    a, b = C.c_double(0.0), C.c_double(0.0)
    _check(lib().tcp_measure_rates(C.byref(a), C.byref(b)))
    return float(a.value), float(b.value)


def tcp_ring_static_setup():
    _check(lib().tcp_ring_static_setup())


def tcp_ring_remove_static(sino_in, sino_out, alpha, stream=None):
    """Ring removal on CUDA tensors [nz][nproj][n] (float32 or float16) without any allocation (tcp_ring_remove_static);
    sino_out may be sino_in."""
    if sino_in.dtype not in (torch.float32, torch.float16):
        raise TcpError("expected float32 or float16 sinograms")
    if sino_in.dim() != 3:
        raise TcpError("expected a sinogram of shape [nz][nproj][n]")
    nz, nproj, n = sino_in.shape
    _check(lib().tcp_ring_remove_static(_dev(sino_in, sino_in.dtype), _dev(sino_out, sino_in.dtype, sino_in.shape), nz, nproj, n,
                                        DTYPES["f16" if sino_in.dtype == torch.float16 else "f32"], float(alpha), _stream(stream)))


def tcp_create_ex(n, nproj, nz_chunk, center, dtype, filter, m):
    h = lib().tcp_create_ex(n, nproj, nz_chunk, float(center), DTYPES.get(dtype, dtype),
                            FILTERS.get(filter, filter), int(m))
    if not h:
        raise TcpError("tcp_create_ex failed: " + tcp_last_error())
    return h


def tcp_create_det(ndet, nproj, nz_chunk, center, dtype, filter, m=0):
    h = lib().tcp_create_det(ndet, nproj, nz_chunk, float(center), DTYPES.get(dtype, dtype),
                             FILTERS.get(filter, filter), int(m))
    if not h:
        raise TcpError("tcp_create_det failed: " + tcp_last_error())
    return h


def tcp_padded_n(h) -> int:
    return int(lib().tcp_padded_n(h))


def tcp_destroy(h):
    lib().tcp_destroy(h)


def tcp_recon(h, raw_u16, flat, dark, theta, out, stream=None):
    """All arguments are CUDA tensors (uint16 as torch.uint16 or int16 storage)."""
    _check(lib().tcp_recon(h, raw_u16.data_ptr(), flat.data_ptr(), dark.data_ptr(), theta.data_ptr(),
                           out.data_ptr(), _stream(stream)))


def tcp_normalize(h, raw_u16, flat, dark, stream=None):
    _check(lib().tcp_normalize(h, raw_u16.data_ptr(), flat.data_ptr(), dark.data_ptr(), _stream(stream)))


def tcp_mean_frames_u16(frames, mean, stream=None):
    k, nz, n = frames.shape
    _check(lib().tcp_mean_frames_u16(frames.data_ptr(), k, nz, n, _dev(mean, torch.float32, (nz, n)), _stream(stream)))


def _host(t: torch.Tensor, dtype, shape=None, what="tensor") -> int:
    """A HOST pointer the library may dereference: CPU tensor, contiguous, right dtype and shape (mirror of _dev)."""
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TcpError("%s: expected a contiguous CPU tensor of dtype %s" % (what, dtype))
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise TcpError("%s: expected shape %s, got %s" % (what, tuple(shape), tuple(t.shape)))
    return t.data_ptr()


def tcp_recon_volume_host(h, raw_host, flat_host, dark_host, theta_host, out_host, nz_total, nbuf=3):
    """Host (pinned) tensors in, host tensor out; returns the device-timed milliseconds."""
    ms = C.c_float(0.0)
    _check(lib().tcp_recon_volume_host(h, raw_host.data_ptr(), flat_host.data_ptr(), dark_host.data_ptr(),
                                       theta_host.data_ptr(), out_host.data_ptr(), int(nz_total), int(nbuf),
                                       C.byref(ms)))
    return float(ms.value)


def tcp_recon_volume_host_rows(h, raw_host, flat_host, dark_host, theta_host, out_host, nz_stack, z_begin, z_end, nbuf=3):
    """Slices [z_begin, z_end) of full-stack host tensors; returns the device-timed milliseconds."""
    ms = C.c_float(0.0)
    _check(lib().tcp_recon_volume_host_rows(h, raw_host.data_ptr(), flat_host.data_ptr(), dark_host.data_ptr(),
                                            theta_host.data_ptr(), out_host.data_ptr(), int(nz_stack), int(z_begin),
                                            int(z_end), int(nbuf), C.byref(ms)))
    return float(ms.value)


def tcp_check_angles(theta_host):
    """Raises TcpError unless the HOST float32 tensor / array of angles is finite, strictly increasing and spans < pi."""
    t = np.ascontiguousarray(theta_host.numpy() if isinstance(theta_host, torch.Tensor) else theta_host, dtype=np.float32)
    _check(lib().tcp_check_angles(t.ctypes.data_as(C.c_void_p), int(t.size)))


def tcp_slice_range(nz_total, rank, world):
    """(z0, z1): the slice range of process `rank` of `world` (host logic in the library, no GPU needed)."""
    z0, z1 = C.c_int(0), C.c_int(0)
    _check(lib().tcp_slice_range(int(nz_total), int(rank), int(world), C.byref(z0), C.byref(z1)))
    return int(z0.value), int(z1.value)


def _as_u16(t: torch.Tensor) -> torch.Tensor:
    if t.dtype == torch.uint16:
        return t
    if t.dtype == torch.int16:
        return t.view(torch.uint16)
    raise TcpError("raw projections must be uint16")


class Recon:
    """Convenience owner of a tcp context (still only marshalling)."""

    def __init__(self, n, nproj, nz_chunk, center, dtype="f32", filter="parzen", m=0):
        if not torch.cuda.is_available():
            raise TcpError("no CUDA device: this library has no CPU fallback")
        self.n, self.nproj, self.nz, self.center = n, nproj, nz_chunk, float(center)
        self.dtype, self.filter = dtype, filter
        # n is the caller's detector width / image side; the library pads it to a power of two if it must
        self.h = tcp_create_det(n, nproj, nz_chunk, center, dtype, filter, m)
        self.npad = tcp_padded_n(self.h)
        self.out_dtype = torch.float16 if dtype == "f16" else torch.float32
        self.store_dtype = torch.float32 if dtype == "f32" else torch.float16

    def close(self):
        if getattr(self, "h", None):
            tcp_destroy(self.h)
            self.h = None

    __del__ = close

    def set_grid_impl(self, name: str):
        _check(lib().tcp_set_option(self.h, 0, GRID_IMPLS[name]))

    def set_weight_cache(self, on: bool):
        """TCP_OPT_WEIGHT_CACHE: reuse the gridding weights across calls with the same angles (default on)."""
        _check(lib().tcp_set_option(self.h, 6, 1 if on else 0))

    def set_fuse_normalize(self, on: bool):
        """TCP_OPT_FUSE_NORMALIZE: S1+S2 inside the row kernel's loader (fp16 storage; default on; same bits)."""
        _check(lib().tcp_set_option(self.h, 8, 1 if on else 0))

    def set_angle_weights(self, on: bool):
        """TCP_OPT_ANGLE_WEIGHTS: trapezoid quadrature weights for unequally spaced angles (off by default)."""
        _check(lib().tcp_set_option(self.h, 7, 1 if on else 0))

    def set_filter_fused(self, on: bool):
        """TCP_OPT_FILTER_FUSED: S3 + S4 as one transform without the crop (a different reading; off by default)."""
        _check(lib().tcp_set_option(self.h, 5, 1 if on else 0))

    def set_pad(self, name: str):
        """TCP_OPT_PAD: "zero" (default) or "edge" padding of the filter stage."""
        _check(lib().tcp_set_option(self.h, 4, {"zero": 0, "edge": 1}[name]))

    def set_algorithm(self, name: str):
        """TCP_OPT_ALGORITHM: "fourier" (FourierRec, default) or "line" (LineRec, direct line summation)."""
        _check(lib().tcp_set_option(self.h, 3, {"fourier": 0, "line": 1}[name]))

    def set_zinger(self, dif: float):
        """TCP_PARAM_ZINGER_DIF: zinger removal threshold on p = -ln t (0 = off)."""
        _check(lib().tcp_set_param(self.h, 0, float(dif)))

    def set_ring(self, alpha: float):
        """TCP_PARAM_RING_ALPHA: regularisation of the closed-form ring estimate (0 = off)."""
        _check(lib().tcp_set_param(self.h, 1, float(alpha)))

    def set_tcfft(self, mask: int):
        """TCP_OPT_TCFFT: which transforms run their butterflies on the tensor cores (1 rows, 6 = both passes of the
        inverse 2D transform; default 7 where available: fp16 storage at M = 4096; 0 = fp32 CUDA-core transforms)."""
        _check(lib().tcp_set_option(self.h, 2, int(mask)))

    STAGES = ("trig", "normalize", "rows", "grid", "ifft_cols", "ifft_rows")

    def set_profile(self, on: bool):
        _check(lib().tcp_set_option(self.h, 1, 1 if on else 0))

    def profile_collect(self):
        """(dict stage -> summed ms, number of tcp_recon calls) since the last collect."""
        ms = (C.c_double * 6)()
        nc = C.c_int(0)
        _check(lib().tcp_profile_collect(self.h, ms, C.byref(nc)))
        return {k: float(ms[i]) for i, k in enumerate(self.STAGES)}, int(nc.value)

    @property
    def scale(self) -> float:
        return float(lib().tcp_scale(self.h))

    @property
    def launches_per_recon(self) -> int:
        return int(lib().tcp_launches_per_recon(self.h))

    @property
    def grid_strip(self) -> int:
        return int(lib().tcp_grid_strip(self.h))

    @property
    def workspace_bytes(self) -> int:
        return int(lib().tcp_workspace_bytes(self.h))

    def recon(self, raw_u16, flat, dark, theta, out=None, stream=None, check_angles=True):
        """tcp_recon on device tensors.  check_angles: tcp_recon cannot validate its DEVICE angles without a synchronisation,
        so the binding checks each distinct theta tensor ONCE (tcp_check_angles on a host copy; cached by data pointer and
        version) -- a 0..2 pi scan or unsorted angles would otherwise give a silently wrong image."""
        if check_angles and isinstance(theta, torch.Tensor) and theta.is_cuda:
            key = (theta.data_ptr(), theta._version, tuple(theta.shape))
            if getattr(self, "_theta_ok", None) != key:
                tcp_check_angles(theta.detach().float().cpu())
                self._theta_ok = key
        raw_u16 = _as_u16(raw_u16)
        _dev(raw_u16, torch.uint16, (self.nproj, self.nz, self.n))
        _dev(flat, torch.float32, (self.nz, self.n))
        _dev(dark, torch.float32, (self.nz, self.n))
        _dev(theta, torch.float32, (self.nproj,))
        if out is None:
            out = torch.empty((self.nz, self.n, self.n), dtype=self.out_dtype, device=raw_u16.device)
        _dev(out, self.out_dtype, (self.nz, self.n, self.n))
        tcp_recon(self.h, raw_u16, flat, dark, theta, out, stream)
        return out

    def recon_try(self, raw_u16, flat, dark, theta, centers, out=None, stream=None):
        """tcp_recon_try: one slice (raw [nproj][1][n], flat / dark [n] or [1][n]) for every centre in `centers`."""
        raw_u16 = _as_u16(raw_u16)
        _dev(raw_u16, torch.uint16, (self.nproj, 1, self.n))
        flat, dark = flat.reshape(1, self.n), dark.reshape(1, self.n)
        _dev(flat, torch.float32, (1, self.n))
        _dev(dark, torch.float32, (1, self.n))
        _dev(theta, torch.float32, (self.nproj,))
        cs = [float(c) for c in centers]
        if out is None:
            out = torch.empty((len(cs), self.n, self.n), dtype=self.out_dtype, device=raw_u16.device)
        _dev(out, self.out_dtype, (len(cs), self.n, self.n))
        arr = (C.c_float * len(cs))(*cs)
        _check(lib().tcp_recon_try(self.h, raw_u16.data_ptr(), flat.data_ptr(), dark.data_ptr(), theta.data_ptr(), arr, len(cs),
                                   out.data_ptr(), _stream(stream)))
        return out

    def fft_lines(self, x_half2: torch.Tensor, inverse=False, stream=None) -> torch.Tensor:
        """tcp_fft_lines: [batch][4096][2] half (re, im) -> [batch][4096] complex64 through the tensor-core transform."""
        _dev(x_half2, torch.float16)
        batch = x_half2.shape[0]
        if tuple(x_half2.shape) != (batch, 4096, 2):
            raise TcpError("expected shape (batch, 4096, 2)")
        out = torch.empty((batch, 4096, 2), dtype=torch.float32, device=x_half2.device)
        _check(lib().tcp_fft_lines(self.h, x_half2.data_ptr(), out.data_ptr(), batch, 1 if inverse else 0, _stream(stream)))
        return torch.view_as_complex(out)

    def normalize(self, raw_u16, flat, dark, stream=None):
        raw_u16 = _as_u16(raw_u16)
        _dev(raw_u16, torch.uint16, (self.nproj, self.nz, self.n))
        tcp_normalize(self.h, raw_u16, flat, dark, stream)
        return self.workspace("sinogram")

    def workspace(self, name: str) -> torch.Tensor:
        """Copy of an intermediate of the last recon, as a torch tensor (tests only)."""
        ptr, nbytes = C.c_void_p(), C.c_size_t()
        _check(lib().tcp_workspace(self.h, WS[name], C.byref(ptr), C.byref(nbytes)))
        npair, M, n = (self.nz + 1) // 2, 2 * self.npad, self.npad
        buf = torch.empty(nbytes.value, dtype=torch.uint8, device="cuda")
        _check(lib().tcp_read_workspace(self.h, WS[name], buf.data_ptr(), nbytes.value, _stream(None)))
        torch.cuda.synchronize()
        if name == "trig":
            return buf.view(torch.float64).view(self.nproj, 2)
        if name == "sinogram":
            return buf.view(self.store_dtype).view(self.nz, self.nproj, n)
        shape = {"spectrum": (npair, self.nproj, M), "grid": (npair, M, M), "pass1": (npair, n, M)}[name]
        v = buf.view(self.store_dtype).view(*shape, 2).float()
        if name == "grid":
            w = int(lib().tcp_grid_strip(self.h))
            if w:       # strip-major [npair][M/w][M l2][w l1] -> [npair][M l2][M l1]
                v = v.view(npair, M // w, M, w, 2)
                if int(lib().tcp_grid_swizzled(self.h)):    # row l2 of a strip is stored at position swz<4>(l2)
                    v = v[:, :, torch.from_numpy(_swz(4, M)).to(v.device)]
                v = v.permute(0, 2, 1, 3, 4).reshape(npair, M, M, 2)
        if name == "pass1" and int(lib().tcp_pass1_layout(self.h)) == 1:
            # row pairs [npair][n/2][position swz<2>(l1)][2 rows] -> [npair][n iy][M l1]
            v = v.view(npair, n // 2, M, 2, 2)[:, :, torch.from_numpy(_swz(2, M)).to(v.device)]
            v = v.permute(0, 1, 3, 2, 4).reshape(npair, n, M, 2)
        elif name == "pass1":   # strip-major [npair][M/w][n iy][w l1] -> [npair][n iy][M l1]
            w = min(32, max(2, 16384 // M))
            v = v.view(npair, M // w, n, w, 2).permute(0, 2, 1, 3, 4).reshape(npair, n, M, 2)
        return torch.complex(v[..., 0], v[..., 1])

    def recon_volume_host(self, raw_host, flat_host, dark_host, theta_host, out_host=None, nbuf=3, rows=None):
        """rows = (z_begin, z_end): only that slice range of the stack (tcp_recon_volume_host_rows), e.g.
        tcp_slice_range(nz_total, rank, world) in a one-process-per-GPU job; out_host keeps the full-stack shape."""
        raw_host = _as_u16(raw_host)
        if raw_host.dim() != 3:
            raise TcpError("raw_host: expected [nproj][nz_total][n]")
        nproj, nz_total, n = raw_host.shape
        if (nproj, n) != (self.nproj, self.n):
            raise TcpError("raw_host: expected %d projections of width %d, got %s" % (self.nproj, self.n, tuple(raw_host.shape)))
        if out_host is None:
            out_host = torch.empty((nz_total, n, n), dtype=self.out_dtype).pin_memory()
        # the library dereferences these on the host and hands them to the copy engines: check them here (a CUDA theta
        # would be read as host memory; a wrong dtype or a non-contiguous view would be misread or overrun)
        _host(raw_host, torch.uint16, (self.nproj, nz_total, self.n), "raw_host")
        _host(flat_host, torch.float32, (nz_total, self.n), "flat_host")
        _host(dark_host, torch.float32, (nz_total, self.n), "dark_host")
        _host(theta_host, torch.float32, (self.nproj,), "theta_host")
        _host(out_host, self.out_dtype, (nz_total, self.n, self.n), "out_host")
        if not (raw_host.is_pinned() and out_host.is_pinned()):
            import warnings
            warnings.warn("tcp_recon_volume_host: pageable host buffers: the copies will not overlap the compute")
        if rows is None:
            ms = tcp_recon_volume_host(self.h, raw_host, flat_host, dark_host, theta_host, out_host, nz_total, nbuf)
        else:
            ms = tcp_recon_volume_host_rows(self.h, raw_host, flat_host, dark_host, theta_host, out_host, nz_total,
                                            rows[0], rows[1], nbuf)
        return out_host, ms
