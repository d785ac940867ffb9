"""paper_2209_08450_b200 -- B200-native parallel-beam FBP by Fourier gridding.

Thin Python binding over the C-ABI library libtcp.so (include/tcp.h): argument
marshalling only; every step of the hot path runs in the library's own sm_100a
kernels.  PyTorch supplies device memory, pinned host memory and streams.
There is no CPU fallback: a missing library or device raises.
"""
from .binding import (  # noqa: F401
    TcpError,
    Recon,
    lib,
    lib_path,
    tcp_create,
    tcp_create_ex,
    tcp_create_det,
    tcp_padded_n,
    tcp_destroy,
    tcp_recon,
    tcp_normalize,
    tcp_mean_frames_u16,
    tcp_recon_volume_host,
    tcp_recon_volume_host_rows,
    tcp_slice_range,
    tcp_check_angles,
    tcp_last_error,
    tcp_measure_rates,
    tcp_ring_static_setup,
    tcp_ring_remove_static,
    DTYPES,
    FILTERS,
    EXPORTS,
)
