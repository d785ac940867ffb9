"""Seeded synthetic inputs for the parallel-beam FBP hot path.

This module is the ONLY code shared by the CPU oracle tests and the CUDA path
tests/bench.  It holds none of the reconstruction method's arithmetic: it only
manufactures detector data (uint16 counts, flat/dark frames, angles) from
analytic ellipsoid phantoms whose line integrals are known in closed form
(the paper checks accuracy "using analytical expressions for the Shepp-Logan
phantom and its projection data"; the performance
workloads are "N 16-bit projections of N x N").

Geometry: image pixel (ix, iy) sits at
x = ix - n/2, y = iy - n/2; slice iz at z = iz - nz_total/2; the ray recorded
by detector pixel i of projection theta is the line
    { (x, y): x cos(theta) + y sin(theta) + c = i },   direction (-sin, cos, 0).
"""
from .phantom import (  # noqa: F401
    Ellipsoids,
    head_phantom,
    random_ellipsoids,
    line_integrals,
    rasterize,
)
from .counts import (  # noqa: F401
    CONFIGS,
    Workload,
    make_theta,
    make_workload,
    make_counts,
    make_counts_torch,
    make_flat_dark,
)
