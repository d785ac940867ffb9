"""Analytic ellipsoid phantoms and their closed-form parallel-beam line integrals.

An ellipsoid is {r : (r - r0)^T A (r - r0) <= 1},  A = Q diag(1/a^2, 1/b^2, 1/c^2) Q^T,
with constant attenuation mu (per pixel length) inside.  The chord of the line
r(t) = p + t d through it has length 2 sqrt(beta^2 - alpha gamma) / alpha with
alpha = d^T A d, beta = d^T A (p - r0), gamma = (p - r0)^T A (p - r0) - 1
(zero when the discriminant is negative).  This is plain analytic geometry, not
part of the reconstruction method; it is the ground truth the oracle is pinned to.

All lengths are in detector pixels.  Works with numpy arrays, or with torch
tensors when ``xp=torch`` (used to manufacture the large configs on the GPU).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class Ellipsoids:
    center: np.ndarray  # (E, 3) x, y, z in pixels, relative to the rotation axis / mid slice
    axes: np.ndarray    # (E, 3) semi-axes in pixels
    rot: np.ndarray     # (E, 3, 3) orthonormal Q (columns = principal directions)
    mu: np.ndarray      # (E,) attenuation per pixel (may be negative: subtractive ellipsoid)

    def __len__(self) -> int:
        return int(self.mu.shape[0])

    def quadric(self) -> np.ndarray:
        """(E,3,3) matrices A."""
        d = 1.0 / self.axes ** 2
        return np.einsum("eij,ej,ekj->eik", self.rot, d, self.rot)

    def scaled(self, s: float) -> "Ellipsoids":
        return Ellipsoids(self.center.copy(), self.axes.copy(), self.rot.copy(), self.mu * s)


def _rotz(deg: float) -> np.ndarray:
    a = np.deg2rad(deg)
    c, s = np.cos(a), np.sin(a)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def head_phantom(n: int, nz_total: int, mu_max: float = 0.02) -> Ellipsoids:
    """Our own 10-ellipsoid head-like phantom (NOT the published Shepp-Logan table,
    which is not in the container).  In-plane sizes are
    fractions of n; z sizes are fractions of max(n, nz_total) so a thin stack of
    slices still cuts every ellipsoid.  Scaled so the largest attenuation is mu_max.
    """
    zs = float(max(n, nz_total))
    rows = [
        # cx,    cy,    cz,    a,     b,     c,    rot,  mu
        (0.000, 0.000, 0.000, 0.360, 0.440, 0.420, 0.0, 1.00),    # skull
        (0.000, -0.010, 0.000, 0.330, 0.405, 0.390, 0.0, -0.80),  # brain (difference of two)
        (-0.105, 0.020, 0.000, 0.050, 0.140, 0.100, 15.0, -0.10),  # left ventricle
        (0.105, 0.020, 0.000, 0.060, 0.160, 0.120, -15.0, -0.10),  # right ventricle
        (0.000, 0.190, 0.010, 0.090, 0.110, 0.100, 0.0, 0.10),
        (0.000, 0.050, 0.000, 0.022, 0.022, 0.030, 0.0, 0.08),
        (0.000, -0.060, 0.000, 0.020, 0.020, 0.030, 0.0, 0.08),
        (-0.040, -0.300, 0.000, 0.025, 0.012, 0.020, 0.0, 0.06),
        (0.000, -0.300, 0.000, 0.012, 0.012, 0.020, 0.0, 0.06),
        (0.045, -0.300, 0.000, 0.012, 0.025, 0.020, 30.0, 0.06),
    ]
    r = np.array(rows, dtype=np.float64)
    center = np.stack([r[:, 0] * n, r[:, 1] * n, r[:, 2] * zs], axis=1)
    axes = np.stack([r[:, 3] * n, r[:, 4] * n, r[:, 5] * zs], axis=1)
    rot = np.stack([_rotz(a) for a in r[:, 6]])
    mu = r[:, 7] * mu_max  # skull (1.0) is the maximum of any sum of overlapping members
    return Ellipsoids(center, axes, rot, mu)


def random_ellipsoids(count: int, n: int, nz_total: int, seed: int,
                      axes_frac=(0.02, 0.12), mu_range=(0.001, 0.01)) -> Ellipsoids:
    """`count` random ellipsoids: centres uniform in the cylinder r < 0.30 n,
    |z| < 0.45 nz_total; semi-axes uniform in axes_frac * n; uniformly random
    rotations; attenuation uniform in mu_range; a draw is rejected when its
    bounding sphere leaves r < 0.48 n (BASELINE.json configs 2-5)."""
    rng = np.random.default_rng(seed)
    cs, ax, qs, mus = [], [], [], []
    while len(mus) < count:
        rad = 0.30 * n * np.sqrt(rng.uniform())
        phi = rng.uniform(0.0, 2.0 * np.pi)
        z = rng.uniform(-0.45, 0.45) * nz_total
        a = rng.uniform(axes_frac[0], axes_frac[1], size=3) * n
        g = rng.standard_normal((3, 3))
        q, rr = np.linalg.qr(g)
        q = q * np.sign(np.diag(rr))
        if np.linalg.det(q) < 0:
            q[:, 0] = -q[:, 0]
        m = rng.uniform(mu_range[0], mu_range[1])
        if rad + a.max() >= 0.48 * n:
            continue
        cs.append([rad * np.cos(phi), rad * np.sin(phi), z])
        ax.append(a)
        qs.append(q)
        mus.append(m)
    return Ellipsoids(np.array(cs), np.array(ax), np.array(qs), np.array(mus))


def line_integrals(ell: Ellipsoids, theta, n: int, center: float, z_rows, nz_total: int,
                   xp=np, dtype=None, device=None):
    """Closed-form line integrals p[j, r, i] for angles theta[j], slice rows
    z_rows[r] (indices into the nz_total stack) and detector pixels i in [0, n).

    Detector pixel i of projection j records the line x cos + y sin + center = i.
    Returns an array of shape (len(theta), len(z_rows), n).
    """
    theta = np.asarray(theta, dtype=np.float64)
    z_rows = np.asarray(z_rows, dtype=np.float64)
    A = ell.quadric()
    if xp is np:
        dt = np.float64 if dtype is None else dtype
        mk = lambda a: np.asarray(a, dtype=dt)  # noqa: E731
    else:  # torch
        dt = xp.float64 if dtype is None else dtype
        mk = lambda a: xp.as_tensor(np.asarray(a, dtype=np.float64), dtype=dt, device=device)  # noqa: E731
    c = mk(np.cos(theta))[:, None, None]
    s = mk(np.sin(theta))[:, None, None]
    u = (mk(np.arange(n, dtype=np.float64)) - center)[None, None, :]
    zz = (mk(z_rows) - nz_total / 2.0)[None, :, None]
    out = None
    # p = (u c, u s, z);  d = (-s, c, 0)
    for e in range(len(ell)):
        a = A[e]
        x0, y0, z0 = ell.center[e]
        # cull: slices the ellipsoid cannot reach contribute nothing (z half-extent of the
        # ellipsoid is sqrt((Q diag(a^2) Q^T)_zz))
        zext = float(np.sqrt(np.sum((ell.rot[e][2, :] * ell.axes[e]) ** 2)))
        if np.all(np.abs(z_rows - nz_total / 2.0 - z0) > zext):
            continue
        vx = u * c - x0
        vy = u * s - y0
        vz = zz - z0
        # A v
        avx = a[0, 0] * vx + a[0, 1] * vy + a[0, 2] * vz
        avy = a[1, 0] * vx + a[1, 1] * vy + a[1, 2] * vz
        avz = a[2, 0] * vx + a[2, 1] * vy + a[2, 2] * vz
        alpha = a[0, 0] * s * s - 2.0 * a[0, 1] * s * c + a[1, 1] * c * c   # d^T A d
        beta = -s * avx + c * avy                                            # d^T A v
        gamma = vx * avx + vy * avy + vz * avz - 1.0
        disc = beta * beta - alpha * gamma
        chord = 2.0 * xp.sqrt(xp.clip(disc, 0.0, None)) / alpha
        term = float(ell.mu[e]) * chord
        out = term if out is None else out + term
    if out is None:
        out = (u * c) * 0.0 + zz * 0.0
    return out


def rasterize(ell: Ellipsoids, n: int, z_rows, nz_total: int) -> np.ndarray:
    """Phantom sampled at voxel centres: f[r, iy, ix] (for mean-value checks only)."""
    z_rows = np.asarray(z_rows, dtype=np.float64)
    A = ell.quadric()
    x = (np.arange(n) - n / 2.0)[None, None, :]
    y = (np.arange(n) - n / 2.0)[None, :, None]
    z = (z_rows - nz_total / 2.0)[:, None, None]
    f = np.zeros((len(z_rows), n, n))
    for e in range(len(ell)):
        a = A[e]
        vx, vy, vz = x - ell.center[e, 0], y - ell.center[e, 1], z - ell.center[e, 2]
        q = (a[0, 0] * vx * vx + a[1, 1] * vy * vy + a[2, 2] * vz * vz
             + 2 * (a[0, 1] * vx * vy + a[0, 2] * vx * vz + a[1, 2] * vy * vz))
        f += ell.mu[e] * (q <= 1.0)
    return f
