"""Seeded synthetic inputs shared by the tests, the bench and the oracle timing.

This module serves BOTH the CPU oracle and the CUDA path, so it holds none of the
method's own arithmetic: it draws random numbers (numpy PCG64), evaluates analytic
shapes, and resamples with a third-party library routine
(`scipy.ndimage.map_coordinates`, order=1, mode='nearest').  It imports neither
`oracle/` nor the CUDA binding.

The inputs stand in for the DIR-Lab 4DCT cases the paper measured on
(Section 3.1 / Table 1: 256x256x94..112 voxels, 0.97-1.16 x 2.5 mm),
which are not available; recipes follow BASELINE.json configs 1-5 and are stated in
DESIGN.md ("Input recipe").

Layout: a scalar volume is a C-contiguous float32 array of shape (nz, ny, nx), i.e.
flat index = x + nx*(y + ny*z) (Section 2.5: "x as rows, y as columns,
z as frames").  A displacement field is float32 of shape (3, nz, ny, nx); component 0
is the x displacement, 1 is y, 2 is z, in voxels.
"""
from __future__ import annotations

import numpy as np
from scipy import ndimage


def _axes(dims):
    nx, ny, nz = dims
    return (np.arange(nx, dtype=np.float64), np.arange(ny, dtype=np.float64),
            np.arange(nz, dtype=np.float64))


def _sum_separable_gaussians(dims, centres, widths, amps):
    """sum_b amps[b, c] * exp(-|x - centres[b]|^2 / (2 widths[b]^2)) -> (C, nz, ny, nx) float64."""
    x, y, z = _axes(dims)
    centres = np.asarray(centres, dtype=np.float64)
    widths = np.asarray(widths, dtype=np.float64)
    amps = np.asarray(amps, dtype=np.float64)
    if amps.ndim == 1:
        amps = amps[:, None]
    gx = np.exp(-(x[None, :] - centres[:, 0:1]) ** 2 / (2.0 * widths[:, None] ** 2))
    gy = np.exp(-(y[None, :] - centres[:, 1:2]) ** 2 / (2.0 * widths[:, None] ** 2))
    gz = np.exp(-(z[None, :] - centres[:, 2:3]) ** 2 / (2.0 * widths[:, None] ** 2))
    out = np.empty((amps.shape[1], dims[2], dims[1], dims[0]), dtype=np.float64)
    gyx = (gy[:, :, None] * gx[:, None, :]).reshape(len(widths), -1)
    for c in range(amps.shape[1]):
        # (z,b) @ (b, y*x) contraction
        out[c] = ((amps[:, c:c + 1] * gz).T @ gyx).reshape(dims[2], dims[1], dims[0])
    return out


def blob_volume(dims, rng, nblobs=20, noise_sd=10.0):
    """BASELINE.json config 1 static volume: 20 Gaussian blobs (sigma U[3,8] voxels,
    amplitude U[-1000,500]) + N(0, noise_sd).  Draw order: centres, sigmas, amplitudes, noise."""
    nx, ny, nz = dims
    centres = rng.uniform(0.0, 1.0, size=(nblobs, 3)) * np.array([nx - 1, ny - 1, nz - 1])
    widths = rng.uniform(3.0, 8.0, size=nblobs)
    amps = rng.uniform(-1000.0, 500.0, size=nblobs)
    vol = _sum_separable_gaussians(dims, centres, widths, amps)[0]
    if noise_sd > 0:
        vol = vol + rng.normal(0.0, noise_sd, size=vol.shape)
    return np.ascontiguousarray(vol, dtype=np.float32)


def bump_field(dims, rng, nbumps, width_range, max_norm, centre_frac=0.5):
    """Smooth displacement field: sum of `nbumps` Gaussian bumps with random 3-vector
    amplitudes, centres uniform in the central `centre_frac` of the volume, scaled so that
    max |d| = max_norm voxels.  Draw order: centres, widths, directions."""
    nx, ny, nz = dims
    ext = np.array([nx - 1, ny - 1, nz - 1], dtype=np.float64)
    lo = 0.5 * (1.0 - centre_frac) * ext
    centres = lo + rng.uniform(0.0, 1.0, size=(nbumps, 3)) * (centre_frac * ext)
    widths = rng.uniform(width_range[0], width_range[1], size=nbumps)
    dirs = rng.normal(0.0, 1.0, size=(nbumps, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    f = _sum_separable_gaussians(dims, centres, widths, dirs)
    norm = np.sqrt((f ** 2).sum(axis=0)).max()
    f *= max_norm / norm
    return np.ascontiguousarray(f, dtype=np.float32)


def resample(vol, field):
    """vol sampled at x + field(x), linear, edge-replicated — library routine, float32 out."""
    nz, ny, nx = vol.shape
    zz, yy, xx = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                             np.arange(nx, dtype=np.float64), indexing="ij")
    coords = np.stack([zz + field[2], yy + field[1], xx + field[0]])
    out = ndimage.map_coordinates(vol.astype(np.float64), coords, order=1, mode="nearest")
    return np.ascontiguousarray(out, dtype=np.float32)


def config1_pair(dims=(64, 64, 32), seed=101, noise_sd=10.0, max_norm=3.0):
    """BASELINE.json config 1: blob static volume; moving = static resampled by a known
    4-bump field with max |d| = 3 voxels.  Returns (S, M, d)."""
    rng = np.random.default_rng(seed)
    S = blob_volume(dims, rng, 20, noise_sd)
    d = bump_field(dims, rng, 4, (6.0, 12.0), max_norm)
    M = resample(S, d)
    return S, M, d


def lung_phantom(dims, rng, noise_sd=20.0):
    """BASELINE.json config 2 phantom: background -1000 HU, body elliptic cylinder at 0 HU,
    two lung ellipsoids at -850 HU, 200 capsule vessels at +50 HU (radius U[1,3]), N(0,20)."""
    nx, ny, nz = dims
    x, y, z = _axes(dims)
    X = x[None, None, :]
    Y = y[None, :, None]
    Z = z[:, None, None]
    cx, cy = 0.5 * (nx - 1), 0.5 * (ny - 1)
    vol = np.full((nz, ny, nx), -1000.0, dtype=np.float64)
    body = ((X - cx) / (0.45 * nx)) ** 2 + ((Y - cy) / (0.35 * ny)) ** 2 <= 1.0
    vol[np.broadcast_to(body, vol.shape)] = 0.0
    lungs = np.zeros(vol.shape, dtype=bool)
    for sgn in (-1.0, 1.0):
        e = (((X - (cx + sgn * 0.2 * nx)) / (0.15 * nx)) ** 2 + ((Y - cy) / (0.22 * ny)) ** 2
             + ((Z - 0.55 * nz) / (0.38 * nz)) ** 2)
        lungs |= e <= 1.0
    vol[lungs] = -850.0
    lung_idx = np.argwhere(lungs)  # (n, 3) as (z, y, x)
    nves = 200
    starts = lung_idx[rng.integers(0, len(lung_idx), size=nves)][:, ::-1].astype(np.float64)
    dirs = rng.normal(0.0, 1.0, size=(nves, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    lengths = rng.uniform(20.0, 60.0, size=nves)
    radii = rng.uniform(1.0, 3.0, size=nves)
    for a, dvec, L, r in zip(starts, dirs, lengths, radii):
        b = a + L * dvec
        lo = np.floor(np.minimum(a, b) - r - 1).astype(int)
        hi = np.ceil(np.maximum(a, b) + r + 1).astype(int)
        lo = np.maximum(lo, 0)
        hi = np.minimum(hi, [nx - 1, ny - 1, nz - 1])
        if np.any(hi < lo):
            continue
        px = x[lo[0]:hi[0] + 1][None, None, :] - a[0]
        py = y[lo[1]:hi[1] + 1][None, :, None] - a[1]
        pz = z[lo[2]:hi[2] + 1][:, None, None] - a[2]
        t = np.clip((px * dvec[0] + py * dvec[1] + pz * dvec[2]) / L, 0.0, 1.0)
        dist2 = (px - t * L * dvec[0]) ** 2 + (py - t * L * dvec[1]) ** 2 + (pz - t * L * dvec[2]) ** 2
        sub = vol[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1]
        sub[dist2 <= r * r] = 50.0
    vol += rng.normal(0.0, noise_sd, size=vol.shape)
    return np.ascontiguousarray(vol, dtype=np.float32)


def breathing_field(dims, rng):
    """Config 2 known field: d_z = 12 exp(-(z - 0.25 nz)^2 / (2 (0.25 nz)^2)) (function of z
    only, slope < 0.3 so invertible) plus lateral x/y bumps of amplitude <= 2 voxels."""
    nx, ny, nz = dims
    z = np.arange(nz, dtype=np.float64)
    dz = 12.0 * np.exp(-(z - 0.25 * nz) ** 2 / (2.0 * (0.25 * nz) ** 2))
    ext = np.array([nx - 1, ny - 1, nz - 1], dtype=np.float64)
    centres = 0.25 * ext + rng.uniform(0.0, 1.0, size=(4, 3)) * (0.5 * ext)
    widths = rng.uniform(20.0, 40.0, size=4)
    ang = rng.uniform(0.0, 2.0 * np.pi, size=4)
    amps = np.stack([np.cos(ang), np.sin(ang)], axis=1)
    lat = _sum_separable_gaussians(dims, centres, widths, amps)
    lat *= 2.0 / np.sqrt((lat ** 2).sum(axis=0)).max()
    f = np.empty((3, nz, ny, nx), dtype=np.float32)
    f[0] = lat[0]
    f[1] = lat[1]
    f[2] = dz[:, None, None]
    return f


def lung_pair(dims=(256, 256, 100), seed=202):
    """BASELINE.json configs 2-4: lung phantom + breathing-like known field.  Returns (S, M, d)."""
    rng = np.random.default_rng(seed)
    S = lung_phantom(dims, rng)
    d = breathing_field(dims, rng)
    M = resample(S, d)
    return S, M, d


def textured_pair(dims=(256, 256, 100), seed=212, max_d=2.0):
    """A WELL-CONDITIONED full-size pair: an analytic texture with intensity gradient almost everywhere (three oblique
    sinusoids, amplitudes of CT-like size), S = tex(x), M = tex(x + d) evaluated analytically for a smooth known field
    d of at most `max_d` voxels (bumps of width 20-40 voxels).  On the lung phantom -- with or without noise, with or
    without softened edges -- large regions are flat, the force there is 0/0-like (d ~ 0, grad ~ 0) and rounding
    differences grow to tenths of a voxel over a registration; here the oracle differs from itself by ~2e-6 voxel when
    the input moves by one ulp, so the END state of a full registration can be held to north_star's plain 1e-2 voxel
    bar.  Returns (S, M, d)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")

    def tex(px, py, pz):
        return (100.0 * np.sin(0.31 * px + 0.05 * pz) * np.cos(0.23 * py) + 60.0 * np.sin(0.27 * pz + 0.11 * px + 0.07 * py)
                + 40.0 * np.cos(0.19 * px - 0.29 * py + 0.13 * pz))

    d = bump_field(dims, rng, 8, (20.0, 40.0), max_d, centre_frac=1.0)
    S = tex(x, y, z).astype(np.float32)
    M = tex(x + d[0], y + d[1], z + d[2]).astype(np.float32)
    return S, M, d


def sweep_inputs(dims, seed):
    """BASELINE.json config 5: blob static, random smooth u (32 bumps, widths U[8,24],
    max |u| = 8 voxels), moving = static resampled by a second such field.  Returns (S, M, u)."""
    rng = np.random.default_rng(seed)
    S = blob_volume(dims, rng, 20, 10.0)
    u = bump_field(dims, rng, 32, (8.0, 24.0), 8.0, centre_frac=1.0)
    other = bump_field(dims, rng, 32, (8.0, 24.0), 8.0, centre_frac=1.0)
    M = resample(S, other)
    return S, M, u


def eval_points(dims, rng, n=1000, margin=16):
    """n integer voxel positions (x, y, z) uniform with >= margin voxels to every face."""
    nx, ny, nz = dims
    m = [min(margin, (nx - 1) // 4), min(margin, (ny - 1) // 4), min(margin, (nz - 1) // 4)]
    pts = np.stack([rng.integers(m[0], nx - m[0], size=n), rng.integers(m[1], ny - m[1], size=n),
                    rng.integers(m[2], nz - m[2], size=n)], axis=1)
    return pts


def true_inverse_at(d, pts, steps=50):
    """Ground truth u* at integer points: the solution of u = -d(p + u) (fixed point, the
    field that undoes `M = S sampled at x + d`), d sampled linearly by the library routine."""
    p = pts.astype(np.float64)
    u = np.zeros_like(p)
    for _ in range(steps):
        q = p + u
        coords = np.stack([q[:, 2], q[:, 1], q[:, 0]])
        dd = np.stack([ndimage.map_coordinates(d[c].astype(np.float64), coords, order=1, mode="nearest")
                       for c in range(3)], axis=1)
        u = -dd
    return u
