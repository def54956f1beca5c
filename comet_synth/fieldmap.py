"""Synthetic solenoid field maps "in the grid format", stand-ins for the COMET field map,
which is not available.  Input generator only: no reconstruction arithmetic lives here."""
import numpy as np


def solenoid_map(b0=1.0, z_edge=90.0, width=12.0, half_xy=96.0, half_z=96.0, spacing=(4.0, 4.0, 4.0)):
    """B on a regular grid covering [-half_xy, half_xy]^2 x [-half_z, half_z] (cm):
    B_z(z) = b0 / (1 + exp((|z| - z_edge) / width)) falls off towards the ends of the solenoid, and
    B_r = -(r/2) dB_z/dz keeps div B = 0 to first order in r.  Inside the CDC (|z| < 75 cm) the field is
    within a few per cent of b0 and grows rougher towards the end plates.
    -> (B [nx][ny][nz][3], origin [3], spacing [3])."""
    d = np.asarray(spacing, dtype=np.float64)
    nx = int(round(2 * half_xy / d[0])) + 1
    ny = int(round(2 * half_xy / d[1])) + 1
    nz = int(round(2 * half_z / d[2])) + 1
    o = np.array([-half_xy, -half_xy, -half_z])
    x = o[0] + d[0] * np.arange(nx)
    y = o[1] + d[1] * np.arange(ny)
    z = o[2] + d[2] * np.arange(nz)
    e = np.exp((np.abs(z) - z_edge) / width)
    bz = b0 / (1.0 + e)
    dbz = -b0 * e / (1.0 + e) ** 2 / width * np.sign(z)
    B = np.empty((nx, ny, nz, 3))
    B[..., 0] = -0.5 * x[:, None, None] * dbz[None, None, :]
    B[..., 1] = -0.5 * y[None, :, None] * dbz[None, None, :]
    B[..., 2] = bz[None, None, :]
    return np.ascontiguousarray(B), o, d


def uniform_map(bz=1.0, half=100.0, spacing=(25.0, 25.0, 25.0)):
    """The uniform field (0, 0, bz) as a grid (pins: the map path must reproduce the uniform-field results)."""
    d = np.asarray(spacing, dtype=np.float64)
    n = int(round(2 * half / d[0])) + 1
    B = np.zeros((n, n, n, 3))
    B[..., 2] = bz
    return B, np.array([-half, -half, -half]), d


def hough_tables(n_phi=256):
    """cos / sin of the Hough directions phi_j = 2 pi j / n_phi (inputs of the transverse seeding: both the
    oracle and the CUDA path read these tables, neither evaluates a trigonometric function)."""
    phi = 2.0 * np.pi * np.arange(n_phi) / n_phi
    return np.cos(phi), np.sin(phi)
