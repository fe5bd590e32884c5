"""Independent numpy statements of the MAC-grid operators, used ONLY by the tests to pin the
oracle (and to check properties of GPU results).  Arrays are (nz, ny, nx); axis 2 is x.
Written with np.roll / slicing, sharing nothing with oracle.c or the CUDA kernels."""
import numpy as np


def spacings(shape, box):
    nz, ny, nx = shape
    return box[0] / nx, box[1] / ny, box[2] / nz


def grad(f, box, wall):
    """(Gx f, Gy f, Gz f) on east / north / top faces; wall: top-face z-gradient is 0."""
    dx, dy, dz = spacings(f.shape, box)
    gx = (np.roll(f, -1, axis=2) - f) / dx
    gy = (np.roll(f, -1, axis=1) - f) / dy
    gz = (np.roll(f, -1, axis=0) - f) / dz
    if wall:
        gz[-1] = 0.0
    return gx, gy, gz


def div(a, b, c, box, wall):
    dx, dy, dz = spacings(a.shape, box)
    cm = np.roll(c, 1, axis=0)
    if wall:
        cm[0] = 0.0          # bottom wall face, not stored
    return (a - np.roll(a, 1, axis=2)) / dx + (b - np.roll(b, 1, axis=1)) / dy + (c - cm) / dz


def lap(f, box, wall):
    return div(*grad(f, box, wall), box, wall)


def face_density(phi, rho1, rho2, wall):
    rc = rho1 * phi + rho2 * (1.0 - phi)
    rx = 0.5 * (rc + np.roll(rc, -1, axis=2))
    ry = 0.5 * (rc + np.roll(rc, -1, axis=1))
    rz = 0.5 * (rc + np.roll(rc, -1, axis=0))
    if wall:
        rz[-1] = rc[-1]      # never multiplies a non-zero gradient
    return rx, ry, rz


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a - b)
