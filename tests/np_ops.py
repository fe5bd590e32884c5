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


# ---- the same operators with a boundary condition per direction: bc = (bc_x, bc_y, bc_z), 0 periodic, 1 Neumann
# (wall: zero normal gradient, zero normal velocity on the boundary faces), 2 Dirichlet (f = 0 ON the boundary faces:
# ghost value = -interior value).  Axis of direction d in an (nz, ny, nx) array: 2 - d.
def grad_bc(f, box, bc):
    out = []
    for d, h in enumerate(spacings(f.shape, box)):
        ax = 2 - d
        g = (np.roll(f, -1, axis=ax) - f) / h
        last = [slice(None)] * 3
        last[ax] = -1
        if bc[d] == 1:
            g[tuple(last)] = 0.0
        elif bc[d] == 2:
            g[tuple(last)] = -2.0 * f[tuple(last)] / h
        out.append(g)
    return out


def div_bc(a, b, c, box, bc, first_face=(None, None, None)):
    """first_face[d]: the flux on the first boundary face of a non-periodic direction d (not a stored face); None = 0"""
    tot = 0.0
    for d, (q, h) in enumerate(zip((a, b, c), spacings(a.shape, box))):
        ax = 2 - d
        qm = np.roll(q, 1, axis=ax)
        if bc[d] != 0:
            first = [slice(None)] * 3
            first[ax] = 0
            qm[tuple(first)] = 0.0 if first_face[d] is None else first_face[d]
        tot = tot + (q - qm) / h
    return tot


def lap_bc(f, box, bc):
    g = grad_bc(f, box, bc)
    first = []
    for d, h in enumerate(spacings(f.shape, box)):
        sl = [slice(None)] * 3
        sl[2 - d] = 0
        first.append(2.0 * f[tuple(sl)] / h if bc[d] == 2 else None)      # Dirichlet: (f_0 - (-f_0)) / h
    return div_bc(*g, box, bc, tuple(first))


def face_density_bc(phi, rho1, rho2, bc):
    rc = rho1 * phi + rho2 * (1.0 - phi)
    out = []
    for d in range(3):
        ax = 2 - d
        r = 0.5 * (rc + np.roll(rc, -1, axis=ax))
        if bc[d] == 1:
            last = [slice(None)] * 3
            last[ax] = -1
            r[tuple(last)] = rc[tuple(last)]      # never multiplies a non-zero gradient
        out.append(r)
    return out
