"""Seeded synthetic inputs for the projection step (numpy, host).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only fabricates fields (u*, v*, w*, phi, p^n, p^(n-1)) with the
shapes, sizes, box dimensions and density ratios of the paper's two application runs,
which are not public data:
  * emulsion in homogeneous isotropic turbulence, 512^3, box 2*pi, triply periodic
                                             -> configs 1, 2, 4
  * two-layer Rayleigh-Benard convection, 1024 x 1024 x 512, walls in z
                                             -> configs 3, 5
The five configs are those of BASELINE.json; the exact recipe is restated in DESIGN.md.

Arrays have shape (nz, ny, nx), C order (x fastest), float64.  Cell centres are at
(i + 1/2) dx; u / v / w[i, j, k] live on the east / north / top face of cell (i, j, k).
Draw order is fixed per config: noise of u*, v*, w*, then p, p_old (when i.i.d.), then the
structure parameters (drop centres, mode tables).  rho1 = 1, dt = 1e-3 everywhere.
"""
from dataclasses import dataclass, field

import numpy as np

BC_Z_PERIODIC = 0
BC_Z_WALL = 1
BC_PERIODIC, BC_NEUMANN, BC_DIRICHLET = 0, 1, 2      # per-direction conditions (NEUMANN = wall)
TWO_PI = 2.0 * np.pi


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    box: tuple          # (lx, ly, lz)
    bc_z: int
    rho1: float
    rho2: float
    dt: float
    seed: int
    u: np.ndarray = field(repr=False, default=None)
    v: np.ndarray = field(repr=False, default=None)
    w: np.ndarray = field(repr=False, default=None)
    phi: np.ndarray = field(repr=False, default=None)
    p: np.ndarray = field(repr=False, default=None)
    p_old: np.ndarray = field(repr=False, default=None)
    bc_x: int = BC_PERIODIC
    bc_y: int = BC_PERIODIC

    @property
    def bc(self):
        return (self.bc_x, self.bc_y, self.bc_z)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def npts(self):
        return self.nx * self.ny * self.nz

    def fields(self):
        return self.u, self.v, self.w, self.phi, self.p, self.p_old


# ----------------------------------------------------------------------------- pieces

def _uniform(rng, shape, lo, hi):
    a = rng.random(shape)
    a *= (hi - lo)
    a += lo
    return a


def _centres(n, length):
    return (np.arange(n) + 0.5) * (length / n)


def _faces(n, length):
    return (np.arange(n) + 1.0) * (length / n)


def _drops_phi(shape, box, centres, radius):
    """phi = min(1, sum_d 0.5*(1 - tanh((r_d - R)/(2 dx)))), each drop evaluated on a cube of
    half-width R + 20 dx around its centre with periodic wrap (min-image by construction)."""
    nz, ny, nx = shape
    lx, ly, lz = box
    dx, dy, dz = lx / nx, ly / ny, lz / nz
    phi = np.zeros(shape)
    # half-width R + 20 dx, capped so that the cube never wraps onto itself (scaled-down test boxes)
    hx, hy, hz = (min(int(np.ceil(radius / d)) + 20, (n - 1) // 2) for d, n in ((dx, nx), (dy, ny), (dz, nz)))
    for cx, cy, cz in centres:
        i0, j0, k0 = int(np.floor(cx / dx)), int(np.floor(cy / dy)), int(np.floor(cz / dz))
        ii, jj, kk = (np.arange(c - h, c + h + 1) for c, h in ((i0, hx), (j0, hy), (k0, hz)))
        ox, oy, oz = (ii + 0.5) * dx - cx, (jj + 0.5) * dy - cy, (kk + 0.5) * dz - cz
        r = np.sqrt(oz[:, None, None] ** 2 + oy[None, :, None] ** 2 + ox[None, None, :] ** 2)
        phi[np.ix_(kk % nz, jj % ny, ii % nx)] += 0.5 * (1.0 - np.tanh((r - radius) / (2.0 * dx)))
    np.minimum(phi, 1.0, out=phi)
    return phi


def _place_drops(rng, n_drops, box, radius, dx):
    """uniform centres by rejection until the min-image centre distance >= 2R + 4dx"""
    lx, ly, lz = box
    L = np.array([lx, ly, lz])
    dmin = 2.0 * radius + 4.0 * dx
    out = np.empty((0, 3))
    tries = 0
    while len(out) < n_drops:
        c = rng.random(3) * L
        tries += 1
        if tries > 2_000_000:
            raise RuntimeError("drop placement did not converge")
        if len(out):
            d = np.abs(out - c)
            d = np.minimum(d, L - d)
            if np.min(np.sqrt((d ** 2).sum(axis=1))) < dmin:
                continue
        out = np.vstack([out, c])
    return out


def _random_modes(rng, n_modes, kmax):
    """integer wave vectors uniform over 1 <= |k| <= kmax, unit amplitudes a perpendicular to k,
    phases uniform in [0, 2 pi)"""
    ks = []
    while len(ks) < n_modes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        if 1 <= np.sqrt(float((k ** 2).sum())) <= kmax:
            ks.append(k)
    ks = np.array(ks)
    g = rng.standard_normal((n_modes, 3))
    kk = (ks ** 2).sum(axis=1, keepdims=True).astype(float)
    a = g - (g * ks).sum(axis=1, keepdims=True) * ks / kk
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    theta = rng.random(n_modes) * TWO_PI
    return ks, a, theta


def _mode_sum(shape, ks, amps, theta, shift):
    """sum_m amps[m] * cos(k_m . x + theta_m) on a (2 pi)^3 periodic box, sampled at
    x = (i + shift_x) dx etc.  Built in spectral space + one inverse real FFT."""
    import scipy.fft as sfft
    nz, ny, nx = shape
    spec = np.zeros((nz, ny, nx // 2 + 1), dtype=np.complex128)
    sx, sy, sz = shift
    for (kx, ky, kz), a, th in zip(ks, amps, theta):
        kx, ky, kz, th = int(kx), int(ky), int(kz), float(th)
        if kx < 0:                                   # cos is even: use -k, -theta
            kx, ky, kz, th = -kx, -ky, -kz, -th
        ph = th + TWO_PI * (kx * sx / nx + ky * sy / ny + kz * sz / nz)
        c = a * np.exp(1j * ph)
        if kx == 0 or 2 * kx == nx:
            # the c2r transform keeps only the real part of these columns
            spec[kz % nz, ky % ny, kx] += c
        else:
            spec[kz % nz, ky % ny, kx] += 0.5 * c
    out = sfft.irfftn(spec, s=shape, axes=(0, 1, 2), workers=-1)
    out *= float(nx) * float(ny) * float(nz)
    return out


def _turbulent_velocity(rng_modes, shape, kmax, n_modes=64):
    ks, a, theta = _random_modes(rng_modes, n_modes, kmax)
    amp = np.sqrt((ks ** 2).sum(axis=1).astype(float)) ** (-5.0 / 6.0)
    # each component sampled at ITS face: u at (i+1, j+1/2, k+1/2) etc.
    u = _mode_sum(shape, ks, amp * a[:, 0], theta, (1.0, 0.5, 0.5))
    v = _mode_sum(shape, ks, amp * a[:, 1], theta, (0.5, 1.0, 0.5))
    w = _mode_sum(shape, ks, amp * a[:, 2], theta, (0.5, 0.5, 1.0))
    return u, v, w


def _smooth_pressure(rng, shape, n_modes=16, kmax=4, peak=0.1):
    ks, _, theta = _random_modes(rng, n_modes, kmax)
    f = _mode_sum(shape, ks, np.ones(n_modes), theta, (0.5, 0.5, 0.5))
    f *= peak / np.max(np.abs(f))
    return f


# ---------------------------------------------------------------------------- configs

def config1(n=32):
    """32^3 triply periodic, (2 pi)^3: one drop R = 0.8 at the centre, rho2/rho1 = 10,
    u*, v*, w* ~ U[-1,1], p, p_old ~ U[-0.1,0.1], seed 0."""
    rng = np.random.default_rng(0)
    shape, box = (n, n, n), (TWO_PI,) * 3
    u, v, w = (_uniform(rng, shape, -1.0, 1.0) for _ in range(3))
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    x = _centres(n, TWO_PI)
    r = np.sqrt((x[:, None, None] - np.pi) ** 2 + (x[None, :, None] - np.pi) ** 2 + (x[None, None, :] - np.pi) ** 2)
    phi = 0.5 * (1.0 - np.tanh((r - 0.8) / (2.0 * (TWO_PI / n))))
    return Workload(f"cfg1_{n}^3_periodic", n, n, n, box, BC_Z_PERIODIC, 1.0, 10.0, 1e-3, 0, u, v, w, phi, p, p_old)


def config2(n=128, n_drops=40, r_cells=8, kmax=8):
    """128^3 triply periodic, emulsion-shaped: 40 drops of radius 8 cells, rho2/rho1 = 1,
    u* = 64 random Fourier modes (|k| <= 8, amplitude |k|^(-5/6)) + U[-0.05,0.05], seed 1."""
    rng = np.random.default_rng(1)
    shape, box = (n, n, n), (TWO_PI,) * 3
    dx = TWO_PI / n
    nu, nv, nw = (_uniform(rng, shape, -0.05, 0.05) for _ in range(3))
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    cent = _place_drops(rng, n_drops, box, r_cells * dx, dx)
    phi = _drops_phi(shape, box, cent, r_cells * dx)
    u, v, w = _turbulent_velocity(rng, shape, kmax)
    u += nu; v += nv; w += nw
    return Workload(f"cfg2_{n}^3_periodic_emulsion", n, n, n, box, BC_Z_PERIODIC, 1.0, 1.0, 1e-3, 1,
                    u, v, w, phi, p, p_old)


def config3(nx=256, ny=256, nz=128):
    """256 x 256 x 128 wall-bounded, box 2 x 2 x 1: two-layer phi, rho2/rho1 = 1.2,
    u*, v*, w* ~ U[-1,1] + one seeded z-mode on w*, w* = 0 at the top wall, seed 2."""
    rng = np.random.default_rng(2)
    shape, box = (nz, ny, nx), (2.0, 2.0, 1.0)
    u, v, w = (_uniform(rng, shape, -1.0, 1.0) for _ in range(3))
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    mx, my = (int(m) for m in rng.integers(1, 5, size=2))
    x, y, zf = _centres(nx, box[0]), _centres(ny, box[1]), _faces(nz, box[2])
    w += 0.5 * (np.sin(np.pi * zf / box[2])[:, None, None]
                * np.cos(TWO_PI * my * y / box[1])[None, :, None]
                * np.cos(TWO_PI * mx * x / box[0])[None, None, :])
    w[nz - 1] = 0.0
    zc = _centres(nz, box[2])
    phi = np.broadcast_to((0.5 * (1.0 + np.tanh((0.5 - zc) / (2.0 * box[2] / nz))))[:, None, None], shape).copy()
    return Workload(f"cfg3_{nx}x{ny}x{nz}_wall", nx, ny, nz, box, BC_Z_WALL, 1.0, 1.2, 1e-3, 2,
                    u, v, w, phi, p, p_old)


def config4(n=512, ratio=50.0, r_cells=16, vol_frac=0.05, kmax=32):
    """512^3 triply periodic (the paper's HIT grid): drops of radius 16 cells at 5 %
    volume fraction, rho2/rho1 in {1, 50}, u* as config 2 with |k| <= 32, smooth p fields, seed 3."""
    rng = np.random.default_rng(3)
    shape, box = (n, n, n), (TWO_PI,) * 3
    dx = TWO_PI / n
    nu, nv, nw = (_uniform(rng, shape, -0.05, 0.05) for _ in range(3))
    n_drops = int(vol_frac * n ** 3 / (4.0 / 3.0 * np.pi * r_cells ** 3))
    cent = _place_drops(rng, n_drops, box, r_cells * dx, dx)
    phi = _drops_phi(shape, box, cent, r_cells * dx)
    u, v, w = _turbulent_velocity(rng, shape, kmax)
    u += nu; v += nv; w += nw
    del nu, nv, nw
    p = _smooth_pressure(rng, shape)
    p_old = _smooth_pressure(rng, shape)
    return Workload(f"cfg4_{n}^3_periodic_r{ratio:g}", n, n, n, box, BC_Z_PERIODIC, 1.0, float(ratio), 1e-3, 3,
                    u, v, w, phi, p, p_old)


def config5(nx=1024, ny=1024, nz=512):
    """1024 x 1024 x 512 wall-bounded (the paper's RB grid), box 4 x 4 x 1: two-layer
    interface at z = 0.5 perturbed by 32 Fourier modes of total amplitude 0.02, rho2/rho1 = 1000,
    u*, v*, w* ~ U[-1,1], p, p_old ~ U[-0.1,0.1], seed 4."""
    rng = np.random.default_rng(4)
    shape, box = (nz, ny, nx), (4.0, 4.0, 1.0)
    u, v, w = (_uniform(rng, shape, -1.0, 1.0) for _ in range(3))
    w[nz - 1] = 0.0
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    ab = rng.integers(1, 9, size=(32, 2))
    theta = rng.random(32) * TWO_PI
    x, y, zc = _centres(nx, box[0]), _centres(ny, box[1]), _centres(nz, box[2])
    eta = np.zeros((ny, nx))
    for (a, b), th in zip(ab, theta):
        eta += np.cos(TWO_PI * (a * x[None, :] / box[0] + b * y[:, None] / box[1]) + th)
    eta *= 0.02 / 32.0
    phi = np.empty(shape)
    dz = box[2] / nz
    for k in range(nz):
        phi[k] = 0.5 * (1.0 + np.tanh((0.5 + eta - zc[k]) / (2.0 * dz)))
    return Workload(f"cfg5_{nx}x{ny}x{nz}_wall", nx, ny, nz, box, BC_Z_WALL, 1.0, 1000.0, 1e-3, 4,
                    u, v, w, phi, p, p_old)


def random_case(nx, ny, nz, bc_z, ratio, seed, box=None):
    """Generic small case for edge-size tests: white-noise velocities and pressures, a tilted
    tanh interface so that rho varies in all three directions."""
    rng = np.random.default_rng(seed)
    shape = (nz, ny, nx)
    if box is None:
        box = (TWO_PI, TWO_PI, TWO_PI) if bc_z == BC_Z_PERIODIC else (2.0, 2.0, 1.0)
    u, v, w = (_uniform(rng, shape, -1.0, 1.0) for _ in range(3))
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    if bc_z == BC_Z_WALL:
        w[nz - 1] = 0.0
    x, y, z = _centres(nx, 1.0), _centres(ny, 1.0), _centres(nz, 1.0)
    s = (z[:, None, None] - 0.5) + 0.2 * np.sin(TWO_PI * y)[None, :, None] + 0.15 * np.cos(TWO_PI * x)[None, None, :]
    phi = 0.5 * (1.0 + np.tanh(-s / 0.1))
    return Workload(f"rand_{nx}x{ny}x{nz}_bc{bc_z}_r{ratio:g}_s{seed}", nx, ny, nz, tuple(box), bc_z, 1.0,
                    float(ratio), 1e-3, seed, u, v, w, phi, p, p_old)


def _zero_wall_faces(W):
    """a walled (NEUMANN) direction stores its far wall face as the last face of every line: no-slip, 0 on entry"""
    if W.bc_x == BC_NEUMANN:
        W.u[:, :, -1] = 0.0
    if W.bc_y == BC_NEUMANN:
        W.v[:, -1, :] = 0.0
    if W.bc_z == BC_NEUMANN:
        W.w[-1] = 0.0
    return W


def random_case_bc(nx, ny, nz, bc, ratio, seed, box=(2.0, 1.5, 1.0)):
    """random_case with a boundary condition per direction, bc = (bc_x, bc_y, bc_z) in {PERIODIC, NEUMANN}"""
    W = random_case(nx, ny, nz, BC_Z_WALL if bc[2] == BC_NEUMANN else BC_Z_PERIODIC, ratio, seed, box=box)
    W.bc_x, W.bc_y = int(bc[0]), int(bc[1])
    W.name = f"rand_{nx}x{ny}x{nz}_bc{bc[0]}{bc[1]}{bc[2]}_r{ratio:g}_s{seed}"
    return _zero_wall_faces(W)


def cavity(nx=256, ny=256, nz=64, ratio=1.0, seed=6):
    """Closed-cavity-shaped case (a box whose boundaries are all solid no-slip walls; the paper's run is a
    256 x 256 plane, this is that plane extruded to nz cells): walls in x, y and z, box 1 x 1 x nz/nx.
    u*, v*, w* ~ U[-1,1] + one smooth circulation cell (the thermally driven roll of the paper's case), wall faces 0;
    a stratified two-layer phi; p, p_old ~ U[-0.1,0.1]."""
    rng = np.random.default_rng(seed)
    shape, box = (nz, ny, nx), (1.0, 1.0, nz / nx)
    u, v, w = (_uniform(rng, shape, -1.0, 1.0) for _ in range(3))
    p, p_old = (_uniform(rng, shape, -0.1, 0.1) for _ in range(2))
    xc, yc, zc = _centres(nx, box[0]), _centres(ny, box[1]), _centres(nz, box[2])
    xf, yf = _faces(nx, box[0]), _faces(ny, box[1])
    # one roll in the (x, y) plane: stream function sin(pi x) sin(pi y) sampled at the faces
    u += 2.0 * (np.sin(np.pi * xf)[None, None, :] * np.cos(np.pi * yc)[None, :, None]) * np.ones((nz, 1, 1))
    v -= 2.0 * (np.cos(np.pi * xc)[None, None, :] * np.sin(np.pi * yf)[None, :, None]) * np.ones((nz, 1, 1))
    phi = np.broadcast_to((0.5 * (1.0 + np.tanh((0.5 - yc) / (2.0 * box[1] / ny))))[None, :, None], shape).copy()
    W = Workload(f"cavity_{nx}x{ny}x{nz}_walls", nx, ny, nz, box, BC_Z_WALL, 1.0, float(ratio), 1e-3, seed,
                 u, v, w, phi, p, p_old, BC_NEUMANN, BC_NEUMANN)
    return _zero_wall_faces(W)


# ------------------------------------------------------------------- z-slab decomposition

def slab_split(a, n_ranks, periodic):
    """Cut a field of shape (nz, ny, nx) into n_ranks local arrays of shape (nz / n_ranks + 2, ny, nx): plane 0 is the
    plane below the slab, planes 1 .. nzl the slab, plane nzl + 1 the plane above (wrapped around when `periodic`, NaN
    beyond a wall so that a kernel that reads it is found out).  Pure data movement: no arithmetic of the method."""
    nz = a.shape[0]
    assert nz % n_ranks == 0
    nzl = nz // n_ranks
    out = []
    for r in range(n_ranks):
        loc = np.full((nzl + 2,) + a.shape[1:], np.nan)
        loc[1:nzl + 1] = a[r * nzl:(r + 1) * nzl]
        lo, hi = r * nzl - 1, (r + 1) * nzl
        if lo >= 0 or periodic:
            loc[0] = a[lo % nz]
        if hi < nz or periodic:
            loc[nzl + 1] = a[hi % nz]
        out.append(loc)
    return out


def slab_gather(parts):
    """the inverse of slab_split for the owned planes: concatenates planes 1 .. nzl of every local array"""
    return np.concatenate([q[1:-1] for q in parts], axis=0)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
