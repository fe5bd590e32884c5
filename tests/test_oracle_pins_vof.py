"""Pins for the oracle's MTHINC volume-of-fluid step (oracle.vof_step / vof_reconstruct; SURVEY.md sec. 8(f) NEXT-4;
PAPER.md:104-132, Appendix A).  The paper prints no worked numbers for one step, so the pins are what the method fixes:
  V1  the reconstruction satisfies its own definition: the cell mean of H^ (A.8) -- evaluated with an INDEPENDENT
      64-point Gauss-Legendre rule along the direction of exact integration -- equals phi to round-off; n is a unit vector
      pointing towards phase 1; pure cells and cells without a gradient are flat
  V2  Youngs' gradient is exact for a linear field (and so is the choice of the integration direction)
  V3  "the mass of each phase [is] conserved up to machine precision" when div u = 0 discretely
  V4  CFL = +-1 along the interface normal moves the profile by exactly one cell (flux = the whole donor cell), in
      each direction: pins upwinding, signs, the swept interval and which velocity component drives which sweep
  V5  a drop in a uniform diagonal flow: 0 <= phi <= 1, volume conserved, centroid moves by u t (consistency)
  V6  a uniform phi stays uniform in a solenoidal flow; donor-cell fluxes for pure cells
  V7  the Youngs stencil itself (A.6: "derivatives at the cell corners ... each corner-value is averaged") on a
      NON-linear field: averaging the eight corner gradients is the 27-point stencil 1/2 (central difference) x 1/4 (1,2,1)
      x 1/4 (1,2,1), written here with numpy.roll -- a plain central difference (or any other consistent stencil) fails
  V8  a partial-CFL flux (A.26-A.27): uniform velocity along one axis, CFL +-0.37, one step; then
      phi' = phi - (F_+ - F_-)/dl with F the integral of the DONOR cell's H^ over [1 - c, 1] (u >= 0) or [0, |c|] (u < 0),
      evaluated with an independent 64-point Gauss-Legendre rule from the oracle's own (n, d) -- the wrong end of the cell,
      the wrong donor or the wrong sign fails
  V9  the one-dimensional integral of the tanh profile, which every volume and flux is made of, against 50-digit values
      (mpmath) -- in particular for normals almost perpendicular to the direction of integration (|alpha| = 1e-11 ... 1e-3),
      where the textbook difference of two ln cosh loses up to nine digits
"""
import numpy as np
import pytest

from tests import np_ops as ops

BETA = 2.0


def _drop(shape, centre, radius, width):
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    d = [np.minimum(np.abs(a - c), n - np.abs(a - c)) for a, c, n in ((x, centre[0], nx), (y, centre[1], ny), (z, centre[2], nz))]
    r = np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)
    return 0.5 * (1.0 - np.tanh((r - radius) / width))


def _solenoidal(shape, box, seed):
    """u = curl of a random vector potential living on the cell edges: discretely divergence free on the MAC grid"""
    rng = np.random.default_rng(seed)
    dx, dy, dz = ops.spacings(shape, box)
    ax, ay, az = (rng.standard_normal(shape) for _ in range(3))
    d = lambda f, axis, h: (f - np.roll(f, 1, axis=axis)) / h
    u = d(az, 1, dy) - d(ay, 0, dz)
    v = d(ax, 0, dz) - d(az, 2, dx)
    w = d(ay, 2, dx) - d(ax, 1, dy)
    assert np.abs(ops.div(u, v, w, box, False)).max() < 1e-10 * np.abs(u).max() / dx
    return u, v, w


def test_v1_reconstruction_satisfies_the_volume_constraint(oracle_mod):
    shape = (12, 14, 16)
    phi = _drop(shape, (8.3, 6.1, 5.7), 4.0, 0.8)
    phi[0, 0, 0] = 0.4                                            # an isolated blip: has a gradient of its own
    n, d, flat = oracle_mod.vof_reconstruct(phi, BETA)
    inter = flat == 0
    assert inter.sum() > 200 and np.all(flat[(phi <= 1e-8) | (phi >= 1 - 1e-8)] == 1)
    assert np.allclose(np.linalg.norm(n[inter], axis=-1), 1.0, atol=1e-14)
    xs, ws = np.polynomial.legendre.leggauss(64)
    xs, ws = 0.5 * (xs + 1.0), 0.5 * ws                           # on [0, 1]
    g2 = np.array([0.5 - 0.5 / np.sqrt(3.0), 0.5 + 0.5 / np.sqrt(3.0)])
    worst = 0.0
    idx = np.argwhere(inter)
    for (k, j, i) in idx[:: max(1, len(idx) // 300)]:
        nn, dd = n[k, j, i], d[k, j, i]
        a = np.abs(nn)
        dr = 0 if (a[0] >= a[1] and a[0] >= a[2]) else (1 if a[1] >= a[2] else 2)
        t1, t2 = (dr + 1) % 3, (dr + 2) % 3
        tot = 0.0
        for p in g2:
            for q in g2:
                tot += 0.25 * np.sum(ws * 0.5 * (1.0 + np.tanh(BETA * (nn[dr] * xs + nn[t1] * p + nn[t2] * q + dd))))
        worst = max(worst, abs(tot - phi[k, j, i]))
    assert worst < 1e-12
    # n points towards phase 1 (phi = 1 inside the drop): against the radial direction
    k, j, i = 6, 6, 12                                            # a cell on the +x side of the drop
    assert flat[k, j, i] == 0 and n[k, j, i, 0] < -0.5


def test_v2_youngs_gradient_is_exact_for_a_linear_field(oracle_mod):
    shape = (8, 9, 10)
    z, y, x = np.meshgrid(np.arange(8.0), np.arange(9.0), np.arange(10.0), indexing="ij")
    for g in ((0.03, 0.01, -0.02), (0.0, -0.04, 0.01), (0.01, 0.01, 0.05), (-0.02, 0.02, 0.02)):
        phi = 0.5 + g[0] * (x - 4.5) + g[1] * (y - 4.0) + g[2] * (z - 3.5)
        n, d, flat = oracle_mod.vof_reconstruct(phi, BETA)
        want = np.array(g) / np.linalg.norm(g)
        inner = n[1:-1, 1:-1, 1:-1]                                # the periodic wrap breaks linearity in the outer layer
        assert np.all(flat[1:-1, 1:-1, 1:-1] == 0) and np.abs(inner - want).max() < 1e-13


@pytest.mark.parametrize("seed", [0, 1])
def test_v3_volume_is_conserved_to_round_off_in_a_solenoidal_flow(oracle_mod, seed):
    shape, box = (10, 12, 16), (1.6, 1.2, 1.0)
    phi = _drop(shape, (7.2, 6.4, 4.9), 3.5, 0.7)
    u, v, w = _solenoidal(shape, box, seed)
    dt = 0.3 * min(ops.spacings(shape, box)) / max(np.abs(a).max() for a in (u, v, w))
    out = oracle_mod.vof_step(phi, u, v, w, box, BETA, dt)
    assert abs(out.sum() - phi.sum()) < 1e-13 * phi.sum()
    assert np.abs(out - phi).max() > 1e-3                         # ... and the step did something
    assert out.min() > -1e-3 and out.max() < 1.0 + 1e-3


@pytest.mark.parametrize("axis,sign", [(2, 1), (2, -1), (1, 1), (1, -1), (0, 1), (0, -1)])
def test_v4_unit_cfl_along_the_normal_is_an_exact_shift(oracle_mod, axis, sign):
    shape, box = (8, 8, 8), (0.8, 1.6, 2.4)
    n = 8
    s = np.arange(n) + 0.5
    prof = 0.5 * (np.tanh((s - 2.0) / 0.9) - np.tanh((s - 6.0) / 0.9))          # a slab, periodic
    sh = [1, 1, 1]
    sh[axis] = n
    phi = np.ascontiguousarray(np.broadcast_to(prof.reshape(sh), shape))
    h = ops.spacings(shape, box)[2 - axis]
    dt = 0.01
    vel = [np.zeros(shape) for _ in range(3)]
    vel[2 - axis] = np.full(shape, sign * h / dt)                   # u dt / dl = +-1
    out = oracle_mod.vof_step(phi, *vel, box, BETA, dt)
    assert np.abs(out - np.roll(phi, sign, axis=axis)).max() < 1e-12


def test_v5_drop_in_a_uniform_diagonal_flow(oracle_mod):
    shape, box = (16, 16, 16), (1.0, 1.0, 1.0)
    phi = _drop(shape, (6.0, 7.0, 8.0), 3.0, 0.7)
    vel = (0.8, -0.5, 0.3)
    u, v, w = (np.full(shape, c) for c in vel)
    dt, steps = 0.25 / 16 / 0.8, 8
    cur = phi
    for _ in range(steps):
        cur = oracle_mod.vof_step(cur, u, v, w, box, BETA, dt)
        assert cur.min() > -1e-6 and cur.max() < 1.0 + 1e-6
    assert abs(cur.sum() - phi.sum()) < 1e-12 * phi.sum()
    z, y, x = np.meshgrid(*(np.arange(16) + 0.5,) * 3, indexing="ij")
    cen = lambda f: np.array([(f * x).sum(), (f * y).sum(), (f * z).sum()]) / f.sum() / 16.0
    shift = cen(cur) - cen(phi)
    want = np.array(vel) * dt * steps
    # the first moment is not an invariant of the scheme (the tanh profile sharpens to the width 1 / beta while it moves):
    # the centroid follows u t to a few per cent -- a wrong component, sign or split order would be off by O(1)
    assert np.all(np.abs(shift - want) < 0.03 * np.abs(want))


def test_v6_uniform_and_pure_states(oracle_mod):
    shape, box = (6, 8, 10), (1.0, 0.8, 0.6)
    u, v, w = _solenoidal(shape, box, 5)
    dt = 0.2 * min(ops.spacings(shape, box)) / max(np.abs(a).max() for a in (u, v, w))
    for val in (0.3, 0.0, 1.0):
        out = oracle_mod.vof_step(np.full(shape, val), u, v, w, box, BETA, dt)
        assert np.abs(out - val).max() < 1e-13


def _bumpy_field(shape, seed):
    """a drop with a smooth random perturbation: curved level sets, 0 < phi < 1, nothing linear about it"""
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    bump = sum(a * np.sin(2 * np.pi * (kx * x / nx + ky * y / ny + kz * z / nz) + ph)
               for a, kx, ky, kz, ph in zip(rng.uniform(0.2, 0.6, 4), rng.integers(1, 3, 4), rng.integers(1, 3, 4),
                                            rng.integers(1, 3, 4), rng.uniform(0, 6.28, 4)))
    r = _drop(shape, (nx * 0.45, ny * 0.55, nz * 0.5), 0.3 * min(shape), 1.1)
    return np.clip(r + 0.08 * bump * r * (1.0 - r) * 4.0, 0.0, 1.0)


def _youngs_by_roll(phi):
    """m = (m_x, m_y, m_z) in cell units: central difference along the component's axis, weights (1, 2, 1) / 4 along the other two"""
    sm = lambda f, ax: 0.25 * (np.roll(f, 1, axis=ax) + 2.0 * f + np.roll(f, -1, axis=ax))
    cd = lambda f, ax: 0.5 * (np.roll(f, -1, axis=ax) - np.roll(f, 1, axis=ax))
    return np.stack([sm(sm(cd(phi, 2), 1), 0), sm(sm(cd(phi, 1), 2), 0), sm(sm(cd(phi, 0), 2), 1)], axis=-1)


def test_v7_youngs_stencil_on_a_curved_field(oracle_mod):
    shape = (10, 12, 14)
    phi = _bumpy_field(shape, 21)
    n, d, flat = oracle_mod.vof_reconstruct(phi, BETA)
    m = _youngs_by_roll(phi)
    mag = np.linalg.norm(m, axis=-1)
    band = (phi > 1e-8) & (phi < 1.0 - 1e-8)
    want_flat = ~band | ~(mag > 1e-12)
    assert np.array_equal(flat == 1, want_flat) and (~want_flat).sum() > 300
    want = m[~want_flat] / mag[~want_flat][:, None]
    assert np.abs(n[~want_flat] - want).max() < 1e-13
    # the field is curved enough for the stencil to matter: plain central differences give a visibly different normal
    cd = np.stack([0.5 * (np.roll(phi, -1, axis=a) - np.roll(phi, 1, axis=a)) for a in (2, 1, 0)], axis=-1)[~want_flat]
    cd /= np.linalg.norm(cd, axis=-1)[:, None]
    assert np.abs(cd - want).max() > 1e-2


def _slice_volume(nn, dd, axis_c, a, b, xs, ws):
    """int_a^b along component axis_c, 2 x 2 Gauss points across it, of 1/2 [1 + tanh(beta (n . x~ + d))] (cell coordinates)"""
    g2 = (0.5 - 0.5 / np.sqrt(3.0), 0.5 + 0.5 / np.sqrt(3.0))
    t1, t2 = (axis_c + 1) % 3, (axis_c + 2) % 3
    x = a + (b - a) * xs
    tot = 0.0
    for p in g2:
        for q in g2:
            tot += 0.25 * (b - a) * np.sum(ws * 0.5 * (1.0 + np.tanh(BETA * (nn[axis_c] * x + nn[t1] * p + nn[t2] * q + dd))))
    return tot


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("cfl", [0.37, -0.37])
def test_v8_partial_cfl_flux_integrates_the_donor_cell_over_the_swept_interval(oracle_mod, comp, cfl):
    shape, box = (8, 9, 10), (1.0, 1.35, 1.6)
    phi = _bumpy_field(shape, 22 + comp)
    axis = 2 - comp                                               # numpy axis of the component (x is the last axis)
    dl = ops.spacings(shape, box)[comp]
    speed, dt = 0.8, abs(cfl) * dl / 0.8
    vel = [np.zeros(shape) for _ in range(3)]
    vel[comp][:] = np.sign(cfl) * speed
    out = oracle_mod.vof_step(phi, vel[0], vel[1], vel[2], box, BETA, dt)
    n, d, flat = oracle_mod.vof_reconstruct(phi, BETA)
    xs, ws = np.polynomial.legendre.leggauss(64)
    xs, ws = 0.5 * (xs + 1.0), 0.5 * ws
    c = abs(cfl)
    a, b = (1.0 - c, 1.0) if cfl > 0 else (0.0, c)                # (A.26): the last c of the donor, or its first |c|
    vol = np.empty(shape)                                         # what every cell gives away
    for idx in np.ndindex(*shape):
        vol[idx] = (b - a) * phi[idx] if flat[idx] else _slice_volume(n[idx], d[idx], comp, a, b, xs, ws)
    # u > 0: a cell loses its own slice and receives that of the cell before it; u < 0: ... of the cell after it
    want = phi - vol + np.roll(vol, 1 if cfl > 0 else -1, axis=axis)
    assert np.abs(out - want).max() < 1e-12
    assert np.abs(out - phi).max() > 1e-2 and (flat == 0).sum() > 100
    # the other end of the donor cell is a different number: the pin can tell them apart
    wrong = np.array([_slice_volume(n[idx], d[idx], comp, 1.0 - b, 1.0 - a, xs, ws) for idx in np.argwhere(flat == 0)[:50].tolist()
                      for idx in [tuple(idx)]])
    right = np.array([vol[tuple(idx)] for idx in np.argwhere(flat == 0)[:50]])
    assert np.abs(wrong - right).max() > 1e-3


@pytest.mark.parametrize("beta", [2.0, 3.0])
def test_v9_tanh_integral_against_high_precision_values(oracle_mod, beta):
    mpmath = pytest.importorskip("mpmath")
    mpmath.mp.dps = 50
    worst = 0.0
    for alpha in (1e-11, -1e-11, 1e-9, -1e-9, 1e-6, 1e-3, -0.02, 0.3, -0.7, 1.0):
        for gamma in (-1.3, -0.2, 0.0, 0.05, 0.9):
            for a, b in ((0.0, 1.0), (0.63, 1.0), (0.0, 0.37), (0.999, 1.0)):
                got = oracle_mod.tanh_integral(a, b, alpha, gamma, beta)
                al, ga, be, aa, bb = (mpmath.mpf(x) for x in (alpha, gamma, beta, a, b))
                want = ((bb - aa) + (mpmath.log(mpmath.cosh(be * (al * bb + ga))) - mpmath.log(mpmath.cosh(be * (al * aa + ga)))) / (be * al)) / 2
                # the integral is a volume fraction of the slice times its length: what matters (it is added to phi = O(1)) is
                # the error relative to (b - a); where the slice is almost empty the relative error of the value itself is larger
                worst = max(worst, abs(float((mpmath.mpf(got) - want) / (bb - aa))))
    assert worst < 1e-15, worst
