"""Host-side checks of the seeded input generators (no method arithmetic here)."""
import numpy as np

import workloads as wl


def test_mode_sum_matches_direct_evaluation():
    rng = np.random.default_rng(0)
    ks, a, theta = wl._random_modes(rng, 12, 5)
    ks[0] = (0, 2, -1)          # exercise the kx = 0 column and a negative kx
    ks[1] = (-3, 1, 2)
    shape, shift = (10, 12, 16), (1.0, 0.5, 0.5)
    got = wl._mode_sum(shape, ks, a[:, 0], theta, shift)
    nz, ny, nx = shape
    x = (np.arange(nx) + shift[0]) * 2 * np.pi / nx
    y = (np.arange(ny) + shift[1]) * 2 * np.pi / ny
    z = (np.arange(nz) + shift[2]) * 2 * np.pi / nz
    want = np.zeros(shape)
    for (kx, ky, kz), amp, th in zip(ks, a[:, 0], theta):
        want += amp * np.cos(kx * x[None, None, :] + ky * y[None, :, None] + kz * z[:, None, None] + th)
    assert np.max(np.abs(got - want)) < 1e-12


def test_configs_are_seeded_and_shaped():
    a, b = wl.config1(), wl.config1()
    for x, y in zip(a.fields(), b.fields()):
        assert x.dtype == np.float64 and x.shape == (32, 32, 32) and np.array_equal(x, y)
    assert 0.0 <= a.phi.min() and a.phi.max() <= 1.0 and a.phi.max() > 0.9
    c = wl.config3(32, 16, 12)
    assert c.bc_z == wl.BC_Z_WALL and np.all(c.w[-1] == 0.0) and c.rho2 == 1.2
    d = wl.config5(32, 16, 24)
    assert np.all(d.w[-1] == 0.0) and d.rho2 == 1000.0 and d.box == (4.0, 4.0, 1.0)
    # interface sits at z = 0.5 +- 0.02
    zc = (np.arange(24) + 0.5) / 24
    assert np.all(d.phi[zc < 0.4] > 0.9) and np.all(d.phi[zc > 0.6] < 0.1)
    e = wl.config2(32, 3, 3, 4)
    assert e.rho1 == e.rho2 == 1.0 and 0.0 <= e.phi.min() and e.phi.max() <= 1.0
    f = wl.config4(32, 50.0, 3, 0.05, 4)
    assert abs(np.max(np.abs(f.p)) - 0.1) < 1e-12 and f.rho2 == 50.0
