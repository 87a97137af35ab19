"""Pins for oracle O3 (Cartesian gradient; Eq. 8, 369-395 Eqs. 20-24)."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs


POLYS = [  # (f, df/dx, df/dy, df/dz) of total degree <= 3
    (lambda x, y, z: x, lambda x, y, z: 1 + 0 * x, lambda x, y, z: 0 * x, lambda x, y, z: 0 * x),
    (lambda x, y, z: x * y, lambda x, y, z: y, lambda x, y, z: x, lambda x, y, z: 0 * x),
    (lambda x, y, z: x * x - y * y, lambda x, y, z: 2 * x, lambda x, y, z: -2 * y, lambda x, y, z: 0 * x),
    (lambda x, y, z: x * x * y + z, lambda x, y, z: 2 * x * y, lambda x, y, z: x * x, lambda x, y, z: 1 + 0 * x),
    (lambda x, y, z: z * z * z - 2 * x * y * z, lambda x, y, z: -2 * y * z, lambda x, y, z: -2 * x * z, lambda x, y, z: 3 * z * z - 2 * x * y),
]


@pytest.mark.parametrize("nr,L", [(4, 3), (6, 5), (8, 8)])
def test_shell_cartesian_polynomials(oracle, nr, L):
    """A Cartesian polynomial of degree p <= min(L, N_r-1) restricted to a shell (centre offset included)
    is band-limited in both r and (theta,phi): its Cartesian gradient must be exact."""
    sd = configs.shell(nr, L, 1.8, 5.0, center=(0.3, -0.2, 0.1))
    xyz = oracle.coords(sd)
    x, y, z = xyz - np.array(sd["center"])[:, None]
    u = np.stack([f(x, y, z) for f, *_ in POLYS])
    g = oracle.gradient(sd, u)
    for c, (_, fx, fy, fz) in enumerate(POLYS):
        for d, fd in enumerate((fx, fy, fz)):
            assert np.abs(g[d, c] - fd(x, y, z)).max() < 5e-12, (c, d)


def test_shell_coords(oracle):
    sd = configs.shell(5, 4, 2.0, 6.0, center=(1.0, 2.0, 3.0))
    xyz = oracle.coords(sd) - np.array(sd["center"])[:, None]
    r = np.sqrt((xyz**2).sum(0)).reshape(5, 5, 10)
    assert np.allclose(r[:, 0, 0], 2.0 + 4.0 * (oracle.cheb_nodes(5) + 1) / 2, atol=1e-14)
    assert np.abs(r - r[:, :1, :1]).max() < 1e-14            # r slowest
    th = np.arccos(xyz[2].reshape(5, 5, 10) / r)
    assert np.allclose(th[0, :, 0], oracle.gl_nodes(4)[0], atol=1e-14)
    ph = np.arctan2(xyz[1], xyz[0]).reshape(5, 5, 10) % (2 * np.pi)
    assert np.allclose(ph[0, 0], 2 * np.pi * np.arange(10) / 10, atol=1e-13)  # phi fastest


def test_block_polynomials_anisotropic(oracle):
    sd = configs.block([5, 7, 6], (1.0, -2.0, 0.5), (3.0, 1.0, 4.5))
    xyz = oracle.coords(sd)
    x, y, z = xyz
    assert np.allclose(x.reshape(5, 7, 6)[:, 0, 0], 1.0 + 2.0 * (oracle.cheb_nodes(5) + 1) / 2)
    assert np.allclose(z.reshape(5, 7, 6)[0, 0, :], 0.5 + 4.0 * (oracle.cheb_nodes(6) + 1) / 2)
    u = np.stack([x**4 * y**2 * z**3 + x * y**6, np.ones_like(x), z**5])
    g = oracle.gradient(sd, u)
    assert np.abs(g[0, 0] - (4 * x**3 * y**2 * z**3 + y**6)).max() < 1e-9
    assert np.abs(g[1, 0] - (2 * x**4 * y * z**3 + 6 * x * y**5)).max() < 1e-9
    assert np.abs(g[2, 0] - (3 * x**4 * y**2 * z**2)).max() < 1e-9
    assert np.abs(g[:, 1]).max() < 1e-12
    assert np.abs(g[2, 2] - 5 * z**4).max() < 1e-10 and np.abs(g[:2, 2]).max() < 1e-10


def test_spectral_convergence_smooth(oracle):
    errs = []
    for n in (6, 10, 14):
        sd = configs.block(n, (3.0, -1.0, -1.0), (5.0, 1.0, 1.0))
        x, y, z = oracle.coords(sd)
        g = oracle.gradient(sd, np.sin(x + 0.5 * y * z)[None])
        errs.append(np.abs(g[0, 0] - np.cos(x + 0.5 * y * z)).max())
    assert errs[0] > 30 * errs[1] > 900 * errs[2]
