"""Pins of the oracle's spectral filter (O9, NEXT-1 of SURVEY.md §8(f); PAPER.md:452-460 blocks, 500-516 shells).
The filter is defined modally (u~_k <- sigma_k u~_k; a_lm <- sigma_l a_lm), so it is pinned by what that definition fixes:
single modes are eigenfunctions with eigenvalue sigma, sigma = 1 is the identity (blocks) / the l <= L projection
(shells), a Heaviside filter is idempotent, the map is linear, and a block filter is the tensor product of line filters."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs


def _cheb_T(k, x):
    return np.cos(k * np.arccos(np.clip(x, -1.0, 1.0)))


def _real_ylm(oracle, L, l, m, th, ph):
    """Y_lm^real on the grid from the oracle's own Pbar table (pinned in test_oracle_ylm.py)."""
    out = np.zeros((len(th), len(ph)))
    for j, t in enumerate(th):
        pb, _ = oracle.pbar(L, float(t))
        out[j] = pb[l, abs(m)] * (np.cos(m * ph) if m >= 0 else np.sin(-m * ph))
    return out


def test_block_single_modes_are_eigenfunctions(oracle):
    d = configs.block([7, 6, 9], (0, 0, 0), (1, 2, 3))
    xyz = oracle.coords(d)
    x = [2 * (xyz[a] - d["lo"][a]) / (d["hi"][a] - d["lo"][a]) - 1 for a in range(3)]
    rng = np.random.default_rng(5)
    sig = [rng.uniform(0.1, 1.0, n) for n in d["n"]]
    for (i, j, k) in [(0, 0, 0), (3, 1, 4), (6, 5, 8), (2, 0, 7)]:
        u = (_cheb_T(i, x[0]) * _cheb_T(j, x[1]) * _cheb_T(k, x[2]))[None]
        got = oracle.spectral_filter(d, u, sig)
        assert np.max(np.abs(got - sig[0][i] * sig[1][j] * sig[2][k] * u)) < 2e-15


def test_block_identity_linearity_and_heaviside(oracle):
    d = configs.block([8, 5, 6], (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(7)
    P = 8 * 5 * 6
    u, v = rng.standard_normal((3, P)), rng.standard_normal((3, P))
    ones = [np.ones(n) for n in d["n"]]
    assert np.max(np.abs(oracle.spectral_filter(d, u, ones) - u)) < 5e-15          # sigma = 1: identity
    sig = [rng.uniform(0, 1, n) for n in d["n"]]
    lin = oracle.spectral_filter(d, 2.0 * u - 3.0 * v, sig)
    assert np.max(np.abs(lin - (2.0 * oracle.spectral_filter(d, u, sig) - 3.0 * oracle.spectral_filter(d, v, sig)))) < 2e-14
    heav = [(np.arange(n) <= n - 3).astype(float) for n in d["n"]]
    once = oracle.spectral_filter(d, u, heav)
    assert np.max(np.abs(oracle.spectral_filter(d, once, heav) - once)) < 5e-15   # projector
    assert np.max(np.abs(once - u)) > 1e-3                                         # and it did remove something
    # filtering only along x leaves every (y, z) line's x-dependence filtered independently: tensor-product structure
    only_x = [heav[0], ones[1], ones[2]]
    fx = oracle.spectral_filter(d, u, only_x).reshape(3, 8, 5, 6)
    line = u.reshape(3, 8, 5, 6)[1, :, 2, 3]
    d1 = configs.block([8, 2, 2], (0, 0, 0), (1, 1, 1))
    rep = np.repeat(line[:, None], 4, axis=1).reshape(1, 32)
    ref = oracle.spectral_filter(d1, rep, [heav[0], np.ones(2), np.ones(2)]).reshape(8, 4)[:, 0]
    assert np.max(np.abs(fx[1, :, 2, 3] - ref)) < 5e-15


def test_shell_single_ylm_and_projection(oracle):
    L = 6
    d = configs.shell(3, L, 2.0, 3.0)
    th, _ = oracle.gl_nodes(L)
    ph = 2 * np.pi * np.arange(2 * L + 2) / (2 * L + 2)
    rng = np.random.default_rng(11)
    sig = rng.uniform(0.1, 1.0, L + 1)
    for (l, m) in [(0, 0), (2, 1), (5, -3), (6, 6), (6, 0)]:
        y = _real_ylm(oracle, L, l, m, th, ph)
        u = np.stack([(i + 1.0) * y for i in range(3)]).reshape(1, -1)      # a different amplitude on each radial plane
        got = oracle.spectral_filter(d, u, [sig])
        assert np.max(np.abs(got - sig[l] * u)) < 5e-15
    # sigma = 1 is the projection onto l <= L (idempotent), not the identity, on non-band-limited data
    w = rng.standard_normal((2, 3 * (L + 1) * (2 * L + 2)))
    p1 = oracle.spectral_filter(d, w, [np.ones(L + 1)])
    for i in range(3):
        plane = slice(i * (L + 1) * (2 * L + 2), (i + 1) * (L + 1) * (2 * L + 2))
        assert np.max(np.abs(p1[0, plane] - oracle.shell_project(L, w[0, plane]))) < 5e-15
    assert np.max(np.abs(oracle.spectral_filter(d, p1, [np.ones(L + 1)]) - p1)) < 5e-14
    assert np.max(np.abs(p1 - w)) > 1e-2
    # Heaviside in l: idempotent, and it annihilates a pure l = L mode
    heav = (np.arange(L + 1) <= L - 2).astype(float)
    once = oracle.spectral_filter(d, w, [heav])
    assert np.max(np.abs(oracle.spectral_filter(d, once, [heav]) - once)) < 5e-14
    yL = _real_ylm(oracle, L, L, 2, th, ph)
    u = np.tile(yL.reshape(-1), 3)[None]
    assert np.max(np.abs(oracle.spectral_filter(d, u, [heav]))) < 5e-15
