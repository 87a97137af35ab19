"""Pins for oracle O2 (shell angular derivatives through Y_lm; Eqs. 23-24)."""
import numpy as np
import pytest
from scipy.special import sph_harm_y


def grid(oracle, L):
    th, w = oracle.gl_nodes(L)
    ph = 2.0 * np.pi * np.arange(2 * L + 2) / (2 * L + 2)
    return th, w, ph


def test_pbar_closed_forms(oracle):
    """Orthonormal Y_lm closed forms for l <= 2 (any textbook), Condon-Shortley phase."""
    for th in [0.3, 1.1, 2.5]:
        pb, dpb = oracle.pbar(4, th)
        s, c = np.sin(th), np.cos(th)
        ref = {(0, 0): np.sqrt(1 / (4 * np.pi)), (1, 0): np.sqrt(3 / (4 * np.pi)) * c, (1, 1): -np.sqrt(3 / (8 * np.pi)) * s,
               (2, 0): np.sqrt(5 / (16 * np.pi)) * (3 * c * c - 1), (2, 1): -np.sqrt(15 / (8 * np.pi)) * s * c,
               (2, 2): np.sqrt(15 / (32 * np.pi)) * s * s}
        dref = {(0, 0): 0.0, (1, 0): -np.sqrt(3 / (4 * np.pi)) * s, (1, 1): -np.sqrt(3 / (8 * np.pi)) * c,
                (2, 0): -np.sqrt(5 / (16 * np.pi)) * 6 * c * s, (2, 1): -np.sqrt(15 / (8 * np.pi)) * (c * c - s * s),
                (2, 2): np.sqrt(15 / (32 * np.pi)) * 2 * s * c}
        for (l, m), v in ref.items():
            assert abs(pb[l, m] - v) < 1e-15
            assert abs(dpb[l, m] - dref[(l, m)]) < 1e-14


@pytest.mark.parametrize("L", [4, 8, 12])
def test_pbar_matches_library_and_unsold(oracle, L):
    for th in [0.2, 1.3, 2.9]:
        pb, _ = oracle.pbar(L, th)
        for l in range(L + 1):
            for m in range(l + 1):
                assert abs(pb[l, m] - sph_harm_y(l, m, th, 0.0).real) < 1e-13
            # Unsold: sum_m |Y_lm|^2 = (2l+1)/(4 pi)
            tot = pb[l, 0] ** 2 + 2.0 * (pb[l, 1 : l + 1] ** 2).sum()
            assert abs(tot - (2 * l + 1) / (4 * np.pi)) < 1e-13


@pytest.mark.parametrize("L", [4, 8])
def test_quadrature_orthonormality(oracle, L):
    th, w, ph = grid(oracle, L)
    P = np.stack([oracle.pbar(L, t)[0] for t in th])  # [j,l,m]
    for m in range(L + 1):
        G = np.einsum("j,jl,jk->lk", w, P[:, m:, m], P[:, m:, m]) * 2 * np.pi
        assert np.abs(G - np.eye(L + 1 - m)).max() < 1e-13


@pytest.mark.parametrize("L", [3, 8, 12])
def test_single_ylm_exact(oracle, L):
    """d_theta, d_phi exact for every real/imag part of each Y_lm, l <= L; library route for the
    expected values: d_phi Y = i m Y;  d_theta Y_lm = m cot(theta) Y_lm + sqrt((l-m)(l+m+1)) e^{-i phi} Y_{l,m+1}."""
    th, w, ph = grid(oracle, L)
    T, Pp = np.meshgrid(th, ph, indexing="ij")
    for l in range(L + 1):
        for m in range(l + 1):
            Y = sph_harm_y(l, m, T, Pp)
            Ynext = sph_harm_y(l, m + 1, T, Pp) if m + 1 <= l else 0.0
            dth = m / np.tan(T) * Y + np.sqrt((l - m) * (l + m + 1.0)) * np.exp(-1j * Pp) * Ynext
            dph = 1j * m * Y
            for part in (np.real, np.imag):
                if m == 0 and part is np.imag:
                    continue
                a, b = oracle.shell_angular(L, part(Y))
                assert np.abs(a - part(dth)).max() < 2e-13 * (l + 1), (l, m)
                assert np.abs(b - part(dph)).max() < 2e-13 * (l + 1), (l, m)


@pytest.mark.parametrize("L", [4, 8])
def test_projection(oracle, L):
    """synthesis(analysis(.)) is a projector, not the identity; rank (L+1)^2 = N_theta N_phi / 2
    (PAPER.md:502 'N_s very roughly N_theta N_phi / 2'); a pure l = L+1 input is annihilated (S6)."""
    rng = np.random.default_rng(7)
    n = (L + 1) * (2 * L + 2)
    u = rng.standard_normal((L + 1, 2 * L + 2))
    p1 = oracle.shell_project(L, u)
    p2 = oracle.shell_project(L, p1)
    assert np.abs(p1 - u).max() > 1e-2          # not the identity on random data
    assert np.abs(p2 - p1).max() < 1e-13        # idempotent
    Pm = np.stack([oracle.shell_project(L, e.reshape(L + 1, -1)).ravel() for e in np.eye(n)], axis=1)
    assert np.linalg.matrix_rank(Pm, tol=1e-9) == (L + 1) ** 2 == n // 2
    th, w, ph = grid(oracle, L)
    T, Pp = np.meshgrid(th, ph, indexing="ij")
    for m in range(0, L + 2):
        y = sph_harm_y(L + 1, m, T, Pp).real
        a, b = oracle.shell_angular(L, y)
        assert np.abs(oracle.shell_project(L, y)).max() < 1e-13
        assert np.abs(a).max() < 1e-12 and np.abs(b).max() < 1e-12


def test_plain_fourier_dphi_differs(oracle):
    """S8 is a real choice: d_phi through a_lm (with the l<=L projection) is not the plain Fourier
    derivative on non-band-limited data."""
    L = 8
    rng = np.random.default_rng(3)
    u = rng.standard_normal((L + 1, 2 * L + 2))
    _, b = oracle.shell_angular(L, u)
    k = np.fft.rfftfreq(2 * L + 2, 1.0 / (2 * L + 2))
    k[-1] = 0
    plain = np.fft.irfft(1j * k * np.fft.rfft(u, axis=1), n=2 * L + 2, axis=1)
    assert np.abs(b - plain).max() > 0.5
